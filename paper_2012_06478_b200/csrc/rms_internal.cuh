// rms_internal.cuh -- shared declarations of the CUDA implementation behind include/rms.h.
// Product code: shares nothing with oracle/ (the random-number counter scheme is restated here
// from DESIGN.md "Random numbers", not included from the oracle).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string>
#include <vector>

#include "../../include/rms.h"

// ------------------------------------------------------------------------------------------------
// error plumbing
// ------------------------------------------------------------------------------------------------
void rms_set_error(const char* fmt, ...);

#define RMS_CUDA_TRY(expr)                                                                         \
    do {                                                                                           \
        cudaError_t _e = (expr);                                                                   \
        if (_e != cudaSuccess) {                                                                   \
            rms_set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
            return (_e == cudaErrorMemoryAllocation) ? RMS_ERR_OOM : RMS_ERR_CUDA;                 \
        }                                                                                          \
    } while (0)

#define RMS_REQUIRE(cond, code, ...)                                                               \
    do {                                                                                           \
        if (!(cond)) {                                                                             \
            rms_set_error(__VA_ARGS__);                                                            \
            return (code);                                                                         \
        }                                                                                          \
    } while (0)

// ------------------------------------------------------------------------------------------------
// device memory (rms_memory.cu): caching allocator behind every handle
// ------------------------------------------------------------------------------------------------
cudaError_t rms_malloc(void** p, size_t bytes);
void rms_free(void* p);                                  // the work on the block has completed
void rms_free_async(void* p, cudaStream_t stream);       // the work on the block is queued on `stream`

// ------------------------------------------------------------------------------------------------
// handles
// ------------------------------------------------------------------------------------------------
struct rms_substrate {
    int nx = 0, ny = 0, nz = 0;
    double voxel_um = 0;
    int n_labels = 0, n_classes = 0;
    uint64_t n_vox = 0;
    const uint16_t* d_labels = nullptr;  // device, x fastest
    bool owns_labels = false;
    // neighbourhood lattice: one 32-bit word per voxel of the lattice padded by a one-voxel periodic ghost
    // shell.  Bit (dx+1) + 3 (dy+1) + 9 (dz+1), d in {-1,0,1}^3, = the voxel at that offset carries the SAME
    // label as this voxel (bit 13 = the voxel itself = 1); a face towards +-k is a membrane iff the
    // bit of the face neighbour is 0.  Bit 27 (RMS_NBR_GHOST) = ghost voxel.
    // Built on demand (rms_substrate_ensure_nbr): only the general fp32 kernel's face-bit mode reads it; the specialised
    // kernel (fp32 and fp64 directions) reads the octant lattice below.
    uint32_t* d_nbr = nullptr;
    // octant lattice (rms_substrate_create, unless RMS_NO_BRICKS): one 64-bit word per padded voxel = 8 bytes, one per octant
    // of hop directions.  Byte o, o = [hop_x < 0] 4 + [hop_y < 0] 2 + [hop_z < 0], holds the same-label bits of the 2x2x2
    // block a hop of that octant can reach: bit c (c = 4 [moved in x] + 2 [moved in y] + [moved in z], 1..7) = the voxel at
    // (sigma_x [c & 4], sigma_y [c & 2], sigma_z [c & 1]) carries the label of this voxel; bit 0 = ghost voxel.  The 26
    // neighbours appear in 4 (faces), 2 (edges) and 1 (corners) of the bytes: the redundancy buys a one-instruction
    // extraction (PRMT by the octant) of everything a hop can ask (at most three faces, all inside the block).
    uint2* d_oct = nullptr;
    uint2* d_oct_alloc = nullptr;        // the allocation behind d_oct (d_oct = d_oct_alloc + oct_margin)
    size_t oct_margin = 0;
    bool want_bricks = false;            // RMS_NO_BRICKS not given: d_nbr may be built on demand
    // dictionary lattice (RMS_LATTICE_DICT; instead of d_oct): one 16-bit code per padded voxel, same geometry, strides and
    // margin; d_dict[code] = the voxel's octant word.  Code 0 = interior voxel (all 26 neighbours carry its label), codes
    // below RMS_DICT_FIXED the prismatic neighbourhoods (rms_fixed_code), codes RMS_DICT_FIXED .. RMS_DICT_TODO - 1 in the order the
    // build met the other neighbourhoods, RMS_DICT_ESCAPE = the lattice has more distinct neighbourhoods than codes: the word
    // of such a voxel is in the hash table d_esc, keyed by its padded index + 1 (slot = {key, 0, word.x, word.y}, linear
    // probing from rms_esc_hash(index) & esc_mask); d_dict[RMS_DICT_ESCAPE] carries the ghost flag (rms_step_fast.cu).
    uint16_t* d_code = nullptr;
    uint16_t* d_code_alloc = nullptr;
    uint2* d_dict = nullptr;             // [RMS_DICT_ESCAPE + 1]
    uint4* d_esc = nullptr;
    uint32_t esc_mask = 0, n_dict = 0, n_esc = 0;
    // memory order of the neighbourhood lattice: index = X SX + Y SY + Z SZ over the padded coordinates.  The axis with
    // the fewest membrane faces normal to it (the direction the cells run along) is made the fastest one, so that
    // the 8 words of a 32-byte sector belong to one compartment; x fastest (1, NX, NX NY) or z fastest (NY NZ, NZ, 1).
    int SX = 0, SY = 0, SZ = 0;
    uint64_t faces_axis[3] = {0, 0, 0};  // membrane faces with normal x, y, z
    int NX = 0, NY = 0, NZ = 0;          // padded dims (n + 2)
    uint64_t n_membrane_faces = 0;
    std::vector<float> D, T2, kappa;     // host copies of the per-label tables
    std::vector<float> conc;             // per label, relative spin concentration (Appendix C.2; R24); empty = all equal
    std::vector<float> T1;               // per label, mixing time of a stimulated echo; empty = none
    std::vector<float> rho;              // surface relaxivity per label pair (absorbing membranes, Eq.4); empty = none
    std::vector<uint16_t> label_class;
    uint16_t* d_label_class = nullptr;
    bool all_impermeable = true;         // every off-diagonal kappa is 0
};

// Walker state between launches, structure of arrays (coalesced): during rms_run's step kernel the
// state lives in registers; it is written back only at launch boundaries (snapshots, end of call).
struct rms_walker_arrays {
    int32_t* w[3];     // voxel inside the box
    int32_t* dI[3];    // whole-voxel displacement since the start (unwrapped - initial)
    float* f[3];       // in-voxel offset [0,1)
    float* f_lo[3];    // fp64 runs (rms_step_precise.cu): offset = f + f_lo to 2^-48; 0 after an fp32 launch
    int32_t* v0[3];    // initial voxel
    float* f0[3];      // initial offset
    uint32_t* lab;     // label | label0 << 16
    float* relax;      // sum t_i / T2_i (Eq.5)
    double* phi;       // [n_wave_alloc*3][n]: Phi_m,k, voxel units
};

struct rms_walkers {
    const rms_substrate* sub = nullptr;
    uint64_t n = 0, first_id = 0, seed = 0;
    uint64_t steps_done = 0;
    bool poisoned = false;     // a run failed after its first launch: the walkers are part-way through it (rms_run refuses them)
    int n_wave_alloc = 0;
    rms_walker_arrays a{};
    void* d_block = nullptr;   // one allocation behind all arrays but phi
    unsigned long long* d_counters = nullptr;  // [8]
};

// ------------------------------------------------------------------------------------------------
// random numbers: Philox4x32-10, key = (seed_lo, seed_hi), counter = (walker_lo, walker_hi, index, stream)
// ------------------------------------------------------------------------------------------------
enum { RMS_STREAM_INIT = 0, RMS_STREAM_DIR = 1, RMS_STREAM_PERM = 2, RMS_STREAM_INIT_OFFSET = 3, RMS_STREAM_MT = 4, RMS_STREAM_ERL = 5 };
#define RMS_MAX_ERL_ATTEMPTS 4096u   // R25

#define RMS_PHILOX_M0 0xD2511F53u
#define RMS_PHILOX_M1 0xCD9E8D57u
#define RMS_PHILOX_W0 0x9E3779B9u
#define RMS_PHILOX_W1 0xBB67AE85u

struct rms_philox_keys { uint32_t k[20]; };  // round keys k0 + r*W0, k1 + r*W1, r = 0..9

static inline rms_philox_keys rms_make_keys(uint64_t seed)
{
    rms_philox_keys rk;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        rk.k[2 * r] = k0 + (uint32_t)r * RMS_PHILOX_W0;
        rk.k[2 * r + 1] = k1 + (uint32_t)r * RMS_PHILOX_W1;
    }
    return rk;
}

#ifdef __CUDACC__
// padded coordinates of an index of the neighbourhood lattice (x fastest: SX == 1, else z fastest)
__device__ __forceinline__ void rms_lattice_coords(int lin, int SX, int SY, int SZ, int& X, int& Y, int& Z)
{
    if (SX == 1) { Z = lin / SZ; const int rem = lin - Z * SZ; Y = rem / SY; X = rem - Y * SY; }
    else         { X = lin / SX; const int rem = lin - X * SX; Y = rem / SY; Z = rem - Y * SY; }
}

__device__ __forceinline__ void rms_philox(const rms_philox_keys& rk, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                           uint32_t& o0, uint32_t& o1, uint32_t& o2, uint32_t& o3)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)RMS_PHILOX_M0 * c0;
        const unsigned long long p1 = (unsigned long long)RMS_PHILOX_M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk.k[2 * r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk.k[2 * r + 1];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

// words -> reals, exact in fp32: sym(w) = (2 (w>>9) + 1 - 2^23) 2^-23, uni(w) = (w>>8) 2^-24
__device__ __forceinline__ float rms_sym(uint32_t w)
{
    const float m = __uint_as_float((w >> 9) | 0x3F800000u);  // 1 + k 2^-23
    return fmaf(m - 1.5f, 2.0f, 1.1920928955078125e-07f);     // exact: odd multiple of 2^-23
}
__device__ __forceinline__ float rms_uni(uint32_t w) { return (float)(w >> 8) * 5.9604644775390625e-08f; }
#endif

// ------------------------------------------------------------------------------------------------
// step kernel parameters
// ------------------------------------------------------------------------------------------------
struct rms_segment {          // a run of steps on which every waveform is constant (integer valued)
    uint32_t n;               // steps in the segment
    uint32_t flags;           // bit 0: some w != 0 ; bit 1: some remaining weight != 0 inside the segment
    float wf[RMS_MAX_WAVES];          // the constant value of each waveform on the segment (specialised kernels)
    int32_t w[RMS_MAX_WAVES];         // the same as integers, and ...
    int32_t wrem_end[RMS_MAX_WAVES];  // ... the sum of w over the steps of this launch after the segment (general kernel, CONST mode)
};

enum { RMS_WMODE_CONST = 0, RMS_WMODE_TABLE = 1 };
// the step kernels are compiled for 0..4, 8 and 16 waveforms; a run with 5..7 or 9..15 is padded with zero-weight waveforms
static inline int rms_kernel_waves(int n_wave) { return n_wave <= 4 ? n_wave : (n_wave <= 8 ? 8 : 16); }
enum { RMS_LAT_LABELS = 0, RMS_LAT_FACES = 1 };
#define RMS_NBR_GHOST (1u << 27)
#define RMS_NBR_SELF 13
#define RMS_DICT_ESCAPE 0xFFFFu
#define RMS_DICT_TODO 0xFFFEu           // not a code (reserved)
#define RMS_OCT_INTERIOR 0xFEFEFEFEu     // both halves of the octant word of an interior voxel
#define RMS_DICT_FIXED 2048u              // codes below this are fixed: interior, prismatic neighbourhoods, and their ghost variants
#define RMS_DICT_NONE 0xFFFFFFFFu
#ifdef __CUDACC__
__host__ __device__ __forceinline__ uint32_t rms_esc_hash(uint32_t lin) { return (lin * 0x9E3779B1u) >> 8; }
// Codes that need no search.  0: the interior voxel (all 27 same-label bits set).  Prismatic neighbourhoods: the 27 bits do not
// change along one lattice axis (the wall of a cell that runs along that axis: 9 in 10 boundary voxels of an axon lattice);
// they get 1 + 256 f + pat8, f = 0 / 1 / 2 for the axis z / y / x, pat8 = the 8 neighbour bits of the 3 x 3 cross-section
// (centre, always 1, left out).  Ghost voxels (RMS_NBR_GHOST set): the same + 1024.  RMS_DICT_NONE for any other word.
__host__ __device__ __forceinline__ uint32_t rms_fixed_code(uint32_t word)
{
    const uint32_t g = (word >> 27) ? 1024u : 0u, m = word & 0x07FFFFFFu;
    if (m == 0x07FFFFFFu) return g;
    const uint32_t p0 = m & 511u, p1 = (m >> 9) & 511u, p2 = m >> 18;        // planes dz = -1, 0, +1
    uint32_t q, f;
    if (p0 == p1 && p2 == p1) { q = p1; f = 0u; }
    else {
        const uint32_t r0 = m & 0x01C0E07u, r1 = (m >> 3) & 0x01C0E07u, r2 = (m >> 6) & 0x01C0E07u;   // rows dy = -1, 0, +1 of the planes
        if (r0 == r1 && r2 == r1) { q = (r1 & 7u) | ((r1 >> 6) & 0x38u) | ((r1 >> 12) & 0x1C0u); f = 1u; }
        else {
            const uint32_t a = m & 0x1249249u, b = (m >> 1) & 0x1249249u, c = (m >> 2) & 0x1249249u;  // dx = -1, 0, +1 of the rows
            if (a != b || c != b) return RMS_DICT_NONE;
            q = 0u;
#pragma unroll
            for (int k = 0; k < 9; ++k) q |= ((b >> (3 * k)) & 1u) << k;
            f = 2u;
        }
    }
    return g + 1u + 256u * f + ((q & 15u) | ((q >> 5) << 4));
}
// the neighbourhood word of a fixed code: 0, 1 .. 768, 1024, 1025 .. 1792 (0 for the unused codes in between)
__host__ __device__ __forceinline__ uint32_t rms_fixed_word(uint32_t code)
{
    const uint32_t g = code >= 1024u ? RMS_NBR_GHOST : 0u;
    code &= 1023u;
    if (code == 0u) return g | 0x07FFFFFFu;
    if (code > 768u) return 0u;
    const uint32_t f = (code - 1u) >> 8, pat = (code - 1u) & 255u;
    const uint32_t q = (pat & 15u) | 16u | ((pat >> 4) << 5);
    uint32_t m = 0u;
    if (f == 0u) m = q | (q << 9) | (q << 18);
    else if (f == 1u) {
        for (int dz = 0; dz < 3; ++dz) { const uint32_t r = (q >> (3 * dz)) & 7u; m |= (r | (r << 3) | (r << 6)) << (9 * dz); }
    } else {
        for (int k = 0; k < 9; ++k) if ((q >> k) & 1u) m |= 7u << (3 * k);
    }
    return g | m;
}
#endif

struct rms_step_params {
    int nx, ny, nz;
    const uint16_t* labels;
    const uint32_t* nbr;
    const uint2* oct;         // octant lattice (rms_substrate::d_oct), same padded geometry and strides as nbr
    const uint16_t* code;     // or the dictionary lattice (rms_substrate::d_code, d_dict, d_esc): oct == NULL then
    const uint2* dict;
    const uint4* esc;
    uint32_t esc_mask;
    const uint32_t* lut1;     // device, [1024]: interaction outcome by (octant byte >> 1, faces reached); rms_step_fast.cu
    const uint16_t* lut2;     // device, [240 * 8]: the outcomes by hit order of the entries lut1 marks order dependent
    int NX, NY;               // padded dims of the neighbourhood lattice
    int SX, SY, SZ;           // its strides: index = X SX + Y SY + Z SZ; SX == 1 (x fastest) or SZ == 1 (z fastest)
    rms_walker_arrays st;
    uint64_t n, first_id;
    rms_philox_keys rk;
    const float* s_tab;       // [n_labels] hop length in voxels
    const float* P512;        // [n_labels^2] 512 * P(a->b)
    const float* PMT;         // [n_labels^2] saturation probability at an encounter a -> b (Eq.4, R20), or NULL
    const float* rate;        // [n_labels] dt / T2
    int n_labels;
    int rejection;            // 1: rejection sampling (R21), 2: equal-step-length random leap (R25); general kernels only
    uint32_t t_ceil;          // ceil(512 max P(a->b)) over the membranes: coarse random bits at or above it cannot permeate
    uint32_t step0;           // steps done before this launch
    uint32_t n_steps;         // steps of this launch
    int n_seg;
    const rms_segment* segs;  // device (CONST mode)
    const float* wave;        // device, [n_wave][wave_stride], element 0 = first step of this launch (TABLE mode)
    const double* wsuf;       // device, same indexing: suffix sum of w from this step to the end of the call
    int64_t wave_stride;
    int64_t wsuf_stride;
    double wsuf_end[RMS_MAX_WAVES];  // suffix sum just after the last step of this launch
    double wtot[RMS_MAX_WAVES];      // sum of w over the steps of this launch
    int n_wave;
    unsigned long long* counters;    // [0] encounters [1] permeations [2] clamps [3] init failures [4] saturations
    const uint32_t* order;           // thread t works on walker order[t] (spatially sorted, rms_sched.cu); NULL = identity
    // specialised kernel, time slices (rms_step_fast.cu): the first n_whole groups of walkers take one block each for all
    // steps, the last n_sliced groups one block per slice of slice_len steps (n_slices of them, the last one shorter);
    // sched = device [1 + n_sliced], zeroed before the launch.  n_slices <= 1: one block per group.
    uint32_t n_slices, slice_len, n_whole, n_sliced;
    uint32_t* sched;
    // four constants of the direction arithmetic, read as constant-bank operands: written as literals, the compiler has to
    // move each into a register again at every step (instructions with two constants) -- 4 of ~120 instructions per step
    uint32_t k_hi7f, k_tau_or;   // 0x7F, 0x3F800080
    float k_two, k_sin3;         // 2.0f, -2.4641574e-06f
};
// fills in the time-slice fields of p for its n walkers x n_steps (n_slices = 0: none); *sched_words = size of p.sched
void rms_fast_slices(rms_step_params* p, size_t* sched_words);

int rms_launch_step(const rms_step_params& p, int n_wave, int wmode, int lat, bool permeable, cudaStream_t stream);
// RMS_LAT_FACES + RMS_WMODE_CONST only; permeable: P(a->b) << 1 expected (rms_step_fast.cu)
int rms_launch_step_fast(const rms_step_params& p, int n_wave, bool permeable, bool fp64, cudaStream_t stream);
// the two look-up tables of the specialised kernel (constants of the method, built once per device)
int rms_fast_luts(const uint32_t** d_lut1, const uint16_t** d_lut2);
// builds rms_substrate::d_nbr if it is not there yet (needs d_labels); rms_substrate.cu
int rms_substrate_ensure_nbr(const rms_substrate* s, cudaStream_t stream);
// fp64, everything else: permeable / variable D / any waveform, RMS_WMODE_TABLE data, label gathers (rms_step_precise_general.cu)
int rms_launch_step_precise_general(const rms_step_params& p, int n_wave, cudaStream_t stream);

// reductions (rms_reduce.cu)
struct rms_reduce_params {
    rms_walker_arrays st;
    uint64_t n;
    const uint16_t* label_class;  // device
    int n_classes;
    const float* rate;           // device [n_labels] (unused: relax is final at launch end)
    int n_dir;
    const double* dirs;          // device [n_dir*3]
    double voxel_um;
};
int rms_launch_moments(const rms_reduce_params& p, double* d_m2, double* d_m4, double* d_alpha,
                       unsigned long long* d_flow, cudaStream_t stream);
// qv: device [nq*3] phase per unit Phi in turns; qwave: device [nq] waveform index
// order_by_class: device [n], needed (and used) only when n_classes > RMS_SIG_SMALL_CLASSES
#define RMS_SIG_SMALL_CLASSES 8
int rms_launch_signal(const rms_reduce_params& p, int n_wave, int nq, int n_terms, const double* d_qv, const int* d_qwave, double* d_re,
                      double* d_im, double* d_sum_alpha, const uint32_t* order_by_class, cudaStream_t stream, unsigned* n_launches);
int rms_compute_tables(const rms_substrate* s, double dt, std::vector<float>& s_tab, std::vector<float>& P_tab,
                       bool rejection_sampling = false);
int rms_walkers_reserve_waves(rms_walkers* w, int n_wave, cudaStream_t stream);
// rms_sched.cu: order[t] = walker index, sorted by the lattice cell the walker sits in (z-major), so that the
// threads of a warp and the blocks resident at one time gather neighbouring words.  d_order: [n] device.
int rms_order_walkers(const rms_substrate* s, const rms_walkers* w, uint32_t* d_order, cudaStream_t stream, unsigned* n_launches);
// order[t] = walker index, sorted by the output class of the walker's initial label (per-cell outputs: hundreds of classes)
int rms_order_by_class(const rms_substrate* s, const rms_walkers* w, uint32_t* d_order, cudaStream_t stream, unsigned* n_launches);
