// rms_substrate.cu -- H0: substrate upload and the derived neighbourhood lattice (include/rms.h, rms_substrate_create).
#include <math.h>
#include <stdarg.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <mutex>

#include "rms_internal.cuh"

// ------------------------------------------------------------------------------------------------
// thread-local error message
// ------------------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

void rms_set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

extern "C" const char* rms_last_error(void) { return g_err; }
extern "C" const char* rms_version(void) { return "rms-b200 0.1 (sm_100a)"; }

// ------------------------------------------------------------------------------------------------
// Neighbourhood lattice.  A membrane is a voxel face whose two sides carry different labels.  A
// hop shorter than a voxel meets at most three faces, all of them inside the 3x3x3 block
// around the walker's voxel, and while the walker stays in its compartment every face test reads "does
// that neighbour carry my label?".  One 32-bit word per voxel answers all of them: bit
// (dx+1) + 3 (dy+1) + 9 (dz+1) = the neighbour at offset d has the same label as this voxel.
// Layout: (nx+2)(ny+2)(nz+2) words, x fastest; voxel (x,y,z) of the box sits at padded (x+1,y+1,z+1);
// the shell replicates the periodic images (R1) so that a walker can step over the box edge without
// any wrap arithmetic and is folded back when it lands on a ghost voxel (RMS_NBR_GHOST).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int rms_wrap1(int a, int n) { return a < 0 ? a + n : (a >= n ? a - n : a); }

// Membrane faces with normal x, y, z on a sample of the lattice (every `sy`-th row of every `sz`-th plane): decides
// the memory order of the neighbourhood lattice (rms_substrate::SX..SZ).
__global__ void __launch_bounds__(256) rms_sample_faces_kernel(const uint16_t* __restrict__ labels, int nx, int ny, int nz,
                                                                int sy, int sz, unsigned long long* __restrict__ counts)
{
    const int rows_y = (ny + sy - 1) / sy, rows_z = (nz + sz - 1) / sz;
    const size_t total = (size_t)rows_z * rows_y * nx;
    unsigned cx = 0, cy = 0, cz = 0;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(t % nx);
        const size_t r = t / nx;
        const int y = (int)(r % rows_y) * sy, z = (int)(r / rows_y) * sz;
        const size_t row = ((size_t)z * ny + y) * nx;
        const uint16_t L = __ldg(labels + row + x);
        cx += __ldg(labels + row + rms_wrap1(x + 1, nx)) != L;
        cy += __ldg(labels + ((size_t)z * ny + rms_wrap1(y + 1, ny)) * nx + x) != L;
        cz += __ldg(labels + ((size_t)rms_wrap1(z + 1, nz) * ny + y) * nx + x) != L;
    }
    for (int o = 16; o > 0; o >>= 1) {
        cx += __shfl_xor_sync(0xffffffffu, cx, o);
        cy += __shfl_xor_sync(0xffffffffu, cy, o);
        cz += __shfl_xor_sync(0xffffffffu, cz, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&counts[0], (unsigned long long)cx);
        atomicAdd(&counts[1], (unsigned long long)cy);
        atomicAdd(&counts[2], (unsigned long long)cz);
    }
}

// One thread owns a column of RMS_NBR_ZCHUNK padded voxels along z at fixed (X, Y): it keeps the 3 x 3 labels of the
// planes z-1, z, z+1 in registers and reads 9 new labels per voxel instead of 27 (consecutive threads = consecutive
// x: coalesced rows, the +-1 neighbours come out of L1).  ZFAST: the words are written z fastest; a warp stages its
// 32 (x) x 32 (z) tile in shared memory and writes it transposed, 128 contiguous bytes per x.
#define RMS_NBR_ZCHUNK 128

__device__ __forceinline__ void rms_nbr_make_word(uint32_t m, bool, const uint32_t*, uint32_t& w) { w = m; }
__device__ __forceinline__ void rms_nbr_make_word(uint32_t m, bool ghost, const uint32_t* quad, uint2& w)
{
    const uint32_t t0 = (quad[(m >> 9) & 511u] & 0xFEFEFEFEu) | (ghost ? 0x01010101u : 0u);   // bit 0: itself -> ghost flag
    const uint32_t e = t0 | (quad[(m >> 18) & 511u] << 1);      // hop_z > 0: the plane above
    const uint32_t f = t0 | (quad[m & 511u] << 1);              // hop_z < 0: the plane below
    w.x = __byte_perm(e, f, 0x5140);                            // bytes o = 2 q + [hop_z < 0]
    w.y = __byte_perm(e, f, 0x7362);
}

//
// OCT: the word written is the 64-bit octant word of rms_substrate::d_oct instead (WORD = uint2), expanded from the 27 bits
// through a 512-entry table in shared memory: entry [9-bit z-plane], byte q = 2 [hop_x < 0] + [hop_y < 0], even bits
// 0, 2, 4, 6 = the plane's same-label bits at (0, 0), (0, sy), (sx, 0), (sx, sy).  The plane of the voxel gives the even
// bits of an octant byte (not moved in z), the plane above or below, shifted by one, the odd ones.
template <bool OCT, bool DICT> struct rms_nbr_word { typedef uint32_t type; };
template <> struct rms_nbr_word<true, false> { typedef uint2 type; };
template <> struct rms_nbr_word<true, true> { typedef uint16_t type; };

// DICT: the word written is the 16-bit code of rms_substrate::d_code; the octant word goes into the dictionary.  A hash
// table in global memory (2 MB, L2 resident) maps the 28-bit neighbourhood word (27 same-label bits + ghost flag, never 0) to
// its code: slot = key | (code + 1) << 32, claimed with a compare-and-swap on the empty slot (0), the code published by the
// claimant afterwards; readers of a claimed slot poll until the code is there.  Interior voxels (9 in 10) never come here, and
// a thread remembers the last neighbourhood it looked up (cells run along its column).
struct rms_dict_build {
    unsigned long long* hash;
    uint32_t hash_mask;
    uint2* dict;
    uint32_t dict_cap;          // codes RMS_DICT_FIXED .. dict_cap - 1 are handed out, then RMS_DICT_ESCAPE
    uint4* esc;
    uint32_t esc_mask, esc_cap;
    uint32_t* counters;         // [0] neighbourhoods met, [1] escaped voxels, [2] gave up (tables full)
};

__device__ __noinline__ uint32_t rms_dict_lookup(const rms_dict_build& B, uint32_t key, uint2 word, uint32_t lin)
{
    uint32_t code = RMS_DICT_ESCAPE;
    bool done = false;
    uint32_t h = ((key * 0x9E3779B1u) >> 10) & B.hash_mask;
    for (int probe = 0; probe < 4096 && !done; ++probe) {
        volatile unsigned long long* slot = B.hash + h;
        unsigned long long cur = *slot;
        if (cur == 0ull) {
            cur = atomicCAS((unsigned long long*)slot, 0ull, (unsigned long long)key);
            if (cur == 0ull) {                                        // claimed: hand out the code, publish it
                const uint32_t idx = atomicAdd(&B.counters[0], 1u) + RMS_DICT_FIXED;   // below: interior and prismatic codes
                code = idx < B.dict_cap ? idx : RMS_DICT_ESCAPE;
                if (code != RMS_DICT_ESCAPE) B.dict[code] = word;
                __threadfence();
                *slot = (unsigned long long)key | ((unsigned long long)(code + 1u) << 32);
                done = true;
            }
        }
        if (!done && (uint32_t)cur == key) {
            while ((cur >> 32) == 0ull) cur = *slot;                 // the claimant publishes without waiting for anyone
            code = (uint32_t)(cur >> 32) - 1u;
            done = true;
        }
        h = (h + 1u) & B.hash_mask;
    }
    if (!done) { B.counters[2] = 1u; return RMS_DICT_ESCAPE; }
    if (code == RMS_DICT_ESCAPE) {
        // more neighbourhoods than codes: this voxel's word goes into the escape table under its own index
        if (atomicAdd(&B.counters[1], 1u) >= B.esc_cap) { B.counters[2] = 1u; return code; }
        uint32_t g = rms_esc_hash(lin) & B.esc_mask;
        for (int probe = 0; probe < 4096; ++probe) {
            if (atomicCAS(&B.esc[g].x, 0u, lin + 1u) == 0u) {
                B.esc[g].z = word.x; B.esc[g].w = word.y;
                return code;
            }
            g = (g + 1u) & B.esc_mask;
        }
        B.counters[2] = 1u;
    }
    return code;
}

template <bool OCT, bool DICT>
__device__ __forceinline__ void rms_nbr_emit(uint32_t m, bool ghost, const uint32_t* quad, typename rms_nbr_word<OCT, DICT>::type& w)
{
    static_assert(!DICT, "the dictionary build has its own, pipelined, path in rms_build_nbr_kernel");
    rms_nbr_make_word(m, ghost, quad, w);
}

// DICT: the code of a neighbourhood whose hash-table slot was read an iteration ago (`val`): the slot's, if it holds this
// neighbourhood with its code published and the code is not the escape code; the full look-up otherwise (first sight of a
// neighbourhood, a collision, an escaped voxel)
__device__ __forceinline__ uint32_t rms_dict_resolve(const rms_dict_build& B, const uint32_t* quad, uint32_t m, unsigned long long val, uint32_t lin)
{
    const uint32_t c = (uint32_t)(val >> 32) - 1u;
    if ((uint32_t)val == m && (val >> 32) != 0ull && c != RMS_DICT_ESCAPE) return c;
    uint2 word;
    rms_nbr_make_word(m, (m & RMS_NBR_GHOST) != 0u, quad, word);
    return rms_dict_lookup(B, m, word, lin);
}

template <bool ZFAST, bool OCT, bool DICT = false>
__global__ void __launch_bounds__(128) rms_build_nbr_kernel(const uint16_t* __restrict__ labels, int nx, int ny, int nz,
                                                             typename rms_nbr_word<OCT, DICT>::type* __restrict__ nbr, int SX, int SY, int SZ,
                                                             int n_labels, unsigned long long* __restrict__ stats,
                                                             const rms_dict_build dictb = rms_dict_build(), int z_chunk0 = 0)
{
    typedef typename rms_nbr_word<OCT, DICT>::type WORD;
    __shared__ WORD tile[ZFAST ? 4 : 1][ZFAST ? 32 : 1][ZFAST ? 33 : 1];
    __shared__ uint32_t quad[OCT ? 512 : 1];
    if (OCT) {
        for (int t = threadIdx.x; t < 512; t += blockDim.x) {
            uint32_t v = 0;
            for (int q = 0; q < 4; ++q) {
                const int sx = (q & 2) ? -1 : 1, sy = (q & 1) ? -1 : 1;
                for (int xy = 0; xy < 4; ++xy) {
                    const int dx = (xy >> 1) * sx, dy = (xy & 1) * sy;
                    v |= ((t >> ((dx + 1) + 3 * (dy + 1))) & 1u) << (8 * q + 2 * xy);
                }
            }
            quad[t] = v;
        }
        __syncthreads();
    }
    const int NX = nx + 2, NY = ny + 2, NZ = nz + 2;
    const int Xt = blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = Xt < NX;
    const int X = active ? Xt : NX - 1;               // idle lanes of the last block shadow the last column (ZFAST needs whole warps)
    const int Y = blockIdx.y;
    const int Z0 = ((int)blockIdx.z + z_chunk0) * RMS_NBR_ZCHUNK, Z1 = min(NZ, Z0 + RMS_NBR_ZCHUNK);   // (z_chunk0: a launch per chunk)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned n_faces = 0, bad = 0;
    if (ZFAST || active) {
        // periodic image of the padded coordinate (|X-1| <= n, so one wrap is enough even for n = 1)
        const int x = rms_wrap1(X - 1, nx), y = rms_wrap1(Y - 1, ny);
        uint32_t off[9];                              // offsets of the 3 x 3 (dx, dy) neighbours inside a z-plane
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) off[a + 3 * b] = (uint32_t)(rms_wrap1(y + b - 1, ny) * nx + rms_wrap1(x + a - 1, nx));
        const uint32_t plane = (uint32_t)nx * (uint32_t)ny;   // voxel indices fit 31 bits (checked by the caller)
        const bool ghost_xy = (X == 0) | (X == NX - 1) | (Y == 0) | (Y == NY - 1);
        uint32_t pa[9], pb[9], pc[9];                  // labels of the planes z-1, z, z+1 (rotating roles)
        int z = rms_wrap1(Z0 - 1, nz);                // box z of the padded plane Z0
        {
            const uint32_t bl = (uint32_t)rms_wrap1(z - 1, nz) * plane, bm = (uint32_t)z * plane;
#pragma unroll
            for (int k = 0; k < 9; ++k) { pa[k] = __ldg(labels + (bl + off[k])); pb[k] = __ldg(labels + (bm + off[k])); }
        }
        WORD* out = nbr + ((size_t)X * SX + (size_t)Y * SY + (size_t)Z0 * SZ);
        int Z = Z0, zi = 0, zbase = Z0;
        // DICT: interior voxels and prismatic neighbourhoods have fixed codes; any other neighbourhood (1 voxel in 14 on an axon
        // lattice, few of them alike within a block) is looked up in the hash table in global memory, and that look-up is
        // pipelined: the slot is read when the neighbourhood is known and used an iteration later, after the label loads of
        // the next voxel have been issued, so that its latency hides behind theirs (looked up on the spot, it doubled the
        // time of the build: 9.7 against 4.0 ms)
        uint32_t last_key = 0u, last_code = 0u;
        const bool give_up = DICT && *(volatile uint32_t*)&dictb.counters[2] != 0u;
        bool pend = false;
        uint32_t pend_m = 0u, pend_lin = 0u;
        unsigned long long pend_val = 0ull;
        int pend_zi = 0;
        WORD* pend_out = nullptr;

        // one voxel: read plane z+1 into HI, compare the 27 labels with the centre of MID, write the word
#define RMS_NBR_ONE(LO, MID, HI)                                                                              \
        if (Z < Z1) {                                                                                         \
            z = (z + 1 == nz) ? 0 : z + 1;                                                                    \
            const uint32_t bh = (uint32_t)z * plane;                                                          \
            _Pragma("unroll") for (int k = 0; k < 9; ++k) HI[k] = __ldg(labels + (bh + off[k]));             \
            const uint32_t L = MID[4];                                                                        \
            uint32_t m = 0;                                                                                   \
            _Pragma("unroll") for (int k = 0; k < 9; ++k)                                                    \
                m += ((LO[k] == L) ? (1u << k) : 0u) + ((MID[k] == L) ? (1u << (k + 9)) : 0u) +                \
                     ((HI[k] == L) ? (1u << (k + 18)) : 0u);                                                  \
            const bool ghost = ghost_xy | (Z == 0) | (Z == NZ - 1);                                           \
            if (ghost) m |= RMS_NBR_GHOST;                                                                    \
            WORD word;                                                                                        \
            if constexpr (DICT) {                                                                             \
                if (pend) {                            /* the look-up of the previous voxel: patch its code in */ \
                    last_code = rms_dict_resolve(dictb, quad, pend_m, pend_val, pend_lin);                    \
                    last_key = pend_m;                                                                        \
                    if (ZFAST) tile[warp][pend_zi][lane] = (WORD)last_code; else *pend_out = (WORD)last_code;  \
                    pend = false;                                                                             \
                }                                                                                             \
                word = 0;                                                                                     \
                if (m != 0x07FFFFFFu && active) {      /* not interior (m carries the ghost flag) */          \
                    const uint32_t pc = rms_fixed_code(m);                                                    \
                    if (pc != RMS_DICT_NONE) word = (WORD)pc;                                                 \
                    else if (m == last_key && last_code != RMS_DICT_ESCAPE) word = (WORD)last_code;           \
                    else if (give_up) word = (WORD)RMS_DICT_ESCAPE;                                           \
                    else {                                                                                    \
                        pend = true; pend_m = m; pend_lin = (uint32_t)(X * SX + Y * SY + Z * SZ);             \
                        pend_val = *(volatile unsigned long long*)(dictb.hash + (((m * 0x9E3779B1u) >> 10) & dictb.hash_mask)); \
                        pend_zi = zi; pend_out = out;                                                         \
                    }                                                                                         \
                }                                                                                             \
            } else {                                                                                          \
                rms_nbr_emit<OCT, DICT>(m, ghost, quad, word);                                                \
            }                                                                                                 \
            if (ZFAST) {                                                                                      \
                tile[warp][zi][lane] = word;                                                                  \
                if (++zi == 32 || Z == Z1 - 1) {       /* warp-uniform: flush the staged tile, transposed */  \
                    if constexpr (DICT) {                                                                     \
                        if (pend) {                    /* no look-up stays open across a flush */             \
                            last_code = rms_dict_resolve(dictb, quad, pend_m, pend_val, pend_lin);            \
                            last_key = pend_m;                                                                \
                            tile[warp][pend_zi][lane] = (WORD)last_code;                                      \
                            pend = false;                                                                     \
                        }                                                                                     \
                    }                                                                                         \
                    __syncwarp();                                                                             \
                    const int Xw = Xt - lane;                                                                 \
                    for (int xx = 0; xx < 32 && Xw + xx < NX; ++xx)                                           \
                        if (lane < zi) nbr[(size_t)(Xw + xx) * SX + (size_t)Y * SY + (size_t)(zbase + lane)] = tile[warp][lane][xx]; \
                    __syncwarp();                                                                             \
                    zbase += zi; zi = 0;                                                                      \
                }                                                                                             \
            } else {                                                                                          \
                *out = word;                                                                                  \
                out += SZ;                                                                                    \
            }                                                                                                 \
            if (!ghost && active) {                                                                           \
                n_faces += 3 - (((m >> 14) & 1u) + ((m >> 16) & 1u) + ((m >> 22) & 1u));                      \
                bad += (L >= (uint32_t)n_labels);                                                             \
            }                                                                                                 \
            ++Z;                                                                                              \
        }
        while (Z < Z1) {
            RMS_NBR_ONE(pa, pb, pc)
            RMS_NBR_ONE(pb, pc, pa)
            RMS_NBR_ONE(pc, pa, pb)
        }
#undef RMS_NBR_ONE
        if constexpr (DICT) {
            if (pend) *pend_out = (WORD)rms_dict_resolve(dictb, quad, pend_m, pend_val, pend_lin);   // (x fastest: the last voxel's)
        }
    }
    // warp-shuffle reduction, then one atomic per warp
    for (int o = 16; o > 0; o >>= 1) {
        n_faces += __shfl_xor_sync(0xffffffffu, n_faces, o);
        bad += __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (n_faces) atomicAdd(&stats[0], (unsigned long long)n_faces);
        if (bad) atomicAdd(&stats[1], (unsigned long long)bad);
    }
}

// the fixed part of the dictionary: code 0 (interior), the prismatic codes, their ghost variants, and -- so that the step kernel needs no test
// for it before the look-up -- the escape code, whose entry carries the ghost flag and so sends the walker to the rare path
__global__ void __launch_bounds__(256) rms_dict_init_kernel(uint2* __restrict__ dict)
{
    __shared__ uint32_t quad[512];
    for (int t = threadIdx.x; t < 512; t += blockDim.x) {
        uint32_t v = 0;
        for (int q = 0; q < 4; ++q) {
            const int sx = (q & 2) ? -1 : 1, sy = (q & 1) ? -1 : 1;
            for (int xy = 0; xy < 4; ++xy) {
                const int dx = (xy >> 1) * sx, dy = (xy & 1) * sy;
                v |= ((t >> ((dx + 1) + 3 * (dy + 1))) & 1u) << (8 * q + 2 * xy);
            }
        }
        quad[t] = v;
    }
    __syncthreads();
    for (uint32_t code = threadIdx.x; code < RMS_DICT_FIXED; code += blockDim.x) {
        uint2 w = make_uint2(0u, 0u);
        const uint32_t m = rms_fixed_word(code);
        if (m) rms_nbr_make_word(m, (m & RMS_NBR_GHOST) != 0u, quad, w);
        dict[code] = w;
    }
    if (threadIdx.x == 0) dict[RMS_DICT_ESCAPE] = make_uint2(0x01010101u, 0x01010101u);
}

// label check + membrane count without building the face lattice (RMS_NO_BRICKS)
__global__ void __launch_bounds__(256) rms_check_labels_kernel(const uint16_t* __restrict__ labels, size_t n, int n_labels,
                                                                unsigned long long* __restrict__ stats)
{
    unsigned bad = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        bad += labels[i] >= n_labels;
    for (int o = 16; o > 0; o >>= 1) bad += __shfl_xor_sync(0xffffffffu, bad, o);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(&stats[1], (unsigned long long)bad);
}

#define RMS_UPLOAD_SLABS 8
// the stream the slabs of a large host lattice are uploaded on, one per device, kept for the life of the process
static int rms_copy_stream(cudaStream_t* out)
{
    static std::mutex mu;
    static cudaStream_t streams[64] = {nullptr};
    int dev = -1;
    RMS_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return RMS_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(mu);
    if (!streams[dev]) RMS_CUDA_TRY(cudaStreamCreateWithFlags(&streams[dev], cudaStreamNonBlocking));
    *out = streams[dev];
    return RMS_OK;
}
static void rms_destroy_events(cudaEvent_t ev_start, cudaEvent_t* ev_slab)
{
    if (ev_start) cudaEventDestroy(ev_start);
    for (int k = 0; k < RMS_UPLOAD_SLABS; ++k)
        if (ev_slab[k]) cudaEventDestroy(ev_slab[k]);
}

extern "C" int rms_substrate_create(const rms_substrate_desc* d, void* cuda_stream, rms_substrate** out)
{
    RMS_REQUIRE(d && out, RMS_ERR_ARG, "rms_substrate_create: null descriptor or output");
    *out = nullptr;
    RMS_REQUIRE(d->nx > 0 && d->ny > 0 && d->nz > 0, RMS_ERR_ARG, "lattice dimensions must be positive");
    RMS_REQUIRE(d->labels, RMS_ERR_ARG, "labels is null");
    RMS_REQUIRE(d->voxel_um > 0, RMS_ERR_ARG, "voxel_um must be positive");
    RMS_REQUIRE(d->n_labels > 0 && d->n_labels <= 65536, RMS_ERR_ARG, "n_labels must be in 1..65536");
    RMS_REQUIRE(d->n_classes > 0 && d->n_classes <= 65535, RMS_ERR_ARG, "n_classes must be in 1..65535");
    RMS_REQUIRE(d->D, RMS_ERR_ARG, "D is null");
    RMS_REQUIRE(!(d->flags & RMS_ADOPT_DEVICE_PTR) || (d->flags & RMS_LABELS_ON_DEVICE), RMS_ERR_ARG,
                "RMS_ADOPT_DEVICE_PTR needs RMS_LABELS_ON_DEVICE");
    const uint64_t n_vox = (uint64_t)d->nx * d->ny * d->nz;
    RMS_REQUIRE((uint64_t)(d->nx + 2) * (d->ny + 2) * (d->nz + 2) < (1ull << 31), RMS_ERR_UNSUPPORTED,
                "lattice too large: padded voxel count must stay below 2^31");
    const int nL = d->n_labels;
    for (int a = 0; a < nL; ++a) {
        RMS_REQUIRE(d->D[a] > 0 && isfinite(d->D[a]), RMS_ERR_ARG, "D[%d] must be positive and finite", a);
        if (d->label_class) RMS_REQUIRE(d->label_class[a] < d->n_classes, RMS_ERR_ARG, "label_class[%d] >= n_classes", a);
    }
    bool all_imp = true;
    if (d->kappa) {
        for (int a = 0; a < nL; ++a)
            for (int b = 0; b < nL; ++b) {
                if (a == b) continue;
                const float k = d->kappa[(size_t)a * nL + b];
                RMS_REQUIRE(k >= 0 && k == k, RMS_ERR_ARG, "kappa[%d][%d] is negative or NaN", a, b);
                RMS_REQUIRE(k == d->kappa[(size_t)b * nL + a], RMS_ERR_ARG, "kappa is not symmetric at (%d,%d)", a, b);
                if (k != 0) all_imp = false;
            }
    }

    if (d->conc)
        for (int a = 0; a < nL; ++a)
            RMS_REQUIRE(d->conc[a] >= 0 && isfinite(d->conc[a]), RMS_ERR_ARG, "conc[%d] is negative, infinite or NaN", a);
    bool any_rho = false;
    if (d->rho)
        for (size_t i = 0; i < (size_t)nL * nL; ++i) {
            RMS_REQUIRE(d->rho[i] >= 0 && d->rho[i] == d->rho[i], RMS_ERR_ARG, "rho[%zu] is negative or NaN", i);
            any_rho |= (i / nL != i % nL) && d->rho[i] > 0;
        }

    int dev_count = 0;
    cudaError_t ce = cudaGetDeviceCount(&dev_count);
    RMS_REQUIRE(ce == cudaSuccess && dev_count > 0, RMS_ERR_CUDA, "no CUDA device: %s (there is no CPU fallback)",
                cudaGetErrorString(ce));
    cudaStream_t stream = (cudaStream_t)cuda_stream;

    rms_substrate* s = new (std::nothrow) rms_substrate();
    RMS_REQUIRE(s, RMS_ERR_OOM, "out of host memory");
    s->nx = d->nx; s->ny = d->ny; s->nz = d->nz; s->voxel_um = d->voxel_um;
    s->n_labels = nL; s->n_classes = d->n_classes; s->n_vox = n_vox;
    s->D.assign(d->D, d->D + nL);
    if (d->T2) s->T2.assign(d->T2, d->T2 + nL); else s->T2.assign(nL, INFINITY);
    if (d->kappa) s->kappa.assign(d->kappa, d->kappa + (size_t)nL * nL); else s->kappa.assign((size_t)nL * nL, 0.f);
    if (d->label_class) s->label_class.assign(d->label_class, d->label_class + nL); else s->label_class.assign(nL, 0);
    if (any_rho) s->rho.assign(d->rho, d->rho + (size_t)nL * nL);
    if (d->T1) s->T1.assign(d->T1, d->T1 + nL);
    if (d->conc) s->conc.assign(d->conc, d->conc + nL);
    s->all_impermeable = all_imp;

    int rc = RMS_OK;
    unsigned long long* d_stats = nullptr;
    unsigned long long* d_hash = nullptr;              // the dictionary build's hash table and counters
    bool piped = false;                                // the labels arrive in slabs (below)
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_start = nullptr, ev_slab[RMS_UPLOAD_SLABS] = {nullptr};
    unsigned long long h_stats[5] = {0, 0, 0, 0, 0};   // membrane faces, bad labels, sampled faces with normal x, y, z
#define SUB_TRY(expr)                                                                                    \
    do {                                                                                                 \
        cudaError_t _e = (expr);                                                                         \
        if (_e != cudaSuccess) {                                                                         \
            rms_set_error("%s failed: %s", #expr, cudaGetErrorString(_e));                               \
            rc = (_e == cudaErrorMemoryAllocation) ? RMS_ERR_OOM : RMS_ERR_CUDA;                         \
            goto fail;                                                                                   \
        }                                                                                                \
    } while (0)

    if (d->flags & RMS_ADOPT_DEVICE_PTR) {
        s->d_labels = d->labels;
        s->owns_labels = false;
    } else {
        uint16_t* buf = nullptr;
        SUB_TRY(rms_malloc((void**)&buf, n_vox * sizeof(uint16_t)));
        s->d_labels = buf;
        s->owns_labels = true;
        // Host labels of a large lattice: uploaded in slabs of z-planes on a stream of the library's own, an event behind each,
        // so that the build below works on the planes that have arrived while the rest is still on the bus (pinned host
        // memory; from pageable memory the copies simply do not overlap anything)
        piped = !(d->flags & (RMS_LABELS_ON_DEVICE | RMS_NO_BRICKS)) && d->nz >= 4 * RMS_NBR_ZCHUNK && n_vox >= (1u << 20) &&
                rms_copy_stream(&copy_stream) == RMS_OK;
        if (piped) {
            const size_t plane = (size_t)d->nx * d->ny;
            SUB_TRY(cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming));
            SUB_TRY(cudaEventRecord(ev_start, stream));
            SUB_TRY(cudaStreamWaitEvent(copy_stream, ev_start, 0));
            for (int k = 0; k < RMS_UPLOAD_SLABS; ++k) {
                const int za = (int)((long long)d->nz * k / RMS_UPLOAD_SLABS), zb = (int)((long long)d->nz * (k + 1) / RMS_UPLOAD_SLABS);
                SUB_TRY(cudaMemcpyAsync(buf + za * plane, d->labels + za * plane, (size_t)(zb - za) * plane * sizeof(uint16_t),
                                        cudaMemcpyHostToDevice, copy_stream));
                SUB_TRY(cudaEventCreateWithFlags(&ev_slab[k], cudaEventDisableTiming));
                SUB_TRY(cudaEventRecord(ev_slab[k], copy_stream));
            }
        } else {
            SUB_TRY(cudaMemcpyAsync(buf, d->labels, n_vox * sizeof(uint16_t),
                                    (d->flags & RMS_LABELS_ON_DEVICE) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, stream));
        }
    }
    {
        uint16_t* lc = nullptr;
        SUB_TRY(rms_malloc((void**)&lc, nL * sizeof(uint16_t)));
        s->d_label_class = lc;
        SUB_TRY(cudaMemcpyAsync(lc, s->label_class.data(), nL * sizeof(uint16_t), cudaMemcpyHostToDevice, stream));
    }
    SUB_TRY(rms_malloc((void**)&d_stats, 5 * sizeof(unsigned long long)));
    SUB_TRY(cudaMemsetAsync(d_stats, 0, 5 * sizeof(unsigned long long), stream));
    if (!(d->flags & RMS_NO_BRICKS)) {
        s->want_bricks = true;
        s->NX = s->nx + 2; s->NY = s->ny + 2; s->NZ = s->nz + 2;
        // a margin on either side: the step kernel asks for the word of the voxel a hop would enter before it knows whether the
        // walker sits on a ghost voxel, whose neighbours may lie outside the padded lattice (the value is never used then)
        s->oct_margin = ((size_t)std::max(s->NX * s->NY, s->NY * s->NZ) + (size_t)std::max(s->NX, s->NZ) + 2 + 7) / 8 * 8;   // (16-byte steps)
        const size_t n_pad = (size_t)s->NX * s->NY * s->NZ;
        dim3 grid((s->NX + 127) / 128, s->NY, (s->NZ + RMS_NBR_ZCHUNK - 1) / RMS_NBR_ZCHUNK);
        if (grid.y > 65535u || grid.z > 65535u) {
            rms_set_error("lattice too large for the neighbourhood-lattice build (ny+2, nz+2 must be <= 65535)");
            rc = RMS_ERR_UNSUPPORTED;
            goto fail;
        }
        // memory order: x fastest unless asked otherwise.  RMS_LAYOUT_AUTO: the axis (x or z) with fewer membrane faces
        // normal to it runs fastest, so that the words of a sector belong to one compartment (cells elongated along
        // z, such as axons, give z); a sample of the lattice decides
        bool zfast = (d->flags & RMS_LAYOUT_AUTO) == RMS_LAYOUT_Z_FASTEST;
        if ((d->flags & RMS_LAYOUT_AUTO) == RMS_LAYOUT_AUTO) {
            const int sy = s->ny >= 256 ? 8 : (s->ny >= 64 ? 4 : 1), sz = s->nz >= 256 ? 8 : (s->nz >= 64 ? 4 : 1);
            // (labels arriving in slabs: the first slab decides)
            if (piped) SUB_TRY(cudaStreamWaitEvent(stream, ev_slab[0], 0));
            const int nz_sample = piped ? s->nz / RMS_UPLOAD_SLABS : s->nz;
            rms_sample_faces_kernel<<<148 * 4, 256, 0, stream>>>(s->d_labels, s->nx, s->ny, nz_sample, sy, sz, d_stats + 2);
            SUB_TRY(cudaGetLastError());
            SUB_TRY(cudaMemcpyAsync(h_stats + 2, d_stats + 2, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, stream));
            SUB_TRY(cudaStreamSynchronize(stream));
            zfast = h_stats[4] < h_stats[2];
        }
        if (zfast) { s->SZ = 1; s->SY = s->NZ; s->SX = s->NY * s->NZ; }
        else       { s->SX = 1; s->SY = s->NX; s->SZ = s->NX * s->NY; }
        bool have_dict = false;
        if (d->flags & RMS_LATTICE_DICT) {
            // dictionary lattice: 16-bit codes + the octant words of the distinct neighbourhoods; abandoned for the octant
            // lattice below if the lattice has more of them than the tables hold (random labels)
            rms_dict_build B;
            memset(&B, 0, sizeof B);
            B.hash_mask = (1u << 18) - 1u;
            B.dict_cap = RMS_DICT_TODO;
            if (const char* cap = getenv("RMS_DICT_CAP"))                  // tests: force escapes
                B.dict_cap = (uint32_t)std::min(std::max(atoi(cap) + (int)RMS_DICT_FIXED, (int)RMS_DICT_FIXED), (int)RMS_DICT_TODO);
            uint32_t esc_slots = 4096u;                                    // one slot per 8 voxels, 2^12 .. 2^20, half of them usable
            while (esc_slots < (1u << 20) && (size_t)esc_slots * 8 < n_pad) esc_slots <<= 1;
            B.esc_mask = esc_slots - 1u;
            B.esc_cap = esc_slots / 2u;
            uint32_t h_cnt[4] = {0, 0, 0, 0};
            SUB_TRY(rms_malloc((void**)&s->d_code_alloc, (n_pad + 2 * s->oct_margin) * sizeof(uint16_t)));
            s->d_code = s->d_code_alloc + s->oct_margin;
            SUB_TRY(rms_malloc((void**)&s->d_dict, ((size_t)RMS_DICT_ESCAPE + 1) * sizeof(uint2)));
            SUB_TRY(rms_malloc((void**)&s->d_esc, ((size_t)B.esc_mask + 1) * sizeof(uint4)));
            SUB_TRY(rms_malloc((void**)&d_hash, ((size_t)B.hash_mask + 1) * sizeof(unsigned long long) + 4 * sizeof(uint32_t)));
            B.hash = d_hash; B.counters = (uint32_t*)(d_hash + B.hash_mask + 1);
            B.dict = s->d_dict; B.esc = s->d_esc;
            SUB_TRY(cudaMemsetAsync(d_hash, 0, ((size_t)B.hash_mask + 1) * sizeof(unsigned long long) + 4 * sizeof(uint32_t), stream));
            SUB_TRY(cudaMemsetAsync(s->d_esc, 0, ((size_t)B.esc_mask + 1) * sizeof(uint4), stream));
            rms_dict_init_kernel<<<1, 256, 0, stream>>>(s->d_dict);
            SUB_TRY(cudaGetLastError());
            if (piped) {                               // chunk by chunk behind the slabs of the upload, as for the octant lattice below
                const dim3 grid1(grid.x, grid.y, 1);
                for (int cc = 1; cc <= (int)grid.z; ++cc) {
                    const int c = cc % (int)grid.z;
                    const int z_hi = c == 0 ? s->nz - 1 : std::min(s->nz - 1, c * RMS_NBR_ZCHUNK + RMS_NBR_ZCHUNK - 1);
                    int k = 0;
                    while ((int)((long long)s->nz * (k + 1) / RMS_UPLOAD_SLABS) <= z_hi) ++k;
                    SUB_TRY(cudaStreamWaitEvent(stream, ev_slab[k], 0));
                    if (zfast)
                        rms_build_nbr_kernel<true, true, true><<<grid1, 128, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, s->d_code, s->SX, s->SY, s->SZ, nL, d_stats, B, c);
                    else
                        rms_build_nbr_kernel<false, true, true><<<grid1, 128, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, s->d_code, s->SX, s->SY, s->SZ, nL, d_stats, B, c);
                }
            } else if (zfast)
                rms_build_nbr_kernel<true, true, true><<<grid, 128, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, s->d_code, s->SX, s->SY, s->SZ, nL, d_stats, B);
            else
                rms_build_nbr_kernel<false, true, true><<<grid, 128, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, s->d_code, s->SX, s->SY, s->SZ, nL, d_stats, B);
            SUB_TRY(cudaGetLastError());
            SUB_TRY(cudaMemcpyAsync(h_cnt, B.counters, sizeof h_cnt, cudaMemcpyDeviceToHost, stream));
            SUB_TRY(cudaStreamSynchronize(stream));
            rms_free(d_hash);
            d_hash = nullptr;
            if (h_cnt[2] == 0) {
                have_dict = true;
                s->esc_mask = B.esc_mask;
                s->n_dict = std::min(h_cnt[0] + RMS_DICT_FIXED, B.dict_cap);
                s->n_esc = h_cnt[1];
            } else {
                rms_free(s->d_code_alloc); rms_free(s->d_dict); rms_free(s->d_esc);
                s->d_code_alloc = s->d_code = nullptr; s->d_dict = nullptr; s->d_esc = nullptr;
                SUB_TRY(cudaMemsetAsync(d_stats, 0, 2 * sizeof(unsigned long long), stream));    // counted again below
            }
        }
        if (!have_dict) {
            SUB_TRY(rms_malloc((void**)&s->d_oct_alloc, (n_pad + 2 * s->oct_margin) * sizeof(uint2)));
            s->d_oct = s->d_oct_alloc + s->oct_margin;
            if (piped) {
                // one launch per chunk of 128 padded planes, each behind the slab that holds the last plane it reads; chunk 0
                // reads the periodic image of the last plane and goes last
                const dim3 grid1(grid.x, grid.y, 1);
                for (int cc = 1; cc <= (int)grid.z; ++cc) {
                    const int c = cc % (int)grid.z;
                    const int z_hi = c == 0 ? s->nz - 1 : std::min(s->nz - 1, c * RMS_NBR_ZCHUNK + RMS_NBR_ZCHUNK - 1);
                    int k = 0;
                    while ((int)((long long)s->nz * (k + 1) / RMS_UPLOAD_SLABS) <= z_hi) ++k;
                    SUB_TRY(cudaStreamWaitEvent(stream, ev_slab[k], 0));
                    if (zfast)
                        rms_build_nbr_kernel<true, true><<<grid1, 128, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, s->d_oct, s->SX, s->SY, s->SZ, nL, d_stats, rms_dict_build(), c);
                    else
                        rms_build_nbr_kernel<false, true><<<grid1, 128, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, s->d_oct, s->SX, s->SY, s->SZ, nL, d_stats, rms_dict_build(), c);
                }
            } else if (zfast)
                rms_build_nbr_kernel<true, true><<<grid, 128, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, s->d_oct, s->SX, s->SY, s->SZ, nL, d_stats);
            else
                rms_build_nbr_kernel<false, true><<<grid, 128, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, s->d_oct, s->SX, s->SY, s->SZ, nL, d_stats);
            SUB_TRY(cudaGetLastError());
        }
    } else {
        rms_check_labels_kernel<<<148 * 8, 256, 0, stream>>>(s->d_labels, (size_t)n_vox, nL, d_stats);
        SUB_TRY(cudaGetLastError());
    }
    SUB_TRY(cudaMemcpyAsync(h_stats, d_stats, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, stream));
    SUB_TRY(cudaStreamSynchronize(stream));
    rms_free(d_stats);
    d_stats = nullptr;
    if (h_stats[1] != 0) {
        rms_set_error("%llu voxels carry a label >= n_labels (%d)", h_stats[1], nL);
        rc = RMS_ERR_ARG;
        goto fail;
    }
    s->n_membrane_faces = h_stats[0];
    rms_destroy_events(ev_start, ev_slab);
    *out = s;
    return RMS_OK;
fail:
    if (piped) cudaStreamSynchronize(copy_stream);     // nothing of ours may still be writing into a block that is about to be freed
    rms_destroy_events(ev_start, ev_slab);
    if (d_stats) rms_free(d_stats);
    if (d_hash) rms_free(d_hash);
    rms_substrate_destroy(s);
    return rc;
#undef SUB_TRY
}

extern "C" int rms_substrate_destroy(rms_substrate* s)
{
    if (!s) return RMS_OK;
    if (s->owns_labels && s->d_labels) rms_free((void*)s->d_labels);
    if (s->d_nbr) rms_free(s->d_nbr);
    if (s->d_oct_alloc) rms_free(s->d_oct_alloc);
    if (s->d_code_alloc) rms_free(s->d_code_alloc);
    if (s->d_dict) rms_free(s->d_dict);
    if (s->d_esc) rms_free(s->d_esc);
    if (s->d_label_class) rms_free(s->d_label_class);
    delete s;
    return RMS_OK;
}

// The 27-bit neighbourhood lattice is read by the fp64 specialised kernel and by the general kernel's face-bit mode only,
// so it is built at the first run that wants it (same padded geometry and memory order as the octant lattice).
int rms_substrate_ensure_nbr(const rms_substrate* cs, cudaStream_t stream)
{
    static std::mutex mu;
    std::lock_guard<std::mutex> lock(mu);
    rms_substrate* s = const_cast<rms_substrate*>(cs);
    if (s->d_nbr) return RMS_OK;
    RMS_REQUIRE(s->want_bricks, RMS_ERR_UNSUPPORTED, "substrate was created with RMS_NO_BRICKS");
    unsigned long long* d_stats = nullptr;
    uint32_t* nbr = nullptr;
    RMS_CUDA_TRY(rms_malloc((void**)&d_stats, 2 * sizeof(unsigned long long)));
    cudaError_t e = rms_malloc((void**)&nbr, (size_t)s->NX * s->NY * s->NZ * sizeof(uint32_t));
    if (e == cudaSuccess) e = cudaMemsetAsync(d_stats, 0, 2 * sizeof(unsigned long long), stream);
    if (e == cudaSuccess) {
        dim3 grid((s->NX + 127) / 128, s->NY, (s->NZ + RMS_NBR_ZCHUNK - 1) / RMS_NBR_ZCHUNK);
        if (s->SZ == 1)
            rms_build_nbr_kernel<true, false><<<grid, 128, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, nbr, s->SX, s->SY, s->SZ, s->n_labels, d_stats);
        else
            rms_build_nbr_kernel<false, false><<<grid, 128, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, nbr, s->SX, s->SY, s->SZ, s->n_labels, d_stats);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);   // d_stats goes back to the cache below
    rms_free(d_stats);
    if (e != cudaSuccess) {
        if (nbr) rms_free(nbr);
        rms_set_error("building the neighbourhood lattice failed: %s", cudaGetErrorString(e));
        return e == cudaErrorMemoryAllocation ? RMS_ERR_OOM : RMS_ERR_CUDA;
    }
    s->d_nbr = nbr;
    return RMS_OK;
}

// Voxels per label (rms_substrate_label_volumes): grid-stride pass over the uint16 lattice; a warp adds each distinct
// label of its 32 voxels once (match_any), into a shared-memory histogram when the labels fit, else into global memory.
#define RMS_VOL_SMEM_LABELS 8192
__global__ void __launch_bounds__(256) rms_label_volumes_kernel(const uint16_t* __restrict__ labels, uint64_t n_vox, int n_labels,
                                                                 unsigned long long* __restrict__ out)
{
    __shared__ unsigned int hist[RMS_VOL_SMEM_LABELS];
    const bool in_smem = n_labels <= RMS_VOL_SMEM_LABELS;
    if (in_smem)
        for (int t = threadIdx.x; t < n_labels; t += blockDim.x) hist[t] = 0u;
    __syncthreads();
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t n_round = (n_vox + 31) / 32 * 32;                 // whole warps stay in the loop together
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += stride) {
        const bool ok = i < n_vox;
        const unsigned L = ok ? labels[i] : 0xFFFFFFFFu;
        const unsigned peers = __match_any_sync(0xFFFFFFFFu, L);
        if (ok && (threadIdx.x & 31) == (unsigned)(__ffs(peers) - 1)) {
            if (in_smem) atomicAdd(&hist[L], (unsigned)__popc(peers));
            else atomicAdd(&out[L], (unsigned long long)__popc(peers));
        }
    }
    __syncthreads();
    if (in_smem)
        for (int t = threadIdx.x; t < n_labels; t += blockDim.x)
            if (hist[t]) atomicAdd(&out[t], (unsigned long long)hist[t]);
}

extern "C" int rms_substrate_label_volumes(const rms_substrate* s, void* cuda_stream, uint64_t* voxels_out)
{
    RMS_REQUIRE(s && voxels_out, RMS_ERR_ARG, "rms_substrate_label_volumes: null argument");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    unsigned long long* d_out = nullptr;
    RMS_CUDA_TRY(rms_malloc((void**)&d_out, (size_t)s->n_labels * sizeof(unsigned long long)));
    cudaError_t e = cudaMemsetAsync(d_out, 0, (size_t)s->n_labels * sizeof(unsigned long long), stream);
    if (e == cudaSuccess) {
        // a block's shared counters are 32 bit: at most 2^32 - 1 voxels per block
        const uint64_t per_block = 1ull << 24;
        unsigned grid = (unsigned)std::min<uint64_t>(std::max<uint64_t>((s->n_vox + per_block - 1) / per_block, 148ull * 8), 1u << 20);
        rms_label_volumes_kernel<<<grid, 256, 0, stream>>>(s->d_labels, s->n_vox, s->n_labels, d_out);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(voxels_out, d_out, (size_t)s->n_labels * sizeof(unsigned long long), cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    rms_free(d_out);
    if (e != cudaSuccess) {
        rms_set_error("rms_substrate_label_volumes failed: %s", cudaGetErrorString(e));
        return e == cudaErrorMemoryAllocation ? RMS_ERR_OOM : RMS_ERR_CUDA;
    }
    return RMS_OK;
}

// ------------------------------------------------------------------------------------------------
// rms_substrate_label_volumes_static: the same count for callers that may not allocate (include/rms.h).  The per-label
// counters live in a file-scope device array instead of a block from rms_malloc; every GPU that loads the library holds
// its RMS_STATIC_MAX_LABELS * 8 bytes until the process exits.  In host code the name `rms_static_label_count` is only a
// stand-in for the symbol: its device address is asked for once per device (cudaGetSymbolAddress, that device current)
// and that address is what the kernel and the copies are given.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned long long rms_static_label_count[RMS_STATIC_MAX_LABELS];

static int rms_static_label_count_ptr(unsigned long long** out)
{
    static std::mutex mu;
    static unsigned long long* ptr_of_device[64] = {nullptr};
    int dev = -1;
    RMS_CUDA_TRY(cudaGetDevice(&dev));
    RMS_REQUIRE(dev >= 0 && dev < 64, RMS_ERR_UNSUPPORTED, "device index %d out of range", dev);
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr_of_device[dev]) {
        unsigned long long* p = nullptr;
        RMS_CUDA_TRY(cudaGetSymbolAddress((void**)&p, rms_static_label_count));
        RMS_REQUIRE(p != nullptr, RMS_ERR_CUDA, "cudaGetSymbolAddress returned no address for the static counters");
        ptr_of_device[dev] = p;
    }
    *out = ptr_of_device[dev];
    return RMS_OK;
}

extern "C" int rms_substrate_label_volumes_static(const rms_substrate* s, void* cuda_stream, uint64_t* voxels_out)
{
    RMS_REQUIRE(s && voxels_out, RMS_ERR_ARG, "rms_substrate_label_volumes_static: null argument");
    RMS_REQUIRE(s->n_labels <= RMS_STATIC_MAX_LABELS, RMS_ERR_UNSUPPORTED,
                "rms_substrate_label_volumes_static: n_labels = %d exceeds the %d labels the static counters hold "
                "(RMS_STATIC_MAX_LABELS); use rms_substrate_label_volumes", s->n_labels, RMS_STATIC_MAX_LABELS);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    unsigned long long* d_count = nullptr;
    const int rc = rms_static_label_count_ptr(&d_count);
    if (rc != RMS_OK) return rc;
    const size_t bytes = (size_t)s->n_labels * sizeof(unsigned long long);
    // the array keeps the counts of the last call: every call starts by clearing the part it uses
    RMS_CUDA_TRY(cudaMemsetAsync(d_count, 0, bytes, stream));
    const uint64_t per_block = 1ull << 24;       // 32-bit shared counters: at most 2^32 - 1 voxels per block
    const unsigned grid = (unsigned)std::min<uint64_t>(std::max<uint64_t>((s->n_vox + per_block - 1) / per_block, 148ull * 8), 1u << 20);
    rms_label_volumes_kernel<<<grid, 256, 0, stream>>>(s->d_labels, s->n_vox, s->n_labels, d_count);
    RMS_CUDA_TRY(cudaGetLastError());
    RMS_CUDA_TRY(cudaMemcpyAsync(voxels_out, d_count, bytes, cudaMemcpyDeviceToHost, stream));
    RMS_CUDA_TRY(cudaStreamSynchronize(stream));
    return RMS_OK;
}

extern "C" int rms_substrate_get_info(const rms_substrate* s, rms_substrate_info* out)
{
    RMS_REQUIRE(s && out, RMS_ERR_ARG, "rms_substrate_get_info: null argument");
    out->nx = s->nx; out->ny = s->ny; out->nz = s->nz;
    out->n_labels = s->n_labels; out->n_classes = s->n_classes;
    out->n_voxels = s->n_vox;
    out->n_membrane_faces = s->n_membrane_faces;
    out->lattice_bytes = s->n_vox * sizeof(uint16_t);
    const uint64_t n_pad = (uint64_t)s->NX * s->NY * s->NZ;
    out->brick_bytes = (s->d_oct ? n_pad * sizeof(uint2) : 0) + (s->d_nbr ? n_pad * sizeof(uint32_t) : 0) +
                       (s->d_code ? n_pad * sizeof(uint16_t) + ((size_t)RMS_DICT_ESCAPE + 1) * sizeof(uint2) + ((size_t)s->esc_mask + 1) * sizeof(uint4) : 0);
    out->has_bricks = s->d_oct != nullptr || s->d_code != nullptr;
    out->dict_entries = s->n_dict;
    out->dict_escaped_voxels = s->n_esc;
    return RMS_OK;
}

// Eq.1 and Eq.3, Eq.C.15 for kappa = inf; fp64 on the host, rounded once to fp32.
// Rejection sampling has its own permeation probability, P_T / (1 - P_T) = kappa ds / D C_d (Appendix B.1 with Eq.2a),
// which the paper derives for equal diffusivities on both sides only (R21).
int rms_compute_tables(const rms_substrate* s, double dt, std::vector<float>& s_tab, std::vector<float>& P_tab,
                       bool rejection_sampling)
{
    const int nL = s->n_labels;
    const double C3 = 2.0 / 3.0;
    RMS_REQUIRE(dt > 0 && isfinite(dt), RMS_ERR_ARG, "dt_ms must be positive and finite");
    s_tab.resize(nL);
    P_tab.assign((size_t)nL * nL, 0.f);
    for (int a = 0; a < nL; ++a) {
        s_tab[a] = (float)(sqrt(6.0 * (double)s->D[a] * dt) / s->voxel_um);
        RMS_REQUIRE(s_tab[a] < 1.0f, RMS_ERR_STEP_TOO_LARGE,
                    "hop length sqrt(6 D dt) = %.4g voxels for label %d: must stay below the voxel size (P:62, P:189)",
                    (double)s_tab[a], a);
    }
    for (int a = 0; a < nL; ++a)
        for (int b = 0; b < nL; ++b) {
            double P;
            if (a == b) {
                P = 1.0;
            } else {
                const double k = s->kappa[(size_t)a * nL + b], Da = s->D[a], Db = s->D[b];
                const double ca = s->conc.empty() ? 1.0 : (double)s->conc[a], cb = s->conc.empty() ? 1.0 : (double)s->conc[b];
                if (k == 0 || ca == 0 || cb == 0) {
                    P = 0;                               // impermeable; nothing enters (or sits in) a medium without spins
                } else if (isinf(k)) {
                    P = fmin(1.0, cb * sqrt(Db) / (ca * sqrt(Da)));      // Eq.C.15
                } else if (ca != cb) {
                    // Eq.C.9 with kappa_0 = kappa (1 - alpha) of Eq.C.13-C.14, lambda = arg min alpha_lambda (R24)
                    RMS_REQUIRE(!rejection_sampling, RMS_ERR_UNSUPPORTED,
                                "rejection sampling with unequal spin concentrations (labels %d, %d)", a, b);
                    const double r = cb / ca, lam = 1.0 / (1.0 + cb * sqrt(Db) / (ca * sqrt(Da)));
                    const double Aab = k * sqrt(6.0 * dt / Da) * C3 * pow(r, lam), Aba = k * sqrt(6.0 * dt / Db) * C3 * pow(r, lam - 1.0);
                    P = Aab / (1.0 + 0.5 * (Aab + Aba));
                    RMS_REQUIRE(P <= 1.0, RMS_ERR_P_RANGE,
                                "Eq.C.9 gives P = %.4g > 1 from label %d into %d: lower kappa or dt (P:624)", P, a, b);
                } else if (rejection_sampling) {
                    RMS_REQUIRE(Da == Db, RMS_ERR_UNSUPPORTED,
                                "rejection sampling with a permeable membrane between unequal diffusivities (labels %d, %d): "
                                "Appendix B.1 gives P_T for equal D only", a, b);
                    const double A = k * sqrt(6.0 * dt / Da) * C3;
                    P = A / (1.0 + A);
                } else {
                    const double Aab = k * sqrt(6.0 * dt / Da) * C3, Aba = k * sqrt(6.0 * dt / Db) * C3;
                    P = Aab / (1.0 + 0.5 * (Aab + Aba));
                    RMS_REQUIRE(P <= 1.0, RMS_ERR_P_RANGE,
                                "Eq.3 gives P = %.4g > 1 from label %d into %d: lower kappa or dt (P:624)", P, a, b);
                }
            }
            P_tab[(size_t)a * nL + b] = (float)P;
        }
    return RMS_OK;
}

extern "C" int rms_tables(const rms_substrate* s, double dt_ms, float* s_out, float* P_out)
{
    RMS_REQUIRE(s, RMS_ERR_ARG, "rms_tables: null substrate");
    std::vector<float> st, pt;
    int rc = rms_compute_tables(s, dt_ms, st, pt);
    if (rc != RMS_OK) return rc;
    if (s_out) memcpy(s_out, st.data(), st.size() * sizeof(float));
    if (P_out) memcpy(P_out, pt.data(), pt.size() * sizeof(float));
    return RMS_OK;
}
