// rms_step_fast.cu -- H2..H5 for the throughput-critical case: impermeable or permeable membranes (built for the
// paper's regime P << 1, and measured to stay ahead of the general kernel at any P; see rms_permeable_step below) and piecewise-constant
// gradient waveforms (PGSE and every other rectangular-lobe sequence, any number of them).  Same method and
// the same numbers as the general kernel of rms_step.cu (section 2.2 steps 2-4; corner
// reflector of Fig.2; elastic collision P:90), organised for the B200 instruction pipes:
//
//   * one thread owns one walker for all steps of a launch, state in registers (position = linear index
//     into the padded neighbourhood lattice + fp32 in-voxel offset);
//   * the walker carries the 27-bit neighbourhood word of its voxel (rms_substrate.cu).  While it stays in
//     its compartment every face test of a hop -- first, second or third interaction, in any order --
//     is one bit of that word: "does the voxel I am about to enter carry my label?".  A step therefore
//     issues at most ONE gather (the word of the voxel it ends in), consumed a whole step later;
//   * the (at most three) interactions are resolved in hit order (R10) by sorting three keys
//     overshoot_k |r_i r_j| (same order as the hit times, no division), with the axis id in the two low
//     mantissa bits, and walking a position code through the word: three short, branch-light slots;
//   * per axis the outcome is applied branch-free: passed -> g -+ 1, reflected -> mirrored;
//   * the direction uses a 256-entry (cos, sin) table in shared memory + a degree-3 residual, accurate to
//     fp32 rounding with 5 ALU-pipe instructions (the ALU pipe, not issue, limits this kernel);
//   * Philox4x32-10: one call serves two steps (R2), both steps fully unrolled.
#include "rms_internal.cuh"

#ifndef RMS_FBLOCK
#define RMS_FBLOCK 128
#endif
#ifndef RMS_FMINB
#define RMS_FMINB 8                  // resident blocks per SM the register allocation is held to
#endif
#define RMS_FCHUNK 512u              // steps per chunk of the phase sums (even; 512 keeps the packed event sums inside int32)
#define RMS_ONE_MINUS 0.99999994f    // 1 - 2^-24

namespace {

__device__ __forceinline__ float rms_sqrt_fast(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// max / min of three signed ints (VIMNMX3 on sm_100)
__device__ __forceinline__ int rms_max3(int a, int b, int c) { return max(max(a, b), c); }
__device__ __forceinline__ int rms_min3(int a, int b, int c) { return min(min(a, b), c); }

// (a & b) | c in one LOP3
__device__ __forceinline__ int rms_and_or(int a, int b, int c)
{
    int r;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
// float bits with the two low mantissa bits replaced by a tag
__device__ __forceinline__ int rms_tag(float v, int tag) { return rms_and_or(__float_as_int(v), ~3, tag); }

// byte `sel` (0..3) of x, zero extended (selector nibbles 1..3 = 0 pick byte 0 of x, which callers keep 0)
__device__ __forceinline__ uint32_t rms_prmt(uint32_t x, uint32_t y, uint32_t sel)
{
    uint32_t r;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(x), "r"(y), "r"(sel));
    return r;
}

// padded linear index of a ghost voxel -> index of its periodic image inside the box, wrap counters updated
__device__ __noinline__ uint2 rms_fold_ghost(int lin, uint32_t wraps, int nx, int ny, int nz, int SX, int SY, int SZ)
{
    int X, Y, Z;
    rms_lattice_coords(lin, SX, SY, SZ, X, Y, Z);
    if (X == 0) { X = nx; wraps -= 1u; } else if (X == nx + 1) { X = 1; wraps += 1u; }
    if (Y == 0) { Y = ny; wraps -= 1u << 10; } else if (Y == ny + 1) { Y = 1; wraps += 1u << 10; }
    if (Z == 0) { Z = nz; wraps -= 1u << 20; } else if (Z == nz + 1) { Z = 1; wraps += 1u << 20; }
    return make_uint2((uint32_t)(X * SX + Y * SY + Z * SZ), wraps);
}

// ------------------------------------------------------------------------------------------------------------------
// Permeable substrates.  An unlike-label face is crossed with the probability of Eq.3, decided by the 33-bit
// uniform of R5 whose 9 coarse bits are the spare low bits of the step's direction words: u_e < P needs coarse bits
// below ceil(512 P_max).  For P << 1 (the paper's regime) that is 1 encounter in several hundred, so the kernel
// below treats every unlike-label face as a wall unless those bits allow a permeation; if they do, the WHOLE step is
// redone here by the interaction loop written out (the same arithmetic as rms_step.cu: labels gathered from the
// uint16 lattice, hop rescaled on entering a compartment of different D, R7).  Rare, so out of line.
//   st  = { fx, fy, fz, s }           in: offsets before the hop, hop length;  out: offsets after it, new hop length
//   ist = { lin, wraps, L, dAx, dAy, dAz, n_enc, n_perm, saturated }   in: lin, wraps, L;  out: all (dA = net voxel move per axis)
// Absorbing membranes (Eq.4; R20) ride on the same path: their saturation draw belongs to every membrane met, so a run with
// a rho table sets ceil(512 P_max) to 512 and every step that meets a membrane comes here.
// ------------------------------------------------------------------------------------------------------------------
__device__ __noinline__ void rms_permeable_step(const rms_step_params* pp, uint32_t id_lo, uint32_t id_hi, uint32_t j,
                                                uint32_t wa, uint32_t wb, float rx, float ry, float rz, float* st, int* ist)
{
    const rms_step_params& p = *pp;
    const float INF = __int_as_float(0x7f800000);
    int X, Y, Z;
    rms_lattice_coords(ist[0], p.SX, p.SY, p.SZ, X, Y, Z);
    int wr[3] = {0, 0, 0};
    if (X == 0) { X = p.nx; --wr[0]; } else if (X == p.nx + 1) { X = 1; ++wr[0]; }     // sitting on a ghost voxel: fold
    if (Y == 0) { Y = p.ny; --wr[1]; } else if (Y == p.ny + 1) { Y = 1; ++wr[1]; }
    if (Z == 0) { Z = p.nz; --wr[2]; } else if (Z == p.nz + 1) { Z = 1; ++wr[2]; }
    int w[3] = {X - 1, Y - 1, Z - 1};
    const int nk3[3] = {p.nx, p.ny, p.nz};
    const int str3[3] = {1, p.nx, p.nx * p.ny};
    float pk3[3] = {st[0], st[1], st[2]};
    float r3[3] = {rx, ry, rz};
    float s = st[3];
    uint32_t L = (uint32_t)ist[2];
    bool done[3] = {false, false, false};
    int dA[3] = {0, 0, 0};
    int e = 0, n_enc = 0, n_perm = 0;
    uint32_t v0 = 0, v1 = 0, v2 = 0, v3 = 0;
    bool have_v = false;
    uint32_t m0 = 0, m1 = 0, m2 = 0, m3 = 0;
    bool have_m = false, saturated = false;
    for (int it = 0; it < 3; ++it) {
        float t3[3];
        bool any = false;
        for (int k = 0; k < 3; ++k) {
            const float g = pk3[k] + r3[k];
            const bool c = !done[k] && __float_as_uint(g) >= 0x3F800000u;
            t3[k] = c ? __fdividef((r3[k] > 0.f ? 1.f : 0.f) - pk3[k], r3[k]) : INF;
            any |= c;
        }
        if (!any) break;
        const float tm = fminf(t3[0], fminf(t3[1], t3[2]));
        const int k = (t3[0] == tm) ? 0 : ((t3[1] == tm) ? 1 : 2);           // ties: lowest axis first (R10)
        const bool neg = r3[k] < 0.f;
        for (int q = 0; q < 3; ++q) pk3[q] = fmaf(tm, r3[q], pk3[q]);
        const float rest = 1.f - tm;
        for (int q = 0; q < 3; ++q) r3[q] *= rest;
        int nwk = w[k] + (neg ? -1 : 1), dwrap = 0;
        if (nwk < 0) { nwk = nk3[k] - 1; dwrap = -1; } else if (nwk == nk3[k]) { nwk = 0; dwrap = 1; }
        const uint32_t Ln = __ldg(p.labels + ((w[2] * p.ny + w[1]) * p.nx + w[0] + (nwk - w[k]) * str3[k]));
        bool pass = true;
        if (Ln != L) {
            ++n_enc;
            if (p.PMT) {                                                     // Eq.4: the encounter saturates the walker with P_MT
                const float Q = __ldg(p.PMT + (size_t)L * p.n_labels + Ln);
                if (Q > 0.f) {
                    if (!have_m) { rms_philox(p.rk, id_lo, id_hi, j + 1u, RMS_STREAM_MT, m0, m1, m2, m3); have_m = true; }
                    if (rms_uni(e == 0 ? m0 : (e == 1 ? m1 : m2)) < Q) saturated = true;
                }
            }
            const float T = __ldg(p.P512 + (size_t)L * p.n_labels + Ln);     // 512 P(L -> Ln), Eq.3
            if (T >= 512.f) pass = true;
            else if (T <= 0.f) pass = false;
            else {
                if (e >= 2 && !have_v) { rms_philox(p.rk, id_lo, id_hi, j + 1u, RMS_STREAM_PERM, v0, v1, v2, v3); have_v = true; }
                const float cf = (float)((e == 0 ? wa : (e == 1 ? wb : v3)) & 511u);
                if (cf + 1.f <= T) pass = true;
                else if (cf >= T) pass = false;
                else {
                    if (!have_v) { rms_philox(p.rk, id_lo, id_hi, j + 1u, RMS_STREAM_PERM, v0, v1, v2, v3); have_v = true; }
                    pass = rms_uni(e == 0 ? v0 : (e == 1 ? v1 : v2)) < (T - cf);
                }
            }
            ++e;
            n_perm += pass;
        }
        const float plane = neg ? 0.f : 1.f;
        if (pass) {
            pk3[k] = 1.f - plane;
            w[k] = nwk;
            wr[k] += dwrap;
            dA[k] += neg ? -1 : 1;
            if (Ln != L) {                   // rest of the hop at the new compartment's speed (R7)
                const float s_new = __ldg(p.s_tab + Ln);
                const float sc = __fdividef(s_new, s);
                for (int q = 0; q < 3; ++q) r3[q] *= sc;
                s = s_new;
                L = Ln;
            }
        } else {
            pk3[k] = plane;
            r3[k] = -r3[k];                  // elastic collision
        }
        done[k] = true;
    }
    for (int k = 0; k < 3; ++k) st[k] = fminf(fmaxf(pk3[k] + r3[k], 0.f), RMS_ONE_MINUS);
    st[3] = s;
    ist[0] = (w[0] + 1) * p.SX + (w[1] + 1) * p.SY + (w[2] + 1) * p.SZ;
    ist[1] = (int)((uint32_t)ist[1] + (uint32_t)wr[0] + ((uint32_t)wr[1] << 10) + ((uint32_t)wr[2] << 20));
    ist[2] = (int)L;
    ist[3] = dA[0]; ist[4] = dA[1]; ist[5] = dA[2];
    ist[6] = n_enc; ist[7] = n_perm; ist[8] = saturated ? 1 : 0;
}

}  // namespace

template <bool XFAST, bool PERM>
__global__ void __launch_bounds__(RMS_FBLOCK, RMS_FMINB) rms_step_fast_kernel(const __grid_constant__ rms_step_params p)
{
    __shared__ float2 sm_trig[256];   // (cos, sin) of the centre of the 256 azimuth bins

    for (int t = threadIdx.x; t < 256; t += RMS_FBLOCK) {
        double sn, cs;
        sincospi(-1.0 + (2.0 * t + 1.0) / 256.0, &sn, &cs);   // bin centre: theta = -pi + (t + 1/2) 2 pi / 256
        sm_trig[t] = make_float2((float)cs, (float)sn);
    }
    __syncthreads();

    // 32-bit shared-window address of the table, held in a register so that the hot loop does not rebuild the
    // window base every step
    // (the "memory" clobber also tells the compiler that the table above is read later: its only readers are the
    // ld.shared of the hot loop, written in PTX)
    int trig_base;
    asm volatile("mov.b32 %0, %1;" : "=r"(trig_base) : "r"((int)__cvta_generic_to_shared(sm_trig)) : "memory");

    const uint64_t t_global = (uint64_t)blockIdx.x * RMS_FBLOCK + threadIdx.x;
    if (t_global >= p.n) return;
    const uint64_t i = p.order ? (uint64_t)p.order[t_global] : t_global;   // walker of this thread (rms_sched.cu)
    const uint64_t id = p.first_id + i;
    const uint32_t id_lo = (uint32_t)id, id_hi = (uint32_t)(id >> 32);
    const size_t n = (size_t)p.n;

    // ---- load state -----------------------------------------------------------------------
    int wx = p.st.w[0][i], wy = p.st.w[1][i], wz = p.st.w[2][i];
    const int wx0 = wx, wy0 = wy, wz0 = wz;
    int dIx = p.st.dI[0][i], dIy = p.st.dI[1][i], dIz = p.st.dI[2][i];
    float fx = p.st.f[0][i], fy = p.st.f[1][i], fz = p.st.f[2][i];
    const uint32_t lab = p.st.lab[i];
    uint32_t L = lab & 0xFFFFu;                 // changes only on a permeation (PERM)
    float s = p.s_tab[L];
    float rate = p.rate[L], relax = p.st.relax[i];
    uint32_t j_rate = p.step0;                  // steps up to here are already in `relax`
    unsigned n_perm = 0, n_sat = 0;
    const uint32_t t_ceil = PERM ? p.t_ceil : 0u;   // permeation needs coarse bits below ceil(512 P_max)

    const int SX = XFAST ? 1 : p.SX, SY = p.SY, SZ = p.SZ;      // x fastest (the default order): unit stride known at compile time
    int lin = (wx + 1) * SX + (wy + 1) * SY + (wz + 1) * SZ;
    uint32_t wraps = 512u | (512u << 10) | (512u << 20);   // packed per-axis counts of box wraps (+512)
    uint32_t nb = __ldg(p.nbr + lin);

    // Phase (Eq.7, R11): Phi_m = sum_i w_m[i] (x_i - x_0).  Inside a segment every waveform is constant, so all of them
    // need the same sum  sum_i (x_i - x_0)  over the segment, taken in chunks of <= RMS_FCHUNK steps:
    //   sum_i f_i              -> SF (fp32, flushed to fp64 per chunk)
    //   sum_i (voxel index)    -> event driven: a face passage at a step adds +-1 to every later x_i of the chunk, i.e.
    //                             +-(steps left in the chunk); A collects that in its low 21 bits and, 2^21 apart, the
    //                             net number of passages, which moves the chunk's starting voxel Dst along
    //   Phi_m += w_m (SF + A_low + (Dst - f_0) len)   at the end of the chunk, for every waveform.
    // The cost per step does not depend on the number of waveforms.
    float SFx = 0.f, SFy = 0.f, SFz = 0.f;
    int Ax = 0, Ay = 0, Az = 0;
    int Dstx = dIx, Dsty = dIy, Dstz = dIz;
    int remK = 0;                               // steps left in the chunk (this one included) + 2^21
    unsigned n_enc = 0;

    // landed on a ghost voxel: fold back into the box (rare; the word of a ghost voxel is its image's word)
    auto fold = [&]() {
        const uint2 lw = rms_fold_ghost(lin, wraps, p.nx, p.ny, p.nz, SX, SY, SZ);
        lin = (int)lw.x; wraps = lw.y;
        nb &= ~RMS_NBR_GHOST;
    };

    // ---- one Monte Carlo step from the two direction words (R3, R4) ------------------------------
    auto step = [&](const uint32_t wa, const uint32_t wb, const uint32_t jj) {
        // z = sym(wa): exact odd multiple of 2^-23
        const float z = fmaf(__uint_as_float(__funnelshift_r(wa, 0x7Fu, 9)) - 1.5f, 2.0f, 1.1920928955078125e-07f);
        // azimuth pi * sym(wb) = bin centre (top 8 bits) + residual (next 15 bits, exact): rotate the table entry
        float2 cs0;                                              // sm_trig[wb >> 24]
        asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(cs0.x), "=f"(cs0.y) : "r"((int)(wb >> 24) * 8 + trig_base));
        const float tau = __int_as_float(rms_and_or((int)(wb >> 1), 0x007FFF00, 0x3F800080)) - 1.5f;   // in (-1/2, 1/2), exact
        const float x2 = tau * tau;
        const float sb = tau * fmaf(x2, -2.4641574e-06f, 0.024543693f);    // sin(tau pi/128)
        const float e = x2 * -3.0119642e-04f;                               // cos(tau pi/128) - 1
        const float cpsi = fmaf(cs0.x, e, -cs0.y * sb) + cs0.x;
        const float spsi = fmaf(cs0.y, e, cs0.x * sb) + cs0.y;
        const float sr = s * rms_sqrt_fast(fmaf(-z, z, 1.0f));
        const float rx = sr * cpsi, ry = sr * spsi, rz = s * z;

        float gx = fx + rx, gy = fy + ry, gz = fz + rz;
        const bool cx = __float_as_uint(gx) >= 0x3F800000u;    // g >= 1 or g < 0: the hop reaches a voxel face
        const bool cy = __float_as_uint(gy) >= 0x3F800000u;
        const bool cz = __float_as_uint(gz) >= 0x3F800000u;
        if (cx | cy | cz) {
            // sign of the hop per axis; plane ahead h = (1 + sigma)/2; overshoot beyond it rho = sigma g - h >= 0
            const float sgx = __uint_as_float((__float_as_uint(rx) & 0x80000000u) | 0x3F800000u);
            const float sgy = __uint_as_float((__float_as_uint(ry) & 0x80000000u) | 0x3F800000u);
            const float sgz = __uint_as_float((__float_as_uint(rz) & 0x80000000u) | 0x3F800000u);
            const float h2x = sgx + 1.f, h2y = sgy + 1.f, h2z = sgz + 1.f;          // 2 h
            const float rhox = fmaf(sgx, gx, -0.5f * h2x), rhoy = fmaf(sgy, gy, -0.5f * h2y), rhoz = fmaf(sgz, gz, -0.5f * h2z);
            // hit order (R10): larger overshoot / |r| = earlier.  key_k = rho_k |r_i r_j| orders the same way;
            // a face not reached has rho < 0 and sorts last.  The two low mantissa bits carry 3 - axis, so
            // ties go to the lower axis and the slot knows its axis.
            const float ax = fabsf(rx), ay = fabsf(ry), az = fabsf(rz);
            const int kx = rms_tag(rhox * (ay * az), 3);
            const int ky = rms_tag(rhoy * (ax * az), 2);
            const int kz = rms_tag(rhoz * (ax * ay), 1);
            const int k_hi = rms_max3(kx, ky, kz), k_lo = rms_min3(kx, ky, kz);
            const int k_mid = kx ^ ky ^ kz ^ k_hi ^ k_lo;
            // per-axis increments of the position code: pass flag (bit 5 + axis) + signed step in the 3x3x3 index,
            // one byte each at byte 3 - axis (byte 0 = 0 serves the upper result bytes of the permute):
            // x: 32 +- 1, y: 64 +- 3, z: 128 +- 9, switched by the sign masks of the hop
            const int mx = __float_as_int(rx) >> 31, my = __float_as_int(ry) >> 31, mz = __float_as_int(rz) >> 31;
            // (integer multiply-adds: they run on the FMA pipe, the ALU pipe is the busy one)
            const int isx = 2 * mx + 1, isy = 2 * my + 1, isz = 2 * mz + 1;
            const uint32_t lut = 0x21438900u + (uint32_t)(mx * 0x02000000 + my * 0x00060000 + mz * 0x00001200);
            int dl = 0;                                             // lattice-index change of this hop
            uint32_t pos = RMS_NBR_SELF;
            // PERM: bit e set = the e-th membrane met in this step may be crossed (its coarse random bits are below
            // ceil(512 P_max); the third draw's bits are not at hand, so it always may)
            const uint32_t pm = PERM ? ((uint32_t)((wa & 511u) < t_ceil) | ((uint32_t)((wb & 511u) < t_ceil) << 1) | 4u) : 0u;
            uint32_t redo = 0;
            auto slot = [&](const int key) {
                const uint32_t q = pos + rms_prmt(lut, 0u, (uint32_t)key & 3u);
                // the voxel ahead carries my label: pass; else a membrane: count the collision in bits 8..9
                if (nb & __funnelshift_l(0u, 1u, q)) pos = q;
                else { if (PERM) redo |= pm >> (pos >> 8); pos += 0x100u; }
            };
            slot(k_hi);
            if (k_mid >= 0) {
                slot(k_mid);
                if (k_lo >= 0) slot(k_lo);
            }
            if (PERM && (redo & 1u)) {
                // a membrane of this step may be permeated: redo the step by the written-out interaction loop
                float st[4] = {fx, fy, fz, s};
                int ist[9] = {lin, (int)wraps, (int)L, 0, 0, 0, 0, 0, 0};
                rms_permeable_step(&p, id_lo, id_hi, jj, wa, wb, rx, ry, rz, st, ist);
                gx = st[0]; gy = st[1]; gz = st[2];
                lin = ist[0]; wraps = (uint32_t)ist[1];
                Ax += ist[3] * remK; Ay += ist[4] * remK; Az += ist[5] * remK;
                n_enc += (unsigned)ist[6]; n_perm += (unsigned)ist[7];
                if (ist[8] && relax != __int_as_float(0x7f800000)) {   // alpha_rho = 0 from here on (Eq.4); the walk goes on
                    relax = __int_as_float(0x7f800000);
                    ++n_sat;
                }
                if ((uint32_t)ist[2] != L) {
                    // Eq.5: the whole dt of this step goes to the compartment at the end of the hop (R12)
                    relax = fmaf(rate, (float)(jj - j_rate), relax);
                    j_rate = jj;
                    L = (uint32_t)ist[2]; s = st[3]; rate = __ldg(p.rate + L);
                }
                nb = __ldg(p.nbr + lin);
            } else {
            // outcome per axis: passed -> g - sigma (enters the neighbour); membrane -> elastic collision,
            // mirrored on the face plane: 2 h - g
            {
                const bool ps = (pos & 32u) != 0, rf = cx && !ps;
                if (ps) {
                    gx -= sgx; dl = isx * SX;
                    Ax += isx * remK;
                }
                if (rf) gx = h2x - gx;
            }
            {
                const bool ps = (pos & 64u) != 0, rf = cy && !ps;
                if (ps) {
                    gy -= sgy; dl += isy * SY;
                    Ay += isy * remK;
                }
                if (rf) gy = h2y - gy;
            }
            {
                const bool ps = (pos & 128u) != 0, rf = cz && !ps;
                if (ps) {
                    gz -= sgz; dl += isz * SZ;
                    Az += isz * remK;
                }
                if (rf) gz = h2z - gz;
            }
            n_enc += pos >> 8;
            if (pos & 0xE0u) {
                // the walker changes voxel.  If it sat on a ghost voxel (it stepped over the box edge earlier; the word of a
                // ghost voxel is its image's, so the tests above were right) fold it back into the box first.  The test
                // sits here, after the slots, so that the gather issued a step ago is not waited for any earlier.
                if (nb & RMS_NBR_GHOST) fold();
                lin += dl;
                nb = __ldg(p.nbr + lin);
            }
            }
        }
        fx = gx; fy = gy; fz = gz;
        // phase: sum of the in-voxel offsets (the voxel part is event driven, above)
        SFx += fx; SFy += fy; SFz += fz;
        --remK;
    };

    uint32_t j = p.step0;                       // steps done so far (absolute)
#pragma unroll 1
    for (int sg = 0; sg < p.n_seg; ++sg) {
        const uint32_t seg_end = j + p.segs[sg].n;
        const bool seg_weighted = (p.segs[sg].flags & 1u) != 0;          // some waveform is non-zero on this segment
#pragma unroll 1
        while (j < seg_end) {
            const uint32_t chunk_end = min(seg_end, (j + RMS_FCHUNK) & ~1u), chunk_begin = j;
            remK = (int)(chunk_end - j) + (1 << 21);
            uint32_t r0, r1, r2, r3;
            if (j & 1u) {                        // second half of a Philox call that an earlier segment began
                rms_philox(p.rk, id_lo, id_hi, j >> 1, RMS_STREAM_DIR, r0, r1, r2, r3);
                step(r2, r3, j);
                ++j;
            }
#pragma unroll 1
            while (j + 2u <= chunk_end) {
                rms_philox(p.rk, id_lo, id_hi, j >> 1, RMS_STREAM_DIR, r0, r1, r2, r3);
                step(r0, r1, j);
                step(r2, r3, j + 1u);
                j += 2u;
            }
            if (j < chunk_end) {
                rms_philox(p.rk, id_lo, id_hi, j >> 1, RMS_STREAM_DIR, r0, r1, r2, r3);
                step(r0, r1, j);
                ++j;
            }
            // end of the chunk: its sum of (x_i - x_0) per axis, in fp64, times the weight of every waveform
            {
                const int netx = (Ax + (1 << 20)) >> 21, nety = (Ay + (1 << 20)) >> 21, netz = (Az + (1 << 20)) >> 21;
                const double len = (double)(chunk_end - chunk_begin);
                const double cx = (double)SFx + (double)(Ax - (netx << 21)) + ((double)Dstx - (double)p.st.f0[0][i]) * len;
                const double cy = (double)SFy + (double)(Ay - (nety << 21)) + ((double)Dsty - (double)p.st.f0[1][i]) * len;
                const double cz = (double)SFz + (double)(Az - (netz << 21)) + ((double)Dstz - (double)p.st.f0[2][i]) * len;
                Dstx += netx; Dsty += nety; Dstz += netz;
                SFx = SFy = SFz = 0.f; Ax = Ay = Az = 0;
                if (seg_weighted)
                    for (int m = 0; m < p.n_wave; ++m) {
                        const double wm = (double)__ldg(&p.segs[sg].wf[m]);
                        if (wm != 0.0) {
                            p.st.phi[(size_t)(3 * m + 0) * n + i] += wm * cx;
                            p.st.phi[(size_t)(3 * m + 1) * n + i] += wm * cy;
                            p.st.phi[(size_t)(3 * m + 2) * n + i] += wm * cz;
                        }
                    }
            }
        }
    }

    // ---- store state --------------------------------------------------------------------------
    {
        int X, Y, Z;
        rms_lattice_coords(lin, SX, SY, SZ, X, Y, Z);
        int wrx = (int)(wraps & 1023u) - 512, wry = (int)((wraps >> 10) & 1023u) - 512, wrz = (int)((wraps >> 20) & 1023u) - 512;
        if (X == 0) { X = p.nx; --wrx; } else if (X == p.nx + 1) { X = 1; ++wrx; }
        if (Y == 0) { Y = p.ny; --wry; } else if (Y == p.ny + 1) { Y = 1; ++wry; }
        if (Z == 0) { Z = p.nz; --wrz; } else if (Z == p.nz + 1) { Z = 1; ++wrz; }
        wx = X - 1; wy = Y - 1; wz = Z - 1;
        dIx += (wx - wx0) + wrx * p.nx;
        dIy += (wy - wy0) + wry * p.ny;
        dIz += (wz - wz0) + wrz * p.nz;
    }
    p.st.w[0][i] = wx; p.st.w[1][i] = wy; p.st.w[2][i] = wz;
    p.st.dI[0][i] = dIx; p.st.dI[1][i] = dIy; p.st.dI[2][i] = dIz;
    // an offset of exactly 1 (a walker left sitting on its upper face by rounding) is legal inside the loop: it
    // crosses at once if it moves on upwards; the stored state keeps the floor convention [0, 1) (R15)
    p.st.f[0][i] = fminf(fx, RMS_ONE_MINUS); p.st.f[1][i] = fminf(fy, RMS_ONE_MINUS); p.st.f[2][i] = fminf(fz, RMS_ONE_MINUS);
    p.st.f_lo[0][i] = 0.f; p.st.f_lo[1][i] = 0.f; p.st.f_lo[2][i] = 0.f;
    p.st.relax[i] = fmaf(rate, (float)(p.step0 + p.n_steps - j_rate), relax);   // Eq.5; the label changes only on a permeation
    if (PERM) p.st.lab[i] = (lab & 0xFFFF0000u) | L;

    // diagnostics: warp-shuffle reduction, one atomic per warp (early-exited lanes are not in the mask)
    const unsigned mask = __activemask();
    n_enc = __reduce_add_sync(mask, n_enc);
    if (PERM) n_perm = __reduce_add_sync(mask, n_perm);
    if (PERM) n_sat = __reduce_add_sync(mask, n_sat);
    if ((threadIdx.x & 31) == (unsigned)(__ffs(mask) - 1)) {
        if (n_enc) atomicAdd(&p.counters[0], (unsigned long long)n_enc);
        if (PERM && n_perm) atomicAdd(&p.counters[1], (unsigned long long)n_perm);
        if (PERM && n_sat) atomicAdd(&p.counters[4], (unsigned long long)n_sat);
    }
}

int rms_launch_step_fast(const rms_step_params& p, int n_wave, bool permeable, cudaStream_t stream)
{
    if (p.n == 0 || p.n_steps == 0) return RMS_OK;
    const unsigned grid = (unsigned)((p.n + RMS_FBLOCK - 1) / RMS_FBLOCK);
    RMS_REQUIRE(n_wave >= 0 && n_wave <= RMS_MAX_WAVES, RMS_ERR_UNSUPPORTED, "n_wave = %d is above RMS_MAX_WAVES = %d", n_wave,
                RMS_MAX_WAVES);
    const bool xf = p.SX == 1;
    if (permeable) {
        if (xf) rms_step_fast_kernel<true, true><<<grid, RMS_FBLOCK, 0, stream>>>(p);
        else rms_step_fast_kernel<false, true><<<grid, RMS_FBLOCK, 0, stream>>>(p);
    } else {
        if (xf) rms_step_fast_kernel<true, false><<<grid, RMS_FBLOCK, 0, stream>>>(p);
        else rms_step_fast_kernel<false, false><<<grid, RMS_FBLOCK, 0, stream>>>(p);
    }
    RMS_CUDA_TRY(cudaGetLastError());
    return RMS_OK;
}
