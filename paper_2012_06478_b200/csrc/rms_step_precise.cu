// rms_step_precise.cu -- the specialised step kernel of rms_step_fast.cu in fp64 arithmetic (RMS_RUN_FP64).
//
// Why it exists: a hop that passes the edge of a convex membrane corner goes round it or is
// reflected by it depending on which of two faces it reaches first, so an fp32 walker and the fp64 oracle walker
// that differ by e in position part company with probability ~ e per such hop.  fp32 positions (error ~1e-6 voxel
// after 1e4 steps) keep 99.98 % of the walkers on the oracle's trajectory at 1e4 steps, 99.8 % at 4e4 and cannot hold
// 99.9 % at the 5e4 .. 5e5 steps of BASELINE.json's configs 1-3.  Here direction, hop, offsets, hit order and
// phase are fp64 (B200 runs DFMA at half the FFMA rate; the fp64 pipe is otherwise idle), which puts the position
// difference at 1e-13 and the trajectories on the oracle's.  Same method, same structure as the fp32 kernel:
// one thread per walker, 27-bit neighbourhood word, keys sorted by hit time, position code walked through the word.
#include "rms_internal.cuh"

#define RMS_PBLOCK 128

namespace {

__device__ __forceinline__ uint32_t rms_prmt_p(uint32_t x, uint32_t y, uint32_t sel)
{
    uint32_t r;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(x), "r"(y), "r"(sel));
    return r;
}

__device__ __noinline__ uint2 rms_fold_ghost_p(int lin, uint32_t wraps, int nx, int ny, int nz, int SX, int SY, int SZ)
{
    int X, Y, Z;
    rms_lattice_coords(lin, SX, SY, SZ, X, Y, Z);
    if (X == 0) { X = nx; wraps -= 1u; } else if (X == nx + 1) { X = 1; wraps += 1u; }
    if (Y == 0) { Y = ny; wraps -= 1u << 10; } else if (Y == ny + 1) { Y = 1; wraps += 1u << 10; }
    if (Z == 0) { Z = nz; wraps -= 1u << 20; } else if (Z == nz + 1) { Z = 1; wraps += 1u << 20; }
    return make_uint2((uint32_t)(X * SX + Y * SY + Z * SZ), wraps);
}

// g >= 1 or g < 0 (or -0): the sign / exponent word of the double, read as unsigned, is >= that of 1.0
__device__ __forceinline__ bool rms_outside_d(double g) { return (uint32_t)__double2hiint(g) >= 0x3FF00000u; }

// bits of v with the two low mantissa bits replaced by a tag
__device__ __forceinline__ long long rms_tag_d(double v, int tag) { return (__double_as_longlong(v) & ~3ll) | (long long)tag; }

}  // namespace

__global__ void __launch_bounds__(RMS_PBLOCK) rms_step_precise_kernel(const __grid_constant__ rms_step_params p)
{
    __shared__ double2 sm_trig[256];   // (cos, sin) of the centre of the 256 azimuth bins

    for (int t = threadIdx.x; t < 256; t += RMS_PBLOCK) {
        double sn, cs;
        sincospi(-1.0 + (2.0 * t + 1.0) / 256.0, &sn, &cs);
        sm_trig[t] = make_double2(cs, sn);
    }
    __syncthreads();

    const uint64_t t_global = (uint64_t)blockIdx.x * RMS_PBLOCK + threadIdx.x;
    if (t_global >= p.n) return;
    const uint64_t i = p.order ? (uint64_t)p.order[t_global] : t_global;
    const uint64_t id = p.first_id + i;
    const uint32_t id_lo = (uint32_t)id, id_hi = (uint32_t)(id >> 32);
    const size_t n = (size_t)p.n;

    // ---- load state -----------------------------------------------------------------------
    int wx = p.st.w[0][i], wy = p.st.w[1][i], wz = p.st.w[2][i];
    const int wx0 = wx, wy0 = wy, wz0 = wz;
    int dIx = p.st.dI[0][i], dIy = p.st.dI[1][i], dIz = p.st.dI[2][i];
    double fx = (double)p.st.f[0][i] + (double)p.st.f_lo[0][i];
    double fy = (double)p.st.f[1][i] + (double)p.st.f_lo[1][i];
    double fz = (double)p.st.f[2][i] + (double)p.st.f_lo[2][i];
    const uint32_t L = p.st.lab[i] & 0xFFFFu;
    const double s = (double)p.s_tab[L];        // the fp32 table value, as on the oracle's side (R6)

    const int SX = p.SX, SY = p.SY, SZ = p.SZ;
    int lin = (wx + 1) * SX + (wy + 1) * SY + (wz + 1) * SZ;
    uint32_t wraps = 512u | (512u << 10) | (512u << 20);
    uint32_t nb = __ldg(p.nbr + lin);

    // Phase (Eq.7, R11), as in rms_step_fast.cu: inside a segment all waveforms are constant and share the sum of
    // (x_i - x_0) over the segment = sum f_i (SF) + event-driven voxel part (A: +-(steps left) per face passage) +
    // (Dst - f_0) x length, Dst = whole-voxel displacement at the start of the segment, moved along by the net passages
    double SFx = 0.0, SFy = 0.0, SFz = 0.0;
    long long Ax = 0, Ay = 0, Az = 0;
    int netx = 0, nety = 0, netz = 0;
    int Dstx = dIx, Dsty = dIy, Dstz = dIz;
    long long rem = 0;                          // steps left in the segment, this one included
    unsigned n_enc = 0;

    auto step = [&](const uint32_t wa, const uint32_t wb) {
        // z = sym(wa), tau = residual of the azimuth: both exact in fp32, widened
        const double z = (double)fmaf(__uint_as_float(__funnelshift_r(wa, 0x7Fu, 9)) - 1.5f, 2.0f, 1.1920928955078125e-07f);
        const double2 cs0 = sm_trig[wb >> 24];
        const double tau = (double)(__uint_as_float(((wb >> 1) & 0x007FFF00u) | 0x3F800080u) - 1.5f);
        const double b = tau * 0.024543692606170259675;            // tau pi / 128, |b| <= 0.0123
        const double b2 = b * b;
        const double sb = b * fma(b2, fma(b2, fma(b2, -1.0 / 5040.0, 1.0 / 120.0), -1.0 / 6.0), 1.0);     // sin b, error < 2e-23
        const double cm = b2 * fma(b2, fma(b2, -1.0 / 720.0, 1.0 / 24.0), -0.5);                         // cos b - 1
        const double cpsi = fma(cs0.x, cm, -cs0.y * sb) + cs0.x;
        const double spsi = fma(cs0.y, cm, cs0.x * sb) + cs0.y;
        const double sr = s * sqrt(fma(-z, z, 1.0));
        const double rx = sr * cpsi, ry = sr * spsi, rz = s * z;

        double gx = fx + rx, gy = fy + ry, gz = fz + rz;
        const bool cx = rms_outside_d(gx), cy = rms_outside_d(gy), cz = rms_outside_d(gz);
        if (cx | cy | cz) {
            const double sgx = copysign(1.0, rx), sgy = copysign(1.0, ry), sgz = copysign(1.0, rz);
            const double h2x = sgx + 1.0, h2y = sgy + 1.0, h2z = sgz + 1.0;
            const double rhox = fma(sgx, gx, -0.5 * h2x), rhoy = fma(sgy, gy, -0.5 * h2y), rhoz = fma(sgz, gz, -0.5 * h2z);
            const double ax = fabs(rx), ay = fabs(ry), az = fabs(rz);
            const long long kx = rms_tag_d(rhox * (ay * az), 3);
            const long long ky = rms_tag_d(rhoy * (ax * az), 2);
            const long long kz = rms_tag_d(rhoz * (ax * ay), 1);
            const long long k_hi = max(max(kx, ky), kz), k_lo = min(min(kx, ky), kz);
            const long long k_mid = kx ^ ky ^ kz ^ k_hi ^ k_lo;
            const int mx = __double2hiint(rx) >> 31, my = __double2hiint(ry) >> 31, mz = __double2hiint(rz) >> 31;
            const int isx = 2 * mx + 1, isy = 2 * my + 1, isz = 2 * mz + 1;
            const uint32_t lut = 0x21438900u + (uint32_t)(mx * 0x02000000 + my * 0x00060000 + mz * 0x00001200);
            int dl = 0;
            uint32_t pos = RMS_NBR_SELF;
            auto slot = [&](const long long key) {
                const uint32_t q = pos + rms_prmt_p(lut, 0u, (uint32_t)key & 3u);
                pos = (nb & __funnelshift_l(0u, 1u, q)) ? q : pos + 0x100u;
            };
            slot(k_hi);
            if (k_mid >= 0) {
                slot(k_mid);
                if (k_lo >= 0) slot(k_lo);
            }
            {
                const bool ps = (pos & 32u) != 0, rf = cx && !ps;
                if (ps) {
                    gx -= sgx; dl = isx * SX;
                    Ax += isx * rem; netx += isx;
                }
                if (rf) gx = h2x - gx;
            }
            {
                const bool ps = (pos & 64u) != 0, rf = cy && !ps;
                if (ps) {
                    gy -= sgy; dl += isy * SY;
                    Ay += isy * rem; nety += isy;
                }
                if (rf) gy = h2y - gy;
            }
            {
                const bool ps = (pos & 128u) != 0, rf = cz && !ps;
                if (ps) {
                    gz -= sgz; dl += isz * SZ;
                    Az += isz * rem; netz += isz;
                }
                if (rf) gz = h2z - gz;
            }
            n_enc += pos >> 8;
            if (pos & 0xE0u) {
                if (nb & RMS_NBR_GHOST) {
                    const uint2 lw = rms_fold_ghost_p(lin, wraps, p.nx, p.ny, p.nz, SX, SY, SZ);
                    lin = (int)lw.x; wraps = lw.y;
                }
                lin += dl;
                nb = __ldg(p.nbr + lin);
            }
        }
        fx = gx; fy = gy; fz = gz;
        SFx += fx; SFy += fy; SFz += fz;
        --rem;
    };

    uint32_t j = p.step0;
#pragma unroll 1
    for (int sg = 0; sg < p.n_seg; ++sg) {
        const uint32_t seg_n = p.segs[sg].n, seg_end = j + seg_n;
        rem = (long long)seg_n;
        uint32_t r0, r1, r2, r3;
        if ((j & 1u) && j < seg_end) {
            rms_philox(p.rk, id_lo, id_hi, j >> 1, RMS_STREAM_DIR, r0, r1, r2, r3);
            step(r2, r3);
            ++j;
        }
#pragma unroll 1
        while (j + 2u <= seg_end) {
            rms_philox(p.rk, id_lo, id_hi, j >> 1, RMS_STREAM_DIR, r0, r1, r2, r3);
            step(r0, r1);
            step(r2, r3);
            j += 2u;
        }
        if (j < seg_end) {
            rms_philox(p.rk, id_lo, id_hi, j >> 1, RMS_STREAM_DIR, r0, r1, r2, r3);
            step(r0, r1);
            ++j;
        }
        // end of the segment: its sum of (x_i - x_0) per axis times the weight of every waveform
        {
            const double len = (double)seg_n;
            const double cx = SFx + (double)Ax + ((double)Dstx - (double)p.st.f0[0][i]) * len;
            const double cy = SFy + (double)Ay + ((double)Dsty - (double)p.st.f0[1][i]) * len;
            const double cz = SFz + (double)Az + ((double)Dstz - (double)p.st.f0[2][i]) * len;
            Dstx += netx; Dsty += nety; Dstz += netz;
            SFx = SFy = SFz = 0.0; Ax = Ay = Az = 0; netx = nety = netz = 0;
            if (p.segs[sg].flags & 1u)
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
    // offset = f + f_lo with f < 1 in fp32 (floor convention R15) and f_lo the fp64 remainder
    {
        const double one_minus = 0.99999999999999988898;   // 1 - 2^-53
        fx = fmin(fx, one_minus); fy = fmin(fy, one_minus); fz = fmin(fz, one_minus);
        const float hx = fminf((float)fx, 0.99999994f), hy = fminf((float)fy, 0.99999994f), hz = fminf((float)fz, 0.99999994f);
        p.st.f[0][i] = hx; p.st.f[1][i] = hy; p.st.f[2][i] = hz;
        p.st.f_lo[0][i] = (float)(fx - (double)hx); p.st.f_lo[1][i] = (float)(fy - (double)hy); p.st.f_lo[2][i] = (float)(fz - (double)hz);
    }
    p.st.relax[i] = fmaf(p.rate[L], (float)p.n_steps, p.st.relax[i]);

    const unsigned mask = __activemask();
    n_enc = __reduce_add_sync(mask, n_enc);
    if ((threadIdx.x & 31) == (unsigned)(__ffs(mask) - 1) && n_enc) atomicAdd(&p.counters[0], (unsigned long long)n_enc);
}

int rms_launch_step_precise(const rms_step_params& p, int n_wave, cudaStream_t stream)
{
    if (p.n == 0 || p.n_steps == 0) return RMS_OK;
    const unsigned grid = (unsigned)((p.n + RMS_PBLOCK - 1) / RMS_PBLOCK);
    RMS_REQUIRE(n_wave >= 0 && n_wave <= RMS_MAX_WAVES, RMS_ERR_UNSUPPORTED, "n_wave = %d is above RMS_MAX_WAVES = %d", n_wave,
                RMS_MAX_WAVES);
    rms_step_precise_kernel<<<grid, RMS_PBLOCK, 0, stream>>>(p);
    RMS_CUDA_TRY(cudaGetLastError());
    return RMS_OK;
}
