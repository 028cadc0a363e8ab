// rms_step.cu -- H2..H5: the walker-persistent Monte Carlo step kernel (section 2.2 steps 2-4).
//
// One thread owns one walker for all steps of a launch; position (integer voxel + fp32 in-voxel offset),
// phase partial sums and the relaxation exponent stay in registers and are written back at launch
// boundaries only.  Per step: Philox4x32-10 words (one call serves two steps) -> unit direction ->
// tentative hop -> if a voxel face is reached, the interaction loop (at most three, ordered by hit
// time, Fig.2): same compartment behind the face -> pass; membrane -> elastic reflection
// or permeation with the probability of Eq.3.
//
// Two lattice paths:
//   RMS_LAT_FACES   impermeable runs: the walker caches the 6 membrane bits of its voxel (from the
//                   neighbourhood lattice); a reflection touches no memory, a pass issues one gather that
//                   is consumed at the NEXT interaction (off the critical path).  This is the general
//                   kernel (any waveform); rms_step_fast.cu serves piecewise-constant gradients.
//   RMS_LAT_LABELS  the paper's lookup table: gather the neighbour's uint16 label at every face.
//                   With PERM it follows the interaction loop literally, including the rescaling of
//                   the remaining hop on entering a compartment of different D (R7).
#include "rms_internal.cuh"

#define RMS_BLOCK 128
#define RMS_FLUSH 64          // steps between flushes of the fp32 / int32 phase partial sums into fp64
#define RMS_ONE_MINUS 0.99999994f   // 1 - 2^-24
#define RMS_INF __int_as_float(0x7f800000)

__device__ __forceinline__ float rms_sqrt_approx(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// hop vector of length s: z = sym(wa), azimuth = pi * sym(wb) (R4)
__device__ __forceinline__ void rms_hop(uint32_t wa, uint32_t wb, float s, float& rx, float& ry, float& rz)
{
    const float z = rms_sym(wa);
    const float a = rms_sym(wb);
    float sn, cs;
#ifdef RMS_FAST_TRIG
    __sincosf(a * 3.14159265358979f, &sn, &cs);
#else
    sincospif(a, &sn, &cs);
#endif
    const float sr = s * rms_sqrt_approx(fmaf(-z, z, 1.0f));
    rx = sr * cs;
    ry = sr * sn;
    rz = s * z;
}

// the 6 membrane bits of a voxel (bit k: face towards +k, bit 3+k: towards -k, bit 6: ghost) from its
// neighbourhood word: a face is a membrane iff the face neighbour does not carry the voxel's label
__device__ __forceinline__ uint32_t rms_face_byte(uint32_t w)
{
    const uint32_t n = ~w;
    return ((n >> 14) & 1u) | (((n >> 16) & 1u) << 1) | (((n >> 22) & 1u) << 2) | (((n >> 12) & 1u) << 3) |
           (((n >> 10) & 1u) << 4) | (((n >> 4) & 1u) << 5) | (((w >> 27) & 1u) << 6);
}

__device__ __forceinline__ bool rms_outside(float g) { return __float_as_uint(g) >= 0x3F800000u; }  // g >= 1 or g < 0

__device__ __forceinline__ float rms_hit_time(bool cross, float f, float r)
{
    return cross ? __fdividef((r > 0.f ? 1.f : 0.f) - f, r) : RMS_INF;
}

// PERM: 0 impermeable (per-axis outcome), 1 the interaction loop written out (permeation, D contrast), 2 the same with the
// absorbing membranes (Eq.4) and the bookkeeping of a cancelled step (rejection sampling, ERL) compiled in
template <int NW, int WMODE, int LAT, int PERM>
__global__ void __launch_bounds__(RMS_BLOCK) rms_step_kernel(const __grid_constant__ rms_step_params p)
{
    const uint64_t t_global = (uint64_t)blockIdx.x * RMS_BLOCK + threadIdx.x;
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
    uint32_t L = lab & 0xFFFFu;
    float s = p.s_tab[L];
    float relax = p.st.relax[i];
    float rate = p.rate[L];
    uint32_t j_rate = p.step0;      // steps up to here are already in `relax`

    // launch prologue of the phase: Phi += (dI - f0) * sum_{launch} w
    if (NW > 0) {
#pragma unroll
        for (int m = 0; m < NW; ++m) {
            const double wt = p.wtot[m];
            if (wt != 0.0) {
                p.st.phi[(size_t)(3 * m + 0) * n + i] += ((double)dIx - (double)p.st.f0[0][i]) * wt;
                p.st.phi[(size_t)(3 * m + 1) * n + i] += ((double)dIy - (double)p.st.f0[1][i]) * wt;
                p.st.phi[(size_t)(3 * m + 2) * n + i] += ((double)dIz - (double)p.st.f0[2][i]) * wt;
            }
        }
    }

    // FACES path: padded linear index + packed wrap counters instead of coordinates
    const int SX = p.SX, SY = p.SY, SZ = p.SZ;
    int lin = 0;
    uint32_t wraps = 512u | (512u << 10) | (512u << 20);
    uint32_t fm = 0;
    if (LAT == RMS_LAT_FACES) {
        lin = (wx + 1) * SX + (wy + 1) * SY + (wz + 1) * SZ;
        fm = rms_face_byte(__ldg(p.nbr + lin));
    }

    float phiF[NW > 0 ? NW : 1][3];
    int A32[NW > 0 ? NW : 1][3];
    double Ad[NW > 0 ? NW : 1][3];
#pragma unroll
    for (int m = 0; m < (NW > 0 ? NW : 1); ++m)
#pragma unroll
        for (int k = 0; k < 3; ++k) { phiF[m][k] = 0.f; A32[m][k] = 0; Ad[m][k] = 0.0; }

    unsigned n_enc = 0, n_perm = 0, n_clamp = 0, n_sat = 0;

    uint32_t j = p.step0;                       // steps done so far (absolute)
    const uint32_t j_launch_end = p.step0 + p.n_steps;
    const int n_seg = (WMODE == RMS_WMODE_CONST) ? p.n_seg : 1;

#pragma unroll 1
    for (int sg = 0; sg < n_seg; ++sg) {
        uint32_t seg_end;
        float wf[NW > 0 ? NW : 1];
        int wi[NW > 0 ? NW : 1];
        int wrem[NW > 0 ? NW : 1];              // CONST: remaining weight of this launch including the current step
        bool acc_w = false, acc_rem = false;
        if (WMODE == RMS_WMODE_CONST) {
            const rms_segment sgm = p.segs[sg];
            seg_end = j + sgm.n;
            acc_w = (sgm.flags & 1u) != 0;
            acc_rem = (sgm.flags & 2u) != 0;
#pragma unroll
            for (int m = 0; m < NW; ++m) {
                wi[m] = sgm.w[m];
                wf[m] = (float)sgm.w[m];
                wrem[m] = sgm.wrem_end[m] + sgm.w[m] * (int)sgm.n;
            }
        } else {
            seg_end = j_launch_end;
            acc_w = NW > 0;
            acc_rem = NW > 0;
        }

#pragma unroll 1
        while (j < seg_end) {
            const uint32_t chunk_end = min(seg_end, j + RMS_FLUSH);
#pragma unroll 1
            while (j < chunk_end) {
                uint32_t r0, r1, r2, r3;
                rms_philox(p.rk, id_lo, id_hi, j >> 1, RMS_STREAM_DIR, r0, r1, r2, r3);
#pragma unroll 1
                for (uint32_t h = j & 1u; h < 2u && j < chunk_end; ++h, ++j) {
                    const uint32_t wa = h ? r2 : r0, wb = h ? r3 : r1;
                    float rx, ry, rz;
                    rms_hop(wa, wb, s, rx, ry, rz);
                    if (WMODE == RMS_WMODE_TABLE && NW > 0) {
#pragma unroll
                        for (int m = 0; m < NW; ++m) wf[m] = __ldg(p.wave + (size_t)m * p.wave_stride + (j - p.step0));
                    }

                    if (!PERM) {
                        // ---------------- impermeable: per-axis independent outcome, faces tested in hit order ----
                        float gx = fx + rx, gy = fy + ry, gz = fz + rz;
                        const bool cx = rms_outside(gx), cy = rms_outside(gy), cz = rms_outside(gz);
                        if (cx | cy | cz) {
                            float tx = rms_hit_time(cx, fx, rx), ty = rms_hit_time(cy, fy, ry), tz = rms_hit_time(cz, fz, rz);
#pragma unroll 1
                            for (;;) {
                                const float tmin = fminf(tx, fminf(ty, tz));
                                if (tmin == RMS_INF) break;
                                const bool isx = (tx == tmin);
                                const bool isy = !isx && (ty == tmin);
                                const float gk = isx ? gx : (isy ? gy : gz);
                                const bool neg = gk < 0.f;
                                bool membrane;
                                int nlin = 0, nwk = 0;
                                if (LAT == RMS_LAT_FACES) {
                                    if (fm & 64u) {
                                        // landed on a ghost voxel earlier: fold back into the box (rare)
                                        int X, Y, Z;
                                        rms_lattice_coords(lin, SX, SY, SZ, X, Y, Z);
                                        if (X == 0) { X = p.nx; wraps -= 1u; } else if (X == p.nx + 1) { X = 1; wraps += 1u; }
                                        if (Y == 0) { Y = p.ny; wraps -= 1u << 10; } else if (Y == p.ny + 1) { Y = 1; wraps += 1u << 10; }
                                        if (Z == 0) { Z = p.nz; wraps -= 1u << 20; } else if (Z == p.nz + 1) { Z = 1; wraps += 1u << 20; }
                                        lin = X * SX + Y * SY + Z * SZ;
                                        fm = rms_face_byte(__ldg(p.nbr + lin));
                                    }
                                    const uint32_t bit = isx ? 1u : (isy ? 2u : 4u);
                                    membrane = ((fm >> (neg ? 3 : 0)) & bit) != 0;
                                } else {
                                    const int wk = isx ? wx : (isy ? wy : wz);
                                    const int nk = isx ? p.nx : (isy ? p.ny : p.nz);
                                    const int stride = isx ? 1 : (isy ? p.nx : p.nx * p.ny);
                                    nwk = wk + (neg ? -1 : 1);
                                    nwk = nwk < 0 ? nk - 1 : (nwk == nk ? 0 : nwk);
                                    nlin = (wz * p.ny + wy) * p.nx + wx + (nwk - wk) * stride;
                                    membrane = __ldg(p.labels + nlin) != L;
                                }
                                const float base = neg ? 0.f : 2.f;
                                float gnew;
                                if (membrane) {
                                    gnew = base - gk;               // mirror on the face plane
                                    ++n_enc;
                                } else {
                                    gnew = gk + (1.f - base);       // same compartment: the face does not exist
                                    if (LAT == RMS_LAT_FACES) {
                                        const int stride = isx ? SX : (isy ? SY : SZ);
                                        lin += neg ? -stride : stride;
                                        fm = rms_face_byte(__ldg(p.nbr + lin));
                                    } else {
                                        if (isx) wx = nwk; else if (isy) wy = nwk; else wz = nwk;
                                        const int sg1 = neg ? -1 : 1;
                                        if (isx) dIx += sg1; else if (isy) dIy += sg1; else dIz += sg1;
                                    }
                                    if (NW > 0 && acc_rem) {
                                        if (WMODE == RMS_WMODE_CONST) {
#pragma unroll
                                            for (int m = 0; m < NW; ++m) {
                                                const int v = neg ? -wrem[m] : wrem[m];
                                                if (isx) A32[m][0] += v; else if (isy) A32[m][1] += v; else A32[m][2] += v;
                                            }
                                        } else {
#pragma unroll
                                            for (int m = 0; m < NW; ++m) {
                                                double v = p.wsuf[(size_t)m * p.wsuf_stride + (j - p.step0)] - p.wsuf_end[m];
                                                v = neg ? -v : v;
                                                if (isx) Ad[m][0] += v; else if (isy) Ad[m][1] += v; else Ad[m][2] += v;
                                            }
                                        }
                                    }
                                }
                                const float gc = fminf(fmaxf(gnew, 0.f), RMS_ONE_MINUS);
                                n_clamp += (gc != gnew);
                                if (isx) { gx = gc; tx = RMS_INF; } else if (isy) { gy = gc; ty = RMS_INF; } else { gz = gc; tz = RMS_INF; }
                            }
                        }
                        fx = gx; fy = gy; fz = gz;
                    } else {
                        // ---------------- permeable / variable D: the interaction loop written out (LABELS only) ----
                        bool saturated = false;
                        constexpr bool REJ = PERM == 2;
                        // equal-step-length random leap (R25): a cancelled attempt is followed by another in a new direction
#pragma unroll 1
                        for (uint32_t attempt = 0;; ++attempt) {
                        if (REJ && attempt) {
                            uint32_t e0, e1, e2, e3;
                            rms_philox(p.rk, id_lo, id_hi, j + 1u, RMS_STREAM_ERL | (attempt << 8), e0, e1, e2, e3);
                            rms_hop(e0, e1, s, rx, ry, rz);
                        }
                        float px = fx, py = fy, pz = fz;
                        bool dx = false, dy = false, dz = false;
                        int e = 0;
                        // rejection sampling (R21): what a cancelled step has to put back
                        const int wx_in = wx, wy_in = wy, wz_in = wz, dIx_in = dIx, dIy_in = dIy, dIz_in = dIz;
                        const uint32_t L_in = L, j_rate_in = j_rate;
                        const float s_in = s, rate_in = rate, relax_in = relax;
                        const unsigned n_perm_in = n_perm;
                        int ev[3] = {0, 0, 0}, n_ev = 0;                // face passages of this step: +-(axis + 1)
                        bool cancelled = false;
                        uint32_t v0 = 0, v1 = 0, v2 = 0, v3 = 0;
                        bool have_v = false;
                        uint32_t m0 = 0, m1 = 0, m2 = 0, m3 = 0;
                        bool have_m = false;
#pragma unroll 1
                        for (int it = 0; it < 3; ++it) {
                            const float gx = px + rx, gy = py + ry, gz = pz + rz;
                            const bool cx = !dx && rms_outside(gx), cy = !dy && rms_outside(gy), cz = !dz && rms_outside(gz);
                            if (!(cx | cy | cz)) break;
                            const float tx = rms_hit_time(cx, px, rx), ty = rms_hit_time(cy, py, ry), tz = rms_hit_time(cz, pz, rz);
                            const float t = fminf(tx, fminf(ty, tz));
                            const bool isx = (tx == t);
                            const bool isy = !isx && (ty == t);
                            const float rk = isx ? rx : (isy ? ry : rz);
                            const bool neg = rk < 0.f;
                            px = fmaf(t, rx, px); py = fmaf(t, ry, py); pz = fmaf(t, rz, pz);
                            const float rest = 1.f - t;
                            rx *= rest; ry *= rest; rz *= rest;
                            const int wk = isx ? wx : (isy ? wy : wz);
                            const int nk = isx ? p.nx : (isy ? p.ny : p.nz);
                            const int stride = isx ? 1 : (isy ? p.nx : p.nx * p.ny);
                            int nwk = wk + (neg ? -1 : 1);
                            nwk = nwk < 0 ? nk - 1 : (nwk == nk ? 0 : nwk);
                            const int nlin = (wz * p.ny + wy) * p.nx + wx + (nwk - wk) * stride;
                            const uint32_t Ln = __ldg(p.labels + nlin);
                            bool pass = true;
                            if (Ln != L) {
                                ++n_enc;
                                if (REJ && p.PMT) {   // absorbing membrane (Eq.4, R20): the encounter saturates the walker with P_MT
                                    const float Q = __ldg(p.PMT + (size_t)L * p.n_labels + Ln);
                                    if (Q > 0.f) {
                                        if (!have_m) {
                                            rms_philox(p.rk, id_lo, id_hi, j + 1u, RMS_STREAM_MT, m0, m1, m2, m3);
                                            have_m = true;
                                        }
                                        if (rms_uni(e == 0 ? m0 : (e == 1 ? m1 : m2)) < Q) saturated = true;
                                    }
                                }
                                const float T = __ldg(p.P512 + (size_t)L * p.n_labels + Ln);   // 512 P
                                if (T >= 512.f) {
                                    pass = true;
                                } else if (T <= 0.f) {
                                    pass = false;
                                } else {
                                    // 33-bit uniform u_e = (c_e + uni(v_e))/512: 9 coarse bits from the spare bits of the
                                    // direction words decide almost always; the fine word is drawn only in between (R5)
                                    if (e >= 2 && !have_v) {
                                        rms_philox(p.rk, id_lo, id_hi, j + 1u, RMS_STREAM_PERM, v0, v1, v2, v3);
                                        have_v = true;
                                    }
                                    const float cf = (float)((e == 0 ? wa : (e == 1 ? wb : v3)) & 511u);
                                    if (cf + 1.f <= T) {
                                        pass = true;
                                    } else if (cf >= T) {
                                        pass = false;
                                    } else {
                                        if (!have_v) {
                                            rms_philox(p.rk, id_lo, id_hi, j + 1u, RMS_STREAM_PERM, v0, v1, v2, v3);
                                            have_v = true;
                                        }
                                        pass = rms_uni(e == 0 ? v0 : (e == 1 ? v1 : v2)) < (T - cf);
                                    }
                                }
                                ++e;
                                n_perm += pass;
                            }
                            const float plane = neg ? 0.f : 1.f;
                            float pk;
                            if (pass) {
                                pk = 1.f - plane;                       // enters the neighbour on its opposite face
                                if (isx) wx = nwk; else if (isy) wy = nwk; else wz = nwk;
                                const int sg1 = neg ? -1 : 1;
                                if (isx) dIx += sg1; else if (isy) dIy += sg1; else dIz += sg1;
                                if (REJ) ev[n_ev++] = sg1 * (isx ? 1 : (isy ? 2 : 3));
                                if (NW > 0 && acc_rem) {
                                    if (WMODE == RMS_WMODE_CONST) {
#pragma unroll
                                        for (int m = 0; m < NW; ++m) {
                                            const int v = neg ? -wrem[m] : wrem[m];
                                            if (isx) A32[m][0] += v; else if (isy) A32[m][1] += v; else A32[m][2] += v;
                                        }
                                    } else {
#pragma unroll
                                        for (int m = 0; m < NW; ++m) {
                                            double v = p.wsuf[(size_t)m * p.wsuf_stride + (j - p.step0)] - p.wsuf_end[m];
                                            v = neg ? -v : v;
                                            if (isx) Ad[m][0] += v; else if (isy) Ad[m][1] += v; else Ad[m][2] += v;
                                        }
                                    }
                                }
                                if (Ln != L) {
                                    // rest of the hop at the new compartment's speed (R7); whole dt of this step is
                                    // attributed to the compartment at the end of the hop (R12)
                                    const float s_new = __ldg(p.s_tab + Ln);
                                    const float sc = __fdividef(s_new, s);
                                    rx *= sc; ry *= sc; rz *= sc;
                                    relax = fmaf(rate, (float)(j - j_rate), relax);
                                    j_rate = j;
                                    rate = __ldg(p.rate + Ln);
                                    s = s_new;
                                    L = Ln;
                                }
                            } else if (REJ && p.rejection) {
                                cancelled = true;                       // rejection sampling: the walker does not move for the step
                                break;
                            } else {
                                pk = plane;
                                if (isx) rx = -rx; else if (isy) ry = -ry; else rz = -rz;   // elastic collision
                            }
                            if (isx) { px = pk; dx = true; } else if (isy) { py = pk; dy = true; } else { pz = pk; dz = true; }
                        }
                        if (REJ && cancelled) {
                            // undo the face passages of the cancelled step (voxel, displacement, event-driven phase part, label)
                            for (int q = 0; q < n_ev; ++q) {
                                const int ax = (ev[q] < 0 ? -ev[q] : ev[q]) - 1;
                                const bool ng = ev[q] < 0;
                                if (NW > 0 && acc_rem) {
                                    if (WMODE == RMS_WMODE_CONST) {
#pragma unroll
                                        for (int m = 0; m < NW; ++m) {
                                            const int v = ng ? -wrem[m] : wrem[m];
                                            if (ax == 0) A32[m][0] -= v; else if (ax == 1) A32[m][1] -= v; else A32[m][2] -= v;
                                        }
                                    } else {
#pragma unroll
                                        for (int m = 0; m < NW; ++m) {
                                            double v = p.wsuf[(size_t)m * p.wsuf_stride + (j - p.step0)] - p.wsuf_end[m];
                                            v = ng ? -v : v;
                                            if (ax == 0) Ad[m][0] -= v; else if (ax == 1) Ad[m][1] -= v; else Ad[m][2] -= v;
                                        }
                                    }
                                }
                            }
                            wx = wx_in; wy = wy_in; wz = wz_in; dIx = dIx_in; dIy = dIy_in; dIz = dIz_in;
                            L = L_in; s = s_in; rate = rate_in; relax = relax_in; j_rate = j_rate_in; n_perm = n_perm_in;
                            px = fx; py = fy; pz = fz; rx = 0.f; ry = 0.f; rz = 0.f;
                        }
                        if (REJ && cancelled && p.rejection == 2 && attempt + 1u < RMS_MAX_ERL_ATTEMPTS) continue;
                        const float gx = px + rx, gy = py + ry, gz = pz + rz;
                        fx = fminf(fmaxf(gx, 0.f), RMS_ONE_MINUS);
                        fy = fminf(fmaxf(gy, 0.f), RMS_ONE_MINUS);
                        fz = fminf(fmaxf(gz, 0.f), RMS_ONE_MINUS);
                        n_clamp += (fx != gx) + (fy != gy) + (fz != gz);
                        break;
                        }
                        if (REJ && saturated && relax != RMS_INF) {   // alpha_rho = 0 from here on (Eq.4); the walk goes on
                            relax = RMS_INF;
                            ++n_sat;
                        }
                    }

                    // ---------------- phase: fractional part, Phi_F += w f (the integer part is event driven) ----
                    if (NW > 0 && acc_w) {
#pragma unroll
                        for (int m = 0; m < NW; ++m) {
                            phiF[m][0] = fmaf(wf[m], fx, phiF[m][0]);
                            phiF[m][1] = fmaf(wf[m], fy, phiF[m][1]);
                            phiF[m][2] = fmaf(wf[m], fz, phiF[m][2]);
                        }
                    }
                    if (WMODE == RMS_WMODE_CONST && NW > 0) {
#pragma unroll
                        for (int m = 0; m < NW; ++m) wrem[m] -= wi[m];
                    }
                }
            }
            // flush the chunk's partial sums into the fp64 accumulators
            if (NW > 0 && (acc_w || acc_rem)) {
#pragma unroll
                for (int m = 0; m < NW; ++m)
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        const double add = (double)phiF[m][k] + (WMODE == RMS_WMODE_CONST ? (double)A32[m][k] : Ad[m][k]);
                        p.st.phi[(size_t)(3 * m + k) * n + i] += add;
                        phiF[m][k] = 0.f; A32[m][k] = 0; Ad[m][k] = 0.0;
                    }
            }
        }
    }

    // ---- store state --------------------------------------------------------------------------
    if (LAT == RMS_LAT_FACES) {
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
    relax = fmaf(rate, (float)(j_launch_end - j_rate), relax);
    p.st.w[0][i] = wx; p.st.w[1][i] = wy; p.st.w[2][i] = wz;
    p.st.dI[0][i] = dIx; p.st.dI[1][i] = dIy; p.st.dI[2][i] = dIz;
    p.st.f[0][i] = fx; p.st.f[1][i] = fy; p.st.f[2][i] = fz;
    p.st.f_lo[0][i] = 0.f; p.st.f_lo[1][i] = 0.f; p.st.f_lo[2][i] = 0.f;
    p.st.lab[i] = (lab & 0xFFFF0000u) | L;
    p.st.relax[i] = relax;

    // diagnostics: warp-shuffle reduction, one atomic per warp (early-exited lanes are not in the mask)
    const unsigned mask = __activemask();
    n_enc = __reduce_add_sync(mask, n_enc);
    n_perm = __reduce_add_sync(mask, n_perm);
    n_clamp = __reduce_add_sync(mask, n_clamp);
    n_sat = __reduce_add_sync(mask, n_sat);
    if ((threadIdx.x & 31) == (unsigned)(__ffs(mask) - 1)) {
        if (n_enc) atomicAdd(&p.counters[0], (unsigned long long)n_enc);
        if (n_perm) atomicAdd(&p.counters[1], (unsigned long long)n_perm);
        if (n_clamp) atomicAdd(&p.counters[2], (unsigned long long)n_clamp);
        if (n_sat) atomicAdd(&p.counters[4], (unsigned long long)n_sat);
    }
}

template <int NW, int WMODE>
static int launch_nw(const rms_step_params& p, int lat, bool permeable, cudaStream_t stream)
{
    const unsigned grid = (unsigned)((p.n + RMS_BLOCK - 1) / RMS_BLOCK);
    if (permeable && (p.rejection || p.PMT))
        rms_step_kernel<NW, WMODE, RMS_LAT_LABELS, 2><<<grid, RMS_BLOCK, 0, stream>>>(p);
    else if (permeable)
        rms_step_kernel<NW, WMODE, RMS_LAT_LABELS, 1><<<grid, RMS_BLOCK, 0, stream>>>(p);
    else if (lat == RMS_LAT_FACES)
        rms_step_kernel<NW, WMODE, RMS_LAT_FACES, 0><<<grid, RMS_BLOCK, 0, stream>>>(p);
    else
        rms_step_kernel<NW, WMODE, RMS_LAT_LABELS, 0><<<grid, RMS_BLOCK, 0, stream>>>(p);
    RMS_CUDA_TRY(cudaGetLastError());
    return RMS_OK;
}

template <int WMODE>
static int launch_wm(const rms_step_params& p, int n_wave, int lat, bool permeable, cudaStream_t stream)
{
    switch (n_wave) {
        case 0: return launch_nw<0, WMODE>(p, lat, permeable, stream);
        case 1: return launch_nw<1, WMODE>(p, lat, permeable, stream);
        case 2: return launch_nw<2, WMODE>(p, lat, permeable, stream);
        case 3: return launch_nw<3, WMODE>(p, lat, permeable, stream);
        case 4: return launch_nw<4, WMODE>(p, lat, permeable, stream);
        case 8: return launch_nw<8, WMODE>(p, lat, permeable, stream);
        case 16: return launch_nw<16, WMODE>(p, lat, permeable, stream);
    }
    rms_set_error("n_wave = %d is above RMS_MAX_WAVES = %d", n_wave, RMS_MAX_WAVES);
    return RMS_ERR_UNSUPPORTED;
}

int rms_launch_step(const rms_step_params& p, int n_wave, int wmode, int lat, bool permeable, cudaStream_t stream)
{
    if (p.n == 0 || p.n_steps == 0) return RMS_OK;
    return wmode == RMS_WMODE_CONST ? launch_wm<RMS_WMODE_CONST>(p, n_wave, lat, permeable, stream)
                                    : launch_wm<RMS_WMODE_TABLE>(p, n_wave, lat, permeable, stream);
}
