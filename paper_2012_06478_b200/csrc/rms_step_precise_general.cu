// rms_step_precise_general.cu -- RMS_RUN_FP64 for everything the specialised fp64 kernel does not serve: permeable
// membranes (Eq.3), compartments of different D (hop rescaled on entry, R7), per-compartment T2, arbitrary gradient
// waveforms.  The interaction loop of P:152-159 written out in fp64, one thread per walker, the neighbour's uint16
// label gathered at every face (the paper's lookup table).  Written for agreement with an fp64 reference over
// 1e4 .. 1e6 steps (rms_step_precise.cu says why fp32 cannot give that), not for speed.
#include "rms_internal.cuh"

#define RMS_GBLOCK 128

namespace {
__device__ __forceinline__ bool rms_outside_g(double g) { return (uint32_t)__double2hiint(g) >= 0x3FF00000u; }   // g >= 1 or g < 0
}

// REJ: the absorbing membranes (Eq.4) and the bookkeeping of a cancelled step (rejection sampling, ERL) compiled in
template <int NW, bool REJ>
__global__ void __launch_bounds__(RMS_GBLOCK) rms_step_precise_general_kernel(const __grid_constant__ rms_step_params p)
{
    const uint64_t t_global = (uint64_t)blockIdx.x * RMS_GBLOCK + threadIdx.x;
    if (t_global >= p.n) return;
    const uint64_t i = p.order ? (uint64_t)p.order[t_global] : t_global;
    const uint64_t id = p.first_id + i;
    const uint32_t id_lo = (uint32_t)id, id_hi = (uint32_t)(id >> 32);
    const size_t n = (size_t)p.n;

    int wx = p.st.w[0][i], wy = p.st.w[1][i], wz = p.st.w[2][i];
    int dIx = p.st.dI[0][i], dIy = p.st.dI[1][i], dIz = p.st.dI[2][i];
    double fx = (double)p.st.f[0][i] + (double)p.st.f_lo[0][i];
    double fy = (double)p.st.f[1][i] + (double)p.st.f_lo[1][i];
    double fz = (double)p.st.f[2][i] + (double)p.st.f_lo[2][i];
    const uint32_t lab = p.st.lab[i];
    uint32_t L = lab & 0xFFFFu;
    double s = (double)p.s_tab[L];
    double rate = (double)p.rate[L];
    double relax = 0.0;                      // added to the stored fp32 exponent at the end
    bool dead = isinf(p.st.relax[i]);        // saturated in an earlier launch (Eq.4)

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
    constexpr int NWA = NW > 0 ? NW : 1;
    double phiD[NWA][3], Ad[NWA][3];
#pragma unroll
    for (int m = 0; m < NWA; ++m)
#pragma unroll
        for (int k = 0; k < 3; ++k) { phiD[m][k] = 0.0; Ad[m][k] = 0.0; }
    unsigned n_enc = 0, n_perm = 0, n_clamp = 0, n_sat = 0;
    const double PI = 3.14159265358979323846;

#pragma unroll 1
    for (uint32_t t = 0; t < p.n_steps; ++t) {
        const uint32_t j = p.step0 + t;                      // steps done before this one
        uint32_t r0, r1, r2, r3;
        rms_philox(p.rk, id_lo, id_hi, j >> 1, RMS_STREAM_DIR, r0, r1, r2, r3);
        uint32_t wa = (j & 1u) ? r2 : r0, wb = (j & 1u) ? r3 : r1;
        double w_now[NWA];
#pragma unroll
        for (int m = 0; m < NW; ++m) w_now[m] = (double)__ldg(p.wave + (size_t)m * p.wave_stride + t);
        const double one_minus = 0.99999999999999988898;
        bool sat_step = false;
        // equal-step-length random leap (R25): a cancelled attempt is followed by another in a new direction
#pragma unroll 1
        for (uint32_t attempt = 0;; ++attempt) {
        // direction (R4): z = sym(wa), azimuth pi sym(wb)
        const double z = (double)rms_sym(wa);
        double sn, cs;
        sincos(PI * (double)rms_sym(wb), &sn, &cs);
        const double rho = sqrt(1.0 - z * z);
        double rx = s * (rho * cs), ry = s * (rho * sn), rz = s * z;

        double px = fx, py = fy, pz = fz;
        bool dx = false, dy = false, dz = false;
        int e = 0;
        uint32_t v0 = 0, v1 = 0, v2 = 0, v3 = 0;
        bool have_v = false;
        uint32_t m0 = 0, m1 = 0, m2 = 0, m3 = 0;
        bool have_m = false, saturated = false;
        // rejection sampling (R21): what a cancelled step has to put back
        const int wx_in = wx, wy_in = wy, wz_in = wz, dIx_in = dIx, dIy_in = dIy, dIz_in = dIz;
        const uint32_t L_in = L;
        const double s_in = s, rate_in = rate;
        const unsigned n_perm_in = n_perm;
        int ev[3] = {0, 0, 0}, n_ev = 0;
        bool cancelled = false;
#pragma unroll 1
        for (int it = 0; it < 3; ++it) {
            const double gx = px + rx, gy = py + ry, gz = pz + rz;
            const bool cx = !dx && rms_outside_g(gx), cy = !dy && rms_outside_g(gy), cz = !dz && rms_outside_g(gz);
            if (!(cx | cy | cz)) break;
            const double INF = __longlong_as_double(0x7ff0000000000000ll);
            const double tx = cx ? ((rx > 0.0 ? 1.0 : 0.0) - px) / rx : INF;
            const double ty = cy ? ((ry > 0.0 ? 1.0 : 0.0) - py) / ry : INF;
            const double tz = cz ? ((rz > 0.0 ? 1.0 : 0.0) - pz) / rz : INF;
            const double tm = fmin(tx, fmin(ty, tz));
            const bool isx = (tx == tm), isy = !isx && (ty == tm);          // ties: lowest axis first (R10)
            const double rk = isx ? rx : (isy ? ry : rz);
            const bool neg = rk < 0.0;
            px = fma(tm, rx, px); py = fma(tm, ry, py); pz = fma(tm, rz, pz);
            const double rest = 1.0 - tm;
            rx *= rest; ry *= rest; rz *= rest;
            const int wk = isx ? wx : (isy ? wy : wz);
            const int nk = isx ? p.nx : (isy ? p.ny : p.nz);
            const int stride = isx ? 1 : (isy ? p.nx : p.nx * p.ny);
            int nwk = wk + (neg ? -1 : 1);
            nwk = nwk < 0 ? nk - 1 : (nwk == nk ? 0 : nwk);
            const uint32_t Ln = __ldg(p.labels + ((wz * p.ny + wy) * p.nx + wx + (nwk - wk) * stride));
            bool pass = true;
            if (Ln != L) {                                                     // a membrane
                ++n_enc;
                if (REJ && p.PMT) {   // absorbing membrane (Eq.4, R20): the encounter saturates the walker with probability P_MT
                    const float Q = __ldg(p.PMT + (size_t)L * p.n_labels + Ln);
                    if (Q > 0.f) {
                        if (!have_m) { rms_philox(p.rk, id_lo, id_hi, j + 1u, RMS_STREAM_MT, m0, m1, m2, m3); have_m = true; }
                        if (rms_uni(e == 0 ? m0 : (e == 1 ? m1 : m2)) < Q) saturated = true;
                    }
                }
                const float T = __ldg(p.P512 + (size_t)L * p.n_labels + Ln);   // 512 P(L -> Ln), Eq.3
                if (T >= 512.f) pass = true;
                else if (T <= 0.f) pass = false;
                else {
                    // R5: u_e = (c_e + uni(v_e)) / 512, c_e = spare low bits of the direction words / of v_3
                    if (!have_v) {
                        rms_philox(p.rk, id_lo, id_hi, j + 1u, RMS_STREAM_PERM, v0, v1, v2, v3);
                        have_v = true;
                    }
                    const double c = (double)((e == 0 ? wa : (e == 1 ? wb : v3)) & 511u);
                    pass = c + (double)rms_uni(e == 0 ? v0 : (e == 1 ? v1 : v2)) < (double)T;
                }
                ++e;
                n_perm += pass;
            }
            const double plane = neg ? 0.0 : 1.0;
            double pk;
            if (pass) {
                pk = 1.0 - plane;
                if (isx) wx = nwk; else if (isy) wy = nwk; else wz = nwk;
                const int sg1 = neg ? -1 : 1;
                if (isx) dIx += sg1; else if (isy) dIy += sg1; else dIz += sg1;
                if (REJ) ev[n_ev++] = sg1 * (isx ? 1 : (isy ? 2 : 3));
#pragma unroll
                for (int m = 0; m < NW; ++m) {
                    double v = p.wsuf[(size_t)m * p.wsuf_stride + t] - p.wsuf_end[m];
                    v = neg ? -v : v;
                    if (isx) Ad[m][0] += v; else if (isy) Ad[m][1] += v; else Ad[m][2] += v;
                }
                if (Ln != L) {           // rest of the hop at the new compartment's speed (R7)
                    const double s_new = (double)__ldg(p.s_tab + Ln);
                    const double sc = s_new / s;
                    rx *= sc; ry *= sc; rz *= sc;
                    s = s_new;
                    rate = (double)__ldg(p.rate + Ln);
                    L = Ln;
                }
            } else if (REJ && p.rejection) {
                cancelled = true;                                              // rejection sampling: the walker does not move for the step
                break;
            } else {
                pk = plane;
                if (isx) rx = -rx; else if (isy) ry = -ry; else rz = -rz;      // elastic collision
            }
            if (isx) { px = pk; dx = true; } else if (isy) { py = pk; dy = true; } else { pz = pk; dz = true; }
        }
        if (REJ && cancelled) {
            for (int q = 0; q < n_ev; ++q) {
                const int ax = (ev[q] < 0 ? -ev[q] : ev[q]) - 1;
#pragma unroll
                for (int m = 0; m < NW; ++m) {
                    double v = p.wsuf[(size_t)m * p.wsuf_stride + t] - p.wsuf_end[m];
                    v = ev[q] < 0 ? -v : v;
                    if (ax == 0) Ad[m][0] -= v; else if (ax == 1) Ad[m][1] -= v; else Ad[m][2] -= v;
                }
            }
            wx = wx_in; wy = wy_in; wz = wz_in; dIx = dIx_in; dIy = dIy_in; dIz = dIz_in;
            L = L_in; s = s_in; rate = rate_in; n_perm = n_perm_in;
            px = fx; py = fy; pz = fz; rx = 0.0; ry = 0.0; rz = 0.0;
        }
        if (!(REJ && cancelled && p.rejection == 2 && attempt + 1u < RMS_MAX_ERL_ATTEMPTS)) {
            const double gx = px + rx, gy = py + ry, gz = pz + rz;
            fx = fmin(fmax(gx, 0.0), one_minus); fy = fmin(fmax(gy, 0.0), one_minus); fz = fmin(fmax(gz, 0.0), one_minus);
            n_clamp += (fx != gx) + (fy != gy) + (fz != gz);
            if (saturated) sat_step = true;
            break;
        }
        {
            uint32_t e0, e1, e2, e3;
            rms_philox(p.rk, id_lo, id_hi, j + 1u, RMS_STREAM_ERL | ((attempt + 1u) << 8), e0, e1, e2, e3);
            wa = e0; wb = e1;
        }
        }
        relax += rate;                                                        // whole dt to the label at the end of the hop (R12)
        if (REJ && sat_step && !dead) {                                              // alpha_rho = 0 from here on (Eq.4); the walk goes on
            relax = __longlong_as_double(0x7ff0000000000000ll);
            dead = true;
            ++n_sat;
        }
#pragma unroll
        for (int m = 0; m < NW; ++m) {
            phiD[m][0] = fma(w_now[m], fx, phiD[m][0]);
            phiD[m][1] = fma(w_now[m], fy, phiD[m][1]);
            phiD[m][2] = fma(w_now[m], fz, phiD[m][2]);
        }
    }
#pragma unroll
    for (int m = 0; m < NW; ++m)
#pragma unroll
        for (int k = 0; k < 3; ++k) p.st.phi[(size_t)(3 * m + k) * n + i] += phiD[m][k] + Ad[m][k];

    p.st.w[0][i] = wx; p.st.w[1][i] = wy; p.st.w[2][i] = wz;
    p.st.dI[0][i] = dIx; p.st.dI[1][i] = dIy; p.st.dI[2][i] = dIz;
    {
        const float hx = fminf((float)fx, 0.99999994f), hy = fminf((float)fy, 0.99999994f), hz = fminf((float)fz, 0.99999994f);
        p.st.f[0][i] = hx; p.st.f[1][i] = hy; p.st.f[2][i] = hz;
        p.st.f_lo[0][i] = (float)(fx - (double)hx); p.st.f_lo[1][i] = (float)(fy - (double)hy); p.st.f_lo[2][i] = (float)(fz - (double)hz);
    }
    p.st.lab[i] = (lab & 0xFFFF0000u) | L;
    p.st.relax[i] = (float)((double)p.st.relax[i] + relax);

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

int rms_launch_step_precise_general(const rms_step_params& p, int n_wave, cudaStream_t stream)
{
    if (p.n == 0 || p.n_steps == 0) return RMS_OK;
    const unsigned grid = (unsigned)((p.n + RMS_GBLOCK - 1) / RMS_GBLOCK);
    switch (n_wave) {
        case 0: if (p.rejection || p.PMT) rms_step_precise_general_kernel<0, true><<<grid, RMS_GBLOCK, 0, stream>>>(p); else rms_step_precise_general_kernel<0, false><<<grid, RMS_GBLOCK, 0, stream>>>(p); break;
        case 1: if (p.rejection || p.PMT) rms_step_precise_general_kernel<1, true><<<grid, RMS_GBLOCK, 0, stream>>>(p); else rms_step_precise_general_kernel<1, false><<<grid, RMS_GBLOCK, 0, stream>>>(p); break;
        case 2: if (p.rejection || p.PMT) rms_step_precise_general_kernel<2, true><<<grid, RMS_GBLOCK, 0, stream>>>(p); else rms_step_precise_general_kernel<2, false><<<grid, RMS_GBLOCK, 0, stream>>>(p); break;
        case 3: if (p.rejection || p.PMT) rms_step_precise_general_kernel<3, true><<<grid, RMS_GBLOCK, 0, stream>>>(p); else rms_step_precise_general_kernel<3, false><<<grid, RMS_GBLOCK, 0, stream>>>(p); break;
        case 4: if (p.rejection || p.PMT) rms_step_precise_general_kernel<4, true><<<grid, RMS_GBLOCK, 0, stream>>>(p); else rms_step_precise_general_kernel<4, false><<<grid, RMS_GBLOCK, 0, stream>>>(p); break;
        case 8: if (p.rejection || p.PMT) rms_step_precise_general_kernel<8, true><<<grid, RMS_GBLOCK, 0, stream>>>(p); else rms_step_precise_general_kernel<8, false><<<grid, RMS_GBLOCK, 0, stream>>>(p); break;
        case 16: if (p.rejection || p.PMT) rms_step_precise_general_kernel<16, true><<<grid, RMS_GBLOCK, 0, stream>>>(p); else rms_step_precise_general_kernel<16, false><<<grid, RMS_GBLOCK, 0, stream>>>(p); break;
        default:
            rms_set_error("n_wave = %d is above RMS_MAX_WAVES = %d", n_wave, RMS_MAX_WAVES);
            return RMS_ERR_UNSUPPORTED;
    }
    RMS_CUDA_TRY(cudaGetLastError());
    return RMS_OK;
}
