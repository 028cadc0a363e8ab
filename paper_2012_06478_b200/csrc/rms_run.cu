// rms_run.cu -- rms_run: host orchestration of the step launches, the reductions and H8 (normalisation).
#include <math.h>
#include <string.h>

#include <algorithm>

#include "rms_internal.cuh"

namespace {

struct DeviceBuf {   // frees on scope exit; work on the block may still be queued on the stream (error returns)
    void* p = nullptr;
    cudaStream_t stream = nullptr;
    ~DeviceBuf() { if (p) rms_free_async(p, stream); }
    template <class T> T* as() { return (T*)p; }
};

// A failure after the first launch leaves the walkers advanced by part of the run while steps_done is not: a later run would
// reuse Philox step indices on moved walkers.  The guard waits for the queued work and marks the handle unusable.
struct RunGuard {
    rms_walkers* w;
    cudaStream_t stream;
    bool armed = false;
    ~RunGuard() { if (armed) { cudaStreamSynchronize(stream); w->poisoned = true; } }
};

struct Events {
    std::vector<cudaEvent_t> ev;
    ~Events() { for (auto e : ev) cudaEventDestroy(e); }
    cudaEvent_t make() { cudaEvent_t e = nullptr; if (cudaEventCreate(&e) != cudaSuccess) e = nullptr; else ev.push_back(e); return e; }
};

// Is every weight an integer small enough for the exact int32 path (piecewise-constant gradients such as PGSE)?
bool wave_is_integer(const float* wave, size_t count)
{
    for (size_t i = 0; i < count; ++i) {
        const float w = wave[i];
        if (!(fabsf(w) <= 32767.f) || w != rintf(w)) return false;
    }
    return true;
}

}  // namespace

// H8: Eq.7 S = <alpha e^{-i phi}> / <alpha>, and the narrow-pulse D, K of P:174 with both moments
// normalised by <alpha> (R14).  Classes are pooled.  Pure host arithmetic on the reduced sums.
// Permeable runs take the specialised kernel when ceil(512 P_max) is at most this.  Measured on the cfg3 lattice (1e6 walkers
// x 1e4 steps, general kernel 176 ms): 65 / 71 / 81 / 90 / 102 / 112 ms at 512 P_max = 0.2 / 23 / 73 / 130 / 213 / 292 -- the
// redo of a step that may permeate is cheaper than the general kernel at any P, so the bound is the largest possible.
#ifndef RMS_FAST_PERM_TCEIL
#define RMS_FAST_PERM_TCEIL 512u
#endif

extern "C" int rms_volume_weighted_signal(int n_classes, int n_q, const double* class_volume, const double* sum_alpha,
                                          const double* sig_re, const double* sig_im, double* S_re, double* S_im)
{
    RMS_REQUIRE(n_classes > 0 && n_q >= 0 && class_volume && sum_alpha, RMS_ERR_ARG, "rms_volume_weighted_signal: bad arguments");
    RMS_REQUIRE(n_q == 0 || (sig_re && sig_im), RMS_ERR_ARG, "rms_volume_weighted_signal: null signal sums");
    double vol = 0.0;
    for (int c = 0; c < n_classes; ++c)
        if (sum_alpha[c] > 0.0) vol += class_volume[c];
    RMS_REQUIRE(vol > 0.0, RMS_ERR_ARG, "rms_volume_weighted_signal: no class holds both walkers and volume");
    for (int q = 0; q < n_q; ++q) {
        double re = 0.0, im = 0.0;
        for (int c = 0; c < n_classes; ++c)
            if (sum_alpha[c] > 0.0) {
                re += class_volume[c] * sig_re[(size_t)q * n_classes + c] / sum_alpha[c];
                im += class_volume[c] * sig_im[(size_t)q * n_classes + c] / sum_alpha[c];
            }
        if (S_re) S_re[q] = re / vol;
        if (S_im) S_im[q] = im / vol;
    }
    return RMS_OK;
}

extern "C" int rms_normalise(int n_classes, int n_q, const double* sum_alpha, const double* sig_re, const double* sig_im,
                             int n_snap, int n_dir, const double* snap_alpha, const double* m2, const double* m4,
                             const double* t_ms, double* S_re, double* S_im, double* Dapp, double* Kapp)
{
    RMS_REQUIRE(n_classes > 0 && n_q >= 0 && n_snap >= 0 && n_dir >= 0, RMS_ERR_ARG, "rms_normalise: bad counts");
    RMS_REQUIRE(n_q == 0 || (sum_alpha && sig_re && sig_im), RMS_ERR_ARG, "rms_normalise: null signal sums");
    RMS_REQUIRE(n_snap * n_dir == 0 || (snap_alpha && m2 && m4 && t_ms), RMS_ERR_ARG, "rms_normalise: null moment sums");
    const int nC = n_classes;
    double tot_alpha = 0.0;
    for (int c = 0; c < nC && sum_alpha; ++c) tot_alpha += sum_alpha[c];
    for (int q = 0; q < n_q; ++q) {
        double re = 0, im = 0;
        for (int c = 0; c < nC; ++c) { re += sig_re[(size_t)q * nC + c]; im += sig_im[(size_t)q * nC + c]; }
        if (S_re) S_re[q] = re / tot_alpha;
        if (S_im) S_im[q] = im / tot_alpha;
    }
    for (int s = 0; s < n_snap; ++s) {
        double al = 0;
        for (int c = 0; c < nC; ++c) al += snap_alpha[(size_t)s * nC + c];
        for (int k = 0; k < n_dir; ++k) {
            double a2 = 0, a4 = 0;
            for (int c = 0; c < nC; ++c) {
                a2 += m2[((size_t)s * n_dir + k) * nC + c];
                a4 += m4[((size_t)s * n_dir + k) * nC + c];
            }
            a2 /= al; a4 /= al;
            if (Dapp) Dapp[(size_t)s * n_dir + k] = a2 / (2.0 * t_ms[s]);
            if (Kapp) Kapp[(size_t)s * n_dir + k] = a4 / (a2 * a2) - 3.0;
        }
    }
    return RMS_OK;
}

extern "C" int rms_run(const rms_substrate* s, rms_walkers* w, const rms_run_desc* d, void* cuda_stream, rms_result* out)
{
    RMS_REQUIRE(s && w && d && out, RMS_ERR_ARG, "rms_run: null argument");
    RMS_REQUIRE(w->sub == s, RMS_ERR_ARG, "rms_run: walkers were initialised on another substrate");
    RMS_REQUIRE(!w->poisoned, RMS_ERR_ARG, "rms_run: an earlier run on these walkers failed part-way; initialise them again");
    RMS_REQUIRE(d->n_steps >= 0, RMS_ERR_ARG, "n_steps is negative");
    RMS_REQUIRE(d->n_wave >= 0 && d->n_g >= 0 && d->n_dir >= 0 && d->n_snap >= 0, RMS_ERR_ARG, "negative count in rms_run_desc");
    RMS_REQUIRE(d->n_wave <= RMS_MAX_WAVES, RMS_ERR_UNSUPPORTED, "n_wave = %d is above RMS_MAX_WAVES = %d", d->n_wave,
                RMS_MAX_WAVES);
    RMS_REQUIRE(d->n_wave == 0 || (d->wave && (d->n_g == 0 || d->gamp)), RMS_ERR_ARG, "wave / gamp is null");
    RMS_REQUIRE(d->n_dir == 0 || d->dirs, RMS_ERR_ARG, "dirs is null");
    RMS_REQUIRE(d->n_snap == 0 || d->snap_steps, RMS_ERR_ARG, "snap_steps is null");
    RMS_REQUIRE(w->steps_done + (uint64_t)d->n_steps < 0xFFFFFFF0ull, RMS_ERR_UNSUPPORTED, "more than 2^32 steps per walker");
    for (int i = 0; i < d->n_dir; ++i) {
        const double* n = d->dirs + 3 * i;
        RMS_REQUIRE(fabs(n[0] * n[0] + n[1] * n[1] + n[2] * n[2] - 1.0) <= 1e-6, RMS_ERR_ARG, "dirs[%d] is not a unit vector", i);
    }
    for (int i = 0; i < d->n_snap; ++i) {
        RMS_REQUIRE(d->snap_steps[i] >= 1 && d->snap_steps[i] <= d->n_steps, RMS_ERR_ARG, "snap_steps[%d] outside 1..n_steps", i);
        RMS_REQUIRE(i == 0 || d->snap_steps[i] > d->snap_steps[i - 1], RMS_ERR_ARG, "snap_steps must be strictly ascending");
    }
    for (size_t i = 0; i < (size_t)d->n_wave * d->n_steps; ++i)
        RMS_REQUIRE(isfinite(d->wave[i]), RMS_ERR_ARG, "wave[%zu] is not finite", i);

    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const int nL = s->n_labels, nC = s->n_classes, nW = d->n_wave, nG = d->n_g, nD = d->n_dir, nS = d->n_snap;
    const int64_t nT = d->n_steps;
    const uint64_t n = w->n;

    // ---- H0 (run-time part): tables from (D, kappa, T2, dt) ---------------------------------------
    std::vector<float> s_tab, P_tab;
    const bool erl = (d->flags & RMS_RUN_ERL) != 0;                  // P:80, Appendix A (R25)
    const bool rs = (d->flags & RMS_RUN_REJECTION_SAMPLING) != 0 || erl;   // P:84, Appendix B (R21); both cancel steps
    RMS_REQUIRE(!(erl && (d->flags & RMS_RUN_REJECTION_SAMPLING)), RMS_ERR_ARG, "RMS_RUN_ERL and RMS_RUN_REJECTION_SAMPLING exclude each other");
    RMS_REQUIRE(!(erl && !s->rho.empty()), RMS_ERR_UNSUPPORTED, "equal-step-length random leap with absorbing membranes (P:80 rules it out)");
    int rc = rms_compute_tables(s, d->dt_ms, s_tab, P_tab, rs && !erl);
    if (rc != RMS_OK) return rc;
    if (erl)    // a face is a wall or no membrane: the paper rules ERL out for exchange
        for (size_t t = 0; t < P_tab.size(); ++t)
            RMS_REQUIRE(!(P_tab[t] > 0.f && P_tab[t] < 1.f), RMS_ERR_UNSUPPORTED,
                        "equal-step-length random leap with a permeable membrane (labels %d, %d)", (int)(t / nL), (int)(t % nL));
    const bool mt = !s->rho.empty();             // absorbing membranes (Eq.4)
    // stimulated echo (R22): the steps of the mixing time relax with T1; its edges become launch boundaries
    const int64_t mix0 = d->mix_first_step, mixN = d->mix_n_steps;
    RMS_REQUIRE(mixN >= 0 && (mixN == 0 || (mix0 >= 1 && mix0 + mixN - 1 <= nT)), RMS_ERR_ARG,
                "mixing time (steps %lld .. %lld) must lie inside 1 .. n_steps", (long long)mix0, (long long)(mix0 + mixN - 1));
    std::vector<float> tabs((size_t)nL * 3 + (size_t)nL * nL * (mt ? 2 : 1));
    float* h_s = tabs.data();
    float* h_rate = h_s + nL;
    float* h_P512 = h_rate + nL;
    float* h_PMT = h_P512 + (size_t)nL * nL;
    float* h_rate1 = h_PMT + (mt ? (size_t)nL * nL : 0);       // dt / T1
    if (mt)       // P_MT(a->b) = rho_ab ds_a / D_a C_d, C_3 = 2/3 (R20), fp64 then rounded once to fp32 (R6)
        for (int a = 0; a < nL; ++a)
            for (int b = 0; b < nL; ++b) {
                const double q = a == b ? 0.0 : (double)s->rho[(size_t)a * nL + b] * sqrt(6.0 * d->dt_ms / (double)s->D[a]) * (2.0 / 3.0);
                RMS_REQUIRE(q <= 1.0, RMS_ERR_P_RANGE, "P_MT = %.4g > 1 from label %d towards %d: lower rho or dt", q, a, b);
                h_PMT[(size_t)a * nL + b] = (float)q;
            }
    bool permeable = false;
    for (int a = 0; a < nL; ++a) {
        h_s[a] = s_tab[a];
        const float t2 = s->T2[a];
        h_rate[a] = (t2 > 0 && isfinite(t2)) ? (float)(d->dt_ms / (double)t2) : 0.f;
        const float t1 = s->T1.empty() ? 0.f : s->T1[a];
        h_rate1[a] = (t1 > 0 && isfinite(t1)) ? (float)(d->dt_ms / (double)t1) : 0.f;
        for (int b = 0; b < nL; ++b) {
            h_P512[(size_t)a * nL + b] = 512.f * P_tab[(size_t)a * nL + b];
            if (a != b && P_tab[(size_t)a * nL + b] > 0.f) permeable = true;
        }
    }
    const bool want_labels = (d->flags & RMS_RUN_LABEL_GATHER) != 0;
    if (mt || rs) permeable = true;              // absorbing membranes and cancelled steps take the kernels' permeable variants
    const int lat = (!permeable && s->want_bricks && !want_labels) ? RMS_LAT_FACES : RMS_LAT_LABELS;
    // permeable runs with P << 1 also take the specialised kernel: ceil(512 P_max) bounds the coarse random
    // bits that can permeate at all (rms_step_fast.cu)
    float t_max = 0.f;
    for (int a = 0; a < nL; ++a)
        for (int b = 0; b < nL; ++b)
            if (a != b) t_max = std::max(t_max, h_P512[(size_t)a * nL + b]);
    const uint32_t t_ceil_P = (uint32_t)ceilf(t_max);
    // absorbing membranes: the saturation draw belongs to every membrane met, so every such step is redone (t_ceil = 512)
    const uint32_t t_ceil = mt ? 512u : t_ceil_P;
    // (rejection sampling and ERL too: the specialised kernel cancels a step at its first uncrossed membrane and, for ERL, tries again)
    // RMS_RUN_FP64: the specialised kernel with fp64 directions and 2^-63 fixed-point offsets serves every run it serves in fp32
    // (piecewise-constant waveforms; impermeable, permeable), the general fp64 kernel (table-driven waveforms, label gathers)
    // everything else
    const bool fp64 = (d->flags & RMS_RUN_FP64) != 0;
    // Where every step that meets a membrane takes the specialised kernel's side path (absorbing membranes, faces with P = 1),
    // fp64 runs go to the general fp64 kernel: that path works on fp32 offsets, and the trajectories would be fp32 ones.
    const bool fast_permeable = permeable && (s->d_oct || s->d_code) && !want_labels && t_ceil <= RMS_FAST_PERM_TCEIL &&
                                !(erl && t_ceil_P > 0u) && !(fp64 && t_ceil >= 512u);

    const int nWk = rms_kernel_waves(nW);        // waveforms the step kernel is compiled for; the extra ones carry zero weight
    rc = rms_walkers_reserve_waves(w, nWk, stream);
    if (rc != RMS_OK) return rc;

    // ---- waveform analysis ---------------------------------------------------------------------------
    // suffix sums S[m][j] = sum_{i > j} w_m[i] (j = 0..nT, steps are 1-based), fp64
    std::vector<double> suf((size_t)std::max(nWk, 1) * (nT + 1), 0.0);
    for (int m = 0; m < nW; ++m) {
        double acc = 0.0;
        double* S = &suf[(size_t)m * (nT + 1)];
        for (int64_t j = nT; j >= 1; --j) { acc += (double)d->wave[(size_t)m * nT + (j - 1)]; S[j - 1] = acc; }
    }
    // integer-valued waveforms: the general kernel's exact int32 path (CONST mode)
    bool int_mode = wave_is_integer(d->wave, (size_t)nW * nT);
    for (size_t i = 0; int_mode && i < suf.size(); ++i) int_mode = fabs(suf[i]) < 1048576.0;   // int32 event sums: <= 64 steps x 2^20 between flushes
    // piecewise-constant waveforms (any amplitudes), segments of >= 32 steps on average: the specialised kernels
    bool const_mode = true;

    // launch boundaries: snapshots and the end of the call
    std::vector<int64_t> bounds;
    for (int i = 0; i < nS; ++i) bounds.push_back(d->snap_steps[i]);
    if (bounds.empty() || bounds.back() != nT) bounds.push_back(nT);
    {
        // the general kernels count box wraps in 10-bit fields per launch (+-511 per axis): on a lattice a few voxels wide a
        // long launch is split so that no walker can wrap more often than that (hop < 1 voxel per step)
        const int64_t max_launch = 511ll * std::min(s->nx, std::min(s->ny, s->nz));
        for (int64_t b = max_launch; b < nT; b += max_launch) bounds.push_back(b);
        std::sort(bounds.begin(), bounds.end());
        bounds.erase(std::unique(bounds.begin(), bounds.end()), bounds.end());
    }
    if (mixN > 0) {
        if (mix0 > 1) bounds.push_back(mix0 - 1);
        bounds.push_back(mix0 + mixN - 1);
        std::sort(bounds.begin(), bounds.end());
        bounds.erase(std::unique(bounds.begin(), bounds.end()), bounds.end());
    }

    std::vector<rms_segment> segs;
    std::vector<std::pair<size_t, size_t>> seg_range;   // per launch: [first, count)
    if (const_mode) {
        int64_t a = 0;
        for (int64_t b : bounds) {
            const size_t first = segs.size();
            int64_t j = a;
            while (j < b) {
                int64_t e = j + 1;
                auto same = [&](int64_t x, int64_t y) {
                    for (int m = 0; m < nW; ++m)
                        if (d->wave[(size_t)m * nT + x] != d->wave[(size_t)m * nT + y]) return false;
                    return true;
                };
                while (e < b && same(j, e)) ++e;
                rms_segment sg;
                memset(&sg, 0, sizeof sg);
                sg.n = (uint32_t)(e - j);
                for (int m = 0; m < nW; ++m) {
                    sg.wf[m] = d->wave[(size_t)m * nT + j];
                    if (int_mode) {
                        sg.w[m] = (int32_t)d->wave[(size_t)m * nT + j];
                        sg.wrem_end[m] = (int32_t)llrint(suf[(size_t)m * (nT + 1) + e] - suf[(size_t)m * (nT + 1) + b]);
                        if (sg.wrem_end[m] != 0) sg.flags |= 2u;
                    }
                    if (sg.wf[m] != 0.f) sg.flags |= 3u;
                }
                segs.push_back(sg);
                j = e;
            }
            seg_range.push_back({first, segs.size() - first});
            a = b;
        }
        if (segs.size() > (1u << 20) || (int64_t)segs.size() > nT / 32 + (int64_t)bounds.size() + 16) {
            const_mode = false; segs.clear(); seg_range.clear();
        }
    }
    // which step kernel: specialised (fp32 / fp64) needs piecewise-constant waveforms and the neighbourhood lattice; the general
    // fp32 kernel runs its CONST mode on integer-valued piecewise-constant waveforms, its TABLE mode otherwise; the general
    // fp64 kernel is table driven
    const bool nbr_fp32 = (!permeable && lat == RMS_LAT_FACES) || fast_permeable;
    // (RMS_RUN_FP64 on the specialised kernel: its direction arithmetic in fp64, rms_step_fast.cu)
    const bool use_fast = const_mode && nbr_fp32 && !(d->flags & RMS_RUN_GENERAL_KERNEL);
    const bool use_general = !use_fast;
    const int wmode = (use_general && !fp64 && const_mode && int_mode) ? RMS_WMODE_CONST : RMS_WMODE_TABLE;
    const bool need_segs = use_fast || wmode == RMS_WMODE_CONST;
    const bool need_table = use_general && wmode == RMS_WMODE_TABLE;
    // the 27-bit neighbourhood lattice serves the general fp32 kernel's face-bit mode only: built on demand
    if (use_general && !fp64 && lat == RMS_LAT_FACES) {
        rc = rms_substrate_ensure_nbr(s, stream);
        if (rc != RMS_OK) return rc;
    }

    // ---- device scratch: tables | segments or wave tables | q vectors | result sums -------------------
    const int nQs = nW * nG * nD;                                    // scalar waveforms x b x direction
    const int nTen = d->n_tensor, nR = d->n_rot;
    RMS_REQUIRE(nTen >= 0 && nR >= 0 && nTen <= 4096 && nR <= 4096, RMS_ERR_ARG, "n_tensor and n_rot must lie in 0 .. 4096");
    const int nQt = nTen * nG * nR;                                  // tensor waveforms x b x rotation (R23)
    if (nQt > 0) {
        RMS_REQUIRE(d->tensor_waves && d->tensor_gamp && d->rots, RMS_ERR_ARG, "tensor_waves, tensor_gamp and rots must be given");
        for (int t = 0; t < 3 * nTen; ++t)
            RMS_REQUIRE(d->tensor_waves[t] >= -1 && d->tensor_waves[t] < nW, RMS_ERR_ARG,
                        "tensor_waves[%d] = %d is no waveform of this run", t, d->tensor_waves[t]);
    }
    const int nQ = nQs + nQt;
    const int nTerms = nQt > 0 ? 3 : 1;
    const size_t n_sig = (size_t)nQ * nC, n_mom = (size_t)nS * nD * nC, n_sal = (size_t)nS * nC, n_flow = (size_t)nS * nC * nC;
    const size_t n_res_d = 2 * n_sig + 2 * n_mom + n_sal + nC;       // doubles
    RMS_REQUIRE(n_flow <= ((size_t)1 << 27) && n_res_d <= ((size_t)1 << 28), RMS_ERR_UNSUPPORTED,
                "n_classes = %d with %d snapshots, %d signals: the result arrays would exceed 1-2 GB", nC, nS, nQ);
    DeviceBuf b_tabs, b_segs, b_wave, b_wsuf, b_q, b_res, b_dirs, b_order, b_sched;
    for (DeviceBuf* b : {&b_tabs, &b_segs, &b_wave, &b_wsuf, &b_q, &b_res, &b_dirs, &b_order, &b_sched}) b->stream = stream;
    RMS_CUDA_TRY(rms_malloc((void**)&b_tabs.p, tabs.size() * sizeof(float)));
    RMS_CUDA_TRY(cudaMemcpyAsync(b_tabs.p, tabs.data(), tabs.size() * sizeof(float), cudaMemcpyHostToDevice, stream));
    if (need_segs) {
        if (!segs.empty()) {
            RMS_CUDA_TRY(rms_malloc((void**)&b_segs.p, segs.size() * sizeof(rms_segment)));
            RMS_CUDA_TRY(cudaMemcpyAsync(b_segs.p, segs.data(), segs.size() * sizeof(rms_segment), cudaMemcpyHostToDevice, stream));
        }
    }
    if (need_table && nW > 0 && nT > 0) {
        RMS_CUDA_TRY(rms_malloc((void**)&b_wave.p, (size_t)nWk * nT * sizeof(float)));
        if (nWk > nW) RMS_CUDA_TRY(cudaMemsetAsync(b_wave.p, 0, (size_t)nWk * nT * sizeof(float), stream));
        RMS_CUDA_TRY(cudaMemcpyAsync(b_wave.p, d->wave, (size_t)nW * nT * sizeof(float), cudaMemcpyHostToDevice, stream));
        RMS_CUDA_TRY(rms_malloc((void**)&b_wsuf.p, (size_t)nWk * (nT + 1) * sizeof(double)));
        RMS_CUDA_TRY(cudaMemcpyAsync(b_wsuf.p, suf.data(), (size_t)nWk * (nT + 1) * sizeof(double), cudaMemcpyHostToDevice, stream));
    }
    // phase per unit Phi, in turns: gamp dt l_p n / (2 pi)   (Eq.7 with the right-endpoint rule, R11)
    // with tensor waveforms every q carries three (vector, waveform) terms, the scalar ones leaving two of them off
    std::vector<double> qv((size_t)std::max(nQ, 1) * nTerms * 3, 0.0);
    std::vector<int> qwave((size_t)std::max(nQ, 1) * nTerms, nTerms == 1 ? 0 : -1);
    const double turn = d->dt_ms * s->voxel_um / (2.0 * 3.14159265358979323846);
    for (int m = 0; m < nW; ++m)
        for (int g = 0; g < nG; ++g)
            for (int k = 0; k < nD; ++k) {
                const size_t q = (((size_t)m * nG + g) * nD + k) * nTerms;
                const double c = d->gamp[(size_t)m * nG + g] * turn;
                for (int x = 0; x < 3; ++x) qv[3 * q + x] = c * d->dirs[3 * k + x];
                qwave[q] = m;
            }
    for (int t = 0; t < nTen; ++t)
        for (int g = 0; g < nG; ++g)
            for (int k = 0; k < nR; ++k) {
                const size_t q = ((size_t)nQs + ((size_t)t * nG + g) * nR + k) * 3;
                const double c = d->tensor_gamp[(size_t)t * nG + g] * turn;
                for (int ax = 0; ax < 3; ++ax) {                     // term ax: the vector R_k e_ax with the waveform on axis ax
                    for (int x = 0; x < 3; ++x) qv[3 * (q + ax) + x] = c * d->rots[9 * k + 3 * x + ax];
                    qwave[q + ax] = d->tensor_waves[3 * t + ax];
                }
            }
    RMS_CUDA_TRY(rms_malloc((void**)&b_q.p, qv.size() * sizeof(double) + qwave.size() * sizeof(int)));
    RMS_CUDA_TRY(cudaMemcpyAsync(b_q.p, qv.data(), qv.size() * sizeof(double), cudaMemcpyHostToDevice, stream));
    int* d_qwave = (int*)(b_q.as<double>() + qv.size());
    RMS_CUDA_TRY(cudaMemcpyAsync(d_qwave, qwave.data(), qwave.size() * sizeof(int), cudaMemcpyHostToDevice, stream));
    RMS_CUDA_TRY(rms_malloc((void**)&b_dirs.p, std::max(nD, 1) * 3 * sizeof(double)));
    if (nD) RMS_CUDA_TRY(cudaMemcpyAsync(b_dirs.p, d->dirs, (size_t)nD * 3 * sizeof(double), cudaMemcpyHostToDevice, stream));
    const size_t res_bytes = n_res_d * sizeof(double) + n_flow * sizeof(unsigned long long);
    RMS_CUDA_TRY(rms_malloc((void**)&b_res.p, res_bytes));
    RMS_CUDA_TRY(cudaMemsetAsync(b_res.p, 0, res_bytes, stream));
    double* d_re = b_res.as<double>();
    double* d_im = d_re + n_sig;
    double* d_m2 = d_im + n_sig;
    double* d_m4 = d_m2 + n_mom;
    double* d_sal = d_m4 + n_mom;
    double* d_sum_alpha = d_sal + n_sal;
    unsigned long long* d_flow = (unsigned long long*)(d_sum_alpha + nC);
    RMS_CUDA_TRY(cudaMemsetAsync(w->d_counters, 0, 64, stream));

    // ---- launches ------------------------------------------------------------------------------------
    Events evs;
    cudaEvent_t ev_begin = evs.make(), ev_end = evs.make();
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> step_ev;
    RMS_CUDA_TRY(cudaEventRecord(ev_begin, stream));
    unsigned n_launches = 0;

    RunGuard guard{w, stream};
    rms_step_params sp;
    memset(&sp, 0, sizeof sp);
    sp.nx = s->nx; sp.ny = s->ny; sp.nz = s->nz;
    sp.labels = s->d_labels; sp.nbr = s->d_nbr; sp.oct = s->d_oct;
    sp.code = s->d_code; sp.dict = s->d_dict; sp.esc = s->d_esc; sp.esc_mask = s->esc_mask;
    sp.k_hi7f = 0x7Fu; sp.k_tau_or = 0x3F800080u; sp.k_two = 2.0f; sp.k_sin3 = -2.4641574e-06f;
    if (use_fast) {
        rc = rms_fast_luts(&sp.lut1, &sp.lut2);
        if (rc != RMS_OK) return rc;
    }
    sp.NX = s->NX; sp.NY = s->NY; sp.SX = s->SX; sp.SY = s->SY; sp.SZ = s->SZ;
    sp.st = w->a; sp.n = n; sp.first_id = w->first_id; sp.rk = rms_make_keys(w->seed);
    sp.s_tab = b_tabs.as<float>(); sp.rate = sp.s_tab + nL; sp.P512 = sp.rate + nL; sp.n_labels = nL;
    sp.PMT = mt ? sp.P512 + (size_t)nL * nL : nullptr;
    const float* rate_T2 = sp.rate;
    const float* rate_T1 = sp.P512 + (size_t)nL * nL * (mt ? 2 : 1);
    sp.t_ceil = t_ceil;
    sp.rejection = erl ? 2 : (rs ? 1 : 0);
    sp.counters = w->d_counters; sp.n_wave = nW; sp.wave_stride = nT; sp.wsuf_stride = nT + 1;

    rms_reduce_params rp;
    memset(&rp, 0, sizeof rp);
    rp.st = w->a; rp.n = n; rp.label_class = s->d_label_class; rp.n_classes = nC; rp.n_dir = nD;
    rp.dirs = b_dirs.as<double>(); rp.voxel_um = s->voxel_um;

    // spatial ordering of the walkers over the threads pays once the lattice outgrows the caches
    const bool ordered = n >= 4096 && s->n_vox >= (1u << 22) && !(d->flags & RMS_RUN_NO_ORDERING);
    if (ordered) RMS_CUDA_TRY(rms_malloc((void**)&b_order.p, n * sizeof(uint32_t)));

    int64_t a = 0;
    int snap = 0;
    for (size_t li = 0; li < bounds.size(); ++li) {
        const int64_t b = bounds[li];
        if (b > a) {
            if (ordered) {
                rc = rms_order_walkers(s, w, b_order.as<uint32_t>(), stream, &n_launches);
                if (rc != RMS_OK) return rc;
                sp.order = b_order.as<uint32_t>();
            }
            const bool mixing = mixN > 0 && a + 1 >= mix0 && b <= mix0 + mixN - 1;
            sp.rate = mixing ? rate_T1 : rate_T2;
            sp.step0 = (uint32_t)(w->steps_done + (uint64_t)a);
            sp.n_steps = (uint32_t)(b - a);
            for (int m = 0; m < nW; ++m) {
                const double* S = &suf[(size_t)m * (nT + 1)];
                sp.wtot[m] = S[a] - S[b];
                sp.wsuf_end[m] = S[b];
            }
            if (need_segs) {
                sp.n_seg = (int)seg_range[li].second;
                sp.segs = b_segs.as<rms_segment>() + seg_range[li].first;
            }
            if (need_table) {
                sp.n_seg = 1;
                sp.wave = b_wave.as<float>() ? b_wave.as<float>() + a : nullptr;
                // wsuf element 0 must be the suffix sum that includes the first step of this launch: S[a]
                sp.wsuf = b_wsuf.as<double>() ? b_wsuf.as<double>() + a : nullptr;
            }
            cudaEvent_t e0 = evs.make(), e1 = evs.make();
            RMS_CUDA_TRY(cudaEventRecord(e0, stream));
            guard.armed = true;
            if (use_fast && !(d->flags & RMS_RUN_NO_SLICES)) {
                // time slices: fill the tail of a launch of many waves of blocks (rms_step_fast.cu)
                size_t words = 0;
                rms_fast_slices(&sp, &words);
                if (sp.n_slices > 1u) {
                    if (!b_sched.p) RMS_CUDA_TRY(rms_malloc((void**)&b_sched.p, words * sizeof(uint32_t)));   // the same size at every launch
                    RMS_CUDA_TRY(cudaMemsetAsync(b_sched.p, 0, words * sizeof(uint32_t), stream));
                    sp.sched = b_sched.as<uint32_t>();
                }
            }
            if (use_fast) rc = rms_launch_step_fast(sp, nW, permeable, fp64, stream);
            else if (fp64) rc = rms_launch_step_precise_general(sp, nWk, stream);
            else rc = rms_launch_step(sp, nWk, wmode, lat, permeable, stream);
            if (rc != RMS_OK) return rc;
            RMS_CUDA_TRY(cudaEventRecord(e1, stream));
            step_ev.push_back({e0, e1});
            ++n_launches;
        }
        while (snap < nS && d->snap_steps[snap] == b) {
            rc = rms_launch_moments(rp, d_m2 + (size_t)snap * nD * nC, d_m4 + (size_t)snap * nD * nC, d_sal + (size_t)snap * nC,
                                    d_flow + (size_t)snap * nC * nC, stream);
            if (rc != RMS_OK) return rc;
            ++n_launches;
            ++snap;
        }
        a = b;
    }
    if (nC > RMS_SIG_SMALL_CLASSES) {     // many classes (per-cell outputs): the signal reduction visits the walkers class by class
        if (!b_order.p) RMS_CUDA_TRY(rms_malloc((void**)&b_order.p, std::max<uint64_t>(n, 1) * sizeof(uint32_t)));
        rc = rms_order_by_class(s, w, b_order.as<uint32_t>(), stream, &n_launches);
        if (rc != RMS_OK) return rc;
    }
    rc = rms_launch_signal(rp, nW, nQ, nTerms, b_q.as<double>(), d_qwave, d_re, d_im, d_sum_alpha, b_order.as<uint32_t>(), stream,
                           &n_launches);
    if (rc != RMS_OK) return rc;
    RMS_CUDA_TRY(cudaEventRecord(ev_end, stream));

    // ---- read back and normalise (H8) -------------------------------------------------------------
    std::vector<double> h_res(n_res_d);
    std::vector<unsigned long long> h_flow(std::max<size_t>(n_flow, 1));
    unsigned long long h_cnt[8] = {0};
    RMS_CUDA_TRY(cudaMemcpyAsync(h_res.data(), b_res.p, n_res_d * sizeof(double), cudaMemcpyDeviceToHost, stream));
    if (n_flow) RMS_CUDA_TRY(cudaMemcpyAsync(h_flow.data(), d_flow, n_flow * sizeof(unsigned long long), cudaMemcpyDeviceToHost, stream));
    RMS_CUDA_TRY(cudaMemcpyAsync(h_cnt, w->d_counters, 64, cudaMemcpyDeviceToHost, stream));
    RMS_CUDA_TRY(cudaStreamSynchronize(stream));
    RMS_CUDA_TRY(cudaGetLastError());

    const double* h_re = h_res.data();
    const double* h_im = h_re + n_sig;
    const double* h_m2 = h_im + n_sig;
    const double* h_m4 = h_m2 + n_mom;
    const double* h_sal = h_m4 + n_mom;
    const double* h_sum_alpha = h_sal + n_sal;
    if (out->sum_alpha) memcpy(out->sum_alpha, h_sum_alpha, nC * sizeof(double));
    const size_t n_sig_s = (size_t)nQs * nC, n_sig_t = (size_t)nQt * nC;
    if (out->sig_re) memcpy(out->sig_re, h_re, n_sig_s * sizeof(double));
    if (out->sig_im) memcpy(out->sig_im, h_im, n_sig_s * sizeof(double));
    if (out->tsig_re) memcpy(out->tsig_re, h_re + n_sig_s, n_sig_t * sizeof(double));
    if (out->tsig_im) memcpy(out->tsig_im, h_im + n_sig_s, n_sig_t * sizeof(double));
    if (out->m2) memcpy(out->m2, h_m2, n_mom * sizeof(double));
    if (out->m4) memcpy(out->m4, h_m4, n_mom * sizeof(double));
    if (out->snap_alpha) memcpy(out->snap_alpha, h_sal, n_sal * sizeof(double));
    if (out->class_flow && n_flow) memcpy(out->class_flow, h_flow.data(), n_flow * sizeof(uint64_t));
    {
        std::vector<double> t_ms(std::max(nS, 1));
        for (int sidx = 0; sidx < nS; ++sidx) t_ms[sidx] = (double)(w->steps_done + (uint64_t)d->snap_steps[sidx]) * d->dt_ms;
        if (nQt > 0)      // Eq.7 for the tensor waveforms: the same normalisation, no moments
            rms_normalise(nC, nQt, h_sum_alpha, h_re + n_sig_s, h_im + n_sig_s, 0, 0, nullptr, nullptr, nullptr, nullptr, out->tS_re,
                          out->tS_im, nullptr, nullptr);
        rms_normalise(nC, nQs, h_sum_alpha, h_re, h_im, nS, nD, h_sal, h_m2, h_m4, t_ms.data(), out->S_re, out->S_im, out->Dapp,
                      out->Kapp);
    }
    out->n_encounters = h_cnt[0];
    out->n_permeations = h_cnt[1];
    out->n_clamps = h_cnt[2];
    out->n_saturations = h_cnt[4];
    float ms = 0.f, tot = 0.f;
    for (auto& pr : step_ev) { float t1 = 0.f; cudaEventElapsedTime(&t1, pr.first, pr.second); ms += t1; }
    cudaEventElapsedTime(&tot, ev_begin, ev_end);
    out->kernel_ms = ms;
    out->total_ms = tot;
    out->n_launches = n_launches;
    guard.armed = false;
    w->steps_done += (uint64_t)nT;
    return RMS_OK;
}
