// rms_reduce.cu -- H6/H7: per-walker epilogue and the reductions to signal and moment sums.
//
//   moments: thread = walker; X = l_p n.(x - x0) per direction; warp-shuffle reduction per class, then
//            shared-memory fp64 accumulators per block, then fp64 atomics (one per block and output).
//   signal:  thread = one (waveform, gradient amplitude, direction) triple; the block stages a tile of
//            walkers in shared memory and every thread sums alpha e^{-i phi} over the tile in registers
//            (the walker is warp-uniform, so class handling never diverges); fp64 throughout the phase
//            reduction to a fraction of a turn, hardware (MUFU) sine / cosine of the reduced phase.
#include "rms_internal.cuh"

#define RED_BLOCK 256

__device__ __forceinline__ double warp_sum(double v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ------------------------------------------------------------------------------------------------
// moments at a snapshot
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(RED_BLOCK) rms_moments_kernel(const rms_reduce_params p, double* __restrict__ g_m2,
                                                                 double* __restrict__ g_m4, double* __restrict__ g_alpha,
                                                                 unsigned long long* __restrict__ g_flow, int use_smem)
{
    extern __shared__ double sm[];   // [n_dir*n_classes] m2, then m4, then [n_classes] alpha
    const int nD = p.n_dir, nC = p.n_classes;
    const int n_acc = 2 * nD * nC + nC;
    if (use_smem) {
        for (int t = threadIdx.x; t < n_acc; t += RED_BLOCK) sm[t] = 0.0;
        __syncthreads();
    }
    double* a_m2 = use_smem ? sm : g_m2;
    double* a_m4 = use_smem ? sm + nD * nC : g_m4;
    double* a_al = use_smem ? sm + 2 * nD * nC : g_alpha;
    const int lane = threadIdx.x & 31;

    const uint64_t n_tiles = (p.n + RED_BLOCK - 1) / RED_BLOCK;
    for (uint64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const uint64_t i = tile * RED_BLOCK + threadIdx.x;
        const bool valid = i < p.n;
        double dx = 0, dy = 0, dz = 0, alpha = 0;
        int c0 = -1, cn = 0;
        if (valid) {
            dx = (double)p.st.dI[0][i] + ((double)p.st.f[0][i] - (double)p.st.f0[0][i]);
            dy = (double)p.st.dI[1][i] + ((double)p.st.f[1][i] - (double)p.st.f0[1][i]);
            dz = (double)p.st.dI[2][i] + ((double)p.st.f[2][i] - (double)p.st.f0[2][i]);
            alpha = exp(-(double)p.st.relax[i]);          // Eq.5
            const uint32_t lab = p.st.lab[i];
            c0 = p.label_class[lab >> 16];
            cn = p.label_class[lab & 0xFFFFu];
        }
        {   // class_flow: one atomic per distinct (initial class, class now) pair in the warp
            const int key = valid ? c0 * nC + cn : -1;
            const unsigned same = __match_any_sync(0xffffffffu, key);
            if (valid && lane == __ffs(same) - 1) atomicAdd(&g_flow[key], (unsigned long long)__popc(same));
        }
        // classes present in this warp, one at a time (2 in the usual intra/extra split)
        unsigned todo = __ballot_sync(0xffffffffu, valid);
        while (todo) {
            const int leader = __ffs(todo) - 1;
            const int cc = __shfl_sync(0xffffffffu, c0, leader);
            const bool mine = valid && (c0 == cc);
            todo &= ~__ballot_sync(0xffffffffu, mine);
            const double a = mine ? alpha : 0.0;
            const double sa = warp_sum(a);
            if (lane == 0) atomicAdd(&a_al[cc], sa);
            for (int d = 0; d < nD; ++d) {
                const double X = p.voxel_um * (p.dirs[3 * d] * dx + p.dirs[3 * d + 1] * dy + p.dirs[3 * d + 2] * dz);
                const double X2 = X * X;
                const double s2 = warp_sum(a * X2);
                const double s4 = warp_sum(a * X2 * X2);
                if (lane == 0) {
                    atomicAdd(&a_m2[d * nC + cc], s2);
                    atomicAdd(&a_m4[d * nC + cc], s4);
                }
            }
        }
    }
    if (use_smem) {
        __syncthreads();
        for (int t = threadIdx.x; t < n_acc; t += RED_BLOCK) {
            const double v = sm[t];
            if (v != 0.0) {
                if (t < nD * nC) atomicAdd(&g_m2[t], v);
                else if (t < 2 * nD * nC) atomicAdd(&g_m4[t - nD * nC], v);
                else atomicAdd(&g_alpha[t - 2 * nD * nC], v);
            }
        }
    }
}

int rms_launch_moments(const rms_reduce_params& p, double* d_m2, double* d_m4, double* d_alpha, unsigned long long* d_flow,
                       cudaStream_t stream)
{
    const size_t n_acc = (size_t)2 * p.n_dir * p.n_classes + p.n_classes;
    const int use_smem = n_acc * sizeof(double) <= 40 * 1024;
    const uint64_t n_tiles = (p.n + RED_BLOCK - 1) / RED_BLOCK;
    const unsigned grid = (unsigned)(n_tiles < 148ull * 4 ? n_tiles : 148ull * 4);
    rms_moments_kernel<<<grid, RED_BLOCK, use_smem ? n_acc * sizeof(double) : 0, stream>>>(p, d_m2, d_m4, d_alpha, d_flow,
                                                                                          use_smem);
    RMS_CUDA_TRY(cudaGetLastError());
    return RMS_OK;
}

// ------------------------------------------------------------------------------------------------
// signal sums at the end of a call
// ------------------------------------------------------------------------------------------------
#define SIG_TILE 256
#define SIG_QPT 3   // q-triples per thread: a launch covers up to RED_BLOCK * SIG_QPT = 768 of them (660 in the bench)

// NT = terms per q: 1 for the scalar waveforms (phi = q . Phi_m), 3 for tensor waveforms (R23: phi = sum_a q_a . Phi_{m_a},
// a term with wave index -1 is off); qv is [q][NT][3], qwave [q][NT]
template <int NT>
__global__ void __launch_bounds__(RED_BLOCK) rms_signal_kernel(const rms_reduce_params p, int n_wave, int nq_l, int q_begin,
                                                                const double* __restrict__ qv, const int* __restrict__ qwave,
                                                                double* __restrict__ g_re, double* __restrict__ g_im,
                                                                double* __restrict__ g_sum_alpha)
{
    extern __shared__ double sm[];
    const int nC = p.n_classes;
    double* s_phi = sm;                                             // [n_wave*3][SIG_TILE]
    double* s_acc = s_phi + (size_t)n_wave * 3 * SIG_TILE;          // [nq_l][nC][2]
    double* s_alsum = s_acc + (size_t)nq_l * nC * 2;                // [nC]
    float* s_alpha = (float*)(s_alsum + nC);                        // [SIG_TILE]
    int* s_cls = (int*)(s_alpha + SIG_TILE);                        // [SIG_TILE]

    for (int t = threadIdx.x; t < nq_l * nC * 2 + nC; t += RED_BLOCK) s_acc[t] = 0.0;

    double qx[SIG_QPT][NT], qy[SIG_QPT][NT], qz[SIG_QPT][NT];
    int qm[SIG_QPT][NT];
    bool qok[SIG_QPT];
#pragma unroll
    for (int c = 0; c < SIG_QPT; ++c) {
        const int jl = c * RED_BLOCK + threadIdx.x;
        const bool ok = jl < nq_l;
        const int j = q_begin + jl;
        qok[c] = ok;
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            const int jt = j * NT + t;
            qx[c][t] = ok ? qv[3 * jt] : 0.0; qy[c][t] = ok ? qv[3 * jt + 1] : 0.0; qz[c][t] = ok ? qv[3 * jt + 2] : 0.0;
            qm[c][t] = ok ? qwave[jt] : -1;
        }
    }

    const uint64_t n_tiles = (p.n + SIG_TILE - 1) / SIG_TILE;
    for (uint64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        __syncthreads();
        const uint64_t i = tile * SIG_TILE + threadIdx.x;
        const int n_in = (int)min((uint64_t)SIG_TILE, p.n - tile * SIG_TILE);
        if (threadIdx.x < n_in) {
            for (int k = 0; k < 3 * n_wave; ++k) s_phi[k * SIG_TILE + threadIdx.x] = p.st.phi[(size_t)k * p.n + i];
            const float al = (float)exp(-(double)p.st.relax[i]);
            const int c0 = p.label_class[p.st.lab[i] >> 16];
            s_alpha[threadIdx.x] = al;
            s_cls[threadIdx.x] = c0;
            if (q_begin == 0) atomicAdd(&s_alsum[c0], (double)al);
        }
        __syncthreads();
        for (int cc = 0; cc < nC; ++cc) {
            double are[SIG_QPT], aim[SIG_QPT];
#pragma unroll
            for (int c = 0; c < SIG_QPT; ++c) { are[c] = 0.0; aim[c] = 0.0; }
            bool any = false;
            for (int w = 0; w < n_in; ++w) {
                if (s_cls[w] != cc) continue;                    // warp-uniform
                any = true;
                const double al = (double)s_alpha[w];
#pragma unroll
                for (int c = 0; c < SIG_QPT; ++c) {
                    if (!qok[c]) continue;
                    double turns = 0.0;
#pragma unroll
                    for (int t = 0; t < NT; ++t) {
                        if (NT > 1 && qm[c][t] < 0) continue;
                        const double* ph = s_phi + (size_t)qm[c][t] * 3 * SIG_TILE + w;
                        turns += qx[c][t] * ph[0] + qy[c][t] * ph[SIG_TILE] + qz[c][t] * ph[2 * SIG_TILE];
                    }
                    // phase reduced in fp64 to [-pi, pi], then the hardware sine / cosine: absolute error < 5e-7 per
                    // walker (random in sign for the sine, mean +2e-8 for the cosine) against the 1e-4 tolerance on S
                    const float ph32 = (float)(6.283185307179586 * (turns - rint(turns)));
                    float sn, cs;
                    __sincosf(ph32, &sn, &cs);
                    are[c] += al * (double)cs;                   // Eq.7: alpha e^{-i phi}
                    aim[c] -= al * (double)sn;
                }
            }
            if (any) {
#pragma unroll
                for (int c = 0; c < SIG_QPT; ++c) {
                    const int jl = c * RED_BLOCK + threadIdx.x;
                    if (jl < nq_l) {
                        s_acc[((size_t)jl * nC + cc) * 2] += are[c];      // (jl, cc) is owned by this thread
                        s_acc[((size_t)jl * nC + cc) * 2 + 1] += aim[c];
                    }
                }
            }
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < nq_l * nC; t += RED_BLOCK) {
        const int jl = t / nC, cc = t - jl * nC;
        const size_t o = (size_t)(q_begin + jl) * nC + cc;
        atomicAdd(&g_re[o], s_acc[2 * t]);
        atomicAdd(&g_im[o], s_acc[2 * t + 1]);
    }
    if (q_begin == 0)
        for (int t = threadIdx.x; t < nC; t += RED_BLOCK)
            if (s_alsum[t] != 0.0) atomicAdd(&g_sum_alpha[t], s_alsum[t]);
}

// ------------------------------------------------------------------------------------------------
// signal sums with many output classes (per-cell outputs: class = label, hundreds of classes).  Per-block accumulators
// for every (q, class) no longer fit anywhere, so the walkers are visited in the order of their class (rms_sched.cu):
// a tile of 256 consecutive walkers is one run of a class, occasionally two or three.  Thread = up to SIG_QPT
// (waveform, b, direction) triples; sums in registers over a run; fp64 atomics into the output at the end of each run.
// ------------------------------------------------------------------------------------------------
template <int NT>
__global__ void __launch_bounds__(RED_BLOCK) rms_signal_runs_kernel(const rms_reduce_params p, int n_wave, int nq_l, int q_begin,
                                                                     const double* __restrict__ qv, const int* __restrict__ qwave,
                                                                     const uint32_t* __restrict__ order, double* __restrict__ g_re,
                                                                     double* __restrict__ g_im, double* __restrict__ g_sum_alpha)
{
    extern __shared__ double sm[];
    const int nC = p.n_classes;
    double* s_phi = sm;                                             // [n_wave*3][SIG_TILE]
    float* s_alpha = (float*)(s_phi + (size_t)n_wave * 3 * SIG_TILE);   // [SIG_TILE]
    int* s_cls = (int*)(s_alpha + SIG_TILE);                        // [SIG_TILE]

    double qx[SIG_QPT][NT], qy[SIG_QPT][NT], qz[SIG_QPT][NT];
    int qm[SIG_QPT][NT];
    bool qok[SIG_QPT];
#pragma unroll
    for (int c = 0; c < SIG_QPT; ++c) {
        const int jl = c * RED_BLOCK + threadIdx.x;
        const bool ok = jl < nq_l;
        const int j = q_begin + jl;
        qok[c] = ok;
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            const int jt = j * NT + t;
            qx[c][t] = ok ? qv[3 * jt] : 0.0; qy[c][t] = ok ? qv[3 * jt + 1] : 0.0; qz[c][t] = ok ? qv[3 * jt + 2] : 0.0;
            qm[c][t] = ok ? qwave[jt] : -1;
        }
    }

    const uint64_t n_tiles = (p.n + SIG_TILE - 1) / SIG_TILE;
    for (uint64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        __syncthreads();
        const int n_in = (int)min((uint64_t)SIG_TILE, p.n - tile * SIG_TILE);
        if (threadIdx.x < n_in) {
            const uint64_t i = order[tile * SIG_TILE + threadIdx.x];
            for (int k = 0; k < 3 * n_wave; ++k) s_phi[k * SIG_TILE + threadIdx.x] = p.st.phi[(size_t)k * p.n + i];
            s_alpha[threadIdx.x] = (float)exp(-(double)p.st.relax[i]);
            s_cls[threadIdx.x] = p.label_class[p.st.lab[i] >> 16];
        }
        __syncthreads();
        double are[SIG_QPT], aim[SIG_QPT], asum = 0.0;
#pragma unroll
        for (int c = 0; c < SIG_QPT; ++c) { are[c] = 0.0; aim[c] = 0.0; }
        int cur = s_cls[0];
        for (int w = 0; w <= n_in; ++w) {
            const int cc = w < n_in ? s_cls[w] : -1;                 // warp-uniform
            if (cc != cur) {                                        // end of a run: flush
#pragma unroll
                for (int c = 0; c < SIG_QPT; ++c) {
                    const int jl = c * RED_BLOCK + threadIdx.x;
                    if (jl < nq_l) {
                        const size_t o = (size_t)(q_begin + jl) * nC + cur;
                        atomicAdd(&g_re[o], are[c]);
                        atomicAdd(&g_im[o], aim[c]);
                    }
                    are[c] = 0.0; aim[c] = 0.0;
                }
                if (q_begin == 0 && threadIdx.x == 0) atomicAdd(&g_sum_alpha[cur], asum);
                asum = 0.0;
                cur = cc;
                if (w == n_in) break;
            }
            const double al = (double)s_alpha[w];
            asum += al;
#pragma unroll
            for (int c = 0; c < SIG_QPT; ++c) {
                if (!qok[c]) continue;
                double turns = 0.0;
#pragma unroll
                for (int t = 0; t < NT; ++t) {
                    if (NT > 1 && qm[c][t] < 0) continue;
                    const double* ph = s_phi + (size_t)qm[c][t] * 3 * SIG_TILE + w;
                    turns += qx[c][t] * ph[0] + qy[c][t] * ph[SIG_TILE] + qz[c][t] * ph[2 * SIG_TILE];
                }
                const float ph32 = (float)(6.283185307179586 * (turns - rint(turns)));
                float sn, cs;
                __sincosf(ph32, &sn, &cs);
                are[c] += al * (double)cs;                       // Eq.7: alpha e^{-i phi}
                aim[c] -= al * (double)sn;
            }
        }
    }
}

int rms_launch_signal(const rms_reduce_params& p, int n_wave, int nq, int n_terms, const double* d_qv, const int* d_qwave, double* d_re,
                      double* d_im, double* d_sum_alpha, const uint32_t* order_by_class, cudaStream_t stream, unsigned* n_launches)
{
    RMS_REQUIRE(n_terms == 1 || n_terms == 3, RMS_ERR_ARG, "signal reduction: 1 or 3 terms per phase");
    auto k_runs = n_terms == 1 ? rms_signal_runs_kernel<1> : rms_signal_runs_kernel<3>;
    auto k_sig = n_terms == 1 ? rms_signal_kernel<1> : rms_signal_kernel<3>;
    const uint64_t n_tiles = (p.n + SIG_TILE - 1) / SIG_TILE;
    // 4 blocks per SM is what the registers allow (58 x 256); measured on 1e6 walkers x 660 signals: 1.78 / 1.47 / 1.33 / 1.45 ms
    // for 2 / 3 / 4 / 6 blocks per SM
    const unsigned grid = (unsigned)(n_tiles < 148ull * 4 ? n_tiles : 148ull * 4);
    const int nw = n_wave > 0 ? n_wave : 1;
    if (p.n_classes > RMS_SIG_SMALL_CLASSES) {
        RMS_REQUIRE(order_by_class, RMS_ERR_ARG, "signal reduction with many classes needs the class ordering");
        const size_t smem = (size_t)nw * 3 * SIG_TILE * sizeof(double) + SIG_TILE * (sizeof(float) + sizeof(int));
        if (smem > 48 * 1024)
            RMS_CUDA_TRY(cudaFuncSetAttribute(k_runs, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        const int q_batch = RED_BLOCK * SIG_QPT;
        int q_begin = 0;
        do {
            const int nq_l = nq - q_begin < q_batch ? nq - q_begin : q_batch;
            k_runs<<<grid, RED_BLOCK, smem, stream>>>(p, nw, nq_l > 0 ? nq_l : 0, q_begin, d_qv, d_qwave, order_by_class,
                                                                      d_re, d_im, d_sum_alpha);
            RMS_CUDA_TRY(cudaGetLastError());
            if (n_launches) ++*n_launches;
            q_begin += q_batch;
        } while (q_begin < nq);
        return RMS_OK;
    }
    const size_t fixed = ((size_t)nw * 3 * SIG_TILE + p.n_classes) * sizeof(double) + SIG_TILE * (sizeof(float) + sizeof(int));
    const size_t budget = 160 * 1024;
    const size_t per_q = (size_t)p.n_classes * 2 * sizeof(double);
    if (fixed + per_q > budget) {
        rms_set_error("signal reduction: n_classes = %d needs more shared memory than a block has", p.n_classes);
        return RMS_ERR_UNSUPPORTED;
    }
    int q_batch = (int)((budget - fixed) / per_q);
    if (q_batch > RED_BLOCK * SIG_QPT) q_batch = RED_BLOCK * SIG_QPT;
    int q_begin = 0;
    do {   // nq == 0: still one launch, for sum_alpha
        const int nq_l = nq - q_begin < q_batch ? nq - q_begin : q_batch;
        const size_t smem = fixed + (size_t)(nq_l > 0 ? nq_l : 0) * per_q;
        if (smem > 48 * 1024)
            RMS_CUDA_TRY(cudaFuncSetAttribute(k_sig, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)budget));
        k_sig<<<grid, RED_BLOCK, smem, stream>>>(p, nw, nq_l, q_begin, d_qv, d_qwave, d_re, d_im, d_sum_alpha);
        RMS_CUDA_TRY(cudaGetLastError());
        if (n_launches) ++*n_launches;
        q_begin += q_batch;
    } while (q_begin < nq);
    return RMS_OK;
}
