// rms_walkers.cu -- H1: walker initialisation and the state arrays / read-back hook.
#include <string.h>
#include <cmath>

#include "rms_internal.cuh"

#define RMS_MAX_INIT_ATTEMPTS (1u << 20)

// One thread per walker.  Proposal a = 0,1,..: voxel = floor(uni(w) * n) per axis from Philox(walker, a, INIT),
// accepted iff its label is allowed; offset from Philox(walker, 0, INIT_OFFSET) (R13).  With spin concentrations
// (Appendix C.2; R24) the proposal is kept with probability accept[L] = c_L / max c, against uni of the spare fourth word.
__global__ void __launch_bounds__(256) rms_init_kernel(const uint16_t* __restrict__ labels, int nx, int ny, int nz,
                                                        const uint8_t* __restrict__ allowed, const float* __restrict__ accept,
                                                        rms_walker_arrays st, uint64_t n,
                                                        uint64_t first_id, rms_philox_keys rk, int n_phi,
                                                        unsigned long long* __restrict__ counters)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint64_t id = first_id + i;
    const uint32_t id_lo = (uint32_t)id, id_hi = (uint32_t)(id >> 32);
    uint32_t w0, w1, w2, w3;
    int x = 0, y = 0, z = 0;
    uint32_t L = 0;
    bool ok = false;
    for (uint32_t a = 0; a < RMS_MAX_INIT_ATTEMPTS; ++a) {
        rms_philox(rk, id_lo, id_hi, a, RMS_STREAM_INIT, w0, w1, w2, w3);
        x = (int)__umulhi(w0 & 0xFFFFFF00u, (uint32_t)nx);  // floor((w>>8) nx / 2^24), integer exact
        y = (int)__umulhi(w1 & 0xFFFFFF00u, (uint32_t)ny);
        z = (int)__umulhi(w2 & 0xFFFFFF00u, (uint32_t)nz);
        L = labels[((size_t)z * ny + y) * nx + x];
        if (allowed && !allowed[L]) continue;
        if (accept && !(rms_uni(w3) < accept[L])) continue;
        ok = true;
        break;
    }
    if (!ok) atomicAdd(&counters[3], 1ull);
    rms_philox(rk, id_lo, id_hi, 0u, RMS_STREAM_INIT_OFFSET, w0, w1, w2, w3);
    const float fx = rms_uni(w0), fy = rms_uni(w1), fz = rms_uni(w2);
    st.w[0][i] = x; st.w[1][i] = y; st.w[2][i] = z;
    st.v0[0][i] = x; st.v0[1][i] = y; st.v0[2][i] = z;
    st.dI[0][i] = 0; st.dI[1][i] = 0; st.dI[2][i] = 0;
    st.f[0][i] = fx; st.f[1][i] = fy; st.f[2][i] = fz;
    st.f0[0][i] = fx; st.f0[1][i] = fy; st.f0[2][i] = fz;
    st.lab[i] = L | (L << 16);
    st.relax[i] = 0.f;
    st.f_lo[0][i] = 0.f; st.f_lo[1][i] = 0.f; st.f_lo[2][i] = 0.f;
    for (int k = 0; k < n_phi; ++k) st.phi[(size_t)k * n + i] = 0.0;
}

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

extern "C" int rms_walkers_init(const rms_substrate* s, uint64_t n_walkers, uint64_t first_walker_id,
                                const uint8_t* label_allowed, uint64_t seed, void* cuda_stream, rms_walkers** out)
{
    return rms_walkers_init_weighted(s, n_walkers, first_walker_id, label_allowed, nullptr, seed, cuda_stream, out);
}

extern "C" int rms_walkers_init_weighted(const rms_substrate* s, uint64_t n_walkers, uint64_t first_walker_id,
                                         const uint8_t* label_allowed, const float* label_weight, uint64_t seed,
                                         void* cuda_stream, rms_walkers** out)
{
    RMS_REQUIRE(s && out, RMS_ERR_ARG, "rms_walkers_init: null substrate or output");
    *out = nullptr;
    RMS_REQUIRE(n_walkers > 0 && n_walkers < (1ull << 31), RMS_ERR_ARG, "n_walkers must be in 1..2^31-1");
    if (label_allowed) {
        bool any = false;
        for (int a = 0; a < s->n_labels; ++a) any |= label_allowed[a] != 0;
        RMS_REQUIRE(any, RMS_ERR_NO_SPACE, "no label is allowed");
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    rms_walkers* w = new (std::nothrow) rms_walkers();
    RMS_REQUIRE(w, RMS_ERR_OOM, "out of host memory");
    w->sub = s; w->n = n_walkers; w->first_id = first_walker_id; w->seed = seed;
    const uint64_t n = n_walkers;
    // 20 arrays of 4 bytes + counters, each 256-byte aligned inside one block
    const size_t a4 = align_up(n * 4, 256);
    const size_t total = 20 * a4 + 256;
    uint8_t* d_allowed = nullptr;
    float* d_accept = nullptr;
    std::vector<float> h_accept;
    if (!s->conc.empty() || label_weight) {
        // initial density proportional to c_L (R24) times the caller's placement weight (R26), over the allowed labels
        auto weight = [&](int a) {
            return (s->conc.empty() ? 1.0 : (double)s->conc[a]) * (label_weight ? (double)label_weight[a] : 1.0);
        };
        double wmax = 0.0;
        for (int a = 0; a < s->n_labels; ++a) {
            RMS_REQUIRE(weight(a) >= 0.0 && std::isfinite(weight(a)), RMS_ERR_ARG, "label_weight[%d] is negative, infinite or NaN", a);
            if ((!label_allowed || label_allowed[a]) && weight(a) > wmax) wmax = weight(a);
        }
        RMS_REQUIRE(wmax > 0.0, RMS_ERR_NO_SPACE, "every allowed label has placement weight or spin concentration 0");
        h_accept.resize(s->n_labels);
        for (int a = 0; a < s->n_labels; ++a) h_accept[a] = (float)(weight(a) / wmax);
    }
    int rc = RMS_OK;
    unsigned long long h_cnt[8] = {0};
#define W_TRY(expr)                                                                                      \
    do {                                                                                                 \
        cudaError_t _e = (expr);                                                                         \
        if (_e != cudaSuccess) {                                                                         \
            rms_set_error("%s failed: %s", #expr, cudaGetErrorString(_e));                               \
            rc = (_e == cudaErrorMemoryAllocation) ? RMS_ERR_OOM : RMS_ERR_CUDA;                         \
            goto fail;                                                                                   \
        }                                                                                                \
    } while (0)
    W_TRY(rms_malloc((void**)&w->d_block, total));
    {
        char* p = (char*)w->d_block;
        auto take = [&](size_t bytes) { char* q = p; p += bytes; return (void*)q; };
        for (int k = 0; k < 3; ++k) w->a.w[k] = (int32_t*)take(a4);
        for (int k = 0; k < 3; ++k) w->a.dI[k] = (int32_t*)take(a4);
        for (int k = 0; k < 3; ++k) w->a.f[k] = (float*)take(a4);
        for (int k = 0; k < 3; ++k) w->a.f_lo[k] = (float*)take(a4);
        for (int k = 0; k < 3; ++k) w->a.v0[k] = (int32_t*)take(a4);
        for (int k = 0; k < 3; ++k) w->a.f0[k] = (float*)take(a4);
        w->a.lab = (uint32_t*)take(a4);
        w->a.relax = (float*)take(a4);
        w->d_counters = (unsigned long long*)take(256);
    }
    w->n_wave_alloc = 1;
    W_TRY(rms_malloc((void**)&w->a.phi, (size_t)3 * w->n_wave_alloc * n * sizeof(double)));
    W_TRY(cudaMemsetAsync(w->d_counters, 0, 64, stream));
    if (label_allowed) {
        W_TRY(rms_malloc((void**)&d_allowed, s->n_labels));
        W_TRY(cudaMemcpyAsync(d_allowed, label_allowed, s->n_labels, cudaMemcpyHostToDevice, stream));
    }
    if (!h_accept.empty()) {
        W_TRY(rms_malloc((void**)&d_accept, s->n_labels * sizeof(float)));
        W_TRY(cudaMemcpyAsync(d_accept, h_accept.data(), s->n_labels * sizeof(float), cudaMemcpyHostToDevice, stream));
    }
    rms_init_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(s->d_labels, s->nx, s->ny, s->nz, d_allowed, d_accept, w->a, n,
                                                                      first_walker_id, rms_make_keys(seed),
                                                                      3 * w->n_wave_alloc, w->d_counters);
    W_TRY(cudaGetLastError());
    W_TRY(cudaMemcpyAsync(h_cnt, w->d_counters, 64, cudaMemcpyDeviceToHost, stream));
    W_TRY(cudaStreamSynchronize(stream));
    if (d_allowed) rms_free(d_allowed);
    d_allowed = nullptr;
    if (d_accept) rms_free(d_accept);
    d_accept = nullptr;
    if (h_cnt[3] != 0) {
        rms_set_error("%llu walkers found no voxel with an allowed label in 2^20 proposals", h_cnt[3]);
        rc = RMS_ERR_NO_SPACE;
        goto fail;
    }
    *out = w;
    return RMS_OK;
fail:
    if (d_allowed) rms_free(d_allowed);
    if (d_accept) rms_free(d_accept);
    rms_walkers_destroy(w);
    return rc;
#undef W_TRY
}

extern "C" int rms_walkers_destroy(rms_walkers* w)
{
    if (!w) return RMS_OK;
    if (w->d_block) rms_free(w->d_block);
    if (w->a.phi) rms_free(w->a.phi);
    delete w;
    return RMS_OK;
}

extern "C" int rms_walkers_steps_done(const rms_walkers* w, uint64_t* out)
{
    RMS_REQUIRE(w && out, RMS_ERR_ARG, "rms_walkers_steps_done: null argument");
    *out = w->steps_done;
    return RMS_OK;
}

// grow the phase accumulators to n_wave waveforms, keeping what is there
int rms_walkers_reserve_waves(rms_walkers* w, int n_wave, cudaStream_t stream)
{
    if (n_wave <= w->n_wave_alloc) return RMS_OK;
    double* np = nullptr;
    RMS_CUDA_TRY(rms_malloc((void**)&np, (size_t)3 * n_wave * w->n * sizeof(double)));
    RMS_CUDA_TRY(cudaMemsetAsync(np, 0, (size_t)3 * n_wave * w->n * sizeof(double), stream));
    RMS_CUDA_TRY(cudaMemcpyAsync(np, w->a.phi, (size_t)3 * w->n_wave_alloc * w->n * sizeof(double), cudaMemcpyDeviceToDevice,
                                 stream));
    RMS_CUDA_TRY(cudaStreamSynchronize(stream));
    rms_free(w->a.phi);
    w->a.phi = np;
    w->n_wave_alloc = n_wave;
    return RMS_OK;
}

extern "C" int rms_walkers_read(const rms_walkers* w, uint64_t first, uint64_t count, rms_walker_state* host_out,
                                void* cuda_stream)
{
    RMS_REQUIRE(w && host_out, RMS_ERR_ARG, "rms_walkers_read: null argument");
    RMS_REQUIRE(first + count <= w->n, RMS_ERR_ARG, "rms_walkers_read: range [%llu, %llu) exceeds %llu walkers",
                (unsigned long long)first, (unsigned long long)(first + count), (unsigned long long)w->n);
    if (count == 0) return RMS_OK;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    std::vector<int32_t> wv(3 * count), dI(3 * count), v0(3 * count);
    std::vector<float> f(3 * count), f0(3 * count), relax(count);
    std::vector<uint32_t> lab(count);
    std::vector<double> phi((size_t)3 * w->n_wave_alloc * count);
    for (int k = 0; k < 3; ++k) {
        RMS_CUDA_TRY(cudaMemcpyAsync(&wv[k * count], w->a.w[k] + first, count * 4, cudaMemcpyDeviceToHost, stream));
        RMS_CUDA_TRY(cudaMemcpyAsync(&dI[k * count], w->a.dI[k] + first, count * 4, cudaMemcpyDeviceToHost, stream));
        RMS_CUDA_TRY(cudaMemcpyAsync(&v0[k * count], w->a.v0[k] + first, count * 4, cudaMemcpyDeviceToHost, stream));
        RMS_CUDA_TRY(cudaMemcpyAsync(&f[k * count], w->a.f[k] + first, count * 4, cudaMemcpyDeviceToHost, stream));
        RMS_CUDA_TRY(cudaMemcpyAsync(&f0[k * count], w->a.f0[k] + first, count * 4, cudaMemcpyDeviceToHost, stream));
    }
    RMS_CUDA_TRY(cudaMemcpyAsync(lab.data(), w->a.lab + first, count * 4, cudaMemcpyDeviceToHost, stream));
    RMS_CUDA_TRY(cudaMemcpyAsync(relax.data(), w->a.relax + first, count * 4, cudaMemcpyDeviceToHost, stream));
    for (int j = 0; j < 3 * w->n_wave_alloc; ++j)
        RMS_CUDA_TRY(cudaMemcpyAsync(&phi[(size_t)j * count], w->a.phi + (size_t)j * w->n + first, count * 8,
                                     cudaMemcpyDeviceToHost, stream));
    RMS_CUDA_TRY(cudaStreamSynchronize(stream));
    for (uint64_t i = 0; i < count; ++i) {
        rms_walker_state& o = host_out[i];
        memset(&o, 0, sizeof o);
        for (int k = 0; k < 3; ++k) {
            o.vox0[k] = v0[k * count + i];
            o.vox[k] = v0[k * count + i] + dI[k * count + i];
            o.off[k] = f[k * count + i];
            o.off0[k] = f0[k * count + i];
        }
        o.label = (uint16_t)(lab[i] & 0xFFFFu);
        o.label0 = (uint16_t)(lab[i] >> 16);
        o.relax = relax[i];
        for (int m = 0; m < w->n_wave_alloc && m < RMS_MAX_WAVES; ++m)
            for (int k = 0; k < 3; ++k) o.phi[m][k] = phi[(size_t)(3 * m + k) * count + i];
    }
    return RMS_OK;
}
