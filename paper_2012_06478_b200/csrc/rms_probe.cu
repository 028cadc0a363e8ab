// rms_probe.cu -- measured ceilings for the second roofline candidate of the step kernel: the rate
// at which the GPU serves random small gathers, each touching its own 32-byte sector, from a table that sits in the L2
// (tens of MB) or in HBM (GB).  Streaming bandwidth says little about that; S: section 8(d) asks for this number.
#include "rms_internal.cuh"

namespace {

template <typename T>
__global__ void __launch_bounds__(256) rms_gather_probe_kernel(const T* __restrict__ table, uint32_t n_elems, uint32_t loads,
                                                                unsigned long long* __restrict__ sink)
{
    // four independent pseudo-random index streams per thread (linear congruential, multiplicative range reduction)
    uint32_t s0 = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
    uint32_t s1 = s0 ^ 0x9E3779B9u, s2 = s0 * 747796405u + 1u, s3 = ~s0;
    unsigned long long acc = 0;
    for (uint32_t i = 0; i < loads; i += 4) {
        s0 = s0 * 1664525u + 1013904223u; s1 = s1 * 1664525u + 1013904223u;
        s2 = s2 * 1664525u + 1013904223u; s3 = s3 * 1664525u + 1013904223u;
        acc += __ldg(table + __umulhi(s0, n_elems));
        acc += __ldg(table + __umulhi(s1, n_elems));
        acc += __ldg(table + __umulhi(s2, n_elems));
        acc += __ldg(table + __umulhi(s3, n_elems));
    }
    if (acc == 0x123456789ull) *sink = acc;   // keeps the loads alive
}

}  // namespace

// Random gathers of `elem_bytes` (2 or 4) from a zero-filled table of `table_bytes`; loads_per_thread each on
// 148 x 2048 threads; *gathers_per_s = gathers (= distinct 32-byte sectors, for tables far larger than the launch)
// per second, timed with CUDA events on `cuda_stream` after one warm-up launch.
extern "C" int rms_gather_probe(uint64_t table_bytes, int elem_bytes, uint32_t loads_per_thread, void* cuda_stream,
                                double* gathers_per_s)
{
    RMS_REQUIRE(gathers_per_s && (elem_bytes == 2 || elem_bytes == 4) && table_bytes >= 4096 && loads_per_thread >= 4 &&
                    table_bytes / elem_bytes < (1ull << 32),
                RMS_ERR_ARG, "rms_gather_probe: bad argument");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    void* table = nullptr;
    unsigned long long* sink = nullptr;
    RMS_CUDA_TRY(rms_malloc(&table, table_bytes));
    cudaError_t e = rms_malloc((void**)&sink, 8);
    if (e != cudaSuccess) { rms_free(table); RMS_CUDA_TRY(e); }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    float ms = 0.f;
    e = cudaMemsetAsync(table, 0, table_bytes, stream);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    const uint32_t n_elems = (uint32_t)(table_bytes / elem_bytes), loads = loads_per_thread & ~3u;
    const unsigned grid = 148 * 8;
    for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) {
        if (rep == 1) e = cudaEventRecord(e0, stream);
        if (elem_bytes == 2) rms_gather_probe_kernel<uint16_t><<<grid, 256, 0, stream>>>((const uint16_t*)table, n_elems, loads, sink);
        else rms_gather_probe_kernel<uint32_t><<<grid, 256, 0, stream>>>((const uint32_t*)table, n_elems, loads, sink);
        if (e == cudaSuccess) e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaEventRecord(e1, stream);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    rms_free(table);
    rms_free(sink);
    RMS_CUDA_TRY(e);
    *gathers_per_s = (double)grid * 256.0 * (double)loads / ((double)ms * 1e-3);
    return RMS_OK;
}
