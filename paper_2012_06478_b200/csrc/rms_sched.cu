// rms_sched.cu -- which thread walks which walker.
//
// Trajectories depend on (seed, walker id, step) only (R2), so the walker -> thread mapping is free.  The step
// kernel's only memory traffic is one gather per voxel change from a lattice far larger than the L2, so the
// mapping is chosen for locality: walkers are binned by the 8 x 8 x 16-voxel cell they sit in, cells ordered z-major
// (a counting sort: histogram, one-block exclusive scan, scatter).  The lanes of a warp then start inside one cell
// (shared sectors and L1 lines), and the blocks resident at one time cover a slab of the lattice instead of all
// of it (L2 reuse).  Walkers drift apart by sqrt(6 D t); rms_run re-sorts at every launch boundary.
#include "rms_internal.cuh"

#define RMS_CELL_XY 8
#define RMS_CELL_Z 16

namespace {

__device__ __forceinline__ uint32_t rms_cell_of(int x, int y, int z, int cx, int cy)
{
    return ((uint32_t)(z / RMS_CELL_Z) * cy + (uint32_t)(y / RMS_CELL_XY)) * cx + (uint32_t)(x / RMS_CELL_XY);
}

__global__ void __launch_bounds__(256) rms_cell_hist_kernel(rms_walker_arrays st, uint64_t n, int cx, int cy, uint32_t* count)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) atomicAdd(&count[rms_cell_of(st.w[0][i], st.w[1][i], st.w[2][i], cx, cy)], 1u);
}

// exclusive prefix sum over n_cells counters, in place, one block
__global__ void __launch_bounds__(1024) rms_cell_scan_kernel(uint32_t* count, uint32_t n_cells)
{
    __shared__ uint32_t part[1024];
    const uint32_t per = (n_cells + 1023u) / 1024u;
    const uint32_t a = min(n_cells, threadIdx.x * per), b = min(n_cells, a + per);
    uint32_t sum = 0;
    for (uint32_t c = a; c < b; ++c) sum += count[c];
    part[threadIdx.x] = sum;
    __syncthreads();
    for (uint32_t o = 1; o < 1024u; o <<= 1) {   // Hillis-Steele inclusive scan of the per-thread sums
        const uint32_t v = threadIdx.x >= o ? part[threadIdx.x - o] : 0u;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    uint32_t run = part[threadIdx.x] - sum;
    for (uint32_t c = a; c < b; ++c) { const uint32_t v = count[c]; count[c] = run; run += v; }
}

__global__ void __launch_bounds__(256) rms_cell_scatter_kernel(rms_walker_arrays st, uint64_t n, int cx, int cy, uint32_t* cursor,
                                                                uint32_t* order)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) order[atomicAdd(&cursor[rms_cell_of(st.w[0][i], st.w[1][i], st.w[2][i], cx, cy)], 1u)] = (uint32_t)i;
}

}  // namespace

int rms_order_walkers(const rms_substrate* s, const rms_walkers* w, uint32_t* d_order, cudaStream_t stream, unsigned* n_launches)
{
    const int cx = (s->nx + RMS_CELL_XY - 1) / RMS_CELL_XY, cy = (s->ny + RMS_CELL_XY - 1) / RMS_CELL_XY;
    const int cz = (s->nz + RMS_CELL_Z - 1) / RMS_CELL_Z;
    const uint64_t n_cells = (uint64_t)cx * cy * cz;
    RMS_REQUIRE(n_cells < (1ull << 31) && w->n < (1ull << 32), RMS_ERR_UNSUPPORTED, "too many cells or walkers to order");
    uint32_t* d_count = nullptr;
    RMS_CUDA_TRY(rms_malloc((void**)&d_count, n_cells * sizeof(uint32_t)));
    cudaError_t e = cudaMemsetAsync(d_count, 0, n_cells * sizeof(uint32_t), stream);
    if (e == cudaSuccess) {
        const unsigned grid = (unsigned)((w->n + 255) / 256);
        rms_cell_hist_kernel<<<grid, 256, 0, stream>>>(w->a, w->n, cx, cy, d_count);
        rms_cell_scan_kernel<<<1, 1024, 0, stream>>>(d_count, (uint32_t)n_cells);
        rms_cell_scatter_kernel<<<grid, 256, 0, stream>>>(w->a, w->n, cx, cy, d_count, d_order);
        e = cudaGetLastError();
        if (n_launches) *n_launches += 3;
    }
    // the block goes back to the cache; later work on this stream is ordered after the kernels above
    rms_free(d_count);
    RMS_CUDA_TRY(e);
    return RMS_OK;
}
