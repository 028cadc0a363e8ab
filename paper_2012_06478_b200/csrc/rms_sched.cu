// rms_sched.cu -- which thread walks which walker.
//
// Trajectories depend on (seed, walker id, step) only (R2), so the walker -> thread mapping is free.  The step
// kernel's only memory traffic is one gather per voxel change from a lattice far larger than the L2, so the
// mapping is chosen for locality: walkers are binned by the 8 x 8 x 16-voxel cell they sit in, cells ordered z-major
// (a counting sort: histogram, one-block exclusive scan, scatter).  The lanes of a warp then start inside one cell
// (shared sectors and L1 lines), and the blocks resident at one time cover a slab of the lattice instead of all
// of it (L2 reuse).  Walkers drift apart by sqrt(6 D t); rms_run re-sorts at every launch boundary.
#include "rms_internal.cuh"

#ifndef RMS_CELL_XY
#define RMS_CELL_XY 8
#endif
#ifndef RMS_CELL_Z
#define RMS_CELL_Z 16
#endif

namespace {

// cells are numbered in the memory order of the neighbourhood lattice: its fastest axis (x or z) runs fastest
__device__ __forceinline__ uint32_t rms_cell_of(int x, int y, int z, int cx, int cy, int cz, bool zfast)
{
    const uint32_t a = (uint32_t)(x / RMS_CELL_XY), b = (uint32_t)(y / RMS_CELL_XY), c = (uint32_t)(z / RMS_CELL_Z);
    return zfast ? (a * cy + b) * cz + c : (c * cy + b) * cx + a;
}

__global__ void __launch_bounds__(256) rms_cell_hist_kernel(rms_walker_arrays st, uint64_t n, int cx, int cy, int cz, bool zfast,
                                                             uint32_t* count)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) atomicAdd(&count[rms_cell_of(st.w[0][i], st.w[1][i], st.w[2][i], cx, cy, cz, zfast)], 1u);
}

// exclusive prefix sum over the counters, in place, one block: tiles of 4096 counters (one uint4 per thread, coalesced;
// the array is padded to a multiple of 4096), scan inside the thread, warp-shuffle scan over the lanes, a second one
// over the 32 warp totals, running carry between tiles
__global__ void __launch_bounds__(1024) rms_cell_scan_kernel(uint4* count4, uint32_t n_tiles)
{
    __shared__ uint32_t wsum[32];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    uint32_t carry = 0;
    uint4 v = count4[threadIdx.x];
    for (uint32_t tile = 0; tile < n_tiles; ++tile) {
        const uint4 cur = v;
        if (tile + 1 < n_tiles) v = count4[(size_t)(tile + 1) * 1024u + threadIdx.x];   // prefetch the next tile
        const uint32_t s1 = cur.x, s2 = s1 + cur.y, s3 = s2 + cur.z, s4 = s3 + cur.w;
        uint32_t x = s4;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= (uint32_t)o) x += y;
        }
        if (lane == 31u) wsum[warp] = x;
        __syncthreads();
        if (warp == 0) {
            uint32_t t = wsum[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_up_sync(0xffffffffu, t, o);
                if (lane >= (uint32_t)o) t += y;
            }
            wsum[lane] = t;
        }
        __syncthreads();
        const uint32_t base = carry + (warp ? wsum[warp - 1] : 0u) + x - s4;
        count4[(size_t)tile * 1024u + threadIdx.x] = make_uint4(base, base + s1, base + s2, base + s3);
        carry += wsum[31];
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256) rms_cell_scatter_kernel(rms_walker_arrays st, uint64_t n, int cx, int cy, int cz, bool zfast,
                                                                uint32_t* cursor, uint32_t* order)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) order[atomicAdd(&cursor[rms_cell_of(st.w[0][i], st.w[1][i], st.w[2][i], cx, cy, cz, zfast)], 1u)] = (uint32_t)i;
}

// the same counting sort keyed on the output class of the walker's initial label (many-class signal reduction)
__global__ void __launch_bounds__(256) rms_class_hist_kernel(rms_walker_arrays st, uint64_t n, const uint16_t* __restrict__ label_class,
                                                              uint32_t* count)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) atomicAdd(&count[label_class[st.lab[i] >> 16]], 1u);
}

__global__ void __launch_bounds__(256) rms_class_scatter_kernel(rms_walker_arrays st, uint64_t n, const uint16_t* __restrict__ label_class,
                                                                 uint32_t* cursor, uint32_t* order)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) order[atomicAdd(&cursor[label_class[st.lab[i] >> 16]], 1u)] = (uint32_t)i;
}

}  // namespace

int rms_order_by_class(const rms_substrate* s, const rms_walkers* w, uint32_t* d_order, cudaStream_t stream, unsigned* n_launches)
{
    RMS_REQUIRE(w->n < (1ull << 32), RMS_ERR_UNSUPPORTED, "too many walkers to order");
    uint32_t* d_count = nullptr;
    const uint64_t n_tiles = ((uint64_t)s->n_classes + 4095) / 4096;
    RMS_CUDA_TRY(rms_malloc((void**)&d_count, n_tiles * 4096 * sizeof(uint32_t)));
    cudaError_t e = cudaMemsetAsync(d_count, 0, n_tiles * 4096 * sizeof(uint32_t), stream);
    if (e == cudaSuccess) {
        const unsigned grid = (unsigned)((w->n + 255) / 256);
        rms_class_hist_kernel<<<grid, 256, 0, stream>>>(w->a, w->n, s->d_label_class, d_count);
        rms_cell_scan_kernel<<<1, 1024, 0, stream>>>((uint4*)d_count, (uint32_t)n_tiles);
        rms_class_scatter_kernel<<<grid, 256, 0, stream>>>(w->a, w->n, s->d_label_class, d_count, d_order);
        e = cudaGetLastError();
        if (n_launches) *n_launches += 3;
    }
    rms_free_async(d_count, stream);
    RMS_CUDA_TRY(e);
    return RMS_OK;
}

int rms_order_walkers(const rms_substrate* s, const rms_walkers* w, uint32_t* d_order, cudaStream_t stream, unsigned* n_launches)
{
    const int cx = (s->nx + RMS_CELL_XY - 1) / RMS_CELL_XY, cy = (s->ny + RMS_CELL_XY - 1) / RMS_CELL_XY;
    const int cz = (s->nz + RMS_CELL_Z - 1) / RMS_CELL_Z;
    const uint64_t n_cells = (uint64_t)cx * cy * cz;
    RMS_REQUIRE(n_cells < (1ull << 31) && w->n < (1ull << 32), RMS_ERR_UNSUPPORTED, "too many cells or walkers to order");
    uint32_t* d_count = nullptr;
    const uint64_t n_tiles = (n_cells + 4095) / 4096;
    RMS_CUDA_TRY(rms_malloc((void**)&d_count, n_tiles * 4096 * sizeof(uint32_t)));
    cudaError_t e = cudaMemsetAsync(d_count, 0, n_tiles * 4096 * sizeof(uint32_t), stream);
    if (e == cudaSuccess) {
        const unsigned grid = (unsigned)((w->n + 255) / 256);
#ifdef RMS_CELL_ORDER_Z
        const bool zfast = RMS_CELL_ORDER_Z != 0;
#else
        const bool zfast = s->SZ == 1 && s->SX != 1;
#endif
        rms_cell_hist_kernel<<<grid, 256, 0, stream>>>(w->a, w->n, cx, cy, cz, zfast, d_count);
        rms_cell_scan_kernel<<<1, 1024, 0, stream>>>((uint4*)d_count, (uint32_t)n_tiles);
        rms_cell_scatter_kernel<<<grid, 256, 0, stream>>>(w->a, w->n, cx, cy, cz, zfast, d_count, d_order);
        e = cudaGetLastError();
        if (n_launches) *n_launches += 3;
    }
    // the block goes back to the cache with an event behind the kernels above
    rms_free_async(d_count, stream);
    RMS_CUDA_TRY(e);
    return RMS_OK;
}
