// rms_memory.cu -- device memory behind the handles of include/rms.h: a small caching allocator.
//
// A pass of the hot path (rms_substrate_create -> rms_walkers_init -> rms_run -> *_destroy) allocates the
// same handful of buffers every time (the 4-byte neighbourhood lattice is the big one).  cudaMalloc /
// cudaFree take the driver's global lock, synchronise the device and cost milliseconds -- tens of
// milliseconds while anything else (a monitoring tool polling the driver) contends for that lock -- so
// freed blocks are kept and handed out again when the same size is asked for.  Blocks are only ever
// released to this cache after the work that used them has completed: every entry point of the library
// synchronises its stream before it returns.
#include <map>
#include <mutex>

#include "rms_internal.cuh"

namespace {
std::mutex g_mu;
std::multimap<size_t, void*> g_free;        // size -> cached block
std::map<void*, size_t> g_live;             // block -> size
size_t g_cached_bytes = 0;
const size_t kMaxCachedBytes = (size_t)24 << 30;
}  // namespace

cudaError_t rms_malloc(void** p, size_t bytes)
{
    if (bytes == 0) bytes = 1;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        auto it = g_free.find(bytes);
        if (it != g_free.end()) {
            *p = it->second;
            g_free.erase(it);
            g_cached_bytes -= bytes;
            g_live[*p] = bytes;
            return cudaSuccess;
        }
    }
    cudaError_t e = cudaMalloc(p, bytes);
    if (e == cudaErrorMemoryAllocation) {   // give the cache back to the driver and try once more
        cudaGetLastError();
        rms_memory_trim();
        e = cudaMalloc(p, bytes);
    }
    if (e == cudaSuccess) {
        std::lock_guard<std::mutex> lk(g_mu);
        g_live[*p] = bytes;
    }
    return e;
}

void rms_free(void* p)
{
    if (!p) return;
    size_t bytes = 0;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        auto it = g_live.find(p);
        if (it != g_live.end()) {
            bytes = it->second;
            g_live.erase(it);
            if (g_cached_bytes + bytes <= kMaxCachedBytes) {
                g_free.emplace(bytes, p);
                g_cached_bytes += bytes;
                return;
            }
        }
    }
    cudaFree(p);
}

extern "C" int rms_memory_trim(void)
{
    std::multimap<size_t, void*> drop;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        drop.swap(g_free);
        g_cached_bytes = 0;
    }
    for (auto& kv : drop) cudaFree(kv.second);
    return RMS_OK;
}
