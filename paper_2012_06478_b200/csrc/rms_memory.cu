// rms_memory.cu -- device memory behind the handles of include/rms.h: a small caching allocator.
//
// A pass of the hot path (rms_substrate_create -> rms_walkers_init -> rms_run -> *_destroy) allocates the
// same handful of buffers every time (the 4-byte neighbourhood lattice is the big one).  cudaMalloc /
// cudaFree take the driver's global lock, synchronise the device and cost milliseconds -- tens of
// milliseconds while anything else (a monitoring tool polling the driver) contends for that lock -- so
// freed blocks are kept, per device, and handed out again when the same size is asked for on that device.
// A block comes back either after the work that used it has completed (rms_free: the entry points of the library
// synchronise their stream before they return) or with an event recorded behind that work (rms_free_async), which
// the next owner waits for.
#include <map>
#include <mutex>

#include "rms_internal.cuh"

namespace {
struct Key {
    int dev; size_t bytes;
    bool operator<(const Key& o) const { return dev != o.dev ? dev < o.dev : bytes < o.bytes; }
};
struct Block { void* p; cudaEvent_t done; };      // done: recorded behind the last work that used the block, or null
std::mutex g_mu;
std::multimap<Key, Block> g_free;           // (device, size) -> cached block
std::map<void*, Key> g_live;                // block -> (device, size)
size_t g_cached_bytes = 0;
const size_t kMaxCachedBytes = (size_t)24 << 30;   // per process; rms_memory_trim() gives it back (invisible to other allocators)
}  // namespace

cudaError_t rms_malloc(void** p, size_t bytes)
{
    if (bytes == 0) bytes = 1;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    {
        std::unique_lock<std::mutex> lk(g_mu);
        auto it = g_free.find(Key{dev, bytes});
        if (it != g_free.end()) {
            const Block b = it->second;
            g_free.erase(it);
            g_cached_bytes -= bytes;
            g_live[b.p] = Key{dev, bytes};
            lk.unlock();
            if (b.done) {       // the block was released while work on it was still queued: wait for that work
                cudaEventSynchronize(b.done);
                cudaEventDestroy(b.done);
            }
            *p = b.p;
            return cudaSuccess;
        }
    }
    e = cudaMalloc(p, bytes);
    if (e == cudaErrorMemoryAllocation) {   // give the cache back to the driver and try once more
        cudaGetLastError();
        rms_memory_trim();
        e = cudaMalloc(p, bytes);
    }
    if (e == cudaSuccess) {
        std::lock_guard<std::mutex> lk(g_mu);
        g_live[*p] = Key{dev, bytes};
    }
    return e;
}

// release a block whose last use is work queued on `stream` (not necessarily finished): an event goes with it
void rms_free_async(void* p, cudaStream_t stream)
{
    if (!p) return;
    cudaEvent_t ev = nullptr;
    if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess || cudaEventRecord(ev, stream) != cudaSuccess) {
        if (ev) cudaEventDestroy(ev);
        cudaStreamSynchronize(stream);
        ev = nullptr;
    }
    {
        std::lock_guard<std::mutex> lk(g_mu);
        auto it = g_live.find(p);
        if (it != g_live.end()) {
            const Key k = it->second;
            g_live.erase(it);
            if (g_cached_bytes + k.bytes <= kMaxCachedBytes) {
                g_free.emplace(k, Block{p, ev});
                g_cached_bytes += k.bytes;
                return;
            }
        }
    }
    if (ev) { cudaEventSynchronize(ev); cudaEventDestroy(ev); }
    cudaFree(p);
}

// release a block whose work has completed (the caller has synchronised)
void rms_free(void* p)
{
    if (!p) return;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        auto it = g_live.find(p);
        if (it != g_live.end()) {
            const Key k = it->second;
            g_live.erase(it);
            if (g_cached_bytes + k.bytes <= kMaxCachedBytes) {
                g_free.emplace(k, Block{p, nullptr});
                g_cached_bytes += k.bytes;
                return;
            }
        }
    }
    cudaFree(p);
}

extern "C" int rms_memory_trim(void)
{
    std::multimap<Key, Block> drop;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        drop.swap(g_free);
        g_cached_bytes = 0;
    }
    for (auto& kv : drop) {
        if (kv.second.done) { cudaEventSynchronize(kv.second.done); cudaEventDestroy(kv.second.done); }
        cudaFree(kv.second.p);
    }
    return RMS_OK;
}
