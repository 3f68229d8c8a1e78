// dfr_context.cu — per-device state between calls: mapped counters, events, the pinned
// staging ring (per host thread) and the private scratch pool (per process). See dfr_context.h.
#include <memory>
#include <mutex>
#include <vector>

#include "dfr_context.h"

namespace dfr {

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_pool_mu;
cudaMemPool_t g_pools[kMaxDevices] = {};

// contexts of this host thread, one per device it has used; never freed at thread exit
// (CUDA may already be gone then) — dfr_release() frees them on request
thread_local std::vector<DevCtx *> t_ctx;

cudaError_t pool_of(int dev, cudaMemPool_t *out)
{
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (!g_pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool;
        cudaError_t err = cudaMemPoolCreate(&pool, &props);
        if (err != cudaSuccess) return err;
        // keep scratch cached between calls (no OS round trip per call); dfr_release trims it
        uint64_t thr = UINT64_MAX;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
        g_pools[dev] = pool;
    }
    *out = g_pools[dev];
    return cudaSuccess;
}

void destroy_ctx(DevCtx *c)
{
    if (c->pinned) cudaFreeHost(c->pinned);
    if (c->done) cudaEventDestroy(c->done);
    if (c->prof.setup_begin) cudaEventDestroy(c->prof.setup_begin);
    if (c->prof.main_begin) cudaEventDestroy(c->prof.main_begin);
    if (c->prof.main_end) cudaEventDestroy(c->prof.main_end);
    if (c->stream_totals) cudaFree(c->stream_totals);
    for (PinnedSlot &s : c->ring) {
        if (s.copied) { cudaEventSynchronize(s.copied); cudaEventDestroy(s.copied); }
        if (s.host) cudaFreeHost(s.host);
    }
    delete c;
}

}  // namespace

cudaError_t current_ctx(DevCtx **out)
{
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    for (DevCtx *c : t_ctx)
        if (c->dev == dev) { *out = c; return cudaSuccess; }
    std::unique_ptr<DevCtx> c(new DevCtx);
    c->dev = dev;
    if ((err = cudaHostAlloc((void **)&c->pinned, 4 * sizeof(int32_t), cudaHostAllocMapped)) != cudaSuccess) return err;
    if ((err = cudaHostGetDevicePointer((void **)&c->pinned_dev, c->pinned, 0)) != cudaSuccess) {
        cudaFreeHost(c->pinned);
        return err;
    }
    if ((err = cudaEventCreateWithFlags(&c->done, cudaEventDisableTiming)) != cudaSuccess) {
        cudaFreeHost(c->pinned);
        return err;
    }
    t_ctx.push_back(c.get());
    *out = c.release();
    return cudaSuccess;
}

cudaError_t ensure_profile_events(DevCtx *c)
{
    cudaError_t err;
    ProfileEvents &p = c->prof;
    if (!p.setup_begin && (err = cudaEventCreate(&p.setup_begin)) != cudaSuccess) return err;
    if (!p.main_begin && (err = cudaEventCreate(&p.main_begin)) != cudaSuccess) return err;
    if (!p.main_end && (err = cudaEventCreate(&p.main_end)) != cudaSuccess) return err;
    return cudaSuccess;
}

cudaError_t scratch_alloc(void **p, size_t bytes, cudaStream_t st)
{
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    cudaMemPool_t pool;
    if ((err = pool_of(dev, &pool)) != cudaSuccess) return err;
    return cudaMallocFromPoolAsync(p, bytes ? bytes : 1, pool, st);
}

cudaError_t stage_acquire(DevCtx *c, size_t bytes, PinnedSlot **slot)
{
    PinnedSlot &s = c->ring[c->ring_next];
    c->ring_next = (c->ring_next + 1) % kRingSlots;
    cudaError_t err;
    if (!s.copied && (err = cudaEventCreateWithFlags(&s.copied, cudaEventDisableTiming)) != cudaSuccess) return err;
    // the upload that last used this slot (kRingSlots calls ago) has normally finished long ago
    if (s.used && (err = cudaEventSynchronize(s.copied)) != cudaSuccess) return err;
    s.used = false;
    if (s.cap < bytes) {
        if (s.host) cudaFreeHost(s.host);
        s.host = nullptr;
        s.cap = 0;
        size_t cap = 4096;
        while (cap < bytes) cap *= 2;
        if ((err = cudaHostAlloc(&s.host, cap, cudaHostAllocMapped)) != cudaSuccess) return err;
        if ((err = cudaHostGetDevicePointer(&s.dev, s.host, 0)) != cudaSuccess) {
            cudaFreeHost(s.host);
            s.host = nullptr;
            return err;
        }
        s.cap = cap;
    }
    *slot = &s;
    return cudaSuccess;
}

cudaError_t stage_done(PinnedSlot *slot, cudaStream_t st)
{
    slot->used = true;
    return cudaEventRecord(slot->copied, st);
}

void release_thread_contexts()
{
    int prev = 0;
    const bool have = cudaGetDevice(&prev) == cudaSuccess;
    for (DevCtx *c : t_ctx) {
        cudaSetDevice(c->dev);
        destroy_ctx(c);
    }
    t_ctx.clear();
    if (have) cudaSetDevice(prev);
}

void release_current_device()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return;
    cudaDeviceSynchronize();
    for (size_t k = 0; k < t_ctx.size(); ++k)
        if (t_ctx[k]->dev == dev) {
            destroy_ctx(t_ctx[k]);
            t_ctx.erase(t_ctx.begin() + (long)k);
            break;
        }
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (dev >= 0 && dev < kMaxDevices && g_pools[dev]) cudaMemPoolTrimTo(g_pools[dev], 0);
}

}  // namespace dfr
