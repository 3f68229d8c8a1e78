// dfr_context.h — state the library keeps between calls (dfr_context.cu). Everything here is
// keyed by DEVICE: a host thread may switch devices between calls, and events, mapped
// counters and scratch belong to the device they were created on.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "dfr_tiled.h"

namespace dfr {

// One slot of the pinned staging ring (per host thread and device): small host->device uploads
// of per-call constants go through pinned memory, so they never block the host on earlier
// work in the stream the way a pageable cudaMemcpyAsync above 64 KB does.
struct PinnedSlot {
    void *host = nullptr;
    void *dev = nullptr;                // the same memory as the device sees it (mapped)
    size_t cap = 0;
    cudaEvent_t copied = nullptr;       // recorded after the last upload out of this slot
    bool used = false;
};
constexpr int kRingSlots = 16;     // a host thread may run this many calls ahead of the device

// Per (host thread, device) state.
struct DevCtx {
    int dev = -1;
    int32_t *pinned = nullptr;          // 4 tile counters in mapped host memory ...
    int32_t *pinned_dev = nullptr;      // ... and the device pointer the setup kernel writes them through
    cudaEvent_t done = nullptr;         // recorded after the last call on this device
    ProfileEvents prof = {nullptr, nullptr, nullptr, false};
    int32_t *stream_totals = nullptr;   // DEVICE int[4]: tile totals of a streaming call
    PinnedSlot ring[kRingSlots];
    int ring_next = 0;
};

// The context of the calling thread for the CURRENT device (created on first use).
cudaError_t current_ctx(DevCtx **out);
// Events of dfr_profile_*: created on the context's device on first use.
cudaError_t ensure_profile_events(DevCtx *c);

// Stream-ordered scratch from the library's own memory pool of the current device (the
// application's default pool is left untouched). Free with cudaFreeAsync.
cudaError_t scratch_alloc(void **p, size_t bytes, cudaStream_t st);

// A pinned, device-mapped staging buffer of at least `bytes` whose previous use has completed.
// Fill it, enqueue the work that reads it on `st` (a cudaMemcpyAsync, or a kernel reading
// slot->dev), then call stage_done(slot, st).
cudaError_t stage_acquire(DevCtx *c, size_t bytes, PinnedSlot **slot);
cudaError_t stage_done(PinnedSlot *slot, cudaStream_t st);

// dfr_release: free what this thread keeps for the current device and trim the scratch pool.
void release_current_device();
// Free every context of the calling thread (all devices). For the library's own short-lived
// worker threads (the *_multi entry points), whose work has been synchronised: without it every
// such thread would leave its events and pinned staging memory behind.
void release_thread_contexts();

}  // namespace dfr
