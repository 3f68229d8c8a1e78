// dfr_api.cu — the C ABI of include/dfr.h: argument validation, host
// pre-composition, stream-ordered scratch, kernel launches. No compute happens
// on the host beyond the O(n) per-exposure constant folding of dfr_host.cu.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

#include "dfr_context.h"
#include "dfr_internal.h"
#include "dfr_tiled.h"

namespace dfr {
const char *last_error_cstr();

static int check_common(int32_t n, int32_t sny, int32_t snx, const dfr_wcs *sw, const dfr_wcs *tw,
                        int32_t ony, int32_t onx, int32_t order)
{
    if (!sw || !tw) { set_error("NULL WCS pointer"); return DFR_ERR_NULL; }
    if (n < 1 || sny < 1 || snx < 1 || ony < 1 || onx < 1 ||
        (int64_t)sny * snx >= (1LL << 31) || (int64_t)ony * onx >= (1LL << 31)) {
        set_error("bad shape: n=%d src=%dx%d out=%dx%d", n, sny, snx, ony, onx);
        return DFR_ERR_SHAPE;
    }
    if (order != DFR_NEAREST && order != DFR_BILINEAR && order != DFR_BICUBIC) {
        set_error("order %d not in {0, 1, 3}", order);
        return DFR_ERR_ORDER;
    }
    int rc = validate_wcs(tw);
    if (rc != DFR_OK) return rc;
    for (int32_t e = 0; e < n; ++e) {
        rc = validate_wcs(&sw[e]);
        if (rc != DFR_OK) return rc;
    }
    return DFR_OK;
}

static int check_weights(const float *weights, int32_t n)
{
    for (int32_t e = 0; weights && e < n; ++e)
        if (!std::isfinite(weights[e])) { set_error("weights[%d] is not finite", e); return DFR_ERR_WEIGHT; }
    return DFR_OK;
}

static bool overlaps(const void *a, size_t na, const void *b, size_t nb)
{
    const char *a0 = (const char *)a, *b0 = (const char *)b;
    return a0 < b0 + nb && b0 < a0 + na;
}

// ---- per-thread record of the last call (dfr_last_stats, dfr_profile_*) ----------------------
// The tile counters land in mapped host memory of the device the call ran on (DevCtx);
// dfr_last_stats waits for that device's `done` event.
struct LastCall {
    DevCtx *ctx = nullptr;
    bool pending = false;
    int64_t kernels = 0;
    bool tiled = false;
};
static thread_local LastCall g_last;
static thread_local bool g_profile = false;                   // dfr_profile_enable (per host thread)
static thread_local int64_t g_stats_acc[4] = {0, 0, 0, 0};    // totals of a streaming call
static thread_local bool g_accumulate = false;                // inside a streaming call

// Streaming calls (dfr_reproject_host, dfr_stack_host): the batches add their tile counters
// into one device array (no host wait between batches); harvested once at the end.
static cudaError_t stream_stats_begin(DevCtx *c)
{
    cudaError_t err;
    if (!c->stream_totals && (err = cudaMalloc((void **)&c->stream_totals, 4 * sizeof(int32_t))) != cudaSuccess) return err;
    if ((err = cudaMemset(c->stream_totals, 0, 4 * sizeof(int32_t))) != cudaSuccess) return err;
    // A device memset returns before it has run, and the pipeline's streams are non-blocking (nothing
    // orders them after the legacy stream): wait here, once per streaming call, so the setup kernels'
    // atomicAdd into stream_totals cannot land before the zeros do.
    if ((err = cudaStreamSynchronize(nullptr)) != cudaSuccess) return err;
    for (int k = 0; k < 4; ++k) g_stats_acc[k] = 0;
    g_last.pending = false;
    g_accumulate = true;
    return cudaSuccess;
}

static void stream_stats_end(DevCtx *c)
{
    g_accumulate = false;
    int32_t t[3] = {0, 0, 0};
    if (cudaMemcpy(t, c->stream_totals, sizeof t, cudaMemcpyDeviceToHost) == cudaSuccess)
        for (int k = 0; k < 3; ++k) g_stats_acc[k] = t[k];
    g_last.pending = false;
    g_last.kernels = -1;                 // marks "use the accumulated totals"
}

// ---- per-call constants -------------------------------------------------------------------
// Host constants -> one stream-ordered device block [SourceDev x n | float weights x n], staged
// through the thread's pinned ring (dfr_context.h) so the upload never blocks the host. `hsrc`
// points into a thread-local host array that the NEXT call on this thread overwrites: valid for the
// launchers of this call, which read it for the staging decision only.
struct CallConsts {
    TargetDev tgt;
    const SourceDev *hsrc = nullptr;
    SourceDev *dsrc = nullptr;
    float *dweights = nullptr;
    void *block = nullptr;
    PinnedSlot *slot = nullptr;
    ConstsCopy cc;                       // set when the tiled path's first kernel is to do the upload
    // after the call's last launch: the staging slot is free once the stream gets here
    cudaError_t finish(cudaStream_t st)
    {
        cudaError_t err = cudaSuccess;
        if (slot) err = stage_done(slot, st);
        slot = nullptr;
        if (block) cudaFreeAsync(block, st);
        block = nullptr;
        return err;
    }
};

// How the constants reach the device (ConstsCopy, dfr_tiled.h). On the tiled path (by_kernel) never
// by a copy-engine transfer in front of the kernels, and never from pageable memory (the runtime does
// not always take the bytes before returning: reusing the buffer made 2 of 8 test runs fail).
// The per-exposure constants are built in a thread-local host array (`hsrc`: the launchers read it for
// the staging decision); then either PACKED (only the coefficients the batch's highest order needs)
// into the parameters of the first setup kernel, which expands them on the device, or — batches too
// large for that — written to the thread's pinned, device-mapped ring and read from there by that
// kernel. The other paths (exact, sky) enqueue a copy from the ring.
static int tri_count(int order) { return (order + 1) * (order + 2) / 2; }

static int upload_consts(DevCtx *c, int32_t n, const dfr_wcs *sw, const dfr_wcs *tw, bool with_weights,
                         const float *weights, cudaStream_t st, bool by_kernel, CallConsts &K)
{
    make_target(tw, &K.tgt);
    const size_t b_src = sizeof(SourceDev) * (size_t)n;
    const size_t bytes = (b_src + (with_weights ? sizeof(float) * (size_t)n : 0) + 15) & ~(size_t)15;
    static thread_local std::vector<SourceDev> t_src;           // host copy (never handed to CUDA)
    if (t_src.size() < (size_t)n) t_src.resize((size_t)n);
    SourceDev *h = t_src.data();
    int maxo = 0;
    for (int32_t e = 0; e < n; ++e) {
        make_source(tw, &sw[e], &h[e]);
        maxo = std::max(maxo, std::max(h[e].ap.order, h[e].bp.order));
    }
    cudaError_t err;
    if ((err = scratch_alloc(&K.block, bytes, st)) != cudaSuccess) return cuda_fail(err, "scratch allocation (constants)");
    K.cc.dst = K.block;
    K.cc.bytes = bytes;
    const int T = tri_count(maxo), stride = kPackedHead + 2 * T;
    const size_t packed_bytes = ((size_t)n * stride * 8 + (with_weights ? 4 * (size_t)n : 0) + 15) & ~(size_t)15;
    if (by_kernel && packed_bytes <= (size_t)kPackedMaxBytes) {
        static thread_local std::vector<unsigned long long> t_pack;
        t_pack.assign(packed_bytes / 8, 0ull);
        for (int32_t e = 0; e < n; ++e) {
            unsigned long long *r = t_pack.data() + (size_t)e * stride;
            std::memcpy(r, h[e].m, 9 * 8);
            std::memcpy(r + 9, &h[e].c1, 8);
            std::memcpy(r + 10, &h[e].c2, 8);
            r[11] = (unsigned long long)(h[e].ap.order & 0xff) | ((unsigned long long)(h[e].bp.order & 0xff) << 8) |
                    ((unsigned long long)(h[e].inv_exact & 0xff) << 16);
            std::memcpy(r + kPackedHead, h[e].ap.c, (size_t)tri_count(h[e].ap.order) * 8);      // rest stays zero
            std::memcpy(r + kPackedHead + T, h[e].bp.c, (size_t)tri_count(h[e].bp.order) * 8);
        }
        if (with_weights) {
            float *hw = reinterpret_cast<float *>(t_pack.data() + (size_t)n * stride);
            for (int32_t e = 0; e < n; ++e) hw[e] = weights ? weights[e] : 1.0f;
        }
        K.cc.packed = t_pack.data();
        K.cc.packed_bytes = (int)packed_bytes;
        K.cc.n = n;
        K.cc.T = T;
        K.cc.nweights = with_weights ? n : 0;
    } else {
        if ((err = stage_acquire(c, bytes, &K.slot)) != cudaSuccess) { K.finish(st); return cuda_fail(err, "pinned staging buffer"); }
        char *stage = static_cast<char *>(K.slot->host);
        std::memcpy(stage, h, b_src);
        if (with_weights) {
            float *hw = reinterpret_cast<float *>(stage + b_src);
            for (int32_t e = 0; e < n; ++e) hw[e] = weights ? weights[e] : 1.0f;
        }
        if (by_kernel) {
            K.cc.mapped = K.slot->dev;
        } else if ((err = cudaMemcpyAsync(K.block, stage, bytes, cudaMemcpyHostToDevice, st)) != cudaSuccess) {
            K.finish(st);
            return cuda_fail(err, "cudaMemcpyAsync(constants)");
        }
    }
    K.hsrc = h;
    K.dsrc = static_cast<SourceDev *>(K.block);
    K.dweights = with_weights ? reinterpret_cast<float *>(static_cast<char *>(K.block) + b_src) : nullptr;
    return DFR_OK;
}

static bool tiled_grid_fits(int32_t ony) { return ((ony + TS * CTA_T - 1) / (TS * CTA_T)) <= 65535; }

static int reproject_impl(const float *src, int32_t n, int32_t sny, int32_t snx,
                          const dfr_wcs *sw, const dfr_wcs *tw, int32_t ony, int32_t onx,
                          int32_t order, float *out, cudaStream_t st, int32_t path, int32_t edge = DFR_EDGE_AREA,
                          float *foot = nullptr)
{
    DevCtx *c = nullptr;
    cudaError_t err = current_ctx(&c);
    if (err != cudaSuccess) return cuda_fail(err, "device context");
    if (g_profile && (err = ensure_profile_events(c)) != cudaSuccess) return cuda_fail(err, "cudaEventCreate");
    c->prof.enabled = g_profile;
    g_last.pending = false;
    g_last.ctx = c;
    // a grid taller than 65535 CTA tiles (out_ny > 4.19 M rows) does not fit the tiled launch
    const bool exact = path == DFR_PATH_EXACT || !tiled_grid_fits(ony);
    CallConsts K;
    int rc = upload_consts(c, n, sw, tw, false, nullptr, st, !exact, K);
    if (rc != DFR_OK) return rc;
    TiledStats ts = {0, 0, 0, 0};
    if (exact) {
        if (c->prof.enabled) cudaEventRecord(c->prof.setup_begin, st), cudaEventRecord(c->prof.main_begin, st);
        err = launch_exact_reproject(src, n, sny, snx, K.tgt, K.dsrc, ony, onx, order, out, st, edge, foot);
        if (c->prof.enabled) cudaEventRecord(c->prof.main_end, st);
        if (g_accumulate) {
            g_stats_acc[3] += 1;
        } else {
            g_last.kernels = 1;
            g_last.tiled = false;
        }
    } else {
        err = launch_tiled_reproject(src, n, sny, snx, K.tgt, K.dsrc, K.hsrc, ony, onx, order, out, st,
                                     g_accumulate ? c->stream_totals : c->pinned_dev, g_accumulate ? 1 : 0,
                                     &ts, &c->prof, K.cc, edge, foot);
        if (g_accumulate) {
            g_stats_acc[3] += ts.kernels;
        } else {
            if (err == cudaSuccess) err = cudaEventRecord(c->done, st);
            g_last.kernels = ts.kernels;
            g_last.tiled = true;
            g_last.pending = (err == cudaSuccess);
        }
    }
    const cudaError_t ferr = K.finish(st);
    if (err == cudaSuccess) err = ferr;
    if (err != cudaSuccess) return cuda_fail(err, "reproject launch");
    return DFR_OK;
}

// validated arguments -> constants, scratch, launches (stream-ordered)
static int stack_impl(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                      const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs, int32_t out_ny, int32_t out_nx,
                      int32_t order, const float *weights, float *sum, float *wsum, int32_t accumulate,
                      cudaStream_t st)
{
    if (!tiled_grid_fits(out_ny)) { set_error("out_ny %d is too tall for the stacking kernel", out_ny); return DFR_ERR_SHAPE; }
    DevCtx *c = nullptr;
    cudaError_t err = current_ctx(&c);
    if (err != cudaSuccess) return cuda_fail(err, "device context");
    if (g_profile && (err = ensure_profile_events(c)) != cudaSuccess) return cuda_fail(err, "cudaEventCreate");
    c->prof.enabled = g_profile;
    g_last.pending = false;
    g_last.ctx = c;
    CallConsts K;
    int rc = upload_consts(c, n, src_wcs, tgt_wcs, true, weights, st, true, K);
    if (rc != DFR_OK) return rc;
    TiledStats ts = {0, 0, 0, 0};
    err = launch_tiled_stack(src_batch, n, src_ny, src_nx, K.tgt, K.dsrc, K.hsrc, out_ny, out_nx, order,
                             K.dweights, sum, wsum, accumulate != 0, st,
                             g_accumulate ? c->stream_totals : c->pinned_dev, g_accumulate ? 1 : 0, &ts, &c->prof, K.cc);
    if (!g_accumulate && err == cudaSuccess) err = cudaEventRecord(c->done, st);
    {
        const cudaError_t ferr = K.finish(st);
        if (err == cudaSuccess) err = ferr;
    }
    if (g_accumulate) {
        g_stats_acc[3] += ts.kernels;
    } else {
        g_last.kernels = ts.kernels;
        g_last.tiled = true;
        g_last.pending = (err == cudaSuccess);
    }
    if (err != cudaSuccess) return cuda_fail(err, "reproject_stack launch");
    return DFR_OK;
}

// ---- host-buffer pipelines ----------------------------------------------
// A pipeline = kSlots (stream, device input buffer, device output buffer) triples on one device:
// H2D(b + 1) || kernels(b) || D2H(b - 1). Pipelines are kept between calls (their buffers are as
// large as the largest batch seen) in a process-wide pool; a call borrows one per shard, so
// concurrent calls, and two shards on one device, never share buffers. dfr_release frees the idle ones.
namespace {
struct Slot {
    cudaStream_t st = nullptr;
    float *din = nullptr, *dout = nullptr;
    size_t in_bytes = 0, out_bytes = 0;
};
constexpr int kSlots = 3;
struct HostPipe {
    int dev = -1;
    bool busy = false;
    Slot slot[kSlots];
};
std::mutex g_pipe_mu;
std::vector<HostPipe *> g_pipes;

HostPipe *pipe_acquire(int dev)
{
    std::lock_guard<std::mutex> lock(g_pipe_mu);
    for (HostPipe *p : g_pipes)
        if (p->dev == dev && !p->busy) { p->busy = true; return p; }
    HostPipe *p = new HostPipe;
    p->dev = dev;
    p->busy = true;
    g_pipes.push_back(p);
    return p;
}

void pipe_release(HostPipe *p)
{
    std::lock_guard<std::mutex> lock(g_pipe_mu);
    p->busy = false;
}

void pipe_free_idle(int dev)
{
    std::lock_guard<std::mutex> lock(g_pipe_mu);
    for (size_t k = 0; k < g_pipes.size();) {
        HostPipe *p = g_pipes[k];
        if (p->dev != dev || p->busy) { ++k; continue; }
        for (Slot &s : p->slot) {
            if (s.din) cudaFree(s.din);
            if (s.dout) cudaFree(s.dout);
            if (s.st) cudaStreamDestroy(s.st);
        }
        delete p;
        g_pipes.erase(g_pipes.begin() + (long)k);
    }
}

cudaError_t ensure_slot(Slot &s, size_t in_bytes, size_t out_bytes)
{
    cudaError_t err;
    if (!s.st && (err = cudaStreamCreateWithFlags(&s.st, cudaStreamNonBlocking)) != cudaSuccess) return err;
    if (s.in_bytes < in_bytes) {
        if (s.din) cudaFree(s.din);
        s.din = nullptr; s.in_bytes = 0;
        if ((err = cudaMalloc((void **)&s.din, in_bytes)) != cudaSuccess) return err;
        s.in_bytes = in_bytes;
    }
    if (s.out_bytes < out_bytes) {
        if (s.dout) cudaFree(s.dout);
        s.dout = nullptr; s.out_bytes = 0;
        if ((err = cudaMalloc((void **)&s.dout, out_bytes)) != cudaSuccess) return err;
        s.out_bytes = out_bytes;
    }
    return cudaSuccess;
}

// Borrowed pipeline of the current device with `used` slots sized for one batch.
struct PipeLease {
    HostPipe *p = nullptr;
    DevCtx *ctx = nullptr;
    int used = 0;
    ~PipeLease() { if (p) pipe_release(p); }
};

int pipe_begin(PipeLease &L, int nb, size_t in_bytes, size_t out_bytes_slot0, size_t out_bytes_other)
{
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err == cudaSuccess) err = current_ctx(&L.ctx);
    if (err != cudaSuccess) return cuda_fail(err, "device context");
    L.p = pipe_acquire(dev);
    L.used = nb < kSlots ? nb : kSlots;
    for (int k = 0; k < L.used; ++k) {
        err = ensure_slot(L.p->slot[k], in_bytes, k == 0 ? out_bytes_slot0 : out_bytes_other);
        if (err != cudaSuccess) return cuda_fail(err, "pipeline buffers");
    }
    if ((err = stream_stats_begin(L.ctx)) != cudaSuccess) return cuda_fail(err, "stream statistics");
    return DFR_OK;
}

int pipe_end(PipeLease &L, int rc)
{
    for (int k = 0; k < L.used; ++k) {
        const cudaError_t err = cudaStreamSynchronize(L.p->slot[k].st);
        if (err != cudaSuccess && rc == DFR_OK) rc = cuda_fail(err, "pipeline sync");
    }
    stream_stats_end(L.ctx);
    return rc;
}

// dfr_reproject_host on the current device (arguments validated by the caller)
int reproject_host_impl(const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                        const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs, int32_t out_ny, int32_t out_nx,
                        int32_t order, float *out_host, int32_t batch)
{
    const size_t in_px = (size_t)src_ny * src_nx, out_px = (size_t)out_ny * out_nx;
    // Batch schedule: the first upload and the last download cannot overlap anything, so the stream
    // starts and ends with small batches (1, 1, 2, ... batch ... 2, 1, 1) — measured on C2 through PCIe:
    // 12.3 -> 12.1 ms per 32 exposures (batch 4) against a 10.8 ms two-way floor.
    std::vector<int32_t> sizes;
    {
        const int32_t ramp[3] = {1, 1, 2};
        int32_t head = 0;
        for (int k = 0; k < 3; ++k) head += std::min(ramp[k], batch);
        if (batch > 2 && n >= 2 * head + batch) {
            for (int k = 0; k < 3; ++k) sizes.push_back(std::min(ramp[k], batch));
            for (int32_t left = n - 2 * head; left > 0; left -= batch) sizes.push_back(std::min(left, batch));
            for (int k = 2; k >= 0; --k) sizes.push_back(std::min(ramp[k], batch));
        } else {
            for (int32_t left = n; left > 0; left -= batch) sizes.push_back(std::min(left, batch));
        }
    }
    const int nb = (int)sizes.size();
    PipeLease L;
    int rc = pipe_begin(L, nb, in_px * batch * sizeof(float), out_px * batch * sizeof(float), out_px * batch * sizeof(float));
    if (rc != DFR_OK) return rc;
    int32_t e0 = 0;
    for (int b = 0; b < nb; ++b) {
        Slot &s = L.p->slot[b % kSlots];
        const int32_t ne = sizes[(size_t)b];
        // slot reuse is ordered by the slot's own stream: H2D(b) waits for D2H(b - kSlots)
        cudaError_t err = cudaMemcpyAsync(s.din, src_host + in_px * e0, in_px * ne * sizeof(float),
                                          cudaMemcpyHostToDevice, s.st);
        if (err != cudaSuccess) { rc = cuda_fail(err, "H2D"); break; }
        rc = reproject_impl(s.din, ne, src_ny, src_nx, src_wcs + e0, tgt_wcs, out_ny, out_nx, order,
                            s.dout, s.st, DFR_PATH_AUTO);
        if (rc != DFR_OK) break;
        err = cudaMemcpyAsync(out_host + out_px * e0, s.dout, out_px * ne * sizeof(float),
                              cudaMemcpyDeviceToHost, s.st);
        if (err != cudaSuccess) { rc = cuda_fail(err, "D2H"); break; }
        e0 += ne;
    }
    return pipe_end(L, rc);
}

// dfr_stack_host on the current device: leaves sum | wsum in the pipeline's slot-0 output buffer
// and copies them to sum_host / wsum_host unless `keep` is given (then *keep receives the device
// pointer, valid until the lease `L` ends — the multi-device form reduces there).
int stack_host_impl(PipeLease &L, const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                    const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs, int32_t out_ny, int32_t out_nx,
                    int32_t order, const float *weights, float *sum_host, float *wsum_host, int32_t batch,
                    float **keep)
{
    const size_t in_px = (size_t)src_ny * src_nx, out_bytes = sizeof(float) * (size_t)out_ny * out_nx;
    const int nb = (n + batch - 1) / batch;
    // slot 0's output buffer holds sum and wsum; every slot needs an input buffer and a stream
    int rc = pipe_begin(L, nb, in_px * batch * sizeof(float), 2 * out_bytes, 0);
    if (rc != DFR_OK) return rc;
    float *dsum = L.p->slot[0].dout, *dwsum = dsum + (size_t)out_ny * out_nx;
    // `turn`: the stacking kernels add into sum / wsum with plain read-modify-writes (one owner per
    // pixel), so batch b's kernels wait for batch b - 1's; the uploads, which are what the pipeline
    // exists for, still overlap them. The first batch overwrites (no memset).
    cudaEvent_t turn = nullptr;
    cudaError_t err = cudaEventCreateWithFlags(&turn, cudaEventDisableTiming);
    if (err != cudaSuccess) rc = cuda_fail(err, "pipeline start");
    for (int b = 0; b < nb && rc == DFR_OK; ++b) {
        Slot &s = L.p->slot[b % kSlots];
        const int32_t e0 = b * batch, ne = (n - e0 < batch) ? n - e0 : batch;
        // the slot's stream orders its own reuse: H2D(b) waits for the kernels of b - kSlots
        err = cudaMemcpyAsync(s.din, src_host + in_px * e0, in_px * ne * sizeof(float), cudaMemcpyHostToDevice, s.st);
        if (err == cudaSuccess && b > 0) err = cudaStreamWaitEvent(s.st, turn, 0);
        if (err != cudaSuccess) { rc = cuda_fail(err, "H2D"); break; }
        rc = stack_impl(s.din, ne, src_ny, src_nx, src_wcs + e0, tgt_wcs, out_ny, out_nx, order,
                        weights ? weights + e0 : nullptr, dsum, dwsum, b > 0 ? 1 : 0, s.st);
        if (rc == DFR_OK && (err = cudaEventRecord(turn, s.st)) != cudaSuccess) rc = cuda_fail(err, "pipeline order");
    }
    rc = pipe_end(L, rc);
    if (turn) cudaEventDestroy(turn);
    if (rc != DFR_OK) return rc;
    if (keep) { *keep = dsum; return DFR_OK; }
    err = cudaMemcpy(sum_host, dsum, out_bytes, cudaMemcpyDeviceToHost);
    if (err == cudaSuccess) err = cudaMemcpy(wsum_host, dwsum, out_bytes, cudaMemcpyDeviceToHost);
    return err == cudaSuccess ? DFR_OK : cuda_fail(err, "D2H");
}

// Contiguous shard k of n exposures over `parts` shards: the first n % parts shards get one more.
void shard_range(int32_t n, int parts, int k, int32_t *lo, int32_t *hi)
{
    const int32_t q = n / parts, r = n % parts;
    *lo = k * q + std::min(k, (int)r);
    *hi = *lo + q + (k < r ? 1 : 0);
}

int check_devices(const int32_t *devices, int32_t ndev)
{
    if (!devices) { set_error("NULL device list"); return DFR_ERR_NULL; }
    if (ndev < 1 || ndev > 64) { set_error("ndev = %d outside [1, 64]", ndev); return DFR_ERR_SHAPE; }
    int count = 0;
    const cudaError_t err = cudaGetDeviceCount(&count);
    if (err != cudaSuccess) return cuda_fail(err, "cudaGetDeviceCount");
    for (int k = 0; k < ndev; ++k)
        if (devices[k] < 0 || devices[k] >= count) {
            set_error("devices[%d] = %d, but %d CUDA device(s) are visible", k, devices[k], count);
            return DFR_ERR_SHAPE;
        }
    return DFR_OK;
}

struct ShardResult {
    int rc = DFR_OK;
    std::string error;
    int64_t stats[4] = {0, 0, 0, 0};
};
}  // namespace
}  // namespace dfr

using namespace dfr;

extern "C" {

int dfr_reproject_fp(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                     const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                     int32_t out_ny, int32_t out_nx, int32_t order, int32_t edge_mode,
                     float *out, float *footprint, void *stream)
{
    if (!src_batch || !out) { set_error("NULL image pointer"); return DFR_ERR_NULL; }
    int rc = check_common(n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order);
    if (rc != DFR_OK) return rc;
    if (edge_mode != DFR_EDGE_AREA && edge_mode != DFR_EDGE_PAPER) {
        set_error("unknown edge mode %d", edge_mode);
        return DFR_ERR_ORDER;
    }
    if (edge_mode == DFR_EDGE_PAPER && order == DFR_BICUBIC) {
        set_error("the paper's footprint normalisation is not defined for bicubic interpolation");
        return DFR_ERR_ORDER;
    }
    const size_t sb = sizeof(float) * (size_t)n * src_ny * src_nx, ob = sizeof(float) * (size_t)n * out_ny * out_nx;
    if (overlaps(out, ob, src_batch, sb)) { set_error("out overlaps src_batch"); return DFR_ERR_ALIAS; }
    if (footprint && (overlaps(footprint, ob, src_batch, sb) || overlaps(footprint, ob, out, ob))) {
        set_error("footprint overlaps src_batch or out");
        return DFR_ERR_ALIAS;
    }
    // nearest: the zero-padded identity is 1 exactly on the area footprint
    const int32_t edge = (order == DFR_NEAREST) ? DFR_EDGE_AREA : edge_mode;
    return reproject_impl(src_batch, n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order,
                          out, (cudaStream_t)stream, DFR_PATH_AUTO, edge, footprint);
}

int dfr_reproject_edge(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                       const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                       int32_t out_ny, int32_t out_nx, int32_t order, int32_t edge_mode,
                       float *out, void *stream)
{
    return dfr_reproject_fp(src_batch, n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order, edge_mode,
                            out, nullptr, stream);
}

int dfr_reproject_ex(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                     const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                     int32_t out_ny, int32_t out_nx, int32_t order,
                     float *out, void *stream, int32_t path)
{
    if (!src_batch || !out) { set_error("NULL image pointer"); return DFR_ERR_NULL; }
    int rc = check_common(n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order);
    if (rc != DFR_OK) return rc;
    if (path != DFR_PATH_AUTO && path != DFR_PATH_EXACT && path != DFR_PATH_TILED) {
        set_error("unknown path %d", path);
        return DFR_ERR_ORDER;
    }
    if (overlaps(out, sizeof(float) * (size_t)n * out_ny * out_nx, src_batch, sizeof(float) * (size_t)n * src_ny * src_nx)) {
        set_error("out overlaps src_batch");
        return DFR_ERR_ALIAS;
    }
    return reproject_impl(src_batch, n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order,
                          out, (cudaStream_t)stream, path);
}

int dfr_reproject(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                  const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                  int32_t out_ny, int32_t out_nx, int32_t order, float *out, void *stream)
{
    return dfr_reproject_ex(src_batch, n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order,
                            out, stream, DFR_PATH_AUTO);
}

int dfr_src_coords(int32_t n, int32_t src_ny, int32_t src_nx,
                   const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                   int32_t out_ny, int32_t out_nx, int32_t order,
                   double *x, double *y, void *stream, int32_t path)
{
    if (!x || !y) { set_error("NULL coordinate pointer"); return DFR_ERR_NULL; }
    int rc = check_common(n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order);
    if (rc != DFR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    DevCtx *c = nullptr;
    cudaError_t err = current_ctx(&c);
    if (err != cudaSuccess) return cuda_fail(err, "device context");
    const bool exact = path == DFR_PATH_EXACT || !tiled_grid_fits(out_ny);
    CallConsts K;
    rc = upload_consts(c, n, src_wcs, tgt_wcs, false, nullptr, st, !exact, K);
    if (rc != DFR_OK) return rc;
    if (exact)
        err = launch_exact_coords(n, K.tgt, K.dsrc, out_ny, out_nx, x, y, st);
    else
        err = launch_tiled_coords(n, src_ny, src_nx, K.tgt, K.dsrc, K.hsrc, out_ny, out_nx, order, x, y, st, K.cc);
    {
        const cudaError_t ferr = K.finish(st);
        if (err == cudaSuccess) err = ferr;
    }
    if (err != cudaSuccess) return cuda_fail(err, "src_coords launch");
    return DFR_OK;
}

int dfr_reproject_stack(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                        const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                        int32_t out_ny, int32_t out_nx, int32_t order,
                        const float *weights, float *sum, float *wsum, int32_t accumulate,
                        void *stream)
{
    if (!src_batch || !sum || !wsum) { set_error("NULL image pointer"); return DFR_ERR_NULL; }
    int rc = check_common(n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order);
    if (rc != DFR_OK) return rc;
    const size_t sb = sizeof(float) * (size_t)n * src_ny * src_nx, ob = sizeof(float) * (size_t)out_ny * out_nx;
    if (overlaps(sum, ob, src_batch, sb) || overlaps(wsum, ob, src_batch, sb) || overlaps(sum, ob, wsum, ob)) {
        set_error("sum / wsum overlap src_batch or each other");
        return DFR_ERR_ALIAS;
    }
    if ((rc = check_weights(weights, n)) != DFR_OK) return rc;
    return stack_impl(src_batch, n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order, weights, sum, wsum,
                      accumulate, (cudaStream_t)stream);
}

int dfr_stack_finalize(const float *sum, const float *wsum, int64_t npix, float *mean, void *stream)
{
    if (npix < 0) { set_error("npix < 0"); return DFR_ERR_SHAPE; }
    if (npix > 0 && (!sum || !wsum || !mean)) { set_error("NULL pointer"); return DFR_ERR_NULL; }
    cudaError_t err = launch_stack_finalize(sum, wsum, (long long)npix, mean, (cudaStream_t)stream);
    return err == cudaSuccess ? DFR_OK : cuda_fail(err, "stack_finalize launch");
}

static int sky_common(const dfr_wcs *w, const void *a, const void *b, const void *c, const void *d,
                      int64_t npts, cudaStream_t st, SkyDev **dev)
{
    if (npts < 0) { set_error("npts < 0"); return DFR_ERR_SHAPE; }
    if (!w || (npts > 0 && (!a || !b || !c || !d))) { set_error("NULL pointer"); return DFR_ERR_NULL; }
    int rc = validate_wcs(w);
    if (rc != DFR_OK) return rc;
    DevCtx *ctx = nullptr;
    cudaError_t err = current_ctx(&ctx);
    if (err != cudaSuccess) return cuda_fail(err, "device context");
    PinnedSlot *slot = nullptr;
    if ((err = stage_acquire(ctx, sizeof(SkyDev), &slot)) != cudaSuccess) return cuda_fail(err, "pinned staging buffer");
    make_sky(w, static_cast<SkyDev *>(slot->host));
    if ((err = scratch_alloc((void **)dev, sizeof(SkyDev), st)) != cudaSuccess) return cuda_fail(err, "scratch allocation (sky)");
    err = cudaMemcpyAsync(*dev, slot->host, sizeof(SkyDev), cudaMemcpyHostToDevice, st);
    if (err == cudaSuccess) err = stage_done(slot, st);
    if (err != cudaSuccess) { cudaFreeAsync(*dev, st); return cuda_fail(err, "cudaMemcpyAsync(sky)"); }
    return DFR_OK;
}

int dfr_pix2world(const dfr_wcs *w, const double *x, const double *y, int64_t npts,
                  double *ra_deg, double *dec_deg, void *stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    SkyDev *d = nullptr;
    int rc = sky_common(w, x, y, ra_deg, dec_deg, npts, st, &d);
    if (rc != DFR_OK) return rc;
    cudaError_t err = launch_pix2world(d, x, y, npts, ra_deg, dec_deg, st);
    cudaFreeAsync(d, st);
    return err == cudaSuccess ? DFR_OK : cuda_fail(err, "pix2world launch");
}

int dfr_world2pix(const dfr_wcs *w, const double *ra_deg, const double *dec_deg, int64_t npts,
                  double *x, double *y, void *stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    SkyDev *d = nullptr;
    int rc = sky_common(w, ra_deg, dec_deg, x, y, npts, st, &d);
    if (rc != DFR_OK) return rc;
    cudaError_t err = launch_world2pix(d, ra_deg, dec_deg, npts, x, y, st);
    cudaFreeAsync(d, st);
    return err == cudaSuccess ? DFR_OK : cuda_fail(err, "world2pix launch");
}

// ---- end-to-end streaming forms ------------------------------------
int dfr_reproject_host(const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                       const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                       int32_t out_ny, int32_t out_nx, int32_t order,
                       float *out_host, int32_t batch)
{
    if (!src_host || !out_host) { set_error("NULL image pointer"); return DFR_ERR_NULL; }
    int rc = check_common(n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order);
    if (rc != DFR_OK) return rc;
    if (batch <= 0) batch = 32;
    if (batch > n) batch = n;
    return reproject_host_impl(src_host, n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order, out_host, batch);
}

int dfr_stack_host(const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                   const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                   int32_t out_ny, int32_t out_nx, int32_t order, const float *weights,
                   float *sum_host, float *wsum_host, int32_t batch)
{
    if (!src_host || !sum_host || !wsum_host) { set_error("NULL image pointer"); return DFR_ERR_NULL; }
    int rc = check_common(n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order);
    if (rc != DFR_OK) return rc;
    if ((rc = check_weights(weights, n)) != DFR_OK) return rc;
    if (batch <= 0) batch = 32;
    if (batch > n) batch = n;
    PipeLease L;
    return stack_host_impl(L, src_host, n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order, weights,
                           sum_host, wsum_host, batch, nullptr);
}

int dfr_shard_range(int32_t n, int32_t parts, int32_t k, int32_t *lo, int32_t *hi)
{
    if (!lo || !hi) { set_error("NULL pointer"); return DFR_ERR_NULL; }
    if (n < 0 || parts < 1 || k < 0 || k >= parts) {
        set_error("bad shard request n=%d parts=%d k=%d", n, parts, k);
        return DFR_ERR_SHAPE;
    }
    shard_range(n, parts, k, lo, hi);
    return DFR_OK;
}

int dfr_reproject_host_multi(const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                             const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                             int32_t out_ny, int32_t out_nx, int32_t order,
                             float *out_host, int32_t batch, const int32_t *devices, int32_t ndev)
{
    if (!src_host || !out_host) { set_error("NULL image pointer"); return DFR_ERR_NULL; }
    int rc = check_common(n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order);
    if (rc != DFR_OK) return rc;
    if ((rc = check_devices(devices, ndev)) != DFR_OK) return rc;
    if (batch <= 0) batch = 32;
    const size_t in_px = (size_t)src_ny * src_nx, out_px = (size_t)out_ny * out_nx;
    std::vector<ShardResult> res((size_t)ndev);
    std::vector<std::thread> workers;
    // exposures are independent: contiguous shards, one host thread and one
    // pipeline per shard, no collective
    for (int k = 0; k < ndev; ++k)
        workers.emplace_back([&, k]() {
            ShardResult &r = res[(size_t)k];
            int32_t lo, hi;
            shard_range(n, ndev, k, &lo, &hi);
            if (hi <= lo) return;
            const cudaError_t err = cudaSetDevice(devices[k]);
            if (err != cudaSuccess) { r.rc = cuda_fail(err, "cudaSetDevice"); r.error = last_error_cstr(); return; }
            r.rc = reproject_host_impl(src_host + in_px * lo, hi - lo, src_ny, src_nx, src_wcs + lo, tgt_wcs, out_ny, out_nx,
                                       order, out_host + out_px * lo, std::min(batch, hi - lo));
            if (r.rc != DFR_OK) r.error = last_error_cstr();
            for (int q = 0; q < 4; ++q) r.stats[q] = g_stats_acc[q];
            g_last = LastCall();
            release_thread_contexts();              // this thread ends here: nothing of it may stay behind
        });
    for (std::thread &t : workers) t.join();
    for (int q = 0; q < 4; ++q) g_stats_acc[q] = 0;
    for (const ShardResult &r : res) {
        if (r.rc != DFR_OK && rc == DFR_OK) { rc = r.rc; set_error("%s", r.error.c_str()); }
        for (int q = 0; q < 4; ++q) g_stats_acc[q] += r.stats[q];
    }
    g_last.pending = false;
    g_last.kernels = -1;
    return rc;
}

int dfr_stack_host_multi(const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                         const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                         int32_t out_ny, int32_t out_nx, int32_t order, const float *weights,
                         float *sum_host, float *wsum_host, int32_t batch, const int32_t *devices, int32_t ndev)
{
    if (!src_host || !sum_host || !wsum_host) { set_error("NULL image pointer"); return DFR_ERR_NULL; }
    int rc = check_common(n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order);
    if (rc != DFR_OK) return rc;
    if ((rc = check_weights(weights, n)) != DFR_OK) return rc;
    if ((rc = check_devices(devices, ndev)) != DFR_OK) return rc;
    if (batch <= 0) batch = 32;
    const size_t in_px = (size_t)src_ny * src_nx, npix = (size_t)out_ny * out_nx;
    std::vector<ShardResult> res((size_t)ndev);
    std::vector<PipeLease> lease((size_t)ndev);
    std::vector<float *> partial((size_t)ndev, nullptr);
    std::vector<std::thread> workers;
    for (int k = 0; k < ndev; ++k)
        workers.emplace_back([&, k]() {
            ShardResult &r = res[(size_t)k];
            int32_t lo, hi;
            shard_range(n, ndev, k, &lo, &hi);
            if (hi <= lo) return;
            const cudaError_t err = cudaSetDevice(devices[k]);
            if (err != cudaSuccess) { r.rc = cuda_fail(err, "cudaSetDevice"); r.error = last_error_cstr(); return; }
            r.rc = stack_host_impl(lease[(size_t)k], src_host + in_px * lo, hi - lo, src_ny, src_nx, src_wcs + lo, tgt_wcs,
                                   out_ny, out_nx, order, weights ? weights + lo : nullptr, nullptr, nullptr,
                                   std::min(batch, hi - lo), &partial[(size_t)k]);
            if (r.rc != DFR_OK) r.error = last_error_cstr();
            for (int q = 0; q < 4; ++q) r.stats[q] = g_stats_acc[q];
            g_last = LastCall();
            release_thread_contexts();              // this thread ends here: nothing of it may stay behind
        });
    for (std::thread &t : workers) t.join();
    for (int q = 0; q < 4; ++q) g_stats_acc[q] = 0;
    for (const ShardResult &r : res) {
        if (r.rc != DFR_OK && rc == DFR_OK) { rc = r.rc; set_error("%s", r.error.c_str()); }
        for (int q = 0; q < 4; ++q) g_stats_acc[q] += r.stats[q];
    }
    g_last.pending = false;
    g_last.kernels = -1;
    if (rc != DFR_OK) return rc;
    // the one exchange step of the stack: the shards' partial sum | wsum pairs are
    // copied to the first shard's device (peer copy) and added there, in shard order
    int first = -1;
    for (int k = 0; k < ndev; ++k)
        if (partial[(size_t)k]) { first = k; break; }
    if (first < 0) { set_error("no exposures"); return DFR_ERR_SHAPE; }
    int prev = 0;
    cudaGetDevice(&prev);
    cudaError_t err = cudaSetDevice(devices[first]);
    float *tmp = nullptr;
    if (err == cudaSuccess) err = cudaMalloc((void **)&tmp, 2 * npix * sizeof(float));
    for (int k = first + 1; k < ndev && err == cudaSuccess; ++k) {
        if (!partial[(size_t)k]) continue;
        err = cudaMemcpyPeer(tmp, devices[first], partial[(size_t)k], devices[k], 2 * npix * sizeof(float));
        if (err == cudaSuccess) err = launch_stack_add(partial[(size_t)first], tmp, (long long)(2 * npix), nullptr);
        if (err == cudaSuccess) err = cudaStreamSynchronize(nullptr);
    }
    if (err == cudaSuccess) err = cudaMemcpy(sum_host, partial[(size_t)first], npix * sizeof(float), cudaMemcpyDeviceToHost);
    if (err == cudaSuccess) err = cudaMemcpy(wsum_host, partial[(size_t)first] + npix, npix * sizeof(float), cudaMemcpyDeviceToHost);
    if (tmp) cudaFree(tmp);
    cudaSetDevice(prev);
    return err == cudaSuccess ? DFR_OK : cuda_fail(err, "multi-device stack reduction");
}

int dfr_wcs_set_pc_cdelt(dfr_wcs *w, const double pc[4], const double cdelt[2])
{
    if (!w || !pc || !cdelt) { set_error("NULL pointer"); return DFR_ERR_NULL; }
    w->cd[0] = cdelt[0] * pc[0];
    w->cd[1] = cdelt[0] * pc[1];
    w->cd[2] = cdelt[1] * pc[2];
    w->cd[3] = cdelt[1] * pc[3];
    return DFR_OK;
}

int dfr_wcs_fit_inverse_sip(dfr_wcs *w, int32_t order, int32_t nx, int32_t ny, double *max_resid_px)
{
    if (!w) { set_error("NULL pointer"); return DFR_ERR_NULL; }
    if (order < 1 || order > DFR_SIP_MAX_ORDER) {
        set_error("inverse SIP order %d outside [1, %d]", order, DFR_SIP_MAX_ORDER);
        return DFR_ERR_SIP_ORDER;
    }
    if (nx < 1 || ny < 1) { set_error("bad image shape %dx%d", ny, nx); return DFR_ERR_SHAPE; }
    dfr_wcs probe = *w;
    probe.ap_order = probe.bp_order = 0;          // only the forward side has to be valid
    const int rc = validate_wcs(&probe);
    if (rc != DFR_OK) return rc;
    return fit_inverse_sip(w, order, nx, ny, max_resid_px);
}

int dfr_last_stats(int64_t stats[4])
{
    if (!stats) return DFR_ERR_NULL;
    if (g_last.kernels == -1) {
        for (int k = 0; k < 4; ++k) stats[k] = g_stats_acc[k];
        return DFR_OK;
    }
    stats[0] = stats[1] = stats[2] = 0;
    stats[3] = g_last.kernels;
    if (g_last.tiled && g_last.pending && g_last.ctx) {
        cudaEventSynchronize(g_last.ctx->done);
        for (int k = 0; k < 3; ++k) stats[k] = g_last.ctx->pinned[k];
    } else if (!g_last.tiled) {
        stats[1] = -1;                                        // exact path: no tiles
    }
    return DFR_OK;
}

int dfr_profile_enable(int on)
{
    g_profile = on != 0;
    return DFR_OK;
}

int dfr_profile_last(float ms[2])
{
    if (!ms) return DFR_ERR_NULL;
    DevCtx *c = g_last.ctx;
    if (!g_profile || !c || !c->prof.main_end) { set_error("profiling is not enabled"); return DFR_ERR_ORDER; }
    cudaError_t err = cudaEventSynchronize(c->prof.main_end);
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms[0], c->prof.setup_begin, c->prof.main_begin);
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms[1], c->prof.main_begin, c->prof.main_end);
    return err == cudaSuccess ? DFR_OK : cuda_fail(err, "profile events");
}

int dfr_release(void)
{
    int dev = 0;
    const cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return cuda_fail(err, "cudaGetDevice");
    if (g_last.ctx && g_last.ctx->dev == dev) g_last = LastCall();
    release_current_device();
    pipe_free_idle(dev);
    return DFR_OK;
}

const char *dfr_strerror(int code)
{
    switch (code) {
    case DFR_OK: return "ok";
    case DFR_ERR_NULL: return "null pointer";
    case DFR_ERR_SHAPE: return "bad shape";
    case DFR_ERR_ORDER: return "bad interpolation order or path";
    case DFR_ERR_SIP_ORDER: return "SIP order out of range";
    case DFR_ERR_SINGULAR_CD: return "singular CD matrix";
    case DFR_ERR_NONFINITE_WCS: return "non-finite WCS field";
    case DFR_ERR_ALIAS: return "output aliases input";
    case DFR_ERR_CUDA: return "CUDA failure";
    case DFR_ERR_WEIGHT: return "non-finite stacking weight";
    default: return "unknown error";
    }
}

const char *dfr_last_error(void) { return dfr::last_error_cstr(); }

int dfr_version(void) { return 200; }

}  // extern "C"
