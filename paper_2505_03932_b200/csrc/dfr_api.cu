// dfr_api.cu — the C ABI of include/dfr.h: argument validation, host
// pre-composition, stream-ordered scratch, kernel launches. No compute happens
// on the host beyond the O(n) per-exposure constant folding of dfr_host.cu.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "dfr_internal.h"
#include "dfr_tiled.h"

namespace dfr {
const char *last_error_cstr();

static std::once_flag g_pool_once;
static void tune_pool()
{
    // keep stream-ordered scratch cached between calls (no OS round trip per call)
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return;
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, dev) != cudaSuccess) return;
    uint64_t thr = UINT64_MAX;
    cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
}

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

// Per-thread record of the last call: tile counters land in pinned host memory through an
// async copy; dfr_last_stats waits for it. Also the optional timing events (dfr_profile_*).
struct LastCall {
    int32_t *pinned = nullptr;          // 3 counters: fast, exact, empty (mapped host memory,
    int32_t *pinned_dev = nullptr;      // written by the setup kernel through this device pointer)
    cudaEvent_t done = nullptr;
    bool pending = false;
    int64_t kernels = 0;
    bool tiled = false;
    ProfileEvents prof = {nullptr, nullptr, nullptr, false};
};
static thread_local LastCall g_last;
static thread_local int64_t g_stats_acc[4] = {0, 0, 0, 0};   // used by dfr_reproject_host
static thread_local bool g_accumulate = false;
static thread_local int32_t *g_stream_totals = nullptr;      // DEVICE int[3]: tile totals of a streaming call

// Streaming calls (dfr_reproject_host, dfr_stack_host): the batches add their tile counters
// into one device array (no host wait between batches); harvested once at the end.
static cudaError_t stream_stats_begin()
{
    cudaError_t err;
    if (!g_stream_totals && (err = cudaMalloc((void **)&g_stream_totals, 4 * sizeof(int32_t))) != cudaSuccess) return err;
    if ((err = cudaMemset(g_stream_totals, 0, 4 * sizeof(int32_t))) != cudaSuccess) return err;
    for (int k = 0; k < 4; ++k) g_stats_acc[k] = 0;
    g_last.pending = false;
    g_accumulate = true;
    return cudaSuccess;
}

static void stream_stats_end()
{
    g_accumulate = false;
    int32_t t[3] = {0, 0, 0};
    if (cudaMemcpy(t, g_stream_totals, sizeof t, cudaMemcpyDeviceToHost) == cudaSuccess)
        for (int k = 0; k < 3; ++k) g_stats_acc[k] = t[k];
    g_last.pending = false;
    g_last.kernels = -1;                 // marks "use the accumulated totals"
}

static int stack_impl(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                      const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs, int32_t out_ny, int32_t out_nx,
                      int32_t order, const float *weights, float *sum, float *wsum, int32_t accumulate,
                      cudaStream_t st);

static cudaError_t ensure_last()
{
    cudaError_t err;
    if (!g_last.pinned) {
        if ((err = cudaHostAlloc((void **)&g_last.pinned, 4 * sizeof(int32_t), cudaHostAllocMapped)) != cudaSuccess) return err;
        if ((err = cudaHostGetDevicePointer((void **)&g_last.pinned_dev, g_last.pinned, 0)) != cudaSuccess) return err;
    }
    if (!g_last.done && (err = cudaEventCreateWithFlags(&g_last.done, cudaEventDisableTiming)) != cudaSuccess) return err;
    return cudaSuccess;
}

static void collect_stats(int64_t out[4])
{
    out[0] = out[1] = out[2] = 0;
    out[3] = g_last.kernels;
    if (g_last.tiled && g_last.pending) {
        cudaEventSynchronize(g_last.done);
        out[0] = g_last.pinned[0];
        out[1] = g_last.pinned[1];
        out[2] = g_last.pinned[2];
    } else if (!g_last.tiled) {
        out[1] = -1;                                          // exact path: no tiles
    }
}

// Host constants -> device scratch (stream-ordered). Caller frees with cudaFreeAsync.
static int upload_sources(int32_t n, const dfr_wcs *sw, const dfr_wcs *tw, cudaStream_t st,
                          std::vector<SourceDev> &h, SourceDev **dev_out)
{
    h.resize((size_t)n);
    for (int32_t e = 0; e < n; ++e) make_source(tw, &sw[e], &h[e]);
    SourceDev *d = nullptr;
    cudaError_t err = cudaMallocAsync((void **)&d, sizeof(SourceDev) * (size_t)n, st);
    if (err != cudaSuccess) return cuda_fail(err, "cudaMallocAsync(sources)");
    // pageable source: the runtime stages the bytes before returning, so `h` may die
    err = cudaMemcpyAsync(d, h.data(), sizeof(SourceDev) * (size_t)n, cudaMemcpyHostToDevice, st);
    if (err != cudaSuccess) { cudaFreeAsync(d, st); return cuda_fail(err, "cudaMemcpyAsync(sources)"); }
    *dev_out = d;
    return DFR_OK;
}

static int reproject_impl(const float *src, int32_t n, int32_t sny, int32_t snx,
                          const dfr_wcs *sw, const dfr_wcs *tw, int32_t ony, int32_t onx,
                          int32_t order, float *out, cudaStream_t st, int32_t path, int32_t edge = DFR_EDGE_AREA)
{
    std::call_once(g_pool_once, tune_pool);
    g_last.pending = false;
    TargetDev tgt;
    make_target(tw, &tgt);
    std::vector<SourceDev> hsrc;
    SourceDev *dsrc = nullptr;
    int rc = upload_sources(n, sw, tw, st, hsrc, &dsrc);
    if (rc != DFR_OK) return rc;
    cudaError_t err;
    TiledStats ts = {0, 0, 0, 0};
    if (path == DFR_PATH_EXACT) {
        if (g_last.prof.enabled) cudaEventRecord(g_last.prof.setup_begin, st), cudaEventRecord(g_last.prof.main_begin, st);
        err = launch_exact_reproject(src, n, sny, snx, tgt, dsrc, ony, onx, order, out, st, edge);
        if (g_last.prof.enabled) cudaEventRecord(g_last.prof.main_end, st);
        g_last.kernels = 1;
        g_last.tiled = false;
    } else {
        err = ensure_last();
        if (err == cudaSuccess)
            err = launch_tiled_reproject(src, n, sny, snx, tgt, dsrc, hsrc.data(), ony, onx, order, out, st,
                                         g_accumulate ? g_stream_totals : g_last.pinned_dev, g_accumulate ? 1 : 0,
                                         &ts, &g_last.prof, edge);
        if (g_accumulate) {
            g_stats_acc[3] += ts.kernels;
        } else {
            if (err == cudaSuccess) err = cudaEventRecord(g_last.done, st);
            g_last.kernels = ts.kernels;
            g_last.tiled = true;
            g_last.pending = (err == cudaSuccess);
        }
    }
    cudaFreeAsync(dsrc, st);
    if (err != cudaSuccess) return cuda_fail(err, "reproject launch");
    return DFR_OK;
}

}  // namespace dfr

using namespace dfr;

extern "C" {

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
    const char *s0 = (const char *)src_batch, *s1 = s0 + sizeof(float) * (size_t)n * src_ny * src_nx;
    const char *o0 = (const char *)out, *o1 = o0 + sizeof(float) * (size_t)n * out_ny * out_nx;
    if (o0 < s1 && s0 < o1) { set_error("out overlaps src_batch"); return DFR_ERR_ALIAS; }
    return reproject_impl(src_batch, n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order,
                          out, (cudaStream_t)stream, path);
}

int dfr_reproject_edge(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                       const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                       int32_t out_ny, int32_t out_nx, int32_t order, int32_t edge_mode,
                       float *out, void *stream)
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
    const char *s0 = (const char *)src_batch, *s1 = s0 + sizeof(float) * (size_t)n * src_ny * src_nx;
    const char *o0 = (const char *)out, *o1 = o0 + sizeof(float) * (size_t)n * out_ny * out_nx;
    if (o0 < s1 && s0 < o1) { set_error("out overlaps src_batch"); return DFR_ERR_ALIAS; }
    // nearest: the zero-padded identity is 1 exactly on the area footprint
    const int32_t edge = (order == DFR_NEAREST) ? DFR_EDGE_AREA : edge_mode;
    return reproject_impl(src_batch, n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order,
                          out, (cudaStream_t)stream, DFR_PATH_AUTO, edge);
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
    std::call_once(g_pool_once, tune_pool);
    cudaStream_t st = (cudaStream_t)stream;
    TargetDev tgt;
    make_target(tgt_wcs, &tgt);
    SourceDev *dsrc = nullptr;
    std::vector<SourceDev> hsrc;
    rc = upload_sources(n, src_wcs, tgt_wcs, st, hsrc, &dsrc);
    if (rc != DFR_OK) return rc;
    cudaError_t err;
    if (path == DFR_PATH_EXACT)
        err = launch_exact_coords(n, tgt, dsrc, out_ny, out_nx, x, y, st);
    else
        err = launch_tiled_coords(n, src_ny, src_nx, tgt, dsrc, hsrc.data(), out_ny, out_nx, order, x, y, st);
    cudaFreeAsync(dsrc, st);
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
    const char *s0 = (const char *)src_batch, *s1 = s0 + sizeof(float) * (size_t)n * src_ny * src_nx;
    const size_t ob = sizeof(float) * (size_t)out_ny * out_nx;
    const char *a0 = (const char *)sum, *b0 = (const char *)wsum;
    if ((a0 < s1 && s0 < a0 + ob) || (b0 < s1 && s0 < b0 + ob) || (a0 < b0 + ob && b0 < a0 + ob)) {
        set_error("sum / wsum overlap src_batch or each other");
        return DFR_ERR_ALIAS;
    }
    for (int32_t e = 0; weights && e < n; ++e)
        if (!std::isfinite(weights[e])) { set_error("weights[%d] is not finite", e); return DFR_ERR_NONFINITE_WCS; }
    return stack_impl(src_batch, n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order, weights, sum, wsum,
                      accumulate, (cudaStream_t)stream);
}

}  // extern "C"

namespace dfr {
// validated arguments -> constants, scratch, launches (stream-ordered)
static int stack_impl(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                      const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs, int32_t out_ny, int32_t out_nx,
                      int32_t order, const float *weights, float *sum, float *wsum, int32_t accumulate,
                      cudaStream_t st)
{
    std::vector<float> hw((size_t)n, 1.0f);
    for (int32_t e = 0; weights && e < n; ++e) hw[e] = weights[e];
    std::call_once(g_pool_once, tune_pool);
    int rc;
    g_last.pending = false;
    TargetDev tgt;
    make_target(tgt_wcs, &tgt);
    std::vector<SourceDev> hsrc;
    SourceDev *dsrc = nullptr;
    rc = upload_sources(n, src_wcs, tgt_wcs, st, hsrc, &dsrc);
    if (rc != DFR_OK) return rc;
    float *dw = nullptr;
    TiledStats ts = {0, 0, 0, 0};
    cudaError_t err = ensure_last();
    if (err == cudaSuccess) err = cudaMallocAsync((void **)&dw, sizeof(float) * (size_t)n, st);
    // pageable source: the runtime stages the bytes before returning, so `hw` may die
    if (err == cudaSuccess) err = cudaMemcpyAsync(dw, hw.data(), sizeof(float) * (size_t)n, cudaMemcpyHostToDevice, st);
    if (err == cudaSuccess)
        err = launch_tiled_stack(src_batch, n, src_ny, src_nx, tgt, dsrc, hsrc.data(), out_ny, out_nx, order,
                                 dw, sum, wsum, accumulate != 0, st,
                                 g_accumulate ? g_stream_totals : g_last.pinned_dev, g_accumulate ? 1 : 0,
                                 &ts, &g_last.prof);
    if (!g_accumulate && err == cudaSuccess) err = cudaEventRecord(g_last.done, st);
    if (dw) cudaFreeAsync(dw, st);
    cudaFreeAsync(dsrc, st);
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
}  // namespace dfr

extern "C" {

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
    std::call_once(g_pool_once, tune_pool);
    SkyDev h;
    make_sky(w, &h);
    cudaError_t err = cudaMallocAsync((void **)dev, sizeof(SkyDev), st);
    if (err != cudaSuccess) return cuda_fail(err, "cudaMallocAsync(sky)");
    err = cudaMemcpyAsync(*dev, &h, sizeof h, cudaMemcpyHostToDevice, st);
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

// ---- end-to-end streaming form ------------------------
namespace {
struct Slot {
    cudaStream_t st = nullptr;
    float *din = nullptr, *dout = nullptr;
    size_t in_bytes = 0, out_bytes = 0;
};
constexpr int kSlots = 3;
struct HostPipe {
    std::mutex mu;
    int dev = -1;
    Slot slot[kSlots];
} g_pipe;

static cudaError_t ensure_slot(Slot &s, size_t in_bytes, size_t out_bytes)
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
}  // namespace

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
    const size_t in_px = (size_t)src_ny * src_nx, out_px = (size_t)out_ny * out_nx;
    std::lock_guard<std::mutex> lock(g_pipe.mu);
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return cuda_fail(err, "cudaGetDevice");
    if (g_pipe.dev != dev) {                       // buffers belong to one device
        for (Slot &s : g_pipe.slot) {
            if (s.din) cudaFree(s.din);
            if (s.dout) cudaFree(s.dout);
            if (s.st) cudaStreamDestroy(s.st);
            s = Slot();
        }
        g_pipe.dev = dev;
    }
    const int nb = (n + batch - 1) / batch;
    const int used = nb < kSlots ? nb : kSlots;
    for (int k = 0; k < used; ++k) {
        err = ensure_slot(g_pipe.slot[k], in_px * batch * sizeof(float), out_px * batch * sizeof(float));
        if (err != cudaSuccess) return cuda_fail(err, "pipeline buffers");
    }
    if ((err = stream_stats_begin()) != cudaSuccess) return cuda_fail(err, "stream statistics");
    for (int b = 0; b < nb; ++b) {
        Slot &s = g_pipe.slot[b % kSlots];
        const int32_t e0 = b * batch, ne = (n - e0 < batch) ? n - e0 : batch;
        // slot reuse is ordered by the slot's own stream: H2D(b) waits for D2H(b - kSlots)
        err = cudaMemcpyAsync(s.din, src_host + in_px * e0, in_px * ne * sizeof(float),
                              cudaMemcpyHostToDevice, s.st);
        if (err != cudaSuccess) { rc = cuda_fail(err, "H2D"); break; }
        rc = reproject_impl(s.din, ne, src_ny, src_nx, src_wcs + e0, tgt_wcs, out_ny, out_nx, order,
                            s.dout, s.st, DFR_PATH_AUTO);
        if (rc != DFR_OK) break;
        err = cudaMemcpyAsync(out_host + out_px * e0, s.dout, out_px * ne * sizeof(float),
                              cudaMemcpyDeviceToHost, s.st);
        if (err != cudaSuccess) { rc = cuda_fail(err, "D2H"); break; }
    }
    for (int k = 0; k < used; ++k) {
        err = cudaStreamSynchronize(g_pipe.slot[k].st);
        if (err != cudaSuccess && rc == DFR_OK) rc = cuda_fail(err, "pipeline sync");
    }
    stream_stats_end();
    return rc;
}

int dfr_stack_host(const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                   const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                   int32_t out_ny, int32_t out_nx, int32_t order, const float *weights,
                   float *sum_host, float *wsum_host, int32_t batch)
{
    if (!src_host || !sum_host || !wsum_host) { set_error("NULL image pointer"); return DFR_ERR_NULL; }
    int rc = check_common(n, src_ny, src_nx, src_wcs, tgt_wcs, out_ny, out_nx, order);
    if (rc != DFR_OK) return rc;
    for (int32_t e = 0; weights && e < n; ++e)
        if (!std::isfinite(weights[e])) { set_error("weights[%d] is not finite", e); return DFR_ERR_NONFINITE_WCS; }
    if (batch <= 0) batch = 32;
    if (batch > n) batch = n;
    const size_t in_px = (size_t)src_ny * src_nx, out_bytes = sizeof(float) * (size_t)out_ny * out_nx;
    std::lock_guard<std::mutex> lock(g_pipe.mu);
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return cuda_fail(err, "cudaGetDevice");
    if (g_pipe.dev != dev) {                       // buffers belong to one device
        for (Slot &s : g_pipe.slot) {
            if (s.din) cudaFree(s.din);
            if (s.dout) cudaFree(s.dout);
            if (s.st) cudaStreamDestroy(s.st);
            s = Slot();
        }
        g_pipe.dev = dev;
    }
    const int nb = (n + batch - 1) / batch;
    const int used = nb < kSlots ? nb : kSlots;
    // slot 0's output buffer holds sum and wsum; every slot needs an input buffer and a stream
    for (int k = 0; k < used; ++k) {
        err = ensure_slot(g_pipe.slot[k], in_px * batch * sizeof(float), k == 0 ? 2 * out_bytes : 0);
        if (err != cudaSuccess) return cuda_fail(err, "pipeline buffers");
    }
    float *dsum = g_pipe.slot[0].dout, *dwsum = dsum + (size_t)out_ny * out_nx;
    cudaEvent_t zeroed = nullptr;
    if ((err = cudaEventCreateWithFlags(&zeroed, cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(err, "event");
    err = cudaMemsetAsync(dsum, 0, 2 * out_bytes, g_pipe.slot[0].st);
    if (err == cudaSuccess) err = cudaEventRecord(zeroed, g_pipe.slot[0].st);
    for (int k = 1; k < used && err == cudaSuccess; ++k) err = cudaStreamWaitEvent(g_pipe.slot[k].st, zeroed, 0);
    if (err != cudaSuccess) { cudaEventDestroy(zeroed); return cuda_fail(err, "pipeline start"); }
    if ((err = stream_stats_begin()) != cudaSuccess) return cuda_fail(err, "stream statistics");
    for (int b = 0; b < nb; ++b) {
        Slot &s = g_pipe.slot[b % kSlots];
        const int32_t e0 = b * batch, ne = (n - e0 < batch) ? n - e0 : batch;
        // the slot's stream orders its own reuse: H2D(b) waits for the kernels of b - kSlots;
        // batches of different slots add into sum / wsum concurrently (atomic adds)
        err = cudaMemcpyAsync(s.din, src_host + in_px * e0, in_px * ne * sizeof(float), cudaMemcpyHostToDevice, s.st);
        if (err != cudaSuccess) { rc = cuda_fail(err, "H2D"); break; }
        rc = stack_impl(s.din, ne, src_ny, src_nx, src_wcs + e0, tgt_wcs, out_ny, out_nx, order,
                        weights ? weights + e0 : nullptr, dsum, dwsum, 1, s.st);
        if (rc != DFR_OK) break;
    }
    for (int k = 0; k < used; ++k) {
        err = cudaStreamSynchronize(g_pipe.slot[k].st);
        if (err != cudaSuccess && rc == DFR_OK) rc = cuda_fail(err, "pipeline sync");
    }
    cudaEventDestroy(zeroed);
    stream_stats_end();
    if (rc != DFR_OK) return rc;
    err = cudaMemcpy(sum_host, dsum, out_bytes, cudaMemcpyDeviceToHost);
    if (err == cudaSuccess) err = cudaMemcpy(wsum_host, dwsum, out_bytes, cudaMemcpyDeviceToHost);
    return err == cudaSuccess ? DFR_OK : cuda_fail(err, "D2H");
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
    collect_stats(stats);
    return DFR_OK;
}

int dfr_profile_enable(int on)
{
    ProfileEvents &p = g_last.prof;
    if (on && !p.setup_begin) {
        cudaError_t err;
        if ((err = cudaEventCreate(&p.setup_begin)) != cudaSuccess ||
            (err = cudaEventCreate(&p.main_begin)) != cudaSuccess ||
            (err = cudaEventCreate(&p.main_end)) != cudaSuccess)
            return cuda_fail(err, "cudaEventCreate");
    }
    p.enabled = on != 0;
    return DFR_OK;
}

int dfr_profile_last(float ms[2])
{
    ProfileEvents &p = g_last.prof;
    if (!ms) return DFR_ERR_NULL;
    if (!p.enabled || !p.main_end) { set_error("profiling is not enabled"); return DFR_ERR_ORDER; }
    cudaError_t err = cudaEventSynchronize(p.main_end);
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms[0], p.setup_begin, p.main_begin);
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms[1], p.main_begin, p.main_end);
    return err == cudaSuccess ? DFR_OK : cuda_fail(err, "profile events");
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
    default: return "unknown error";
    }
}

const char *dfr_last_error(void) { return dfr::last_error_cstr(); }

int dfr_version(void) { return 100; }

}  // extern "C"
