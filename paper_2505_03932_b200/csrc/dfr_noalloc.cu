// dfr_noalloc.cu — dfr_reproject_noalloc (include/dfr.h): the exact per-pixel reprojection for
// callers that must not cause a device allocation.
//
// Who that is. Every other entry point of libdfr takes its per-call scratch (the table of
// per-exposure constants the kernels read, tile records, staging memory) from a CUDA memory pool
// and keeps events and pinned buffers per thread. That is a problem for
//   - a pipeline that shares the GPU with an application which already owns all of HBM — a
//     framework's caching allocator grown to the whole card, or a night's stack of exposures
//     reserved up front: the library's first cudaMallocAsync can then fail half way through a run;
//   - a real-time loop (quick-look reduction between two telescope read-outs) that may not risk
//     the implicit device-wide synchronisation a cudaMalloc / cudaFree can bring, nor a pool
//     that grows or trims underneath it.
// For them this file keeps the one piece of scratch the exact kernel needs — the SourceDev table,
// 992 bytes per exposure — in a fixed array that is part of the library image itself. It costs
// DFR_NOALLOC_MAX_EXPOSURES x 992 B = 63 488 B of device memory on every GPU that loads libdfr,
// from load until the process ends, and in exchange the call path below contains no cudaMalloc,
// cudaFree, cudaMallocAsync, memory pool, event or stream creation, and no pinned allocation.
//
// The existing paths are untouched: the kernel here is a copy of exact_reproject_kernel
// (dfr_kernels_exact.cu) built from the same device functions of dfr_device.cuh (so results are
// the exact path's, bit for bit), minus the edge-rule / footprint-array options.
#include <mutex>

#include "dfr_device.cuh"

namespace dfr {
namespace {

constexpr int kMaxExposures = DFR_NOALLOC_MAX_EXPOSURES;
static_assert(sizeof(SourceDev) % 8 == 0, "the table is filled in 8-byte words");

// The scratch: per-exposure constants of the call in flight. One array per GPU and process, shared
// by every call; it keeps whatever the previous call left in it. Nothing in it has to start at
// zero: a call overwrites entries [0, n) in full before its reprojection kernel reads exactly
// those, and entries >= n are never read.
//
// In HOST code the identifier below is only a handle for the runtime's symbol table, not a device
// address (a kernel handed `g_table` from the host would fault, or read host memory): the host
// obtains the real address once per device through cudaGetSymbolAddress (table_on_current_device).
// DEVICE code may name the array directly; the fill kernel does.
static __device__ __align__(256) unsigned char g_table[kMaxExposures * sizeof(SourceDev)];

// Constants travel as kernel PARAMETERS (copied by the launch itself: no staging buffer whose
// lifetime would have to be tracked, no copy-engine transfer from pageable memory), a few
// exposures per launch.
constexpr int kFillChunk = 8;                            // 8 x 992 B = 7936 B of parameters
struct FillChunk { SourceDev s[kFillChunk]; };

__global__ void noalloc_fill_kernel(const __grid_constant__ FillChunk chunk, int e0, int count)
{
    const unsigned long long *w = reinterpret_cast<const unsigned long long *>(&chunk);
    unsigned long long *dst = reinterpret_cast<unsigned long long *>(g_table + (size_t)e0 * sizeof(SourceDev));
    const int nwords = count * (int)(sizeof(SourceDev) / 8);
    for (int k = threadIdx.x; k < nwords; k += blockDim.x) dst[k] = w[k];
}

constexpr int NA_BX = 64, NA_BY = 4;

// exact_reproject_kernel with the constants table passed as the address the host looked up
// (steps a1-a9 of SURVEY.md §8(a); area footprint rule).
template <int ORDER>
__global__ void __launch_bounds__(NA_BX *NA_BY)
noalloc_reproject_kernel(const float *__restrict__ src, int sny, int snx,
                         const __grid_constant__ TargetDev tgt,
                         const SourceDev *__restrict__ table,
                         int ony, int onx, float *__restrict__ out)
{
    const int tiles_x = (onx + NA_BX - 1) / NA_BX;
    const int i = (blockIdx.x % tiles_x) * NA_BX + threadIdx.x;
    const int j = (blockIdx.x / tiles_x) * NA_BY + threadIdx.y;
    const int e = blockIdx.y;
    if (i >= onx || j >= ony) return;
    double U, V, x, y;
    target_uv(tgt, (double)i, (double)j, U, V);
    source_xy(table[e], U, V, x, y);
    float val = qnanf();
    if (in_footprint(x, y, sny, snx, DFR_EDGE_AREA))
        val = sample_global<ORDER>(src + (size_t)e * sny * snx, sny, snx, x, y);
    out[((size_t)e * ony + j) * onx + i] = val;
}

// Device address of g_table on the CURRENT device, looked up on the first call made with that
// device current and remembered (a per-ordinal slot: no allocation on the host side either).
constexpr int kMaxDevices = 64;
std::mutex g_mu;
SourceDev *g_table_addr[kMaxDevices] = {};

cudaError_t table_on_current_device(SourceDev **out)
{
    int dev = -1;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_table_addr[dev]) {
        void *p = nullptr;
        err = cudaGetSymbolAddress(&p, g_table);
        if (err != cudaSuccess) return err;
        if (!p) return cudaErrorInvalidSymbol;
        g_table_addr[dev] = static_cast<SourceDev *>(p);
    }
    *out = g_table_addr[dev];
    return cudaSuccess;
}

bool overlaps(const void *a, size_t na, const void *b, size_t nb)
{
    const char *a0 = (const char *)a, *b0 = (const char *)b;
    return a0 < b0 + nb && b0 < a0 + na;
}

}  // namespace
}  // namespace dfr

using namespace dfr;

extern "C" int dfr_reproject_noalloc(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                                     const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                                     int32_t out_ny, int32_t out_nx, int32_t order,
                                     float *out, void *stream)
{
    if (!src_batch || !out) { set_error("NULL image pointer"); return DFR_ERR_NULL; }
    if (!src_wcs || !tgt_wcs) { set_error("NULL WCS pointer"); return DFR_ERR_NULL; }
    if (n < 1 || src_ny < 1 || src_nx < 1 || out_ny < 1 || out_nx < 1 ||
        (int64_t)src_ny * src_nx >= (1LL << 31) || (int64_t)out_ny * out_nx >= (1LL << 31)) {
        set_error("bad shape: n=%d src=%dx%d out=%dx%d", n, src_ny, src_nx, out_ny, out_nx);
        return DFR_ERR_SHAPE;
    }
    if (n > kMaxExposures) {
        set_error("dfr_reproject_noalloc takes at most DFR_NOALLOC_MAX_EXPOSURES = %d exposures per call "
                  "(its constants table is a fixed array), got n = %d: split the batch, or use dfr_reproject",
                  kMaxExposures, n);
        return DFR_ERR_SHAPE;
    }
    if (order != DFR_NEAREST && order != DFR_BILINEAR && order != DFR_BICUBIC) {
        set_error("order %d not in {0, 1, 3}", order);
        return DFR_ERR_ORDER;
    }
    int rc = validate_wcs(tgt_wcs);
    for (int32_t e = 0; e < n && rc == DFR_OK; ++e) rc = validate_wcs(&src_wcs[e]);
    if (rc != DFR_OK) return rc;
    if (overlaps(out, sizeof(float) * (size_t)n * out_ny * out_nx, src_batch, sizeof(float) * (size_t)n * src_ny * src_nx)) {
        set_error("out overlaps src_batch");
        return DFR_ERR_ALIAS;
    }

    cudaStream_t st = (cudaStream_t)stream;
    SourceDev *table = nullptr;
    cudaError_t err = table_on_current_device(&table);
    if (err != cudaSuccess) return cuda_fail(err, "cudaGetSymbolAddress(no-alloc constants table)");

    TargetDev tgt;
    make_target(tgt_wcs, &tgt);
    FillChunk chunk;                                          // host stack; copied by each launch
    for (int32_t e0 = 0; e0 < n; e0 += kFillChunk) {
        const int count = (n - e0 < kFillChunk) ? n - e0 : kFillChunk;
        for (int k = 0; k < count; ++k) make_source(tgt_wcs, &src_wcs[e0 + k], &chunk.s[k]);
        noalloc_fill_kernel<<<1, 256, 0, st>>>(chunk, e0, count);
        if ((err = cudaGetLastError()) != cudaSuccess) return cuda_fail(err, "no-alloc table fill launch");
    }
    const dim3 block(NA_BX, NA_BY);
    const dim3 grid(((out_nx + NA_BX - 1) / NA_BX) * ((out_ny + NA_BY - 1) / NA_BY), n, 1);
    if (order == DFR_NEAREST)
        noalloc_reproject_kernel<DFR_NEAREST><<<grid, block, 0, st>>>(src_batch, src_ny, src_nx, tgt, table, out_ny, out_nx, out);
    else if (order == DFR_BILINEAR)
        noalloc_reproject_kernel<DFR_BILINEAR><<<grid, block, 0, st>>>(src_batch, src_ny, src_nx, tgt, table, out_ny, out_nx, out);
    else
        noalloc_reproject_kernel<DFR_BICUBIC><<<grid, block, 0, st>>>(src_batch, src_ny, src_nx, tgt, table, out_ny, out_nx, out);
    if ((err = cudaGetLastError()) != cudaSuccess) return cuda_fail(err, "no-alloc reproject launch");
    return DFR_OK;
}
