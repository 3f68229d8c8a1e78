// dfr_tiled_main.cu — the main kernel of the tiled fast path:
//
//   tiled_reproject_kernel (fp32) per 64x64 CTA tile: the source bounding box is staged
//                         into shared memory by one TMA box load issued before the tile
//                         records arrive; each warp walks one 32x32 tile. INTERIOR tiles
//                         (every tap inside the image and the box, by the record's bound)
//                         run the packed loop: two rows per step in FFMA2/FADD2 pairs,
//                         floor by a round-down add, no range test, one folded address
//                         per pixel, 4 LDS, coalesced 128-byte row stores. Other FAST
//                         tiles run the checked scalar loop; pixels whose taps leave the
//                         staged box or touch the image rim, and all pixels of EXACT
//                         tiles, take the exact/global-gather code of dfr_device.cuh.
#include <algorithm>
#include <atomic>
#include <cstring>

#include "dfr_tiled_device.cuh"

namespace dfr {

// ---------------------------------------------------------------------------------
// main kernel: one CTA per 64x64 output tile per exposure, one warp per 32x32 tile
// ---------------------------------------------------------------------------------
// EDGE (DFR_EDGE_*) is a template parameter so that the default kernel is compiled exactly as
// without it (a run-time flag cost 3 % through register allocation alone).
// Bicubic gets 80 registers (6 CTAs / SM): with 64 the 32 taps of a row pair cannot all be in flight
// (measured on B200, C3: 0.102 -> 0.094 ms; 96 registers / 5 CTAs: 0.093 ms).
template <int ORDER, bool STAGE, int EDGE = DFR_EDGE_AREA>
__global__ void __launch_bounds__(32 * CTA_T * CTA_T, ORDER == DFR_BICUBIC ? 6 : 8)
tiled_reproject_kernel(const __grid_constant__ TiledParams P, const __grid_constant__ TargetDev tgt,
                       const __grid_constant__ CUtensorMap tmap)
{
    extern __shared__ __align__(128) float box[];
    __shared__ __align__(8) unsigned long long mbar;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int e = P.e0 + blockIdx.z;                  // grid = (ctas_x, ctas_y, exposures): no divisions
    const int ttx = blockIdx.x * CTA_T + (warp % CTA_T), tty = blockIdx.y * CTA_T + (warp / CTA_T);
    const bool active = ttx < P.tiles_x && tty < P.tiles_y;
    const int ntile = P.tiles_x * P.tiles_y;
    const TileRec *rec = P.recs + ((size_t)e * ntile + (active ? tty * P.tiles_x + ttx : 0));

    pdl_wait();                         // the setup kernel's records and box origins are complete
    // ---- stage the CTA tile's source box first: its origin was reduced by the setup kernel
    // (cta_box), so the TMA load does not wait for the tile records, which load meanwhile.
    int ox = 0, oy = 0;                 // origin of the staged box in source pixels
    bool has_box = false;
    if (STAGE) {
        const int2 cb = __ldg(P.cta_box + ((size_t)e * P.ctas_y + blockIdx.y) * P.ctas_x + blockIdx.x);
        has_box = cb.x != kNoBox;
        // TMA wants a 16-byte aligned start along x (measured on B200: an unaligned inner
        // coordinate faults with "illegal instruction"): round down to 4 floats
        ox = (cb.x - (Taps<ORDER>::lo + 1)) & ~3;
        oy = cb.y - (Taps<ORDER>::lo + 1);
        if (threadIdx.x == 0 && has_box) {
            const uint32_t bar = smem_u32(&mbar), dst = smem_u32(box);
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            const uint32_t bytes = (uint32_t)(P.BW * P.BH * sizeof(float));
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
            asm volatile(
                "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                ::"r"(dst), "l"(&tmap), "r"(ox), "r"(oy), "r"(e), "r"(bar) : "memory");
        }
        // L2 prefetch of the box of the CTA tile that will be scheduled about one wave from now
        // (blocks are issued in linear order), so that its own TMA load finds the lines in L2
        if (threadIdx.x == 0 && P.prefetch_dist > 0) {
            const long long ctas = (long long)P.ctas_x * P.ctas_y;
            const long long lin = ((long long)blockIdx.z * P.ctas_y + blockIdx.y) * P.ctas_x + blockIdx.x + P.prefetch_dist;
            if (lin < ctas * (long long)gridDim.z) {
                const int2 cf = __ldg(P.cta_box + (size_t)P.e0 * ctas + lin);
                if (cf.x != kNoBox) {
                    const int fx = (cf.x - (Taps<ORDER>::lo + 1)) & ~3, fy = cf.y - (Taps<ORDER>::lo + 1);
                    const int fe = P.e0 + (int)(lin / ctas);
                    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];"
                                 ::"l"(&tmap), "r"(fx), "r"(fy), "r"(fe) : "memory");
                }
            }
        }
    }

    int flag = TILE_EMPTY, ix0 = 0, iy0 = 0, bx0 = 0, by0 = 0, bx1 = 0, by1 = 0, deg = 3;
    if (active) {
        const int4 h0 = __ldg(reinterpret_cast<const int4 *>(&rec->ix0));       // ix0 iy0 bx0 by0
        const int4 h1 = __ldg(reinterpret_cast<const int4 *>(&rec->bx1));       // bx1 by1 flag deg
        ix0 = h0.x; iy0 = h0.y; bx0 = h0.z; by0 = h0.w; bx1 = h1.x; by1 = h1.y; flag = h1.z; deg = h1.w;
    }
    // per-lane column polynomials in dj (FAST tiles; harmless otherwise)
    float X[4], Y[4];
    column_polys(rec, lane, X, Y);
    if (STAGE) {
        __syncthreads();                // the mbarrier is initialised before anybody polls it
        if (has_box) {
            const uint32_t bar = smem_u32(&mbar);
            uint32_t done = 0;
            while (!done) {
                asm volatile(
                    "{\n\t.reg .pred p;\n\t"
                    "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                    "selp.u32 %0, 1, 0, p;\n\t}"
                    : "=r"(done) : "r"(bar), "r"(0u) : "memory");
            }
        }
    }
    if (!active) return;
    TileHead H;
    H.flag = flag; H.ix0 = ix0; H.iy0 = iy0; H.bx0 = bx0; H.by0 = by0; H.bx1 = bx1; H.by1 = by1; H.deg = deg;
    dfr_chk_set(has_box ? smem_u32(box) : 0u, has_box ? smem_u32(box) + (uint32_t)(P.BW * P.BH * sizeof(float)) : 0u);
    StoreSink sink;
    sink.orow = P.out + ((size_t)e * P.ony + (size_t)tty * TS) * P.onx + (ttx * TS + lane);
    sink.opitch = (size_t)P.onx;
    warp_tile<ORDER, STAGE, EDGE>(P, tgt, e, ttx, tty, lane, H, X, Y, smem_u32(box), ox, oy, sink);
}

#ifdef DFR_BOUNDS_CHECK
}  // namespace dfr
extern "C" unsigned long long dfr_dev_oob_main()
{
    unsigned long long v = 0, zero = 0;
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(&v, dfr::dfr_oob_count, sizeof v);
    cudaMemcpyToSymbol(dfr::dfr_oob_count, &zero, sizeof zero);
    return v;
}
namespace dfr {
#endif

// coordinates the tiled path uses (dfr_src_coords): same records, same polynomial code
__global__ void __launch_bounds__(32 * CTA_T * CTA_T)
tiled_coords_kernel(const __grid_constant__ TiledParams P, const __grid_constant__ TargetDev tgt,
                    double *__restrict__ xo, double *__restrict__ yo)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int e = P.e0 + blockIdx.z;
    const int ttx = blockIdx.x * CTA_T + (warp % CTA_T), tty = blockIdx.y * CTA_T + (warp / CTA_T);
    if (!(ttx < P.tiles_x && tty < P.tiles_y)) return;
    const int ntile = P.tiles_x * P.tiles_y;
    const TileRec *rec = P.recs + ((size_t)e * ntile + tty * P.tiles_x + ttx);
    const int flag = rec->flag, ix0 = rec->ix0, iy0 = rec->iy0, deg = rec->deg;
    const int tx0 = ttx * TS, ty0 = tty * TS, col = tx0 + lane;
    if (col >= P.onx) return;
    const int rows = min(TS, P.ony - ty0);
    const size_t o = ((size_t)e * P.ony + ty0) * P.onx + col;
    if (flag == TILE_EXACT) {
        for (int r = 0; r < rows; ++r) {
            double U, V, x, y;
            target_uv(tgt, (double)col, (double)(ty0 + r), U, V);
            source_xy(P.srcdev[e], U, V, x, y);
            xo[o + (size_t)r * P.onx] = x;
            yo[o + (size_t)r * P.onx] = y;
        }
        return;
    }
    float X[4], Y[4];
    column_polys(rec, lane, X, Y);                              // the main kernel's own functions
    truncate_degree(deg, X, Y);
    for (int r = 0; r < rows; ++r) {
        float xl, yl;
        tile_coord(X, Y, r, xl, yl);
        xo[o + (size_t)r * P.onx] = (double)ix0 + (double)xl;
        yo[o + (size_t)r * P.onx] = (double)iy0 + (double)yl;
    }
}

// The footprint array of dfr_reproject_fp (footprint_value, dfr_device.cuh) from the same tile records
// and the same polynomial coordinates as the main kernel, so it is consistent with `out` pixel by
// pixel: EMPTY tiles are 0, EXACT tiles use the fp64 map, FAST tiles the polynomial coordinate. A
// separate pass over the records (no image reads, 4 B written per pixel) keeps the main kernel,
// and with it `out`, exactly as it is without a footprint.
__global__ void __launch_bounds__(32 * CTA_T * CTA_T)
tiled_footprint_kernel(const __grid_constant__ TiledParams P, const __grid_constant__ TargetDev tgt,
                       int order, int edge, float *__restrict__ foot)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int e = P.e0 + blockIdx.z;
    const int ttx = blockIdx.x * CTA_T + (warp % CTA_T), tty = blockIdx.y * CTA_T + (warp / CTA_T);
    if (!(ttx < P.tiles_x && tty < P.tiles_y)) return;
    const int ntile = P.tiles_x * P.tiles_y;
    const TileRec *rec = P.recs + ((size_t)e * ntile + tty * P.tiles_x + ttx);
    const int flag = rec->flag, ix0 = rec->ix0, iy0 = rec->iy0, deg = rec->deg;
    const int tx0 = ttx * TS, ty0 = tty * TS, col = tx0 + lane;
    if (col >= P.onx) return;
    const int rows = min(TS, P.ony - ty0);
    float *__restrict__ o = foot + ((size_t)e * P.ony + ty0) * P.onx + col;
    if (flag == TILE_EMPTY) {
        for (int r = 0; r < rows; ++r) o[(size_t)r * P.onx] = 0.0f;
        return;
    }
    if (flag == TILE_EXACT) {
        for (int r = 0; r < rows; ++r) {
            double U, V, x, y;
            target_uv(tgt, (double)col, (double)(ty0 + r), U, V);
            source_xy(P.srcdev[e], U, V, x, y);
            o[(size_t)r * P.onx] = footprint_value(x, y, P.sny, P.snx, order, edge);
        }
        return;
    }
    float X[4], Y[4];
    column_polys(rec, lane, X, Y);                              // the main kernel's own functions
    truncate_degree(deg, X, Y);
    for (int r = 0; r < rows; ++r) {
        float xl, yl;
        tile_coord(X, Y, r, xl, yl);
        o[(size_t)r * P.onx] = footprint_value((double)ix0 + (double)xl, (double)iy0 + (double)yl, P.sny, P.snx, order, edge);
    }
}

template <int ORDER, bool STAGE, int EDGE = DFR_EDGE_AREA>
static cudaError_t launch_main(const TiledParams &P, const TargetDev &tgt, const CUtensorMap &tmap,
                               size_t smem, cudaStream_t st)
{
    auto kern = tiled_reproject_kernel<ORDER, STAGE, EDGE>;
    if (P.ctas_y > 65535) return cudaErrorInvalidConfiguration;
    TiledParams Q = P;
    if (STAGE) {
        // per (kernel, device): the shared-memory opt-in once, the resident-CTA count per box size
        // (the occupancy query costs microseconds of host time per call otherwise)
        constexpr int kDevs = 64, kSlots = kMaxBoxBytes / 1024 + 2;
        static std::atomic<int> per_sm_cache[kDevs][kSlots];       // 0 = unknown; indexed by KB of box
        static std::atomic<bool> opted_in[kDevs];
        int dev = 0;
        cudaError_t err = cudaGetDevice(&dev);
        if (err != cudaSuccess) return err;
        const int d = (dev >= 0 && dev < kDevs) ? dev : 0, slot = (int)std::min<size_t>((smem + 1023) / 1024, kSlots - 1);
        if (!opted_in[d].load(std::memory_order_acquire) || dev != d) {
            if ((err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxBoxBytes)) != cudaSuccess) return err;
            opted_in[d].store(true, std::memory_order_release);
        }
        int waves = per_sm_cache[d][slot].load(std::memory_order_relaxed);
        if (waves == 0 || dev != d) {
            int sms = 0, per_sm = 0;
            if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
                cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 32 * CTA_T * CTA_T, (size_t)slot * 1024) == cudaSuccess)
                waves = sms * per_sm;
            per_sm_cache[d][slot].store(waves, std::memory_order_relaxed);
        }
        Q.prefetch_dist = waves / 2;        // measured on B200, C2: flat optimum between 1/2 and 3/4 of a wave
#ifdef DFR_DEV_HOOKS                                                 // A-B timing builds only (never the shipped library)
        static const char *pd = std::getenv("DFR_PREFETCH");
        if (pd) Q.prefetch_dist = std::atoi(pd);
#endif
    }
    for (int e0 = 0; e0 < P.n; e0 += 65535) {
        Q.e0 = e0;
        const dim3 grid((unsigned)P.ctas_x, (unsigned)P.ctas_y, (unsigned)std::min(P.n - e0, 65535));
        const cudaError_t err = launch_pdl(kern, grid, dim3(32 * CTA_T * CTA_T), smem, st, Q, tgt, tmap);
        if (err != cudaSuccess) return err;
    }
    return cudaSuccess;
}

cudaError_t launch_tiled_reproject(const float *src, int n, int sny, int snx,
                                   const TargetDev &tgt, const SourceDev *srcdev,
                                   const SourceDev *srchost,
                                   int ony, int onx, int order, float *out, cudaStream_t st,
                                   int32_t *host_stats, int stats_add, TiledStats *stats, ProfileEvents *prof,
                                   const ConstsCopy &cc, int edge, float *foot)
{
    Prepared R;
    if (prof && prof->enabled) cudaEventRecord(prof->setup_begin, st);
    cudaError_t err = prepare_tiled(src, n, sny, snx, tgt, srcdev, srchost, ony, onx, order, st, host_stats, stats_add, R, cc);
    if (err != cudaSuccess) { free_scratch(R.sc, st); return err; }
    R.P.out = out;
    if (prof && prof->enabled) cudaEventRecord(prof->main_begin, st);
#define DFR_LAUNCH(O)                                                                     \
    err = R.stage ? launch_main<O, true>(R.P, tgt, R.tmap, R.box_bytes, st) : launch_main<O, false>(R.P, tgt, R.tmap, 0, st)
    if (order == DFR_NEAREST) DFR_LAUNCH(DFR_NEAREST);
    else if (order == DFR_BILINEAR && edge == DFR_EDGE_PAPER)
        err = R.stage ? launch_main<DFR_BILINEAR, true, DFR_EDGE_PAPER>(R.P, tgt, R.tmap, R.box_bytes, st)
                      : launch_main<DFR_BILINEAR, false, DFR_EDGE_PAPER>(R.P, tgt, R.tmap, 0, st);
    else if (order == DFR_BILINEAR) DFR_LAUNCH(DFR_BILINEAR);
    else DFR_LAUNCH(DFR_BICUBIC);
#undef DFR_LAUNCH
    if (prof && prof->enabled) cudaEventRecord(prof->main_end, st);
    stats->kernels = 3;
    if (foot && err == cudaSuccess) {
        TiledParams Q = R.P;
        for (int e0 = 0; e0 < n && err == cudaSuccess; e0 += 65535) {
            Q.e0 = e0;
            const dim3 grid((unsigned)Q.ctas_x, (unsigned)Q.ctas_y, (unsigned)std::min(n - e0, 65535));
            tiled_footprint_kernel<<<grid, 32 * CTA_T * CTA_T, 0, st>>>(Q, tgt, order, edge, foot);
            err = cudaGetLastError();
        }
        stats->kernels = 4;
    }
    free_scratch(R.sc, st);
    stats->tiles_fast = stats->tiles_exact = stats->tiles_empty = -1;   // written to host_stats by the setup kernel
    return err;
}

cudaError_t launch_tiled_coords(int n, int sny, int snx, const TargetDev &tgt,
                                const SourceDev *srcdev, const SourceDev *srchost, int ony, int onx, int order,
                                double *x, double *y, cudaStream_t st, const ConstsCopy &cc)
{
    (void)order;
    TiledParams P;
    std::memset(&P, 0, sizeof P);
    Scratch sc;
    cudaError_t err = run_setup(n, sny, snx, tgt, srcdev, srchost, ony, onx, st, nullptr, 0, sc, P, cc);
    if (err == cudaSuccess) {
        for (int e0 = 0; e0 < n && err == cudaSuccess; e0 += 65535) {
            P.e0 = e0;
            const dim3 grid((unsigned)P.ctas_x, (unsigned)P.ctas_y, (unsigned)std::min(n - e0, 65535));
            tiled_coords_kernel<<<grid, 32 * CTA_T * CTA_T, 0, st>>>(P, tgt, x, y);
            err = cudaGetLastError();
        }
    }
    free_scratch(sc, st);
    return err;
}

}  // namespace dfr
