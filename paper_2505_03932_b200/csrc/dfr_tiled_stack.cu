// dfr_tiled_stack.cu — fused reproject-and-stack (dfr_reproject_stack).
#include <algorithm>
#include <cmath>
#include <atomic>
#include <cstring>
#include <mutex>

#include "dfr_tiled_device.cuh"

namespace dfr {

// ---------------------------------------------------------------------------------
// fused reproject-and-stack (dfr_reproject_stack)
//
// One WARP per 32x32 output tile loops over the exposures; the per-pixel accumulators
//   sum += w_e v_e,  wsum += w_e   (only where v_e is not NaN)
// of its tile (2 x 32 rows per lane) live in TENSOR MEMORY: 64 TMEM columns per CTA, the
// warp's lane quarter, lane = output column, column = row (sum) / 32 + row (wsum part), read
// and written four rows at a time with tcgen05.ld / tcgen05.st (32x32b.x4). They never occupy
// registers for longer than four pixels, there is no per-exposure output in HBM, and the
// row loop stays a loop.
// ---------------------------------------------------------------------------------
// Accumulators of one warp's 32x32 tile in TMEM: column r = sum of row r, column 32 + r = the
// per-pixel part `c` of wsum. wsum itself = tileW + c, where tileW (one scalar per warp) is the sum of
// the weights of the exposures whose tile was INTERIOR (every tap of every pixel inside the image,
// by the record's bound): there a pixel can only be invalid through NaN source pixels, so the
// per-pixel work is reduced to `sum` — `c` records deficits (-w) and is touched only when a NaN
// shows up. Other tiles (image rim, box edge, EXACT) count per pixel: c += w where valid.
struct StackSink {
    static constexpr bool kAllLanes = true;        // tcgen05.ld/st are warp-wide: nobody leaves
    uint32_t taddr;                                // TMEM address of this warp's row 0 (sum)
    float w;                                       // weight of the current exposure
    float tileW;                                   // see above
    bool uniform;                                  // the current (tile, exposure) is counted through tileW
    int r;                                         // next row
    float s0, s1, s2, s3;                          // sums of rows r .. r + 3 in flight
    __device__ __forceinline__ void begin_exposure(float weight)
    {
        w = weight; r = 0; uniform = false;
    }
    __device__ __forceinline__ void set_uniform()   // called once per (tile, exposure), before any row
    {
        uniform = true; tileW += w;
    }
    __device__ __forceinline__ void prefetch4()
    {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=f"(s0), "=f"(s1), "=f"(s2), "=f"(s3) : "r"(taddr + (uint32_t)r));
    }
    // c of rows r .. r + 3 (warp-wide; `any` is warp-uniform)
    __device__ __forceinline__ void update_c4(bool ok0, bool ok1, bool ok2, bool ok3)
    {
        float c0, c1, c2, c3;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=f"(c0), "=f"(c1), "=f"(c2), "=f"(c3) : "r"(taddr + (uint32_t)(TS + r)));
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        // what a valid / an invalid pixel adds to c: (w, 0) per pixel, or (0, -w) against tileW
        const float cw_ok = uniform ? 0.0f : w, cw_bad = uniform ? -w : 0.0f;
        c0 += ok0 ? cw_ok : cw_bad; c1 += ok1 ? cw_ok : cw_bad; c2 += ok2 ? cw_ok : cw_bad; c3 += ok3 ? cw_ok : cw_bad;
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                     ::"r"(taddr + (uint32_t)(TS + r)), "f"(c0), "f"(c1), "f"(c2), "f"(c3) : "memory");
    }
    __device__ __forceinline__ void rows4(float v0, float v1, float v2, float v3)
    {
        const bool ok0 = v0 == v0, ok1 = v1 == v1, ok2 = v2 == v2, ok3 = v3 == v3;   // NaN: outside the footprint, or NaN taps
        // uniform tiles: c changes only where a pixel is invalid (rare: one warp vote decides)
        if (!uniform || __any_sync(0xffffffffu, !(ok0 && ok1 && ok2 && ok3))) update_c4(ok0, ok1, ok2, ok3);
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        s0 = ok0 ? fmaf(w, v0, s0) : s0; s1 = ok1 ? fmaf(w, v1, s1) : s1;
        s2 = ok2 ? fmaf(w, v2, s2) : s2; s3 = ok3 ? fmaf(w, v3, s3) : s3;
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                     ::"r"(taddr + (uint32_t)r), "f"(s0), "f"(s1), "f"(s2), "f"(s3) : "memory");
        r += 4;
    }
    // the packed interior loop: rows (r, r + 1) = va, (r + 2, r + 3) = vb. One NaN test for the four
    // values (their sum: a NaN anywhere, or +inf - inf, sends the group to the per-pixel form).
    __device__ __forceinline__ void rows4p(f32x2 va, f32x2 vb)
    {
        float t0, t1;
        unpk2(add2(va, vb), t0, t1);
        const float t = t0 + t1;
        if (__any_sync(0xffffffffu, !(t == t) || !uniform)) {
            float v0, v1, v2, v3;
            unpk2(va, v0, v1);
            unpk2(vb, v2, v3);
            rows4(v0, v1, v2, v3);
            return;
        }
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        const f32x2 w2 = splat2(w);
        float a0, a1, a2, a3;
        unpk2(fma2(w2, va, pk2(s0, s1)), a0, a1);
        unpk2(fma2(w2, vb, pk2(s2, s3)), a2, a3);
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                     ::"r"(taddr + (uint32_t)r), "f"(a0), "f"(a1), "f"(a2), "f"(a3) : "memory");
        r += 4;
    }
    __device__ __forceinline__ void row1(float v)
    {
        float s, c;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=f"(s) : "r"(taddr + (uint32_t)r));
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=f"(c) : "r"(taddr + (uint32_t)(TS + r)));
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        const bool ok = v == v;
        s = ok ? fmaf(w, v, s) : s;
        c += ok ? (uniform ? 0.0f : w) : (uniform ? -w : 0.0f);
        asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr + (uint32_t)r), "f"(s) : "memory");
        asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr + (uint32_t)(TS + r)), "f"(c) : "memory");
        r += 1;
    }
    __device__ __forceinline__ void empty_tile(int) {}           // an empty tile adds nothing
};

constexpr int kStackCols = 2 * TS;                 // TMEM columns per CTA (power of two >= 32)
constexpr int kStackWarps = 4;                     // one per TMEM lane quarter
constexpr int kStackThreads = 32 * kStackWarps;
constexpr size_t kStackMaxBoxBytes = 14 * 1024;    // per warp: keeps >= 4 CTAs (16 warps) per SM

struct StackParams {
    const float *weights;                          // DEVICE [n]
    float *sum, *wsum;                             // DEVICE [ony][onx]
    float *partial;                                // DEVICE [nchunk][ntile][2][32][32] (nchunk > 1), else NULL
    int32_t *ticket;                               // DEVICE [ntile], zeroed (nchunk > 1), else NULL
    int add;                                       // 0: overwrite sum / wsum; 1: add to their contents
    int nchunk;                                    // exposure chunks = gridDim.y
};

// Every warp is autonomous: it owns one 32x32 output tile (its TMEM lane quarter holds the tile's
// accumulators), one box buffer and one mbarrier, and walks the exposures of its chunk by itself:
//   lane 0 issues the TMA load of its own tile's source box for exposure e (origin from the tile
//   record, read one exposure ahead) and an L2 prefetch of the box of e + 1; all lanes load the
//   record and build their column polynomials while the box is in flight; wait; accumulate.
// No producer warp, no barrier between warps inside the loop: a warp waiting for its box is covered
// by the other resident warps (7 CTAs x 4 warps per SM at the C2 box size), and tiles of different
// cost (image rim, empty) never hold each other up. All warps of the grid move through the exposure
// list roughly together, so the halo a box shares with its neighbours is served by L2 and every source
// pixel comes from HBM once. One chunk (nchunk = 1) needs no reduction: every pixel has one owner, so
// the result is the same on every run; with exposure chunks (small outputs) the partial tiles go to
// scratch and the last chunk to arrive (ticket) adds them in chunk order — deterministic as well.
// 7 CTAs = 28 warps per SM (72 registers): measured best on B200 (C2: 0.249 ms; 6 CTAs / 80 registers
// 0.276, 8 CTAs / 64 registers with spills 0.262).
template <int ORDER, bool STAGE>
__global__ void __launch_bounds__(kStackThreads, STAGE ? 7 : 8)
tiled_stack_kernel(const __grid_constant__ TiledParams P, const __grid_constant__ TargetDev tgt,
                   const __grid_constant__ CUtensorMap tmap, const __grid_constant__ StackParams S)
{
    extern __shared__ __align__(128) unsigned char boxes[];
    __shared__ __align__(8) unsigned long long mbar[kStackWarps];
    __shared__ uint32_t tmem_base;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ntile = P.tiles_x * P.tiles_y;
    // four consecutive tiles of one tile row per CTA (neighbouring boxes share L2 lines)
    const int groups_x = (P.tiles_x + kStackWarps - 1) / kStackWarps;
    const int tty = blockIdx.x / groups_x, ttx = (blockIdx.x - tty * groups_x) * kStackWarps + warp;
    const bool active = ttx < P.tiles_x;
    const int tile = tty * P.tiles_x + (active ? ttx : 0);
    const int chunk = blockIdx.y;
    const int e_lo = (int)((long long)chunk * P.n / S.nchunk);
    const int e_hi = (int)((long long)(chunk + 1) * P.n / S.nchunk);

    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     ::"r"(smem_u32(&tmem_base)), "n"(kStackCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    const uint32_t bar = smem_u32(&mbar[warp]);
    if (lane == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    pdl_wait();                         // the setup kernel's records are complete

    StackSink sink;
    sink.taddr = tmem_base + ((uint32_t)(warp * 32) << 16);
    sink.tileW = 0.0f;
    sink.begin_exposure(0.0f);
    for (int g = 0; g < kStackCols; g += 4)                    // zero sum and c
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %1, %1, %1};"
                     ::"r"(sink.taddr + (uint32_t)g), "f"(0.0f) : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");

    if (active) {
        const uint32_t box_smem = smem_u32(boxes) + (uint32_t)warp * (uint32_t)P.stage_bytes;
        const uint32_t box_bytes = (uint32_t)(P.BW * P.BH * sizeof(float));
        const TileRec *rec0 = P.recs + tile;                   // exposure e: rec0 + e * ntile
        // (bx0, by0, flag) of the record one exposure ahead: the box origin without waiting for it
        int nbx = 0, nby = 0, nflag = TILE_EMPTY;
        if (e_lo < e_hi) {
            const TileRec *r0 = rec0 + (size_t)e_lo * ntile;
            nbx = __ldg(&r0->bx0); nby = __ldg(&r0->by0); nflag = __ldg(&r0->flag);
        }
        uint32_t phase = 0;
        for (int e = e_lo; e < e_hi; ++e) {
            const TileRec *rec = rec0 + (size_t)e * ntile;
            // TMA wants a 16-byte aligned start along x (measured on B200): round down to 4 floats
            const int ox = (nbx - (Taps<ORDER>::lo + 1)) & ~3, oy = nby - (Taps<ORDER>::lo + 1);
            const bool has_box = STAGE && nflag == TILE_FAST;
            if (has_box && lane == 0) {
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(box_bytes) : "memory");
                asm volatile(
                    "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                    ::"r"(box_smem), "l"(&tmap), "r"(ox), "r"(oy), "r"(e), "r"(bar) : "memory");
            }
            // the next exposure's box origin, and an L2 prefetch of that box
            if (e + 1 < e_hi) {
                nbx = __ldg(&(rec + ntile)->bx0); nby = __ldg(&(rec + ntile)->by0); nflag = __ldg(&(rec + ntile)->flag);
                if (STAGE && lane == 0 && nflag == TILE_FAST) {
                    const int fx = (nbx - (Taps<ORDER>::lo + 1)) & ~3, fy = nby - (Taps<ORDER>::lo + 1);
                    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];"
                                 ::"l"(&tmap), "r"(fx), "r"(fy), "r"(e + 1) : "memory");
                }
            }
            TileHead H;
            {
                const int4 h0 = __ldg(reinterpret_cast<const int4 *>(&rec->ix0));       // ix0 iy0 bx0 by0
                const int4 h1 = __ldg(reinterpret_cast<const int4 *>(&rec->bx1));       // bx1 by1 flag deg
                H.ix0 = h0.x; H.iy0 = h0.y; H.bx0 = h0.z; H.by0 = h0.w; H.bx1 = h1.x; H.by1 = h1.y; H.flag = h1.z; H.deg = h1.w;
            }
            sink.begin_exposure(__ldg(S.weights + e));
            // per-lane column polynomials in dj, while the box is in flight
            float X[4], Y[4];
            column_polys(rec, lane, X, Y);
            if (has_box) {
                mbar_wait(bar, phase);
                phase ^= 1u;
            }
            dfr_chk_set(has_box ? box_smem : 0u, has_box ? box_smem + box_bytes : 0u);
            warp_tile<ORDER, STAGE>(P, tgt, e, ttx, tty, lane, H, X, Y, box_smem, ox, oy, sink);
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            __syncwarp();                                   // every lane is done with the box
        }
    }

    // ---- epilogue: accumulators -> sum, wsum (one coalesced 128-byte row per warp and row)
    if (active) {
        const int col = ttx * TS + lane, ty0 = tty * TS;
        const int rows = min(TS, P.ony - ty0);
        float *part = S.nchunk > 1 ? S.partial + ((size_t)chunk * ntile + tile) * (2 * TS * TS) : nullptr;
        for (int r = 0; r < TS; r += 4) {
            float a[4], c[4];
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                         : "=f"(a[0]), "=f"(a[1]), "=f"(a[2]), "=f"(a[3]) : "r"(sink.taddr + (uint32_t)r));
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                         : "=f"(c[0]), "=f"(c[1]), "=f"(c[2]), "=f"(c[3]) : "r"(sink.taddr + (uint32_t)(TS + r)));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float ws = sink.tileW + c[k];
                if (S.nchunk > 1) {
                    part[(r + k) * TS + lane] = a[k];
                    part[TS * TS + (r + k) * TS + lane] = ws;
                } else if (r + k < rows && col < P.onx) {
                    const size_t o = (size_t)(ty0 + r + k) * P.onx + col;
                    S.sum[o] = S.add ? S.sum[o] + a[k] : a[k];
                    S.wsum[o] = S.add ? S.wsum[o] + ws : ws;
                }
            }
        }
        if (S.nchunk > 1) {
            // the last chunk of this tile to arrive adds the partial tiles in chunk order
            __threadfence();
            __syncwarp();
            int t = 0;
            if (lane == 0) t = atomicAdd(S.ticket + tile, 1);
            t = __shfl_sync(0xffffffffu, t, 0);
            if (t == S.nchunk - 1) {
                __threadfence();
                const float *p0 = S.partial + (size_t)tile * (2 * TS * TS);
                const size_t cs = (size_t)ntile * (2 * TS * TS);
                for (int r = 0; r < rows; ++r) {
                    if (col >= P.onx) break;
                    float a = 0.0f, c = 0.0f;
                    for (int q = 0; q < S.nchunk; ++q) {
                        a += __ldcg(p0 + q * cs + r * TS + lane);
                        c += __ldcg(p0 + q * cs + TS * TS + r * TS + lane);
                    }
                    const size_t o = (size_t)(ty0 + r) * P.onx + col;
                    S.sum[o] = S.add ? S.sum[o] + a : a;
                    S.wsum[o] = S.add ? S.wsum[o] + c : c;
                }
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kStackCols) : "memory");
}

#ifdef DFR_BOUNDS_CHECK
}  // namespace dfr
extern "C" unsigned long long dfr_dev_oob_stack()
{
    unsigned long long v = 0, zero = 0;
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(&v, dfr::dfr_oob_count, sizeof v);
    cudaMemcpyToSymbol(dfr::dfr_oob_count, &zero, sizeof zero);
    return v;
}
namespace dfr {
#endif

__global__ void stack_finalize_kernel(const float *__restrict__ sum, const float *__restrict__ wsum,
                                      long long npix, float *__restrict__ mean)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < npix) {
        const float w = wsum[i];
        mean[i] = (w != 0.0f) ? sum[i] / w : qnanf();
    }
}

// a[k] += b[k]: the reduction step of the multi-device stack (partial sums of two shards)
__global__ void stack_add_kernel(float *__restrict__ a, const float *__restrict__ b, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] += b[i];
}

template <int ORDER, bool STAGE>
static cudaError_t launch_stack(TiledParams P, const TargetDev &tgt, const CUtensorMap &tmap, size_t box_bytes,
                                const StackParams &S, cudaStream_t st, void **scratch)
{
    auto kern = tiled_stack_kernel<ORDER, STAGE>;
    P.stage_bytes = (int)((box_bytes + 127) & ~(size_t)127);
    P.rec_off = 0;
    const size_t smem = (size_t)kStackWarps * P.stage_bytes;
    P.e0 = 0;
    // Per (kernel, device), once: the shared-memory opt-in to the constant maximum (never to this call's
    // own size — the attribute is per function and device, so two host threads stacking on one device
    // with different box sizes would otherwise lower each other's limit between set and launch) and the
    // resource figures the resident-CTA estimate below needs (no runtime queries on later calls).
    struct DevInfo {
        std::atomic<int> ready{0};
        int sms = 0, smem_sm = 0, regs_sm = 0, static_smem = 0, regs = 0;
    };
    constexpr int kDevs = 64;
    constexpr size_t kMaxSmem = (size_t)kStackWarps * ((kStackMaxBoxBytes + 127) & ~(size_t)127);
    static DevInfo info[kDevs];
    static std::mutex info_mu;
    if (smem > kMaxSmem) return cudaErrorInvalidValue;
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    DevInfo uncached;                                    // device ordinals beyond the table: queried every call
    DevInfo *I = (dev >= 0 && dev < kDevs) ? &info[dev] : &uncached;
    if (!I->ready.load(std::memory_order_acquire)) {
        std::lock_guard<std::mutex> lock(info_mu);
        if (!I->ready.load(std::memory_order_relaxed)) {
            cudaFuncAttributes fa;
            err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
            if (err == cudaSuccess) err = cudaDeviceGetAttribute(&I->sms, cudaDevAttrMultiProcessorCount, dev);
            if (err == cudaSuccess) err = cudaFuncGetAttributes(&fa, kern);
            if (err == cudaSuccess) err = cudaDeviceGetAttribute(&I->smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
            if (err == cudaSuccess) err = cudaDeviceGetAttribute(&I->regs_sm, cudaDevAttrMaxRegistersPerMultiprocessor, dev);
            if (err != cudaSuccess) return err;
            I->static_smem = (int)fa.sharedSizeBytes;
            I->regs = fa.numRegs;
            I->ready.store(1, std::memory_order_release);
        }
    }
    // resident CTAs per SM from the kernel's own resources: shared memory, registers, TMEM columns
    const int sms = I->sms, smem_sm = I->smem_sm, regs_sm = I->regs_sm;
    struct { size_t sharedSizeBytes; int numRegs; } fa = {(size_t)I->static_smem, I->regs};
    int per_sm = std::min(512 / kStackCols, 32);
    per_sm = (int)std::min<long long>(per_sm, smem_sm / (long long)(smem + fa.sharedSizeBytes + 1024));
    per_sm = std::max(1, std::min(per_sm, regs_sm / std::max(1, ((fa.numRegs + 7) & ~7) * kStackThreads)));
    // Exposure chunks: a CTA runs for (exposures in its chunk) x (one tile's time). With enough
    // tiles to fill the machine one chunk is best (no reduction at all); small outputs are cut
    // along the exposure list until the waves fill evenly.
    const int groups_x = (P.tiles_x + kStackWarps - 1) / kStackWarps;
    const long long ctas = (long long)groups_x * P.tiles_y;
    const double slots = (double)sms * per_sm;
    int best = 1;
    double best_cost = 1e300;
    for (int z = 1; z <= std::min(P.n, 16); ++z) {
        const double per_cta = std::ceil((double)P.n / z) + 1.0;          // + prologue, epilogue, reduction
        const double cost = std::ceil((double)ctas * z / slots) * per_cta;
        if (cost < best_cost * 0.97) { best_cost = cost; best = z; }
    }
    StackParams S2 = S;
#ifdef DFR_DEV_HOOKS
    if (const char *zc = std::getenv("DFR_STACK_Z")) best = std::max(1, std::min(std::atoi(zc), std::min(P.n, 64)));
#endif
    if (ctas * best > 0x7fffffffLL || best > 65535) return cudaErrorInvalidConfiguration;
    S2.nchunk = best;
    S2.partial = nullptr;
    S2.ticket = nullptr;
    if (best > 1) {
        const size_t ntile = (size_t)P.tiles_x * P.tiles_y, b_part = sizeof(float) * 2 * TS * TS * ntile * best;
        if ((err = scratch_alloc(scratch, b_part + sizeof(int32_t) * ntile, st)) != cudaSuccess) return err;
        S2.partial = static_cast<float *>(*scratch);
        S2.ticket = reinterpret_cast<int32_t *>(static_cast<char *>(*scratch) + b_part);
        if ((err = cudaMemsetAsync(S2.ticket, 0, sizeof(int32_t) * ntile, st)) != cudaSuccess) return err;
    }
    return launch_pdl(kern, dim3((unsigned)ctas, (unsigned)best), dim3(kStackThreads), smem, st, P, tgt, tmap, S2);
}

cudaError_t launch_tiled_stack(const float *src, int n, int sny, int snx, const TargetDev &tgt,
                               const SourceDev *srcdev, const SourceDev *srchost, int ony, int onx, int order,
                               const float *dev_weights, float *sum, float *wsum, int accumulate,
                               cudaStream_t st, int32_t *host_stats, int stats_add, TiledStats *stats, ProfileEvents *prof,
                               const ConstsCopy &cc)
{
    Prepared R;
    if (prof && prof->enabled) cudaEventRecord(prof->setup_begin, st);
    // the staged boxes are per 32x32 tile (one per warp)
    cudaError_t err = prepare_tiled(src, n, sny, snx, tgt, srcdev, srchost, ony, onx, order, st, host_stats, stats_add, R,
                                    cc, 1, kStackMaxBoxBytes);
    if (err != cudaSuccess) { free_scratch(R.sc, st); return err; }
    StackParams S;
    S.weights = dev_weights; S.sum = sum; S.wsum = wsum; S.partial = nullptr; S.ticket = nullptr;
    S.add = accumulate; S.nchunk = 1;
    void *red_scratch = nullptr;
    if (prof && prof->enabled) cudaEventRecord(prof->main_begin, st);
#define DFR_LAUNCH(O)                                                                     \
    err = R.stage ? launch_stack<O, true>(R.P, tgt, R.tmap, R.box_bytes, S, st, &red_scratch)                        \
                  : launch_stack<O, false>(R.P, tgt, R.tmap, 0, S, st, &red_scratch)
    if (order == DFR_NEAREST) DFR_LAUNCH(DFR_NEAREST);
    else if (order == DFR_BILINEAR) DFR_LAUNCH(DFR_BILINEAR);
    else DFR_LAUNCH(DFR_BICUBIC);
#undef DFR_LAUNCH
    if (prof && prof->enabled) cudaEventRecord(prof->main_end, st);
    if (red_scratch) cudaFreeAsync(red_scratch, st);
    free_scratch(R.sc, st);
    stats->kernels = 3;
    stats->tiles_fast = stats->tiles_exact = stats->tiles_empty = -1;
    return err;
}

cudaError_t launch_stack_add(float *a, const float *b, long long n, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    stack_add_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(a, b, n);
    return cudaGetLastError();
}

cudaError_t launch_stack_finalize(const float *sum, const float *wsum, long long npix, float *mean, cudaStream_t st)
{
    if (npix <= 0) return cudaSuccess;
    stack_finalize_kernel<<<(unsigned)((npix + 255) / 256), 256, 0, st>>>(sum, wsum, npix, mean);
    return cudaGetLastError();
}


}  // namespace dfr
