// dfr_tiled_stack.cu — fused reproject-and-stack (dfr_reproject_stack).
#include <algorithm>
#include <cmath>
#include <cstring>

#include "dfr_tiled_device.cuh"

namespace dfr {

// ---------------------------------------------------------------------------------
// fused reproject-and-stack (dfr_reproject_stack)
//
// One CTA per 64x64 output tile loops over the exposures; the per-pixel accumulators
//   sum += w_e v_e,  wsum += w_e   (only where v_e is not NaN)
// of each warp's 32x32 tile (2 x 32 rows per lane) live in TENSOR MEMORY: 64 TMEM columns
// per CTA, lane = output column, column = row (sum) / 32 + row (wsum), read and written
// four rows at a time with tcgen05.ld / tcgen05.st (32x32b.x4). They never occupy
// registers for longer than four pixels, there is no per-exposure output in HBM, and the
// row loop stays a loop. The source boxes arrive through a two-stage TMA ring: while
// exposure e is accumulated out of stage e & 1, the box of e + 1 is in flight.
// ---------------------------------------------------------------------------------
struct StackSink {
    static constexpr bool kAllLanes = true;        // tcgen05.ld/st are warp-wide: nobody leaves
    uint32_t taddr;                                // TMEM address of this warp's row 0 (sum)
    float w;                                       // weight of the current exposure
    int r;                                         // next row
    float s0, s1, s2, s3, c0, c1, c2, c3;          // accumulators of rows r .. r + 3 in flight
    __device__ __forceinline__ void prefetch4()
    {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=f"(s0), "=f"(s1), "=f"(s2), "=f"(s3) : "r"(taddr + (uint32_t)r));
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=f"(c0), "=f"(c1), "=f"(c2), "=f"(c3) : "r"(taddr + (uint32_t)(TS + r)));
    }
    __device__ __forceinline__ void add(float &s, float &c, float v) const
    {
        const bool ok = v == v;                    // NaN: outside the footprint, or NaN taps
        s = ok ? fmaf(w, v, s) : s;
        c = ok ? c + w : c;
    }
    __device__ __forceinline__ void rows4(float v0, float v1, float v2, float v3)
    {
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        add(s0, c0, v0); add(s1, c1, v1); add(s2, c2, v2); add(s3, c3, v3);
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                     ::"r"(taddr + (uint32_t)r), "f"(s0), "f"(s1), "f"(s2), "f"(s3) : "memory");
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                     ::"r"(taddr + (uint32_t)(TS + r)), "f"(c0), "f"(c1), "f"(c2), "f"(c3) : "memory");
        r += 4;
    }
    __device__ __forceinline__ void row1(float v)
    {
        float s, c;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=f"(s) : "r"(taddr + (uint32_t)r));
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=f"(c) : "r"(taddr + (uint32_t)(TS + r)));
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        add(s, c, v);
        asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr + (uint32_t)r), "f"(s) : "memory");
        asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr + (uint32_t)(TS + r)), "f"(c) : "memory");
        r += 1;
    }
    __device__ __forceinline__ void empty_tile(int) {}           // an empty tile adds nothing
};

constexpr int kStackCols = 2 * TS;                 // TMEM columns per CTA (power of two >= 32)

struct StackParams {
    const float *weights;                          // DEVICE [n]
    float *sum, *wsum;                             // DEVICE [ony][onx]
    int add;                                       // 0: plain stores (one chunk, overwrite); 1: atomic adds
    int nchunk;                                    // exposure chunks = gridDim.z
};

constexpr int kStackConsumers = CTA_T * CTA_T;                  // compute warps per CTA
constexpr int kStackThreads = 32 * (kStackConsumers + 1);       // + one producer warp
constexpr int kRecBytes = kStackConsumers * (int)sizeof(TileRec);

// the producer's wait: let the hardware suspend the thread (time hint) instead of spinning,
// so the wait takes no issue slots from the compute warps
__device__ __forceinline__ void mbar_wait_sleep(uint32_t bar, uint32_t parity)
{
    for (;;) {
        uint32_t done;
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(bar), "r"(parity), "r"(20000u) : "memory");
        if (done) break;
    }
}

// stage = [ box BW x BH floats | the CTA tile's 4 TileRec | head ]; STAGE = false: records only
template <int ORDER, bool STAGE>
__global__ void __launch_bounds__(kStackThreads)
tiled_stack_kernel(const __grid_constant__ TiledParams P, const __grid_constant__ TargetDev tgt,
                   const __grid_constant__ CUtensorMap tmap, const __grid_constant__ StackParams S)
{
    extern __shared__ __align__(128) unsigned char stages[];
    __shared__ __align__(8) unsigned long long full[2], empty[2];
    __shared__ int4 head[2];                                       // has_box, ox, oy
    __shared__ uint32_t tmem_base;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ntile = P.tiles_x * P.tiles_y, ctas = P.ctas_x * P.ctas_y;
    const int cta = blockIdx.y * P.ctas_x + blockIdx.x;
    // this CTA's chunk of the exposure list (grid.z chunks balance the waves; partial sums
    // of different chunks meet in global memory through atomic adds)
    const int e_lo = (int)((long long)blockIdx.z * P.n / S.nchunk);
    const int e_hi = (int)((long long)(blockIdx.z + 1) * P.n / S.nchunk);

    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     ::"r"(smem_u32(&tmem_base)), "n"(kStackCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < 2; ++s) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&full[s])));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(&empty[s])), "r"(kStackConsumers));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    pdl_wait();                         // the setup kernel's records and box origins are complete

    if (warp == kStackConsumers) {
        // ------------------------------ producer (one lane) ------------------------------
        if (lane == 0) {
            const uint32_t box_bytes = (uint32_t)(P.BW * P.BH * sizeof(float));
            // the CTA tile's records: up to two runs (tile rows) of up to two records
            const int tx0 = blockIdx.x * CTA_T, ty0 = blockIdx.y * CTA_T;
            const uint32_t run = (uint32_t)min(CTA_T, P.tiles_x - tx0) * (uint32_t)sizeof(TileRec);
            const int nrun = min(CTA_T, P.tiles_y - ty0);
            for (int e = e_lo; e < e_hi; ++e) {
                const int k = e - e_lo, s = k & 1;
                int2 cb = make_int2(kNoBox, kNoBox);
                if (STAGE) cb = __ldg(P.cta_box + (size_t)e * ctas + cta);
                if (k >= 2) mbar_wait_sleep(smem_u32(&empty[s]), ((uint32_t)(k >> 1) & 1u) ^ 1u);
                const int hb = STAGE && cb.x != kNoBox;
                // TMA wants a 16-byte aligned start along x (measured on B200): round down to 4 floats
                const int ox = (cb.x - (Taps<ORDER>::lo + 1)) & ~3, oy = cb.y - (Taps<ORDER>::lo + 1);
                head[s] = make_int4(hb, ox, oy, 0);
                unsigned char *st = stages + (size_t)s * P.stage_bytes;
                const uint32_t bar = smem_u32(&full[s]);
                const uint32_t bytes = (hb ? box_bytes : 0u) + run * (uint32_t)nrun;
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
                for (int q = 0; q < nrun; ++q)
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                 ::"r"(smem_u32(st + P.rec_off + q * CTA_T * (int)sizeof(TileRec))),
                                   "l"(P.recs + ((size_t)e * ntile + (size_t)(ty0 + q) * P.tiles_x + tx0)), "r"(run), "r"(bar)
                                 : "memory");
                if (hb)
                    asm volatile(
                        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                        ::"r"(smem_u32(st)), "l"(&tmap), "r"(ox), "r"(oy), "r"(e), "r"(bar) : "memory");
            }
        }
    } else {
        // ------------------------------ consumers ------------------------------
        const int ttx = blockIdx.x * CTA_T + (warp % CTA_T), tty = blockIdx.y * CTA_T + (warp / CTA_T);
        const bool active = ttx < P.tiles_x && tty < P.tiles_y;
        StackSink sink;
        sink.taddr = tmem_base + ((uint32_t)(warp * 32) << 16);
        sink.w = 0.0f;
        sink.r = 0;
        for (int g = 0; g < kStackCols; g += 4)                    // zero sum and wsum
            asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %1, %1, %1};"
                         ::"r"(sink.taddr + (uint32_t)g), "f"(0.0f) : "memory");
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");

        for (int e = e_lo; e < e_hi; ++e) {
            const int k = e - e_lo, s = k & 1;
            sink.w = __ldg(S.weights + e);
            sink.r = 0;
            mbar_wait(smem_u32(&full[s]), (uint32_t)(k >> 1) & 1u);
            if (active) {
                const unsigned char *st = stages + (size_t)s * P.stage_bytes;
                const TileRec *rec = reinterpret_cast<const TileRec *>(st + P.rec_off) + warp;
                const int4 h0 = *reinterpret_cast<const int4 *>(&rec->ix0);    // ix0 iy0 bx0 by0
                const int4 h1 = *reinterpret_cast<const int4 *>(&rec->bx1);    // bx1 by1 flag deg
                TileHead H;
                H.ix0 = h0.x; H.iy0 = h0.y; H.bx0 = h0.z; H.by0 = h0.w; H.bx1 = h1.x; H.by1 = h1.y; H.flag = h1.z; H.deg = h1.w;
                float X[4], Y[4];
                const float di = (float)lane - (float)kCentre;
                const float4 *c4 = reinterpret_cast<const float4 *>(rec->cx);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float4 a = c4[q], b = c4[4 + q];
                    X[q] = fmaf(fmaf(fmaf(a.w, di, a.z), di, a.y), di, a.x);
                    Y[q] = fmaf(fmaf(fmaf(b.w, di, b.z), di, b.y), di, b.x);
                }
                const int4 hd = head[s];
                warp_tile<ORDER, STAGE>(P, tgt, e, ttx, tty, lane, H, X, Y, smem_u32(st), hd.y, hd.z, sink);
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            __syncwarp();                                   // every lane is done with stage s
            if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&empty[s])) : "memory");
        }

        // ---- epilogue: accumulators -> sum, wsum (one coalesced 128-byte row per warp and row)
        if (active) {
            const int col = ttx * TS + lane, ty0 = tty * TS;
            const int rows = min(TS, P.ony - ty0);
            for (int r = 0; r < TS; r += 4) {
                float a[4], c[4];
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                             : "=f"(a[0]), "=f"(a[1]), "=f"(a[2]), "=f"(a[3]) : "r"(sink.taddr + (uint32_t)r));
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                             : "=f"(c[0]), "=f"(c[1]), "=f"(c[2]), "=f"(c[3]) : "r"(sink.taddr + (uint32_t)(TS + r)));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (r + k < rows && col < P.onx) {
                        const size_t o = (size_t)(ty0 + r + k) * P.onx + col;
                        if (S.add) {
                            atomicAdd(S.sum + o, a[k]);
                            atomicAdd(S.wsum + o, c[k]);
                        } else {
                            S.sum[o] = a[k];
                            S.wsum[o] = c[k];
                        }
                    }
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kStackCols) : "memory");
}

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
                                const StackParams &S, cudaStream_t st)
{
    auto kern = tiled_stack_kernel<ORDER, STAGE>;
    P.rec_off = (int)((box_bytes + 127) & ~(size_t)127);
    P.stage_bytes = (int)((P.rec_off + kRecBytes + 127) & ~(size_t)127);
    const size_t smem = 2 * (size_t)P.stage_bytes;
    {
        cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (err != cudaSuccess) return err;
    }
    if (P.ctas_y > 65535) return cudaErrorInvalidConfiguration;
    P.e0 = 0;
    // Exposure chunks: every CTA runs for (exposures in its chunk) x (one tile's time), so the
    // grid is cut along the exposure list until its waves fill the machine evenly.
    int dev = 0, sms = 0, per_sm = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err == cudaSuccess) err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // resident CTAs per SM from the kernel's own resources (the occupancy API returned 1 for
    // this kernel on B200 / CUDA 12.9): shared memory, registers, TMEM columns
    cudaFuncAttributes fa;
    int smem_sm = 0, regs_sm = 0;
    if (err == cudaSuccess) err = cudaFuncGetAttributes(&fa, kern);
    if (err == cudaSuccess) err = cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
    if (err == cudaSuccess) err = cudaDeviceGetAttribute(&regs_sm, cudaDevAttrMaxRegistersPerMultiprocessor, dev);
    if (err != cudaSuccess) return err;
    const int threads = kStackThreads;
    per_sm = std::min(512 / kStackCols, 32);
    per_sm = std::min<long long>(per_sm, smem_sm / (long long)(smem + fa.sharedSizeBytes + 1024));
    per_sm = std::min(per_sm, regs_sm / std::max(1, ((fa.numRegs + 7) & ~7) * threads));
    const double slots = (double)sms * std::max(per_sm, 1), tiles = (double)P.ctas_x * P.ctas_y;
    int best = 1;
    double best_eff = 0.0;
    for (int z = 1; z <= std::min(P.n, 8); ++z) {
        const double waves = tiles * z / slots, eff = waves / std::ceil(waves);
        if (eff > best_eff + 0.02) { best_eff = eff; best = z; }
    }
    StackParams S2 = S;
    S2.nchunk = best;
    if (best > 1 && !S.add) {                       // partial sums meet by atomic adds: start from zero
        const size_t bytes = sizeof(float) * (size_t)P.ony * P.onx;
        if ((err = cudaMemsetAsync(S.sum, 0, bytes, st)) != cudaSuccess) return err;
        if ((err = cudaMemsetAsync(S.wsum, 0, bytes, st)) != cudaSuccess) return err;
        S2.add = 1;
    }
    const dim3 grid((unsigned)P.ctas_x, (unsigned)P.ctas_y, (unsigned)best);
    return launch_pdl(kern, grid, dim3(kStackThreads), smem, st, P, tgt, tmap, S2);
}

cudaError_t launch_tiled_stack(const float *src, int n, int sny, int snx, const TargetDev &tgt,
                               const SourceDev *srcdev, const SourceDev *srchost, int ony, int onx, int order,
                               const float *dev_weights, float *sum, float *wsum, int accumulate,
                               cudaStream_t st, int32_t *host_stats, int stats_add, TiledStats *stats, ProfileEvents *prof)
{
    Prepared R;
    if (prof && prof->enabled) cudaEventRecord(prof->setup_begin, st);
    cudaError_t err = prepare_tiled(src, n, sny, snx, tgt, srcdev, srchost, ony, onx, order, st, host_stats, stats_add, R);
    if (err != cudaSuccess) { free_scratch(R.sc, st); return err; }
    StackParams S;
    S.weights = dev_weights; S.sum = sum; S.wsum = wsum; S.add = accumulate; S.nchunk = 1;
    if (prof && prof->enabled) cudaEventRecord(prof->main_begin, st);
#define DFR_LAUNCH(O)                                                                     \
    err = R.stage ? launch_stack<O, true>(R.P, tgt, R.tmap, R.box_bytes, S, st) : launch_stack<O, false>(R.P, tgt, R.tmap, 0, S, st)
    if (order == DFR_NEAREST) DFR_LAUNCH(DFR_NEAREST);
    else if (order == DFR_BILINEAR) DFR_LAUNCH(DFR_BILINEAR);
    else DFR_LAUNCH(DFR_BICUBIC);
#undef DFR_LAUNCH
    if (prof && prof->enabled) cudaEventRecord(prof->main_end, st);
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
