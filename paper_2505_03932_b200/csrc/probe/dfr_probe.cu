// dfr_probe.cu — register-only instruction-rate probes. NOT part of libdfr or of include/dfr.h: a
// measurement tool built into its own libdfr_probe.so, which only `bench.py --mode probes` loads
// (through paper_2505_03932_b200.dfr_probe_rates).
//
// The roofline of SURVEY.md §8(d) has an ALU side whose denominator must be MEASURED on the
// device ("register-only FMA micro-benchmark and the actual SM clock recorded"). These
// kernels measure, per SM and per clock, how many thread-level operations of each class the
// B200 retires when nothing else competes: the numbers DESIGN.md §8 uses to say which pipe
// bounds a kernel. Every probe runs kBlocksPerSm x 256 threads per SM, each thread kChains
// independent dependency chains of one instruction class (or an interleaved mix), and the
// cycle count is %clock64 of the longest block.
#include <algorithm>
#include <vector>

#include <cuda_runtime.h>

// Probe classes: out[k] of dfr_probe_rates receives the thread-level INSTRUCTIONS retired per clock
// per SM (every SM loaded with 32 warps of independent chains); a packed FFMA2 counts as one
// instruction (two fp32 FMAs). The three mixed classes interleave two instruction kinds 1:1 and
// report their combined rate: a rate above either kind alone means the two do not share a pipe.
enum { DFR_PROBE_FFMA = 0, DFR_PROBE_FFMA2 = 1, DFR_PROBE_FADD2_RM = 2, DFR_PROBE_DFMA = 3,
       DFR_PROBE_IMAD = 4, DFR_PROBE_LOP3 = 5, DFR_PROBE_LDS = 6,
       DFR_PROBE_FFMA_FFMA2 = 7, DFR_PROBE_FFMA2_IMAD = 8, DFR_PROBE_FFMA2_LOP3 = 9,
       DFR_PROBE_FFMA_3REG = 10, DFR_PROBE_FFMA2_3REG = 11,   /* three distinct, changing register operands */
       DFR_PROBE_COUNT = 12 };

namespace dfr {

constexpr int kProbeThreads = 256;
constexpr int kBlocksPerSm = 4;          // 32 warps per SM
constexpr int kChains = 8;
constexpr int kUnroll = 16;

typedef unsigned long long u64;

__device__ __forceinline__ u64 p_fma2(u64 a, u64 b, u64 c)
{
    u64 r;
    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ u64 p_add2_rm(u64 a, u64 b)
{
    u64 r;
    asm volatile("add.rm.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ float p_fma(float a, float b, float c)
{
    float r;
    asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}
__device__ __forceinline__ double p_dfma(double a, double b, double c)
{
    double r;
    asm volatile("fma.rn.f64 %0, %1, %2, %3;" : "=d"(r) : "d"(a), "d"(b), "d"(c));
    return r;
}
__device__ __forceinline__ unsigned p_imad(unsigned a, unsigned b, unsigned c)
{
    unsigned r;
    asm volatile("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ unsigned p_lop(unsigned a, unsigned b, unsigned c)
{
    unsigned r;
    asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ unsigned p_lds(unsigned addr)
{
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

// KIND: see dfr.h (DFR_PROBE_*). ops = thread-level operations per thread per iteration.
template <int KIND>
__global__ void __launch_bounds__(kProbeThreads)
probe_kernel(int iters, long long *__restrict__ cycles, float *__restrict__ sink)
{
    __shared__ unsigned sm[kProbeThreads];          // per warp: a 32-entry permutation (index chase, conflict-free)
    sm[threadIdx.x] = 4u * ((threadIdx.x + 7u) & 31u);
    __syncthreads();
    float f[kChains];
    u64 p[kChains];
    double d[kChains];
    unsigned u[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) {
        f[k] = 1.0f + 0.001f * (float)(threadIdx.x + k);
        p[k] = ((u64)__float_as_uint(f[k]) << 32) | __float_as_uint(f[k]);
        d[k] = (double)f[k];
        u[k] = (KIND == DFR_PROBE_LDS) ? 4u * ((threadIdx.x + (unsigned)k) & 31u) : threadIdx.x * 4u + (unsigned)k;
    }
    const float fa = 0.999f, fb = 1e-3f;
    const u64 pa = ((u64)__float_as_uint(fa) << 32) | __float_as_uint(fa), pb = ((u64)__float_as_uint(fb) << 32) | __float_as_uint(fb);
    const unsigned lbase = (unsigned)__cvta_generic_to_shared(sm) + 4u * (threadIdx.x & ~31u);
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < kUnroll; ++r) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) {
                if (KIND == DFR_PROBE_FFMA) f[k] = p_fma(f[k], fa, fb);
                if (KIND == DFR_PROBE_FFMA2) p[k] = p_fma2(p[k], pa, pb);
                if (KIND == DFR_PROBE_FADD2_RM) p[k] = p_add2_rm(p[k], pb);
                if (KIND == DFR_PROBE_DFMA) d[k] = p_dfma(d[k], 0.999, 1e-3);
                if (KIND == DFR_PROBE_IMAD) u[k] = p_imad(u[k], 3u, u[(k + 1) % kChains]);
                if (KIND == DFR_PROBE_LOP3) u[k] = p_lop(u[k], u[(k + 1) % kChains], 0x5a5a5a5au);
                if (KIND == DFR_PROBE_LDS) u[k] = p_lds(lbase + u[k]);      // the lanes of a warp always hold a permutation
                if (KIND == DFR_PROBE_FFMA_FFMA2) {   // one scalar + one packed per slot: do they share a pipe?
                    f[k] = p_fma(f[k], fa, fb);
                    p[k] = p_fma2(p[k], pa, pb);
                }
                if (KIND == DFR_PROBE_FFMA2_IMAD) {
                    p[k] = p_fma2(p[k], pa, pb);
                    u[k] = p_imad(u[k], 3u, u[(k + 1) % kChains]);
                }
                // three DISTINCT, changing register operands per instruction (no operand-reuse hits):
                // what the interpolation code looks like, unlike the chains above whose multiplier and
                // addend never change
                if (KIND == DFR_PROBE_FFMA_3REG) f[k] = p_fma(f[(k + 1) % kChains], f[(k + 2) % kChains], f[k]);
                if (KIND == DFR_PROBE_FFMA2_3REG) p[k] = p_fma2(p[(k + 1) % kChains], p[(k + 2) % kChains], p[k]);
                if (KIND == DFR_PROBE_FFMA2_LOP3) {
                    p[k] = p_fma2(p[k], pa, pb);
                    u[k] = p_lop(u[k], u[(k + 1) % kChains], 0x5a5a5a5au);
                }
            }
        }
    }
    const long long t1 = clock64();
    float acc = 0.0f;
#pragma unroll
    for (int k = 0; k < kChains; ++k)
        acc += f[k] + __uint_as_float((unsigned)p[k]) + __uint_as_float((unsigned)(p[k] >> 32)) + (float)d[k] + (float)u[k];
    if (acc == 123.456f) sink[0] = acc;              // keeps the chains alive
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

template <int KIND>
static cudaError_t run_probe(int sms, int iters, long long *dcyc, float *dsink, double *instr_per_clk_sm)
{
    const int blocks = sms * kBlocksPerSm;
    probe_kernel<KIND><<<blocks, kProbeThreads>>>(8, dcyc, dsink);           // warm-up
    probe_kernel<KIND><<<blocks, kProbeThreads>>>(iters, dcyc, dsink);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    std::vector<long long> h((size_t)blocks);
    if ((err = cudaMemcpy(h.data(), dcyc, sizeof(long long) * (size_t)blocks, cudaMemcpyDeviceToHost)) != cudaSuccess) return err;
    const long long worst = *std::max_element(h.begin(), h.end());
    const int per_slot = (KIND >= DFR_PROBE_FFMA_FFMA2 && KIND <= DFR_PROBE_FFMA2_LOP3) ? 2 : 1;         // thread-level INSTRUCTIONS per chain step
    const double instr = (double)iters * kUnroll * kChains * per_slot * kProbeThreads * kBlocksPerSm;
    *instr_per_clk_sm = instr / (double)worst;
    return cudaSuccess;
}

cudaError_t probe_rates(double *out /* [DFR_PROBE_COUNT] thread-instructions per clock per SM */)
{
    int dev = 0, sms = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err == cudaSuccess) err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (err != cudaSuccess) return err;
    long long *dcyc = nullptr;
    float *dsink = nullptr;
    if ((err = cudaMalloc((void **)&dcyc, sizeof(long long) * (size_t)sms * kBlocksPerSm)) != cudaSuccess) return err;
    if ((err = cudaMalloc((void **)&dsink, sizeof(float))) != cudaSuccess) { cudaFree(dcyc); return err; }
    const int iters = 2000;
#define DFR_RUN(K) if (err == cudaSuccess) err = run_probe<K>(sms, iters, dcyc, dsink, &out[K])
    DFR_RUN(DFR_PROBE_FFMA);
    DFR_RUN(DFR_PROBE_FFMA2);
    DFR_RUN(DFR_PROBE_FADD2_RM);
    DFR_RUN(DFR_PROBE_DFMA);
    DFR_RUN(DFR_PROBE_IMAD);
    DFR_RUN(DFR_PROBE_LOP3);
    DFR_RUN(DFR_PROBE_LDS);
    DFR_RUN(DFR_PROBE_FFMA_FFMA2);
    DFR_RUN(DFR_PROBE_FFMA2_IMAD);
    DFR_RUN(DFR_PROBE_FFMA2_LOP3);
    DFR_RUN(DFR_PROBE_FFMA_3REG);
    DFR_RUN(DFR_PROBE_FFMA2_3REG);
#undef DFR_RUN
    cudaFree(dcyc);
    cudaFree(dsink);
    return err;
}

}  // namespace dfr

// HOST out[n], n >= DFR_PROBE_COUNT. Synchronous, ~50 ms on the current device. Returns 0, -1 (NULL),
// -2 (n too small) or -8 (CUDA failure: dfr_probe_error() has the text).
static thread_local cudaError_t g_probe_err = cudaSuccess;
extern "C" int dfr_probe_rates(double *out, int n)
{
    if (!out) return -1;
    if (n < DFR_PROBE_COUNT) return -2;
    g_probe_err = dfr::probe_rates(out);
    return g_probe_err == cudaSuccess ? 0 : -8;
}
extern "C" const char *dfr_probe_error(void) { return cudaGetErrorString(g_probe_err); }
