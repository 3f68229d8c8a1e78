// dfr_tiled_device.cuh — device code shared by the tiled kernels:
// programmatic dependent launch, the packed fp32 pair arithmetic, the per-pixel gathers
// from the TMA-staged box, and warp_tile (one 32x32 tile by one warp) with its sinks.
#pragma once
#include <cuda.h>

#include "dfr_device.cuh"
#include "dfr_tiled.h"

namespace dfr {

// Programmatic dependent launch (PDL): a kernel launched with launch_pdl() may start while
// its predecessor in the stream is still running; it must call pdl_wait() before touching
// anything the predecessor writes. pdl_trigger() in the predecessor allows that early start.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <class... KArgs, class... Args>
static cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

constexpr double kHalf = 0.5 * TS;            // 16: pixel offset of s = 1
constexpr double kCentre = 0.5 * (TS - 1);    // 15.5: tile centre relative to its first pixel

// ---------------------------------------------------------------------------------
// pieces of the main kernel
// ---------------------------------------------------------------------------------
// The source coordinate of a FAST tile, ONE definition for every kernel that needs it (the
// reprojection and stacking kernels, the footprint pass, and dfr_src_coords, which SURVEY.md §8(b)
// requires to run "the same __device__ function as dfr_reproject"):
//   x(lane, r) = ix0 + sum_q X[q] dj^q,   dj = r - kCentre,   X[q] = sum_p cx[q][p] di^p,   di = lane - kCentre
// (and y likewise), all in fp32 with the fused multiply-adds in exactly this order.
// column_polys: the per-lane polynomials in dj from the tile record's 2 x 16 coefficients.
__device__ __forceinline__ void column_polys(const TileRec *__restrict__ rec, int lane, float X[4], float Y[4])
{
    const float di = (float)lane - (float)kCentre;
    const float4 *c4 = reinterpret_cast<const float4 *>(rec->cx);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float4 a = __ldg(c4 + q), b = __ldg(c4 + 4 + q);
        X[q] = fmaf(fmaf(fmaf(a.w, di, a.z), di, a.y), di, a.x);
        Y[q] = fmaf(fmaf(fmaf(b.w, di, b.z), di, b.y), di, b.x);
    }
}
// truncate_degree: the setup kernel found that the dj^3 (dj^2) terms cannot move a coordinate of this
// tile by 2.5e-7 px (TileRec::deg): they are dropped, on every path alike.
__device__ __forceinline__ void truncate_degree(int deg, float X[4], float Y[4])
{
    if (deg < 3) { X[3] = 0.0f; Y[3] = 0.0f; }
    if (deg < 2) { X[2] = 0.0f; Y[2] = 0.0f; }
}
// tile_coord: the coordinate (relative to ix0, iy0) in row r of the tile, scalar form (the packed
// interior loop of warp_tile evaluates the same Horner chain two rows at a time).
__device__ __forceinline__ void tile_coord(const float X[4], const float Y[4], int r, float &xl, float &yl)
{
    const float dj = (float)r - (float)kCentre;
    xl = fmaf(fmaf(fmaf(X[3], dj, X[2]), dj, X[1]), dj, X[0]);
    yl = fmaf(fmaf(fmaf(Y[3], dj, Y[2]), dj, Y[1]), dj, Y[0]);
}

constexpr float kMagic = 12582912.0f;              // 1.5 * 2^23: ulp 1 on [2^23, 2^24)
constexpr int kMagicBits = 0x4B400000;

template <int ORDER> struct Taps;
template <> struct Taps<DFR_NEAREST>  { static constexpr int lo = 0, hi = 1; };   // rint in {floor, floor+1}
template <> struct Taps<DFR_BILINEAR> { static constexpr int lo = 0, hi = 1; };
template <> struct Taps<DFR_BICUBIC>  { static constexpr int lo = 1, hi = 2; };


__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}

// index range [A_lo, A_hi] of the base tap for which every tap is inside the image AND
// inside the staged box [o, o + B)
template <int ORDER>
__device__ __forceinline__ void axis_range(int n, int o, int B, int &A_lo, int &A_hi)
{
    if (ORDER == DFR_NEAREST) { A_lo = max(0, o); A_hi = min(n - 1, o + B - 1); }
    else if (ORDER == DFR_BILINEAR) { A_lo = max(0, o); A_hi = min(n - 2, o + B - 2); }
    else { A_lo = max(1, o + 1); A_hi = min(n - 3, o + B - 3); }
}

// Slow pixel of a FAST tile: polynomial coordinate, rim/out-of-box handling by the exact
// footprint rule and edge-replicated global gathers.
template <int ORDER, int EDGE>
__device__ __noinline__ float slow_poly_pixel(const float *__restrict__ img, int sny, int snx,
                                              int ix0, int iy0, float xl, float yl)
{
    const double x = (double)ix0 + (double)xl, y = (double)iy0 + (double)yl;
    if (!in_footprint(x, y, sny, snx, EDGE)) return qnanf();
    return sample_global<ORDER>(img, sny, snx, x, y);
}

template <int ORDER, int EDGE>
__device__ __noinline__ float exact_pixel(const float *__restrict__ img, int sny, int snx,
                                          const TargetDev &tgt, const SourceDev &s, int i, int j)
{
    double U, V, x, y;
    target_uv(tgt, (double)i, (double)j, U, V);
    source_xy(s, U, V, x, y);
    if (!in_footprint(x, y, sny, snx, EDGE)) return qnanf();
    return sample_global<ORDER>(img, sny, snx, x, y);
}

// Where the fast path gathers from: the TMA-staged box in shared memory (STAGE) or the
// source image itself (no staging). Shared loads use 32-bit shared-window addresses so
// the address arithmetic is one IMAD + one LEA per pixel.
template <bool STAGE> struct GatherSrc {
    int pitch;                       // floats per row
    uint32_t sbase;                  // STAGE: shared address of element (0, 0)
    const float *gbase;              // !STAGE: global address of element (0, 0)
};

#ifdef DFR_BOUNDS_CHECK
// Checked build (never shipped): compute-sanitizer is not available on the GPU pool, so the
// unchecked gathers of the packed loops are verified by an instrumented build instead. Every staged
// load checks its address against the box the current warp may read — set by the kernels with
// dfr_chk_set: the CTA's box (reproject) or the warp's own box (stack) — and against 4-byte
// alignment; violations are counted in dfr_oob_count and the load is redirected to the box start.
// dfr_dev_oob_main() / dfr_dev_oob_stack() (extern "C") return and clear the counts.
static __device__ unsigned long long dfr_oob_count;
__device__ __forceinline__ uint2 &dfr_chk_range()
{
    __shared__ uint2 r[8];
    return r[(threadIdx.x >> 5) & 7];
}
__device__ __forceinline__ void dfr_chk_set(uint32_t lo, uint32_t hi)
{
#ifdef DFR_BOUNDS_SELFTEST                      // negative control: declare a box 256 bytes long
    hi = hi > lo + 256u ? lo + 256u : hi;
#endif
    dfr_chk_range() = make_uint2(lo, hi);
    __syncwarp();
}
__device__ __forceinline__ uint32_t dfr_chk(uint32_t a)
{
    const uint2 r = dfr_chk_range();
    if (a < r.x || a + 4u > r.y || (a & 3u)) {
        atomicAdd(&dfr_oob_count, 1ull);
        return r.x;
    }
    return a;
}
#else
__device__ __forceinline__ void dfr_chk_set(uint32_t, uint32_t) {}
__device__ __forceinline__ uint32_t dfr_chk(uint32_t a) { return a; }
#endif

__device__ __forceinline__ float lds_f32(uint32_t a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(dfr_chk(a)));
    return v;
}
__device__ __forceinline__ float lds_f32_4(uint32_t a)
{
#ifdef DFR_BOUNDS_CHECK
    return lds_f32(a + 4u);
#else
    float v;
    asm volatile("ld.shared.f32 %0, [%1+4];" : "=f"(v) : "r"(a));
    return v;
#endif
}

// One pixel of a FAST tile: floor/rint by a magic add, range test, gather, interpolate.
// `ok` = every tap is inside the image and inside the staged box; when it is false the
// loads are redirected to element (0, 0) and the value is discarded by the caller.
template <int ORDER, bool STAGE>
__device__ __forceinline__ float fast_pixel(const GatherSrc<STAGE> &G, float xl, float yl, int Cx, int Cy,
                                            unsigned cntx, unsigned cnty, bool &ok)
{
    float Tx, Ty;
    if (ORDER == DFR_NEAREST) { Tx = xl + kMagic; Ty = yl + kMagic; }             // rint (half-even)
    else { Tx = __fadd_rd(xl, kMagic); Ty = __fadd_rd(yl, kMagic); }               // floor
    const float fx = xl - (Tx - kMagic), fy = yl - (Ty - kMagic);
    const int kx = __float_as_int(Tx) - Cx, ky = __float_as_int(Ty) - Cy;
    ok = ((unsigned)kx < cntx) && ((unsigned)ky < cnty);
    const int idx = ok ? ky * G.pitch + kx : 0;
    if (STAGE) {
        const uint32_t a0 = G.sbase + 4u * (unsigned)idx;
        if (ORDER == DFR_NEAREST) return lds_f32(a0);
        const uint32_t p4 = 4u * (unsigned)G.pitch;
        if (ORDER == DFR_BILINEAR) {
            const uint32_t a1 = a0 + p4;
            const float s00 = lds_f32(a0), s10 = lds_f32_4(a0), s01 = lds_f32(a1), s11 = lds_f32_4(a1);
            const float top = fmaf(fx, s10 - s00, s00);
            const float bot = fmaf(fx, s11 - s01, s01);
            return fmaf(fy, bot - top, top);
        }
        float wx[4], wy[4];
        keys_weights(fx, wx);
        keys_weights(fy, wy);
        float acc = 0.0f;
        uint32_t a = a0;
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            float row = wx[0] * lds_f32(a);
            row = fmaf(wx[1], lds_f32_4(a), row);
            row = fmaf(wx[2], lds_f32(a + 8), row);
            row = fmaf(wx[3], lds_f32_4(a + 8), row);
            acc = fmaf(wy[m], row, acc);
            a += p4;
        }
        return acc;
    } else {
        const float *__restrict__ p = G.gbase + idx;
        if (ORDER == DFR_NEAREST) return __ldg(p);
        if (ORDER == DFR_BILINEAR) {
            const float s00 = __ldg(p), s10 = __ldg(p + 1), s01 = __ldg(p + G.pitch), s11 = __ldg(p + G.pitch + 1);
            const float top = fmaf(fx, s10 - s00, s00);
            const float bot = fmaf(fx, s11 - s01, s01);
            return fmaf(fy, bot - top, top);
        }
        float wx[4], wy[4];
        keys_weights(fx, wx);
        keys_weights(fy, wy);
        float acc = 0.0f;
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const float *__restrict__ q = p + m * G.pitch;
            float row = wx[0] * __ldg(q);
            row = fmaf(wx[1], __ldg(q + 1), row);
            row = fmaf(wx[2], __ldg(q + 2), row);
            row = fmaf(wx[3], __ldg(q + 3), row);
            acc = fmaf(wy[m], row, acc);
        }
        return acc;
    }
}

// ---------------------------------------------------------------------------------
// packed fp32 pairs (sm_100a FFMA2 / FADD2 / FMUL2): one issue slot for two pixels.
// The main kernel is issue-bound, not FMA-pipe-bound (ncu, profiles/), so the rows of
// an interior tile are walked two at a time with every FP step packed over the pair.
// ---------------------------------------------------------------------------------
typedef unsigned long long f32x2;

__device__ __forceinline__ f32x2 pk2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpk2(f32x2 v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 add2_rm(f32x2 a, f32x2 b)      // round toward -inf
{
    f32x2 r;
    asm("add.rm.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 splat2(float v) { return pk2(v, v); }

// Keys weights (a = -0.75) on a packed pair of fractions t in [0, 1): the same cubics as
// keys_weights, factored so the outer taps share u = t (1 - t):
//   w0 = a t (1-t)^2 = (a u)(1-t),  w3 = a t^2 (1-t) = (a u) t,
//   w1 = ((a+2) t - (a+3)) t^2 + 1,  w2 = ((a+2)(1-t) - (a+3)) (1-t)^2 + 1      (11 packed ops, was 15)
__device__ __forceinline__ void keys_weights2(f32x2 t, f32x2 w[4])
{
    const float A = -0.75f;
    const f32x2 one = splat2(1.0f);
    const f32x2 s = sub2(one, t);
    const f32x2 au = mul2(mul2(t, s), splat2(A));
    w[0] = mul2(au, s);
    w[3] = mul2(au, t);
    w[1] = fma2(fma2(splat2(A + 2.0f), t, splat2(-(A + 3.0f))), mul2(t, t), one);
    w[2] = fma2(fma2(splat2(A + 2.0f), s, splat2(-(A + 3.0f))), mul2(s, s), one);
}

// Two rows (dj, dj + 1) of an INTERIOR tile of a STAGE kernel: every tap of every pixel is
// inside the image and inside the staged box (bounded rigorously by the tile record), so
// there is no range test and no address guard. K folds the shared base address and both
// index biases: address of the first tap = Ty_bits * pitch4 + Tx_bits * 4 + K (mod 2^32).
template <int ORDER, int DEG>
__device__ __forceinline__ f32x2 interior_pair(const f32x2 (&X)[4], const f32x2 (&Y)[4], f32x2 d,
                                               uint32_t pitch4, uint32_t K)
{
    f32x2 xl, yl;
    if (DEG == 1) {
        xl = fma2(X[1], d, X[0]);
        yl = fma2(Y[1], d, Y[0]);
    } else if (DEG == 2) {
        xl = fma2(fma2(X[2], d, X[1]), d, X[0]);
        yl = fma2(fma2(Y[2], d, Y[1]), d, Y[0]);
    } else {
        xl = fma2(fma2(fma2(X[3], d, X[2]), d, X[1]), d, X[0]);
        yl = fma2(fma2(fma2(Y[3], d, Y[2]), d, Y[1]), d, Y[0]);
    }
    const f32x2 magic = splat2(kMagic);
    f32x2 Tx, Ty;
    if (ORDER == DFR_NEAREST) { Tx = add2(xl, magic); Ty = add2(yl, magic); }          // rint (half-even)
    else { Tx = add2_rm(xl, magic); Ty = add2_rm(yl, magic); }                           // floor
    float txa, txb, tya, tyb;
    unpk2(Tx, txa, txb);
    unpk2(Ty, tya, tyb);
    const uint32_t aA = __float_as_uint(tya) * pitch4 + K + (__float_as_uint(txa) << 2);
    const uint32_t aB = __float_as_uint(tyb) * pitch4 + K + (__float_as_uint(txb) << 2);
    if (ORDER == DFR_NEAREST) return pk2(lds_f32(aA), lds_f32(aB));
    const f32x2 fx = sub2(xl, sub2(Tx, magic)), fy = sub2(yl, sub2(Ty, magic));
    if (ORDER == DFR_BILINEAR) {
        const uint32_t a1A = aA + pitch4, a1B = aB + pitch4;
        const f32x2 s00 = pk2(lds_f32(aA), lds_f32(aB)), s10 = pk2(lds_f32_4(aA), lds_f32_4(aB));
        const f32x2 s01 = pk2(lds_f32(a1A), lds_f32(a1B)), s11 = pk2(lds_f32_4(a1A), lds_f32_4(a1B));
        const f32x2 top = fma2(fx, sub2(s10, s00), s00);
        const f32x2 bot = fma2(fx, sub2(s11, s01), s01);
        return fma2(fy, sub2(bot, top), top);
    }
    f32x2 wx[4], wy[4];
    keys_weights2(fx, wx);
    keys_weights2(fy, wy);
    f32x2 acc = 0ull;                                   // (+0.0f, +0.0f)
    uint32_t a = aA, b = aB;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        f32x2 row = mul2(wx[0], pk2(lds_f32(a), lds_f32(b)));
        row = fma2(wx[1], pk2(lds_f32_4(a), lds_f32_4(b)), row);
        row = fma2(wx[2], pk2(lds_f32(a + 8), lds_f32(b + 8)), row);
        row = fma2(wx[3], pk2(lds_f32_4(a + 8), lds_f32_4(b + 8)), row);
        acc = fma2(wy[m], row, acc);
        a += pitch4;
        b += pitch4;
    }
    return acc;
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    }
}

// Where the values of a tile go. A sink receives the rows of a tile in increasing order:
// rows4(v) = the next four rows, row1(v) = the next single row (ragged bottom edge).
// StoreSink: the per-exposure output of dfr_reproject (one coalesced 128-byte row per warp).
struct StoreSink {
    static constexpr bool kAllLanes = false;       // lanes beyond the right edge may leave early
    float *__restrict__ orow;
    size_t opitch;
    __device__ __forceinline__ void prefetch4() {}
    __device__ __forceinline__ void rows4(float v0, float v1, float v2, float v3)
    {
        orow[0] = v0;
        orow[opitch] = v1;
        orow[2 * opitch] = v2;
        orow[3 * opitch] = v3;
        orow += 4 * opitch;
    }
    __device__ __forceinline__ void rows4p(f32x2 va, f32x2 vb)
    {
        float v0, v1, v2, v3;
        unpk2(va, v0, v1);
        unpk2(vb, v2, v3);
        rows4(v0, v1, v2, v3);
    }
    __device__ __forceinline__ void set_uniform() {}
    __device__ __forceinline__ void row1(float v)
    {
        *orow = v;
        orow += opitch;
    }
    __device__ __forceinline__ void empty_tile(int rows)
    {
        for (int r = 0; r < rows; ++r) orow[r * opitch] = qnanf();
    }
};

// All complete groups of U rows of an interior tile; advances r.
template <int ORDER, int DEG, class Sink>
__device__ __forceinline__ void interior_rows(const f32x2 (&X2)[4], const f32x2 (&Y2)[4], uint32_t pitch4,
                                              uint32_t K, int rows, int &r, Sink &sink)
{
    f32x2 d = pk2(-(float)kCentre, 1.0f - (float)kCentre);
    const f32x2 step = splat2(2.0f);
    for (; r + 4 <= rows; r += 4) {
        sink.prefetch4();
        const f32x2 va = interior_pair<ORDER, DEG>(X2, Y2, d, pitch4, K);
        d = add2(d, step);
        const f32x2 vb = interior_pair<ORDER, DEG>(X2, Y2, d, pitch4, K);
        d = add2(d, step);
        sink.rows4p(va, vb);
    }
}

// One 32x32 tile by one warp (lane = output column): EMPTY -> NaN, EXACT -> fp64 map per
// pixel, FAST -> polynomial coordinates + gathers from the staged box (STAGE) or the image.
// (ox, oy) is the source pixel of the staged box's element (0, 0); box_smem its shared address.
struct TileHead {
    int flag, ix0, iy0, bx0, by0, bx1, by1, deg;
};

template <int ORDER, bool STAGE, int EDGE = DFR_EDGE_AREA, class Sink>
__device__ __forceinline__ void warp_tile(const TiledParams &P, const TargetDev &tgt, int e, int ttx, int tty,
                                          int lane, const TileHead &H, float (&X)[4], float (&Y)[4],
                                          uint32_t box_smem, int ox, int oy, Sink &sink)
{
    const int flag = H.flag, ix0 = H.ix0, iy0 = H.iy0, bx0 = H.bx0, by0 = H.by0, bx1 = H.bx1, by1 = H.by1,
              deg = H.deg;
    const int tx0 = ttx * TS, ty0 = tty * TS;
    const int col = tx0 + lane;
    if (!Sink::kAllLanes && col >= P.onx) return;      // ragged right edge (no block-level sync below)
    const int rows = min(TS, P.ony - ty0);
    const float *__restrict__ img = P.src + (size_t)e * P.sny * P.snx;

    if (flag == TILE_EMPTY) {
        sink.empty_tile(rows);
        return;
    }
    if (flag == TILE_EXACT) {
        for (int r = 0; r < rows; ++r)
            sink.row1(exact_pixel<ORDER, EDGE>(img, P.sny, P.snx, tgt, P.srcdev[e], col, ty0 + r));
        return;
    }

    // ---- per-axis fast-gather constants (a FAST tile in a STAGE kernel always has a box)
    int Alx, Ahx, Aly, Ahy;
    if (STAGE) {
        axis_range<ORDER>(P.snx, ox, P.BW, Alx, Ahx);
        axis_range<ORDER>(P.sny, oy, P.BH, Aly, Ahy);
    } else {
        axis_range<ORDER>(P.snx, -(1 << 28), 1 << 30, Alx, Ahx);
        axis_range<ORDER>(P.sny, -(1 << 28), 1 << 30, Aly, Ahy);
    }
    const unsigned cntx = (unsigned)max(Ahx - Alx + 1, 0), cnty = (unsigned)max(Ahy - Aly + 1, 0);
    const int Cx = kMagicBits - ix0 + Alx, Cy = kMagicBits - iy0 + Aly;
    // gather array: element (k = 0) = first tap of base index (Alx, Aly)
    const int tlo = (ORDER == DFR_BICUBIC) ? 1 : 0;
    GatherSrc<STAGE> G;
    if (STAGE) {
        G.pitch = P.BW;
        G.sbase = box_smem + 4u * (unsigned)((Aly - tlo - oy) * P.BW + (Alx - tlo - ox));
        G.gbase = nullptr;
    } else {
        G.pitch = P.snx;
        G.sbase = 0;
        G.gbase = img + ((long long)(Aly - tlo) * P.snx + (Alx - tlo));
    }

    truncate_degree(deg, X, Y);                                 // same polynomial on every path
    constexpr int U = 4;                      // rows in flight per thread
    float dj = -(float)kCentre;
    int r = 0;
    if (STAGE) {
        // INTERIOR tile: the record's rigorous index range lies inside [Al, Ah] on both axes
        // (image interior AND staged box), so no pixel needs a range test or the rim rule.
        const int top = (ORDER == DFR_NEAREST) ? 1 : 0;          // rint(x) <= floor(x) + 1
        const bool interior = bx0 >= Alx && bx1 + top <= Ahx && by0 >= Aly && by1 + top <= Ahy;
        if (interior) {
            sink.set_uniform();                  // no pixel of this tile can leave the footprint
            f32x2 X2[4], Y2[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) { X2[q] = splat2(X[q]); Y2[q] = splat2(Y[q]); }
            const uint32_t pitch4 = 4u * (unsigned)G.pitch;
            const uint32_t K = G.sbase - pitch4 * (unsigned)Cy - 4u * (unsigned)Cx;
            if (deg == 1) interior_rows<ORDER, 1>(X2, Y2, pitch4, K, rows, r, sink);
            else if (deg == 2) interior_rows<ORDER, 2>(X2, Y2, pitch4, K, rows, r, sink);
            else interior_rows<ORDER, 3>(X2, Y2, pitch4, K, rows, r, sink);
            dj += (float)r;
        }
    }
    for (; r + U <= rows; r += U) {
        sink.prefetch4();
        float xl[U], yl[U], val[U];
        bool ok[U];
#pragma unroll
        for (int k = 0; k < U; ++k) {
            const float d = dj + (float)k;
            xl[k] = fmaf(fmaf(fmaf(X[3], d, X[2]), d, X[1]), d, X[0]);
            yl[k] = fmaf(fmaf(fmaf(Y[3], d, Y[2]), d, Y[1]), d, Y[0]);
            val[k] = fast_pixel<ORDER, STAGE>(G, xl[k], yl[k], Cx, Cy, cntx, cnty, ok[k]);
        }
        bool all_ok = true;
#pragma unroll
        for (int k = 0; k < U; ++k) all_ok = all_ok && ok[k];
        if (!all_ok) {                        // rare: image rim, outside the staged box, NaN
#pragma unroll
            for (int k = 0; k < U; ++k)
                if (!ok[k]) val[k] = slow_poly_pixel<ORDER, EDGE>(img, P.sny, P.snx, ix0, iy0, xl[k], yl[k]);
        }
        sink.rows4(val[0], val[1], val[2], val[3]);
        dj += (float)U;
    }
    for (; r < rows; ++r) {                   // ragged bottom edge
        const float xs = fmaf(fmaf(fmaf(X[3], dj, X[2]), dj, X[1]), dj, X[0]);
        const float ys = fmaf(fmaf(fmaf(Y[3], dj, Y[2]), dj, Y[1]), dj, Y[0]);
        bool ok1;
        float v = fast_pixel<ORDER, STAGE>(G, xs, ys, Cx, Cy, cntx, cnty, ok1);
        if (!ok1) v = slow_poly_pixel<ORDER, EDGE>(img, P.sny, P.snx, ix0, iy0, xs, ys);
        sink.row1(v);
        dj += 1.0f;
    }
}


}  // namespace dfr
