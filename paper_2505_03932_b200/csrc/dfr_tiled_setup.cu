// dfr_tiled_setup.cu — setup kernels of the tiled fast path and the host
// side they share with the main kernels (scratch, staging decision, tensor map).
//
//   target_nodes_kernel      (fp64) a1-a2 at the sample points — shared by the whole batch, as
//                            SURVEY.md §8(a) a10 notes: 16 nodes + 16 check points per 128x128
//                            super-tile for the cooperative kernel, 25 points per 64x64 CTA tile
//                            for the wide one.
//   tile_setup_kernel        (fp64, the default) cooperative: 16 lanes per 128x128 super-tile, one
//                            node, one check point and one 32x32 tile each. a3-a6 at the 16
//                            Chebyshev nodes, bicubic fit through shuffles, compared with the exact
//                            map at 16 other points (centre, T4 extrema on the axes, corners, edge
//                            mid-points, three generic points); if accepted, every lane re-centres
//                            the cubic on its own tile; if not, every lane fits its own tile from
//                            25 points (16 nodes + 9 check points), and a tile whose own fit fails
//                            is classified EXACT.
//   tile_setup_wide_kernel   (fp64) the round-1 form, a thread per 64x64 CTA tile (25 points: 16
//                            nodes + 9 check points, refit per 32x32 tile when the 64x64 fit
//                            fails); chosen by run_setup when the launch fills the GPU anyway.
//   Both then bound each tile's source footprint rigorously, classify it FAST / EXACT / EMPTY,
//   pick the dj degree the main kernel must keep, and reduce the origin of the CTA tile's
//   staged box.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "dfr_tiled_device.cuh"

namespace dfr {

// ---------------------------------------------------------------------------------
// constants of the fit
// ---------------------------------------------------------------------------------
constexpr int SUP_T = 2;               // a super-tile is SUP_T x SUP_T CTA tiles (128 x 128 px)
constexpr int kSupLanes = 16;          // = its 4 x 4 tiles = the 16 nodes = the 16 check points: one lane each
constexpr int kSupEdge = TS * CTA_T * SUP_T;

struct FitConsts {
    double W[4][4];            // monomial coefficients of the Lagrange basis: L_a(s) = sum_p W[p][a] s^p
    double pts[NPTS][2];       // sample points (s, t) in [-1, 1]^2; pixel offset = 16 s
    double sup[2 * kSupLanes][2];  // the 128x128 super-tile fit: 16 nodes, then 16 check points
};

static FitConsts make_fit_consts()
{
    FitConsts f;
    double s[4];
    for (int a = 0; a < 4; ++a) s[a] = std::cos((2 * a + 1) * 3.14159265358979323846 / 8.0);
    for (int a = 0; a < 4; ++a) {
        double b[3];
        int m = 0;
        for (int k = 0; k < 4; ++k)
            if (k != a) b[m++] = s[k];
        const double den = (s[a] - b[0]) * (s[a] - b[1]) * (s[a] - b[2]);
        f.W[3][a] = 1.0 / den;
        f.W[2][a] = -(b[0] + b[1] + b[2]) / den;
        f.W[1][a] = (b[0] * b[1] + b[0] * b[2] + b[1] * b[2]) / den;
        f.W[0][a] = -(b[0] * b[1] * b[2]) / den;
    }
    for (int b = 0; b < 4; ++b)
        for (int a = 0; a < 4; ++a) {
            f.pts[4 * b + a][0] = s[a];
            f.pts[4 * b + a][1] = s[b];
        }
    const double h = 0.70710678118654752440;
    // check points: extrema of T4 (0, +-1/sqrt2, +-1) where the interpolation error of a cubic
    // through Chebyshev nodes peaks. The axis points matter: at the centre, on the diagonals
    // and at the corners |T4(s)| = |T4(t)| with equal signs, so fourth-order errors of
    // opposite sign in s and t (u^4 - v^4) cancel there; (+-h, 0) and (0, +-h) separate them.
    const double chk[9][2] = {{0, 0}, {h, 0}, {-h, 0}, {0, h}, {0, -h}, {1, 1}, {-1, 1}, {1, -1}, {-1, -1}};
    for (int k = 0; k < 9; ++k) {
        f.pts[16 + k][0] = chk[k][0];
        f.pts[16 + k][1] = chk[k][1];
    }
    // super-tile: the same nodes; 16 check points = the 9 above + the 4 edge mid-points (|T4| = 1 in
    // one direction, 0 offset in the other) + 3 interior points off every symmetry line
    for (int k = 0; k < 16; ++k) { f.sup[k][0] = f.pts[k][0]; f.sup[k][1] = f.pts[k][1]; }
    const double more[7][2] = {{1, 0}, {-1, 0}, {0, 1}, {0, -1}, {h, -0.38}, {-0.38, h}, {-0.55, -0.8}};
    for (int k = 0; k < 9; ++k) { f.sup[16 + k][0] = chk[k][0]; f.sup[16 + k][1] = chk[k][1]; }
    for (int k = 0; k < 7; ++k) { f.sup[25 + k][0] = more[k][0]; f.sup[25 + k][1] = more[k][1]; }
    return f;
}

// ---------------------------------------------------------------------------------
// setup kernels (fp64)
// ---------------------------------------------------------------------------------
// Expansion of the packed constants (ConstsCopy, dfr_tiled.h): word j of the full-size block.
__device__ __forceinline__ unsigned long long expand_word(const unsigned long long *__restrict__ pk, int stride, int T, int j)
{
    constexpr int W = (int)(sizeof(SourceDev) / 8);             // 124 words per exposure
    const int e = j / W, k = j - e * W;
    const unsigned long long *r = pk + (size_t)e * stride;
    const unsigned long long hdr = r[11];                        // ap.order | bp.order << 8 | inv_exact << 16
    if (k < 11) return r[k];
    if (k == 11) return hdr & 0xffull;                           // Poly ap: { int32 order, int32 pad }
    if (k < 67) return (k - 12 < T) ? r[kPackedHead + (k - 12)] : 0ull;
    if (k == 67) return (hdr >> 8) & 0xffull;
    if (k < 123) return (k - 68 < T) ? r[kPackedHead + T + (k - 68)] : 0ull;
    return (hdr >> 16) & 0xffull;                                // { int32 inv_exact, int32 pad }
}

template <int BYTES>
__global__ void __launch_bounds__(128)
target_nodes_kernel(const __grid_constant__ TargetDev tgt, const __grid_constant__ FitConsts fc,
                    int ctas_x, int ctas, double2 *__restrict__ uv, int32_t *__restrict__ counters,
                    const uint4 *__restrict__ cc_mapped, void *__restrict__ cc_dst, int cc_bytes,
                    int pk_n, int pk_T, int pk_nw, const __grid_constant__ PackedConsts<BYTES> pk, int wide)
{
    // tile counters + ticket of the setup kernel start from zero (no memset in the stream)
    if (blockIdx.x == 0 && threadIdx.x < 4) counters[threadIdx.x] = 0;
    // the call's constants (per-exposure maps, weights) -> device scratch
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    if (cc_mapped) {
        for (int k = tid; k < cc_bytes / 16; k += nth) static_cast<uint4 *>(cc_dst)[k] = cc_mapped[k];
    } else if (pk_n > 0) {
        const unsigned long long *src = reinterpret_cast<const unsigned long long *>(pk.q);
        const int stride = kPackedHead + 2 * pk_T, words = pk_n * (int)(sizeof(SourceDev) / 8);
        for (int j = tid; j < words; j += nth) static_cast<unsigned long long *>(cc_dst)[j] = expand_word(src, stride, pk_T, j);
        const float *w = reinterpret_cast<const float *>(src + (size_t)pk_n * stride);
        float *wd = reinterpret_cast<float *>(static_cast<char *>(cc_dst) + (size_t)pk_n * sizeof(SourceDev));
        for (int j = tid; j < pk_nw; j += nth) wd[j] = w[j];
    }
    pdl_trigger();                                  // the setup kernel may stage its constants meanwhile
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (wide) {
        // sample points of the 64x64 CTA tiles (tile_setup_wide_kernel): (ctas_x, ctas) count CTA tiles
        if (idx >= ctas * NPTS) return;
        const int c = idx / NPTS, k = idx - c * NPTS;
        constexpr double edge = TS * CTA_T;
        const double cx0 = (c % ctas_x) * edge + 0.5 * (edge - 1), cy0 = (c / ctas_x) * edge + 0.5 * (edge - 1);
        double U, V;
        target_uv(tgt, cx0 + 0.5 * edge * fc.pts[k][0], cy0 + 0.5 * edge * fc.pts[k][1], U, V);
        uv[(size_t)k * ctas + c] = make_double2(U, V);          // [point][CTA tile]: coalesced for the setup kernel
        return;
    }
    // (ctas_x, ctas) here count SUPER-tiles
    if (idx >= ctas * 2 * kSupLanes) return;
    const int c = idx / (2 * kSupLanes), k = idx - c * (2 * kSupLanes);
    constexpr double edge = kSupEdge;
    const double cx0 = (c % ctas_x) * edge + 0.5 * (edge - 1), cy0 = (c / ctas_x) * edge + 0.5 * (edge - 1);
    double U, V;
    target_uv(tgt, cx0 + 0.5 * edge * fc.sup[k][0], cy0 + 0.5 * edge * fc.sup[k][1], U, V);
    uv[(size_t)k * ctas + c] = make_double2(U, V);          // [point][super-tile]
}

// Triangle size and row offset of an order-N packed polynomial (see Poly).
__host__ __device__ constexpr int tri(int n) { return (n + 1) * (n + 2) / 2; }
__host__ __device__ constexpr int tri_off(int n, int p) { return p * (n + 1) - (p * (p - 1)) / 2; }

// a3-a6 with the exposure's constants in shared memory, SIP order fixed at compile time
// (lower orders are zero-padded): sm = { m[9], c1, c2, ap[tri(N)], bp[tri(N)] }.
// The reciprocal is a float seed + two Newton steps (c is O(1) for any valid point);
// invalid points (c <= 0, NaN) come out as NaN.
template <int N>
__device__ __forceinline__ void source_xy_sm(const double *__restrict__ sm, bool inv_exact, double U, double V,
                                             double &x, double &y)
{
    const double a = fma(sm[0], U, fma(sm[1], V, sm[2]));
    const double b = fma(sm[3], U, fma(sm[4], V, sm[5]));
    const double c = fma(sm[6], U, fma(sm[7], V, sm[8]));
    float rf;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rf) : "f"((float)c));
    double r = (double)rf;
    r = r * fma(-c, r, 2.0);
    r = r * fma(-c, r, 2.0);
    if (!(c > 0.0)) r = __longlong_as_double(0x7ff8000000000000LL);
    const double us = a * r, vs = b * r;
    x = us + sm[9];
    y = vs + sm[10];
    if (N > 0) {
        if (inv_exact) {                         // DFR_SIP_INVERSE_EXACT: sm holds A, B; solve at this sample point
            double u, v;
            invert_sip([&](double p, double q) { return poly_eval_fixed<N>(sm + 11, p, q); },
                       [&](double p, double q) { return poly_eval_fixed<N>(sm + 11 + tri(N), p, q); }, us, vs, u, v);
            x = u + sm[9];
            y = v + sm[10];
        } else {
            x += poly_eval_fixed<N>(sm + 11, us, vs);
            y += poly_eval_fixed<N>(sm + 11 + tri(N), us, vs);
        }
    }
}

// Cubic fit of the pixel map over one square region: 16 Chebyshev nodes -> tensor-product
// cubic in (s, t) in [-1, 1]^2 (separably: along s within each node row, then along t),
// then VERIFIED against the exact map at 9 other points (centre, T4 extrema on the axes, corners).
// uvf(k) returns the target-side (U, V) of sample point k. C[4q + p] = coefficient of s^p t^q.
template <int N, class UVF>
__device__ __forceinline__ bool fit_cubic(const double *__restrict__ sm, bool inv_exact, const FitConsts &fc, UVF uvf,
                                          double (&Cx)[16], double (&Cy)[16])
{
    double Rx[4][4], Ry[4][4];                  // [node row b][power of s]
    double nanacc = 0.0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        double xs[4], ys[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            const double2 q = uvf(4 * b + a);
            source_xy_sm<N>(sm, inv_exact, q.x, q.y, xs[a], ys[a]);
            nanacc = fma(xs[a], 0.0, fma(ys[a], 0.0, nanacc));
        }
#pragma unroll
        for (int pp = 0; pp < 4; ++pp) {
            Rx[b][pp] = fma(fc.W[pp][0], xs[0], fma(fc.W[pp][1], xs[1], fma(fc.W[pp][2], xs[2], fc.W[pp][3] * xs[3])));
            Ry[b][pp] = fma(fc.W[pp][0], ys[0], fma(fc.W[pp][1], ys[1], fma(fc.W[pp][2], ys[2], fc.W[pp][3] * ys[3])));
        }
    }
#pragma unroll
    for (int qq = 0; qq < 4; ++qq)
#pragma unroll
        for (int pp = 0; pp < 4; ++pp) {
            Cx[4 * qq + pp] = fma(fc.W[qq][0], Rx[0][pp], fma(fc.W[qq][1], Rx[1][pp], fma(fc.W[qq][2], Rx[2][pp], fc.W[qq][3] * Rx[3][pp])));
            Cy[4 * qq + pp] = fma(fc.W[qq][0], Ry[0][pp], fma(fc.W[qq][1], Ry[1][pp], fma(fc.W[qq][2], Ry[2][pp], fc.W[qq][3] * Ry[3][pp])));
        }
    bool good = true;
#pragma unroll
    for (int k = 16; k < NPTS; ++k) {
        const double2 q = uvf(k);
        double x, y;
        source_xy_sm<N>(sm, inv_exact, q.x, q.y, x, y);
        const double ss = fc.pts[k][0], tt = fc.pts[k][1];
        double px = 0.0, py = 0.0;
#pragma unroll
        for (int qq = 3; qq >= 0; --qq) {
            const double rx = fma(fma(fma(Cx[4 * qq + 3], ss, Cx[4 * qq + 2]), ss, Cx[4 * qq + 1]), ss, Cx[4 * qq]);
            const double ry = fma(fma(fma(Cy[4 * qq + 3], ss, Cy[4 * qq + 2]), ss, Cy[4 * qq + 1]), ss, Cy[4 * qq]);
            px = fma(px, tt, rx);
            py = fma(py, tt, ry);
        }
        good = good && (fabs(px - x) <= (double)FIT_TOL) && (fabs(py - y) <= (double)FIT_TOL);   // false on NaN
    }
    return good && (nanacc == 0.0);
}

// p(s0 + s'/2) as a cubic in s': the re-centring of a parent cubic (unit = 32 px) on one of
// its halves (unit = 16 px). Exact up to fp64 rounding.
__device__ __forceinline__ void shift_half(double &c0, double &c1, double &c2, double &c3, double s0)
{
    const double d0 = fma(s0, fma(s0, fma(s0, c3, c2), c1), c0);
    const double d1 = 0.5 * fma(s0, fma(3.0 * s0, c3, 2.0 * c2), c1);
    const double d2 = 0.25 * fma(3.0 * s0, c3, c2);
    c0 = d0; c1 = d1; c2 = d2; c3 = 0.125 * c3;
}

__device__ __forceinline__ void shift_quarter(double &c0, double &c1, double &c2, double &c3, double s0)
{
    // p(s0 + s'/4) as a cubic in s': a 128-px parent (unit = 64 px) re-centred on a 32-px tile (unit = 16 px)
    const double d0 = fma(s0, fma(s0, fma(s0, c3, c2), c1), c0);
    const double d1 = 0.25 * fma(s0, fma(3.0 * s0, c3, 2.0 * c2), c1);
    const double d2 = 0.0625 * fma(3.0 * s0, c3, c2);
    c0 = d0; c1 = d1; c2 = d2; c3 = 0.015625 * c3;
}

// The record of one 32x32 tile from its cubic (unit = 16 px about the tile centre):
// footprint bound, classification, dj degree, integer base, fp32 coefficients.
// Returns the flag; (bx0, by0) is the first floor index the tile can touch.
__device__ __forceinline__ int emit_tile(double (&Cx)[16], double (&Cy)[16], bool finite, int sny, int snx,
                                         TileRec *__restrict__ out, int &bx0, int &by0)
{
    // Rigorous range of the fitted polynomial over the tile: |s|, |t| <= 31/32 < 1, so
    // |x - C00| <= sum of the other |C_pq|. The main kernel evaluates exactly this
    // polynomial (in fp32: + kBoxSlack), which is what makes its unchecked gathers safe.
    double ex = 0.0, ey = 0.0;
#pragma unroll
    for (int k = 1; k < 16; ++k) { ex += fabs(Cx[k]); ey += fabs(Cy[k]); }
    constexpr double kBoxSlack = 1e-3;
    const double xmin = Cx[0] - ex - kBoxSlack, xmax = Cx[0] + ex + kBoxSlack;
    const double ymin = Cy[0] - ey - kBoxSlack, ymax = Cy[0] + ey + kBoxSlack;
    // Degree of the per-lane column polynomials in dj: the t^2, t^3 terms (any power of s)
    // are dropped by the main kernel when they cannot move a coordinate by kDegTol px.
    double q2x = 0.0, q2y = 0.0, q3x = 0.0, q3y = 0.0;
#pragma unroll
    for (int pp = 0; pp < 4; ++pp) {
        q2x += fabs(Cx[8 + pp]); q2y += fabs(Cy[8 + pp]);
        q3x += fabs(Cx[12 + pp]); q3y += fabs(Cy[12 + pp]);
    }
    constexpr double kDegTol = 2.5e-7;
    TileRec r;
    r.deg = fmax(q3x, q3y) >= kDegTol ? 3 : (fmax(q2x, q2y) >= kDegTol ? 2 : 1);
    int flag = TILE_EXACT;
    r.ix0 = r.iy0 = r.bx0 = r.by0 = r.bx1 = r.by1 = 0;
    double bx = 0.0, by = 0.0;
    if (finite && fabs(xmin) < 1e9 && fabs(xmax) < 1e9 && fabs(ymin) < 1e9 && fabs(ymax) < 1e9) {
        // EVEN integer base: the main kernel rounds the tile-relative coordinate x - ix0 half-to-even
        // (nearest neighbour), which is the rounding of x itself only when ix0 is even
        bx = 2.0 * floor(0.5 * Cx[0]); by = 2.0 * floor(0.5 * Cy[0]);
        r.ix0 = (int)bx; r.iy0 = (int)by;
        r.bx0 = (int)floor(xmin); r.bx1 = (int)floor(xmax);
        r.by0 = (int)floor(ymin); r.by1 = (int)floor(ymax);
        const bool small = (r.bx1 - r.bx0) < 2048 && (r.by1 - r.by0) < 2048 &&
                           abs(r.bx0 - r.ix0) < 2048 && abs(r.bx1 - r.ix0) < 2048 &&
                           abs(r.by0 - r.iy0) < 2048 && abs(r.by1 - r.iy0) < 2048;
        if (small) {
            // outside the footprint [-0.5, n-0.5) by a 2 px margin on one side => all NaN
            const bool outside = (xmax + 2.0 < -0.5) || (xmin - 2.0 >= snx - 0.5) ||
                                 (ymax + 2.0 < -0.5) || (ymin - 2.0 >= sny - 0.5);
            flag = outside ? TILE_EMPTY : TILE_FAST;
        } else {
            bx = by = 0.0;
        }
    }
    r.flag = flag;
    bx0 = r.bx0; by0 = r.by0;
    // s = di / 16: coefficient of di^p dj^q is C[p][q] / 16^(p+q)
    double sq = 1.0;
#pragma unroll
    for (int qq = 0; qq < 4; ++qq) {
        double sp = sq;
#pragma unroll
        for (int pp = 0; pp < 4; ++pp) {
            const double c0x = (qq == 0 && pp == 0) ? Cx[0] - bx : Cx[4 * qq + pp];
            const double c0y = (qq == 0 && pp == 0) ? Cy[0] - by : Cy[4 * qq + pp];
            r.cx[4 * qq + pp] = (float)(c0x * sp);
            r.cy[4 * qq + pp] = (float)(c0y * sp);
            sp *= 1.0 / kHalf;
        }
        sq *= 1.0 / kHalf;
    }
    *out = r;
    return flag;
}

// Sixteen lanes per (128x128 super-tile, exposure) — its 4 x 4 tiles, its 16 interpolation nodes and
// its 16 check points, one of each per lane. A block is 8 consecutive super-tiles of ONE exposure, so
// the exposure's constants are staged once in shared memory and every coefficient read is a
// broadcast LDS. Two levels:
//   1. every lane evaluates the exact map (a3-a6) at one Chebyshev node; the tensor-product cubic over
//      the whole super-tile comes out of two rounds of 4-lane shuffles (Lagrange -> monomial along s,
//      then along t), is gathered by all lanes, and is compared with the exact map at 16 other points
//      (one per lane: centre, T4 extrema on the axes, corners, edge mid-points, three generic points);
//      if it holds everywhere, each lane re-centres it on its own 32x32 tile — no further map
//      evaluations: 2 per lane instead of the 25 (+ fit) a tile of its own would need;
//   2. if it does not (strongly curved maps), each lane fits its own tile from 25 points with the
//      target side (a1-a2) evaluated on the fly; a tile whose own fit fails is EXACT.
// Round 1 ran one thread per 64x64 tile (a serial chain of ~2600 fp64 operations, 17 us on C2, and as
// long for a single frame, where the GPU was nearly empty); here the chain is ~400 operations.
constexpr int kSetupThreads = 128;
constexpr long long kWideThreshold = 16384;      // (CTA tiles x exposures) from which tile_setup_wide_kernel is used
constexpr int kSupPerBlock = kSetupThreads / kSupLanes;

__device__ __forceinline__ double shfl16(double v, int src_lane_in_group)
{
    return __shfl_sync(0xffffffffu, v, src_lane_in_group, kSupLanes);
}

template <int N, bool INV>
__global__ void __launch_bounds__(kSetupThreads)
tile_setup_kernel(const double2 *__restrict__ uv, const SourceDev *__restrict__ srcdev,
                  const __grid_constant__ TargetDev tgt, const __grid_constant__ FitConsts fc, int e0,
                  int tiles_x, int tiles_y, int ctas_x, int ctas_y, int sups_x, int nsup, int sny, int snx,
                  TileRec *__restrict__ recs, int2 *__restrict__ cta_box, int32_t *__restrict__ counters,
                  int total_blocks, int32_t *__restrict__ host_stats, int stats_add, int late_consts)
{
    __shared__ double sm[11 + 2 * tri(N)];
    const int e = e0 + blockIdx.y;
    // The exposure's constants -> shared memory. When they were uploaded by a copy earlier in the
    // stream they are staged BEFORE waiting for the node kernel (this kernel's launch overlaps it);
    // when the node kernel itself brings them in (late_consts), after.
    if (late_consts) {
        pdl_trigger();
        pdl_wait();
    }
    const bool inv_exact = INV && N > 0 && srcdev[e].inv_exact != 0;
    {
        const SourceDev &s = srcdev[e];
        for (int k = threadIdx.x; k < 11 + 2 * tri(N); k += blockDim.x) {
            double v;
            if (k < 9) v = s.m[k];
            else if (k == 9) v = s.c1;
            else if (k == 10) v = s.c2;
            else {
                // slot of the order-N layout -> (p, q) -> slot of the stored order-n layout
                const int t = (k - 11) % tri(N);
                const Poly &P = (k - 11) < tri(N) ? s.ap : s.bp;
                int p = 0;
                while (p < N && tri_off(N, p + 1) <= t) ++p;
                const int q = t - tri_off(N, p), n = P.order;
                v = (p + q <= n) ? P.c[tri_off(n, p) + q] : 0.0;
            }
            sm[k] = v;
        }
    }
    if (!late_consts) pdl_trigger();                // the main kernel's launch may overlap this one
    __syncthreads();
    if (!late_consts) pdl_wait();                   // the node table is complete

    const int l = threadIdx.x & (kSupLanes - 1);                // lane of the group: node / check point / tile
    const int a = l & 3, b = l >> 2;
    const int sidx_raw = blockIdx.x * kSupPerBlock + (threadIdx.x / kSupLanes);
    const bool live = sidx_raw < nsup;                          // dead groups compute on super-tile 0 and write nothing
    const int sidx = live ? sidx_raw : 0;
    const int sy = sidx / sups_x, sx = sidx - sy * sups_x;

    // ---- level 1: one node per lane, the fit through shuffles
    double xs, ys;
    {
        const double2 q = __ldg(uv + (size_t)l * nsup + sidx);
        source_xy_sm<N>(sm, inv_exact, q.x, q.y, xs, ys);
    }
    double Rx = 0.0, Ry = 0.0;                                  // row b, power a of s
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double w = fc.W[a][k];
        Rx = fma(w, shfl16(xs, (b << 2) | k), Rx);
        Ry = fma(w, shfl16(ys, (b << 2) | k), Ry);
    }
    double cxl = 0.0, cyl = 0.0;                                // coefficient of s^a t^b
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double w = fc.W[b][k];
        cxl = fma(w, shfl16(Rx, (k << 2) | a), cxl);
        cyl = fma(w, shfl16(Ry, (k << 2) | a), cyl);
    }
    double Cx[16], Cy[16];                                      // C[4q + p]: s^p t^q, unit = 64 px
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        Cx[k] = shfl16(cxl, k);
        Cy[k] = shfl16(cyl, k);
    }
    bool ok;
    {
        const double2 q = __ldg(uv + (size_t)(kSupLanes + l) * nsup + sidx);
        double x, y;
        source_xy_sm<N>(sm, inv_exact, q.x, q.y, x, y);
        const double ss = fc.sup[kSupLanes + l][0], tt = fc.sup[kSupLanes + l][1];
        double px = 0.0, py = 0.0;
#pragma unroll
        for (int qq = 3; qq >= 0; --qq) {
            const double rx = fma(fma(fma(Cx[4 * qq + 3], ss, Cx[4 * qq + 2]), ss, Cx[4 * qq + 1]), ss, Cx[4 * qq]);
            const double ry = fma(fma(fma(Cy[4 * qq + 3], ss, Cy[4 * qq + 2]), ss, Cy[4 * qq + 1]), ss, Cy[4 * qq]);
            px = fma(px, tt, rx);
            py = fma(py, tt, ry);
        }
        // false on NaN; a NaN at a node poisons every coefficient, hence every lane's comparison
        ok = (fabs(px - x) <= (double)FIT_TOL) && (fabs(py - y) <= (double)FIT_TOL);
    }
    const unsigned votes = __ballot_sync(0xffffffffu, ok);
    const bool parent = ((votes >> (threadIdx.x & 16)) & 0xffffu) == 0xffffu;

    // ---- this lane's tile
    const int ttx = (sx * SUP_T * CTA_T) + a, tty = (sy * SUP_T * CTA_T) + b;
    const bool mine = live && ttx < tiles_x && tty < tiles_y;
    bool good = true;
    if (parent) {
        const double s0 = 0.5 * a - 0.75, t0 = 0.5 * b - 0.75;
#pragma unroll
        for (int q = 0; q < 4; ++q) {           // along s, each power of t
            shift_quarter(Cx[4 * q], Cx[4 * q + 1], Cx[4 * q + 2], Cx[4 * q + 3], s0);
            shift_quarter(Cy[4 * q], Cy[4 * q + 1], Cy[4 * q + 2], Cy[4 * q + 3], s0);
        }
#pragma unroll
        for (int pp = 0; pp < 4; ++pp) {        // along t, each power of s
            shift_quarter(Cx[pp], Cx[4 + pp], Cx[8 + pp], Cx[12 + pp], t0);
            shift_quarter(Cy[pp], Cy[4 + pp], Cy[8 + pp], Cy[12 + pp], t0);
        }
    } else if (mine) {
        // ---- level 2: this tile's own fit, target side on the fly
        const double cx0 = ttx * TS + kCentre, cy0 = tty * TS + kCentre;
        good = fit_cubic<N>(sm, inv_exact, fc, [&](int k) {
            double U, V;
            target_uv(tgt, cx0 + kHalf * fc.pts[k][0], cy0 + kHalf * fc.pts[k][1], U, V);
            return make_double2(U, V);
        }, Cx, Cy);
    }
    int nflag[3] = {0, 0, 0};
    int box_x = kNoBox, box_y = kNoBox;
    if (mine) {
        int bx0, by0;
        const int flag = emit_tile(Cx, Cy, good, sny, snx,
                                   recs + ((size_t)e * tiles_x * tiles_y + (size_t)tty * tiles_x + ttx), bx0, by0);
        ++nflag[flag];
        if (flag == TILE_FAST) { box_x = bx0; box_y = by0; }
    }
    // origin of each CTA tile's staged box = min over its 2 x 2 FAST tiles (kNoBox: none)
    box_x = min(box_x, __shfl_xor_sync(0xffffffffu, box_x, 1));
    box_y = min(box_y, __shfl_xor_sync(0xffffffffu, box_y, 1));
    box_x = min(box_x, __shfl_xor_sync(0xffffffffu, box_x, 4));
    box_y = min(box_y, __shfl_xor_sync(0xffffffffu, box_y, 4));
    if (live && (a & 1) == 0 && (b & 1) == 0) {
        const int ctx = sx * SUP_T + (a >> 1), cty = sy * SUP_T + (b >> 1);
        if (ctx < ctas_x && cty < ctas_y)
            cta_box[(size_t)e * ctas_x * ctas_y + (size_t)cty * ctas_x + ctx] = make_int2(box_x, box_y);
    }
    // tile statistics: per-warp sums -> device counters; the last block of the last launch
    // (ticket) writes the totals straight into the caller's mapped host memory, so
    // dfr_last_stats needs neither a memset nor a copy in the stream
#pragma unroll
    for (int f = 0; f < 3; ++f) {
        const int w = __reduce_add_sync(0xffffffffu, nflag[f]);
        if ((threadIdx.x & 31) == 0 && w) atomicAdd(&counters[f], w);
    }
    __syncthreads();
    if (threadIdx.x == 0 && host_stats) {
        __threadfence();
        if (atomicAdd(&counters[3], 1) == total_blocks - 1) {
            __threadfence();
            for (int f = 0; f < 3; ++f) {
                const int32_t v = *(volatile int32_t *)&counters[f];
                if (stats_add) atomicAdd(&host_stats[f], v);     // streaming calls: device-side totals
                else host_stats[f] = v;
            }
        }
    }
}

// The WIDE form of the setup kernel, for launches that fill the GPU (C2: 32 768 CTA tiles):
// one thread per (64x64 CTA tile, exposure); a block is 128 consecutive CTA tiles of ONE
// exposure, so the exposure's constants are staged once in shared memory and every
// coefficient read is a broadcast LDS. Two levels:
//   1. the cubic is fitted and verified over the whole 64x64 CTA tile (25 map evaluations);
//      if it holds, the four 32x32 tile records are its exact re-centrings (no more map
//      evaluations) — 4x less fp64 work than fitting each tile;
//   2. if it does not (strongly curved maps), each 32x32 tile gets its own fit, with the
//      target side (a1-a2) evaluated on the fly; a tile whose own fit fails is EXACT.
// Measured on B200, C2: 19.3 us under ncu against 25.7 us for the cooperative kernel above, whose
// strength is its short serial chain when the grid is small (single frames).

// INV: the batch contains DFR_SIP_INVERSE_EXACT sources (a separate instantiation, so the common
// kernel is compiled exactly as without that feature: as a run-time flag alone it cost 6 us per call).
template <int N, bool INV>
__global__ void __launch_bounds__(kSetupThreads)
tile_setup_wide_kernel(const double2 *__restrict__ uv, const SourceDev *__restrict__ srcdev,
                  const __grid_constant__ TargetDev tgt, const __grid_constant__ FitConsts fc, int e0,
                  int tiles_x, int tiles_y, int ctas_x, int ctas, int sny, int snx,
                  TileRec *__restrict__ recs, int2 *__restrict__ cta_box, int32_t *__restrict__ counters,
                  int total_blocks, int32_t *__restrict__ host_stats, int stats_add, int late_consts)
{
    __shared__ double sm[11 + 2 * tri(N)];
    const int e = e0 + blockIdx.y;
    // The exposure's constants -> shared memory. When they were uploaded by a copy earlier in the
    // stream they are staged BEFORE waiting for the node kernel (this kernel's launch overlaps it);
    // when the node kernel itself brings them in (late_consts), after.
    if (late_consts) {
        pdl_trigger();
        pdl_wait();
    }
    const bool inv_exact = INV && N > 0 && srcdev[e].inv_exact != 0;
    {
        const SourceDev &s = srcdev[e];
        for (int k = threadIdx.x; k < 11 + 2 * tri(N); k += blockDim.x) {
            double v;
            if (k < 9) v = s.m[k];
            else if (k == 9) v = s.c1;
            else if (k == 10) v = s.c2;
            else {
                // slot of the order-N layout -> (p, q) -> slot of the stored order-n layout
                const int t = (k - 11) % tri(N);
                const Poly &P = (k - 11) < tri(N) ? s.ap : s.bp;
                int p = 0;
                while (p < N && tri_off(N, p + 1) <= t) ++p;
                const int q = t - tri_off(N, p), n = P.order;
                v = (p + q <= n) ? P.c[tri_off(n, p) + q] : 0.0;
            }
            sm[k] = v;
        }
    }
    if (!late_consts) pdl_trigger();                // the main kernel's launch may overlap this one
    __syncthreads();
    if (!late_consts) pdl_wait();                   // the node table is complete
    const int c = blockIdx.x * kSetupThreads + threadIdx.x;
    int nflag[3] = {0, 0, 0};
    if (c < ctas) {
        const int cty = c / ctas_x, ctx = c - cty * ctas_x;
        double Px[16], Py[16];                      // parent cubic, unit = 32 px
        const bool parent = fit_cubic<N>(sm, inv_exact, fc, [&](int k) { return __ldg(uv + (size_t)k * ctas + c); }, Px, Py);
        int box_x = kNoBox, box_y = kNoBox;
#pragma unroll 1
        for (int sub = 0; sub < CTA_T * CTA_T; ++sub) {
            const int ttx = ctx * CTA_T + (sub % CTA_T), tty = cty * CTA_T + (sub / CTA_T);
            if (ttx >= tiles_x || tty >= tiles_y) continue;
            double Cx[16], Cy[16];
            bool good = true;
            if (parent) {
                const double s0 = (sub % CTA_T) ? 0.5 : -0.5, t0 = (sub / CTA_T) ? 0.5 : -0.5;
#pragma unroll
                for (int k = 0; k < 16; ++k) { Cx[k] = Px[k]; Cy[k] = Py[k]; }
#pragma unroll
                for (int q = 0; q < 4; ++q) {       // along s, each power of t
                    shift_half(Cx[4 * q], Cx[4 * q + 1], Cx[4 * q + 2], Cx[4 * q + 3], s0);
                    shift_half(Cy[4 * q], Cy[4 * q + 1], Cy[4 * q + 2], Cy[4 * q + 3], s0);
                }
#pragma unroll
                for (int pp = 0; pp < 4; ++pp) {    // along t, each power of s
                    shift_half(Cx[pp], Cx[4 + pp], Cx[8 + pp], Cx[12 + pp], t0);
                    shift_half(Cy[pp], Cy[4 + pp], Cy[8 + pp], Cy[12 + pp], t0);
                }
            } else {
                const double cx0 = ttx * TS + kCentre, cy0 = tty * TS + kCentre;
                good = fit_cubic<N>(sm, inv_exact, fc, [&](int k) {
                    double U, V;
                    target_uv(tgt, cx0 + kHalf * fc.pts[k][0], cy0 + kHalf * fc.pts[k][1], U, V);
                    return make_double2(U, V);
                }, Cx, Cy);
            }
            int bx0, by0;
            const int flag = emit_tile(Cx, Cy, good, sny, snx,
                                       recs + ((size_t)e * tiles_x * tiles_y + (size_t)tty * tiles_x + ttx), bx0, by0);
            ++nflag[flag];
            if (flag == TILE_FAST) { box_x = min(box_x, bx0); box_y = min(box_y, by0); }
        }
        // origin of the CTA tile's staged box = min over its FAST tiles (kNoBox: none)
        cta_box[(size_t)e * ctas + c] = make_int2(box_x, box_y);
    }
    // tile statistics: per-warp sums -> device counters; the last block of the last launch
    // (ticket) writes the totals straight into the caller's mapped host memory, so
    // dfr_last_stats needs neither a memset nor a copy in the stream
#pragma unroll
    for (int f = 0; f < 3; ++f) {
        const int w = __reduce_add_sync(0xffffffffu, nflag[f]);
        if ((threadIdx.x & 31) == 0 && w) atomicAdd(&counters[f], w);
    }
    __syncthreads();
    if (threadIdx.x == 0 && host_stats) {
        __threadfence();
        if (atomicAdd(&counters[3], 1) == total_blocks - 1) {
            __threadfence();
            for (int f = 0; f < 3; ++f) {
                const int32_t v = *(volatile int32_t *)&counters[f];
                if (stats_add) atomicAdd(&host_stats[f], v);     // streaming calls: device-side totals
                else host_stats[f] = v;
            }
        }
    }
}

// ---------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                  const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode()
{
    // function-local static initialiser: run once, and every thread that gets here meanwhile waits for
    // it (the *_multi entry points start several worker threads that all reach this on first use)
    static const EncodeTiledFn fn = []() -> EncodeTiledFn {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            return (EncodeTiledFn)p;
        return nullptr;
    }();
    return fn;
}


// Source-pixel extent of an output region of span_tiles x span_tiles tiles, from the Jacobian of the map probed in fp64
// on the host at the centre of the output grid, per exposure (3 map evaluations each; the
// Jacobian varies by well under 1 % over a frame, the caller adds 2 % + fixed margins, and
// the kernel checks every pixel against the staged box anyway). False if no probe is finite.
static bool probe_extent(const TargetDev &tgt, const SourceDev *hs, int n, int ony, int onx, int span_tiles,
                         double &ext_x, double &ext_y)
{
    const double span = TS * span_tiles - 1;
    const double ci = 0.5 * (onx - 1), cj = 0.5 * (ony - 1), h = 16.0;
    double U0, V0, U1, V1, U2, V2;
    target_uv(tgt, ci, cj, U0, V0);
    target_uv(tgt, ci + h, cj, U1, V1);
    target_uv(tgt, ci, cj + h, U2, V2);
    const int step = n > 256 ? n / 256 : 1;
    bool any = false;
    ext_x = ext_y = 0.0;
    for (int e = 0; e < n; e += step) {
        double x0, y0, x1, y1, x2, y2;
        source_xy(hs[e], U0, V0, x0, y0);
        source_xy(hs[e], U1, V1, x1, y1);
        source_xy(hs[e], U2, V2, x2, y2);
        const double jxx = (x1 - x0) / h, jxy = (x2 - x0) / h, jyx = (y1 - y0) / h, jyy = (y2 - y0) / h;
        if (!(std::isfinite(jxx) && std::isfinite(jxy) && std::isfinite(jyx) && std::isfinite(jyy))) continue;
        any = true;
        ext_x = std::fmax(ext_x, span * (std::fabs(jxx) + std::fabs(jxy)));
        ext_y = std::fmax(ext_y, span * (std::fabs(jyx) + std::fabs(jyy)));
    }
    return any;
}

cudaError_t run_setup(int n, int sny, int snx, const TargetDev &tgt, const SourceDev *srcdev,
                             const SourceDev *srchost, int ony, int onx, cudaStream_t st,
                             int32_t *host_stats, int stats_add, Scratch &sc, TiledParams &P, const ConstsCopy &cc)
{
    static const FitConsts fc = make_fit_consts();
    P.n = n; P.sny = sny; P.snx = snx; P.ony = ony; P.onx = onx;
    P.tiles_x = (onx + TS - 1) / TS;
    P.tiles_y = (ony + TS - 1) / TS;
    P.ctas_x = (P.tiles_x + CTA_T - 1) / CTA_T;
    P.ctas_y = (P.tiles_y + CTA_T - 1) / CTA_T;
    P.srcdev = srcdev;
    const int ntile = P.tiles_x * P.tiles_y;
    cudaError_t err;
    const int ctas = P.ctas_x * P.ctas_y;
    // one stream-ordered allocation from the library's pool, carved up (256-byte aligned pieces)
    auto up = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const int sups_x = (P.ctas_x + SUP_T - 1) / SUP_T, sups_y = (P.ctas_y + SUP_T - 1) / SUP_T, nsup = sups_x * sups_y;
    // which setup kernel: the wide one (a thread per 64x64 tile) when the launch fills the GPU anyway,
    // the cooperative one (16 lanes per 128x128 super-tile, short serial chain) otherwise
    const bool wide = (long long)ctas * n >= kWideThreshold;
    const size_t b_uv = up(sizeof(double2) * std::max((size_t)nsup * 2 * kSupLanes, (size_t)ctas * NPTS)), b_recs = up(sizeof(TileRec) * (size_t)ntile * n),
                 b_box = up(sizeof(int2) * (size_t)ctas * n), b_cnt = up(4 * sizeof(int32_t));
    if ((err = scratch_alloc(&sc.block, b_uv + b_recs + b_box + b_cnt, st)) != cudaSuccess) return err;
    char *base = static_cast<char *>(sc.block);
    sc.uv = reinterpret_cast<double2 *>(base);
    sc.recs = reinterpret_cast<TileRec *>(base + b_uv);
    sc.cta_box = reinterpret_cast<int2 *>(base + b_uv + b_recs);
    sc.counters = reinterpret_cast<int32_t *>(base + b_uv + b_recs + b_box);
    P.recs = sc.recs;
    P.cta_box = sc.cta_box;
    {
        const unsigned nb = (unsigned)(((wide ? ctas * NPTS : nsup * 2 * kSupLanes) + 127) / 128);
        const int nx_ = wide ? P.ctas_x : sups_x, nn_ = wide ? ctas : nsup;
        const uint4 *mp = static_cast<const uint4 *>(cc.mapped);
        if (cc.packed && cc.packed_bytes > kPackedSmallBytes) {
            static thread_local PackedConsts<kPackedMaxBytes> pk;         // kernel parameters are copied at launch
            std::memcpy(&pk, cc.packed, (size_t)cc.packed_bytes);
            target_nodes_kernel<kPackedMaxBytes><<<nb, 128, 0, st>>>(tgt, fc, nx_, nn_, sc.uv, sc.counters, mp, cc.dst,
                                                                     (int)cc.bytes, cc.n, cc.T, cc.nweights, pk, wide ? 1 : 0);
        } else {
            static thread_local PackedConsts<kPackedSmallBytes> pk;
            if (cc.packed) std::memcpy(&pk, cc.packed, (size_t)cc.packed_bytes);
            target_nodes_kernel<kPackedSmallBytes><<<nb, 128, 0, st>>>(tgt, fc, nx_, nn_, sc.uv, sc.counters, mp, cc.dst,
                                                                       (int)cc.bytes, cc.packed ? cc.n : 0, cc.T, cc.nweights, pk, wide ? 1 : 0);
        }
    }
    if ((err = cudaGetLastError()) != cudaSuccess) return err;
    // SIP order class of the batch: inverse polynomials are zero-padded up to N
    int maxo = 0;
    bool inv = false;
    for (int e = 0; e < n; ++e) {
        maxo = std::max(maxo, std::max(srchost[e].ap.order, srchost[e].bp.order));
        inv = inv || srchost[e].inv_exact != 0;
    }
    const unsigned bx = wide ? (unsigned)((ctas + kSetupThreads - 1) / kSetupThreads) : (unsigned)((nsup + kSupPerBlock - 1) / kSupPerBlock);
    const long long total_blocks = (long long)bx * n;
    if (total_blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    for (int e0 = 0; e0 < n; e0 += 65535) {
        const dim3 grid(bx, (unsigned)std::min(n - e0, 65535));
#define DFR_SETUP(NN, II)                                                                                           \
    (wide ? launch_pdl(tile_setup_wide_kernel<NN, II>, grid, dim3(kSetupThreads), 0, st, (const double2 *)sc.uv, srcdev,  \
                       tgt, fc, e0, P.tiles_x, P.tiles_y, P.ctas_x, ctas, sny, snx, sc.recs, sc.cta_box, sc.counters,     \
                       (int)total_blocks, host_stats, stats_add, cc.any() ? 1 : 0)                                        \
          : launch_pdl(tile_setup_kernel<NN, II>, grid, dim3(kSetupThreads), 0, st, (const double2 *)sc.uv, srcdev, tgt,  \
                       fc, e0, P.tiles_x, P.tiles_y, P.ctas_x, P.ctas_y, sups_x, nsup, sny, snx, sc.recs, sc.cta_box,     \
                       sc.counters, (int)total_blocks, host_stats, stats_add, cc.any() ? 1 : 0))
        if (maxo == 0) err = DFR_SETUP(0, false);
        else if (maxo <= 3) err = inv ? DFR_SETUP(3, true) : DFR_SETUP(3, false);
        else if (maxo <= 4) err = inv ? DFR_SETUP(4, true) : DFR_SETUP(4, false);
        else if (maxo <= 5) err = inv ? DFR_SETUP(5, true) : DFR_SETUP(5, false);
        else err = inv ? DFR_SETUP(9, true) : DFR_SETUP(9, false);
#undef DFR_SETUP
        if (err != cudaSuccess) return err;
    }
    return cudaSuccess;
}

void free_scratch(Scratch &sc, cudaStream_t st)
{
    if (sc.block) cudaFreeAsync(sc.block, st);
    sc = Scratch();
}

cudaError_t prepare_tiled(const float *src, int n, int sny, int snx, const TargetDev &tgt,
                                 const SourceDev *srcdev, const SourceDev *srchost, int ony, int onx,
                                 int order, cudaStream_t st, int32_t *host_stats, int stats_add, Prepared &R,
                                 const ConstsCopy &cc, int span_tiles, size_t max_box_bytes)
{
    std::memset(&R.P, 0, sizeof R.P);
    std::memset(&R.tmap, 0, sizeof R.tmap);
    R.P.src = src;
    cudaError_t err = run_setup(n, sny, snx, tgt, srcdev, srchost, ony, onx, st, host_stats, stats_add, R.sc, R.P, cc);
    if (err != cudaSuccess) return err;
    // ---- staging decision: box size from a host probe; TMA needs 16-byte rows
    double ex, ey;
    const int tlo = (order == DFR_BICUBIC) ? 1 : 0, thi = (order == DFR_BICUBIC) ? 2 : 1;
    EncodeTiledFn enc = get_encode();
    bool no_stage = false;
    // Row pitch of the staged box. Bicubic: a multiple of 32 floats (128 B), so the lanes of a warp,
    // whose taps span two or three box rows under any rotation, never meet in a bank — its 16 LDS per
    // pixel made shared-memory wavefronts the wall (ncu, C3: 13.5 M conflicts on 26.8 M wavefronts, data
    // pipe 79 %; 0.131 -> 0.102 ms). Nearest / bilinear read 1 / 4 taps and are HBM-bound: the narrower
    // box (fewer L2 -> shared bytes, more CTAs per SM) measured equal or better there.
    int bw_align = (order == DFR_BICUBIC) ? 32 : 4;
#ifdef DFR_DEV_HOOKS                                                 // A-B timing builds only (never the shipped library)
    no_stage = std::getenv("DFR_NO_STAGE") != nullptr;
    if (const char *a = std::getenv("DFR_BW_ALIGN")) bw_align = std::atoi(a);
#endif
    if (!no_stage && enc && (snx % 4 == 0) && ((uintptr_t)src % 16 == 0) && probe_extent(tgt, srchost, n, ony, onx, span_tiles, ex, ey)) {
        // floor-range spread + taps + 1 px safety each side; + 3: the origin is rounded down
        // to a multiple of 4 floats; then the width itself is rounded up to 16 bytes
        int bw = ((int)std::ceil(ex * 1.02) + 2 + tlo + thi + 2 + 3 + 3) & ~3;
        const int bh = (int)std::ceil(ey * 1.02) + 2 + tlo + thi + 2;
        const int bwa = (bw + bw_align - 1) / bw_align * bw_align;
        if (bwa <= 256 && (size_t)bwa * bh * sizeof(float) <= max_box_bytes) bw = bwa;
        if (bw <= 256 && bh <= 256 && (size_t)bw * bh * sizeof(float) <= max_box_bytes) {
            const cuuint64_t dims[3] = {(cuuint64_t)snx, (cuuint64_t)sny, (cuuint64_t)n};
            const cuuint64_t strides[2] = {(cuuint64_t)snx * 4, (cuuint64_t)snx * sny * 4};
            const cuuint32_t boxd[3] = {(cuuint32_t)bw, (cuuint32_t)bh, 1};
            const cuuint32_t estr[3] = {1, 1, 1};
            CUresult r = enc(&R.tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)src, dims, strides, boxd, estr,
                             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                             CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r == CUDA_SUCCESS) { R.stage = true; R.P.BW = bw; R.P.BH = bh; }
        }
    }
    R.box_bytes = R.stage ? (size_t)R.P.BW * R.P.BH * sizeof(float) : 0;
    return cudaSuccess;
}

}  // namespace dfr
