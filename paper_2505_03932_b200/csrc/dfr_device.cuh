// dfr_device.cuh — device functions shared by the kernels of libdfr:
// the exact fp64 pixel map (steps a1-a6 of SURVEY.md §8(a)) and the
// interpolators with the footprint rule (a7-a8).
#pragma once

#include <cuda_runtime.h>
#include <math.h>

#include "dfr_internal.h"

namespace dfr {

// fma() on the host is a libm call unless the build enables FMA; the host only needs
// these functions for coarse geometry probes, so plain a*b+c is fine there.
#ifdef __CUDA_ARCH__
#define DFR_FMA(a, b, c) fma((a), (b), (c))
#else
#define DFR_FMA(a, b, c) ((a) * (b) + (c))
#endif

// sum_{p+q<=order} c[p][q] u^p v^q by nested Horner (north_star
// "SIP is evaluated by Horner's rule"). Works for Poly in param or global space.
// The common orders are fully unrolled (no loop or index arithmetic survives).
template <int N>
__host__ __device__ __forceinline__ double poly_eval_fixed(const double *__restrict__ c, double u, double v)
{
    double r = 0.0;
#pragma unroll
    for (int p = N; p >= 0; --p) {
        const int off = p * (N + 1) - (p * (p - 1)) / 2;
        const int len = N - p + 1;
        double inner = c[off + len - 1];
#pragma unroll
        for (int q = len - 2; q >= 0; --q) inner = DFR_FMA(inner, v, c[off + q]);
        r = DFR_FMA(r, u, inner);
    }
    return r;
}

__host__ __device__ __forceinline__ double poly_eval(const Poly &P, double u, double v)
{
    const int n = P.order;
    switch (n) {
    case 0: return 0.0;
    case 2: return poly_eval_fixed<2>(P.c, u, v);
    case 3: return poly_eval_fixed<3>(P.c, u, v);
    case 4: return poly_eval_fixed<4>(P.c, u, v);
    case 5: return poly_eval_fixed<5>(P.c, u, v);
    default: break;
    }
    if (n < 0) return 0.0;
    double r = 0.0;
    for (int p = n; p >= 0; --p) {
        const int off = p * (n + 1) - (p * (p - 1)) / 2;
        const int len = n - p + 1;
        double inner = P.c[off + len - 1];
        for (int q = len - 2; q >= 0; --q) inner = DFR_FMA(inner, v, P.c[off + q]);
        r = DFR_FMA(r, u, inner);
    }
    return r;
}

// a1-a2: target pixel (i, j) -> distorted offsets (U, V).
__host__ __device__ __forceinline__ void target_uv(const TargetDev &t, double i, double j,
                                          double &U, double &V)
{
    const double u = i - t.c1, v = j - t.c2;
    U = u + poly_eval(t.a, u, v);
    V = v + poly_eval(t.b, u, v);
}

// DFR_SIP_INVERSE_EXACT: solve u + A(u, v) = U, v + B(u, v) = V by fixed-point iteration
// (u, v) <- (U - A(u, v), V - B(u, v)) to 1e-11 px. Contraction rate = the distortion's gradient
// (1e-3 ... 3e-2 for real optics): 4-8 steps; NaN if 32 steps do not converge.
constexpr int kInvIters = 32;
constexpr double kInvTol = 1e-11;
template <class PA, class PB>
__host__ __device__ __forceinline__ void invert_sip(PA polyA, PB polyB, double U, double V, double &u, double &v)
{
    u = U;
    v = V;
    bool done = false;
    for (int it = 0; it < kInvIters && !done; ++it) {
        const double un = U - polyA(u, v), vn = V - polyB(u, v);
        done = fabs(un - u) + fabs(vn - v) < kInvTol;
        u = un;
        v = vn;
    }
    if (!done) u = v = NAN;                     // includes NaN input
}

// a3-a6: (U, V) -> fractional source pixel (x, y) for one exposure
// (PAPER.md:91-121 in the projective form of dfr_host.cu). NaN when the sky
// point is >= 90 deg from the source tangent point.
__host__ __device__ __forceinline__ void source_xy(const SourceDev &s, double U, double V,
                                          double &x, double &y)
{
    const double a = DFR_FMA(s.m[0], U, DFR_FMA(s.m[1], V, s.m[2]));
    const double b = DFR_FMA(s.m[3], U, DFR_FMA(s.m[4], V, s.m[5]));
    const double c = DFR_FMA(s.m[6], U, DFR_FMA(s.m[7], V, s.m[8]));
    if (!(c > 0.0)) {
        x = y = NAN;
        return;
    }
    const double rc = 1.0 / c;
    const double us = a * rc, vs = b * rc;
    if (s.inv_exact) {
        double u, v;
        invert_sip([&](double p, double q) { return poly_eval(s.ap, p, q); },
                   [&](double p, double q) { return poly_eval(s.bp, p, q); }, us, vs, u, v);
        x = u + s.c1;
        y = v + s.c2;
        return;
    }
    x = us + poly_eval(s.ap, us, vs) + s.c1;
    y = vs + poly_eval(s.bp, us, vs) + s.c2;
}

__device__ __forceinline__ float qnanf() { return __int_as_float(0x7fc00000); }

// a7: footprint. edge = DFR_EDGE_AREA: union of source pixel areas, half-open (G6);
// edge = DFR_EDGE_PAPER: where the paper's zero-padded projected identity is positive for
// bilinear interpolation, the open square (-1, n) x (-1, n) (G19). Taps are
// edge-replicated under both, which for the second IS the ratio image / identity.
__device__ __forceinline__ bool in_footprint(double x, double y, int ny, int nx, int edge = DFR_EDGE_AREA)
{
    if (edge == DFR_EDGE_PAPER) return (x > -1.0) && (x < (double)nx) && (y > -1.0) && (y < (double)ny);
    return (x >= -0.5) && (x < (double)nx - 0.5) && (y >= -0.5) && (y < (double)ny - 0.5);
}

// The footprint array of dfr_reproject_fp ("projecting an identity
// tensor called the footprint"). DFR_EDGE_PAPER with bilinear interpolation: the zero-padded
// interpolation of an all-ones image, i.e. the product over the two axes of the weight of the taps
// that fall inside the image (1 on [0, n-1], falling linearly to 0 at -1 and at n). Every other
// mode: 1 inside the area footprint, 0 outside (nearest: the paper's identity is exactly that).
__device__ __forceinline__ float footprint_value(double x, double y, int ny, int nx, int order, int edge)
{
    if (!(x == x) || !(y == y)) return 0.0f;
    if (edge == DFR_EDGE_PAPER && order == DFR_BILINEAR) {
        if (!(x > -1.0 && x < (double)nx && y > -1.0 && y < (double)ny)) return 0.0f;
        const double wx = x < 0.0 ? 1.0 + x : (x > (double)nx - 1.0 ? (double)nx - x : 1.0);
        const double wy = y < 0.0 ? 1.0 + y : (y > (double)ny - 1.0 ? (double)ny - y : 1.0);
        return (float)(wx * wy);
    }
    return in_footprint(x, y, ny, nx, DFR_EDGE_AREA) ? 1.0f : 0.0f;
}

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return min(max(v, lo), hi); }

// Keys cubic-convolution weights for taps -1, 0, +1, +2 at fraction t, a = -0.75 (G7).
__device__ __forceinline__ void keys_weights(float t, float w[4])
{
    const float A = -0.75f;
    const float t1 = t + 1.0f, s = 1.0f - t, s1 = 2.0f - t;
    w[0] = fmaf(fmaf(fmaf(A, t1, -5.0f * A), t1, 8.0f * A), t1, -4.0f * A);
    w[1] = fmaf(fmaf(A + 2.0f, t, -(A + 3.0f)), t * t, 1.0f);
    w[2] = fmaf(fmaf(A + 2.0f, s, -(A + 3.0f)), s * s, 1.0f);
    w[3] = fmaf(fmaf(fmaf(A, s1, -5.0f * A), s1, 8.0f * A), s1, -4.0f * A);
}

// a8 with direct global gathers (taps edge-replicated). (x, y) must be in the footprint.
template <int ORDER>
__device__ __forceinline__ float sample_global(const float *__restrict__ src, int ny, int nx,
                                               double x, double y)
{
    if (ORDER == DFR_NEAREST) {
        const int ix = clampi(__double2int_rn(x), 0, nx - 1);      // round-half-even (G8)
        const int iy = clampi(__double2int_rn(y), 0, ny - 1);
        return __ldg(src + (size_t)iy * nx + ix);
    }
    const double fx0 = floor(x), fy0 = floor(y);
    const int ix = (int)fx0, iy = (int)fy0;
    const float fx = (float)(x - fx0), fy = (float)(y - fy0);
    if (ORDER == DFR_BILINEAR) {
        const int x0 = max(ix, 0), x1 = min(ix + 1, nx - 1);
        const int y0 = max(iy, 0), y1 = min(iy + 1, ny - 1);
        const float *r0 = src + (size_t)y0 * nx, *r1 = src + (size_t)y1 * nx;
        const float s00 = __ldg(r0 + x0), s10 = __ldg(r0 + x1);
        const float s01 = __ldg(r1 + x0), s11 = __ldg(r1 + x1);
        const float top = fmaf(fx, s10 - s00, s00);
        const float bot = fmaf(fx, s11 - s01, s01);
        return fmaf(fy, bot - top, top);
    }
    // bicubic, separable 4x4
    float wx[4], wy[4];
    keys_weights(fx, wx);
    keys_weights(fy, wy);
    int xs[4];
#pragma unroll
    for (int l = 0; l < 4; ++l) xs[l] = clampi(ix - 1 + l, 0, nx - 1);
    float acc = 0.0f;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        const float *r = src + (size_t)clampi(iy - 1 + m, 0, ny - 1) * nx;
        float row = wx[0] * __ldg(r + xs[0]);
        row = fmaf(wx[1], __ldg(r + xs[1]), row);
        row = fmaf(wx[2], __ldg(r + xs[2]), row);
        row = fmaf(wx[3], __ldg(r + xs[3]), row);
        acc = fmaf(wy[m], row, acc);
    }
    return acc;
}

}  // namespace dfr
