/*
 * orc.c — the oracle (see orc.h: test infrastructure, independent of the CUDA
 * path). Literal restatement of PAPER.md §3.1-§3.2 in IEEE double, one pixel
 * at a time. Step numbers O1..O13 are those of DESIGN.md §3.
 *
 * Readings of garbled / silent passages used here (G1..G16):
 *   G1  "\det" = dec, "atan^2" = atan2(y, x)
 *   G2  u', v', r in degrees; r0 = 180/pi
 *   G3  SIP sign is PLUS (Shupe 2005), not the paper's minus
 *   G4  both SIP polynomials see the pre-update (u, v)
 *   G5  full triangle 0 <= p+q <= order is evaluated
 *   G6  footprint = [-0.5, n-0.5) per axis, taps edge-replicated
 *   G7  bicubic = Keys cubic convolution, a = -0.75
 *   G8  nearest = round-half-even (rint)
 *   G12 sin(theta) <= 0 -> NaN
 */
#include "orc.h"

#include <math.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static const double ORC_PI = 3.14159265358979323846264338327950288;

static double deg2rad(double d) { return d * (ORC_PI / 180.0); }
static double rad2deg(double r) { return r * (180.0 / ORC_PI); }

/* x^k for a small non-negative integer k, by repeated multiplication. */
static double ipow(double x, int k)
{
    double r = 1.0;
    for (int i = 0; i < k; ++i) r *= x;
    return r;
}

/* Sum_{0 <= p+q <= order} c[p][q] u^p v^q   (reading G5). */
static double sip_poly(const double *c, int order, double u, double v)
{
    double s = 0.0;
    if (order <= 0) return 0.0;
    for (int p = 0; p <= order; ++p)
        for (int q = 0; q + p <= order; ++q)
            s += c[p * ORC_SIP_DIM + q] * ipow(u, p) * ipow(v, q);
    return s;
}

static double clamp1(double s) { return s > 1.0 ? 1.0 : (s < -1.0 ? -1.0 : s); }

/* O1-O5: pixel (x, y) -> (ra, dec) in RADIANS with WCS w. */
static void pix2sky_rad(const orc_wcs *w, double x, double y, double *ra, double *dec)
{
    /* O1: shift, FITS 1-based CRPIX with 0-based pixels */
    double u = x - (w->crpix[0] - 1.0);
    double v = y - (w->crpix[1] - 1.0);
    /* O2 (G3, G4): forward SIP, both at the same (u, v) */
    double f = sip_poly(w->a, w->a_order, u, v);
    double g = sip_poly(w->b, w->b_order, u, v);
    u = u + f;
    v = v + g;
    /* O3: CD matrix, degrees */
    double up = w->cd[0] * u + w->cd[1] * v;
    double vp = w->cd[2] * u + w->cd[3] * v;
    /* O4 */
    double r = sqrt(up * up + vp * vp);
    double r0 = 180.0 / ORC_PI;
    double phi = atan2(-up, vp);
    double theta = atan2(r0, r);
    /* O5 */
    double ra0 = deg2rad(w->crval[0]);
    double dec0 = deg2rad(w->crval[1]);
    *dec = asin(clamp1(sin(theta) * sin(dec0) + cos(theta) * cos(dec0) * cos(phi)));
    *ra = ra0 + atan2(-cos(theta) * sin(phi),
                      sin(theta) * cos(dec0) - cos(theta) * sin(dec0) * cos(phi));
}

/* O6-O10: (ra, dec) in RADIANS -> pixel with WCS w.
 * Returns 0 and NaNs when sin(theta) <= 0 (G12). */
static int sky2pix_rad(const orc_wcs *w, double ra, double dec, double *x, double *y)
{
    double ra0 = deg2rad(w->crval[0]);
    double dec0 = deg2rad(w->crval[1]);
    /* O6 */
    double dra = ra - ra0;
    double phi = atan2(-cos(dec) * sin(dra),
                       sin(dec) * cos(dec0) - cos(dec) * sin(dec0) * cos(dra));
    double theta = asin(clamp1(sin(dec) * sin(dec0) + cos(dec) * cos(dec0) * cos(dra)));
    /* O7 */
    if (!(sin(theta) > 0.0)) { *x = NAN; *y = NAN; return 0; }
    double r0 = 180.0 / ORC_PI;
    double r = r0 * cos(theta) / sin(theta);
    double up = -r * sin(phi);
    double vp = r * cos(phi);
    /* O8: explicit 2x2 inverse */
    double det = w->cd[0] * w->cd[3] - w->cd[1] * w->cd[2];
    double u = (w->cd[3] * up - w->cd[1] * vp) / det;
    double v = (-w->cd[2] * up + w->cd[0] * vp) / det;
    /* O9 (G3, G4) */
    double f = sip_poly(w->ap, w->ap_order, u, v);
    double g = sip_poly(w->bp, w->bp_order, u, v);
    u = u + f;
    v = v + g;
    /* O10 */
    *x = u + (w->crpix[0] - 1.0);
    *y = v + (w->crpix[1] - 1.0);
    return 1;
}

void orc_pix2world(const orc_wcs *w, const double *x, const double *y, int64_t n,
                   double *ra_deg, double *dec_deg)
{
    for (int64_t k = 0; k < n; ++k) {
        double ra, dec;
        pix2sky_rad(w, x[k], y[k], &ra, &dec);
        double rd = fmod(rad2deg(ra), 360.0);      /* G11: RA in [0, 360) */
        if (rd < 0.0) rd += 360.0;
        if (rd >= 360.0) rd -= 360.0;
        ra_deg[k] = rd;
        dec_deg[k] = rad2deg(dec);
    }
}

void orc_world2pix(const orc_wcs *w, const double *ra_deg, const double *dec_deg, int64_t n,
                   double *x, double *y)
{
    for (int64_t k = 0; k < n; ++k)
        sky2pix_rad(w, deg2rad(ra_deg[k]), deg2rad(dec_deg[k]), &x[k], &y[k]);
}

void orc_src_coords(const orc_wcs *tgt, const orc_wcs *src, int32_t out_ny, int32_t out_nx,
                    double *x, double *y)
{
#pragma omp parallel for schedule(static)
    for (int32_t j = 0; j < out_ny; ++j)
        for (int32_t i = 0; i < out_nx; ++i) {
            double ra, dec;
            pix2sky_rad(tgt, (double)i, (double)j, &ra, &dec);
            size_t k = (size_t)j * (size_t)out_nx + (size_t)i;
            sky2pix_rad(src, ra, dec, &x[k], &y[k]);
        }
}

/* Tap with the index clamped to the image (edge replication, G6). */
static double tap(const float *src, int32_t ny, int32_t nx, long iy, long ix)
{
    if (ix < 0) ix = 0;
    if (ix > nx - 1) ix = nx - 1;
    if (iy < 0) iy = 0;
    if (iy > ny - 1) iy = ny - 1;
    return (double)src[(size_t)iy * (size_t)nx + (size_t)ix];
}

/* Keys (1981) cubic convolution kernel with free parameter a (G7). */
static double keys(double d, double a)
{
    d = fabs(d);
    if (d <= 1.0) return (a + 2.0) * d * d * d - (a + 3.0) * d * d + 1.0;
    if (d < 2.0) return a * d * d * d - 5.0 * a * d * d + 8.0 * a * d - 4.0 * a;
    return 0.0;
}

/* O11-O12 for one point. */
static double interp_one(const float *src, int32_t ny, int32_t nx, double x, double y,
                         int32_t order, double a)
{
    /* O11 (G6): footprint = union of source pixel areas */
    if (!isfinite(x) || !isfinite(y)) return NAN;
    if (!(x >= -0.5 && x < (double)nx - 0.5)) return NAN;
    if (!(y >= -0.5 && y < (double)ny - 0.5)) return NAN;
    /* O12 */
    if (order == ORC_NEAREST) {
        long ix = (long)rint(x), iy = (long)rint(y);          /* G8 */
        return tap(src, ny, nx, iy, ix);
    }
    if (order == ORC_BILINEAR) {
        double fx0 = floor(x), fy0 = floor(y);
        long ix = (long)fx0, iy = (long)fy0;
        double fx = x - fx0, fy = y - fy0;
        double s00 = tap(src, ny, nx, iy, ix), s10 = tap(src, ny, nx, iy, ix + 1);
        double s01 = tap(src, ny, nx, iy + 1, ix), s11 = tap(src, ny, nx, iy + 1, ix + 1);
        return (1.0 - fy) * ((1.0 - fx) * s00 + fx * s10)
             + fy * ((1.0 - fx) * s01 + fx * s11);
    }
    /* bicubic: separable 4x4, taps i0-1 .. i0+2 */
    {
        double fx0 = floor(x), fy0 = floor(y);
        long ix = (long)fx0, iy = (long)fy0;
        double fx = x - fx0, fy = y - fy0;
        double acc = 0.0;
        for (int m = -1; m <= 2; ++m) {
            double wy = keys(fy - (double)m, a);
            double row = 0.0;
            for (int l = -1; l <= 2; ++l)
                row += keys(fx - (double)l, a) * tap(src, ny, nx, iy + m, ix + l);
            acc += wy * row;
        }
        return acc;
    }
}

void orc_interp(const float *src, int32_t ny, int32_t nx, const double *x, const double *y,
                int64_t n, int32_t order, double a, double *val)
{
    for (int64_t k = 0; k < n; ++k)
        val[k] = interp_one(src, ny, nx, x[k], y[k], order, a);
}

int orc_interp_paper(const float *src, int32_t ny, int32_t nx, const double *x, const double *y,
                     int64_t n, int32_t order, double *val, double *foot)
{
    if (order != ORC_NEAREST && order != ORC_BILINEAR) return -1;
    for (int64_t k = 0; k < n; ++k) {
        double num = 0.0, den = 0.0;
        if (x[k] == x[k] && y[k] == y[k]) {
            if (order == ORC_NEAREST) {
                const double rx = rint(x[k]), ry = rint(y[k]);      /* half-even (G8) */
                if (rx >= 0.0 && rx <= nx - 1.0 && ry >= 0.0 && ry <= ny - 1.0) {
                    num = (double)src[(size_t)ry * (size_t)nx + (size_t)rx];
                    den = 1.0;
                }
            } else {
                const double fx0 = floor(x[k]), fy0 = floor(y[k]);
                const double fx = x[k] - fx0, fy = y[k] - fy0;
                for (int m = 0; m < 2; ++m)
                    for (int l = 0; l < 2; ++l) {
                        const double ix = fx0 + l, iy = fy0 + m;
                        if (ix < 0.0 || ix > nx - 1.0 || iy < 0.0 || iy > ny - 1.0) continue;   /* zero padding */
                        const double w = (l ? fx : 1.0 - fx) * (m ? fy : 1.0 - fy);
                        num += w * (double)src[(size_t)iy * (size_t)nx + (size_t)ix];
                        den += w;
                    }
            }
        }
        val[k] = den > 0.0 ? num / den : NAN;
        if (foot) foot[k] = den;
    }
    return 0;
}

int orc_reproject(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                  const orc_wcs *src_wcs, const orc_wcs *tgt_wcs,
                  int32_t out_ny, int32_t out_nx, int32_t order, float *out)
{
    if (order != ORC_NEAREST && order != ORC_BILINEAR && order != ORC_BICUBIC) return -1;
    for (int32_t e = 0; e < n; ++e) {
        const float *src = src_batch + (size_t)e * (size_t)src_ny * (size_t)src_nx;
        float *dst = out + (size_t)e * (size_t)out_ny * (size_t)out_nx;
        const orc_wcs *sw = &src_wcs[e];
#pragma omp parallel for schedule(static)
        for (int32_t j = 0; j < out_ny; ++j)
            for (int32_t i = 0; i < out_nx; ++i) {
                double ra, dec, x, y;
                pix2sky_rad(tgt_wcs, (double)i, (double)j, &ra, &dec);   /* O1-O5  */
                sky2pix_rad(sw, ra, dec, &x, &y);                         /* O6-O10 */
                double val = interp_one(src, src_ny, src_nx, x, y, order, -0.75); /* O11-O12 */
                dst[(size_t)j * (size_t)out_nx + (size_t)i] = (float)val; /* O13    */
            }
    }
    return 0;
}

int orc_stack(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
              const orc_wcs *src_wcs, const orc_wcs *tgt_wcs,
              int32_t out_ny, int32_t out_nx, int32_t order, const double *weight,
              float *sum, float *wsum)
{
    if (order != ORC_NEAREST && order != ORC_BILINEAR && order != ORC_BICUBIC) return -1;
#pragma omp parallel for schedule(static)
    for (int32_t j = 0; j < out_ny; ++j)
        for (int32_t i = 0; i < out_nx; ++i) {
            double ra, dec, s = 0.0, W = 0.0;
            pix2sky_rad(tgt_wcs, (double)i, (double)j, &ra, &dec);            /* O1-O5  */
            for (int32_t e = 0; e < n; ++e) {                                  /* exposure order */
                const float *src = src_batch + (size_t)e * (size_t)src_ny * (size_t)src_nx;
                double x, y;
                sky2pix_rad(&src_wcs[e], ra, dec, &x, &y);                     /* O6-O10 */
                double val = interp_one(src, src_ny, src_nx, x, y, order, -0.75); /* O11-O12 */
                if (val == val) {                                              /* not NaN */
                    const double w = weight ? weight[e] : 1.0;
                    s += w * val;
                    W += w;
                }
            }
            sum[(size_t)j * (size_t)out_nx + (size_t)i] = (float)s;
            wsum[(size_t)j * (size_t)out_nx + (size_t)i] = (float)W;
        }
    return 0;
}

void orc_cd_from_pc_cdelt(const double pc[4], const double cdelt[2], double cd[4])
{
    cd[0] = cdelt[0] * pc[0];
    cd[1] = cdelt[0] * pc[1];
    cd[2] = cdelt[1] * pc[2];
    cd[3] = cdelt[1] * pc[3];
}

void orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_get_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
