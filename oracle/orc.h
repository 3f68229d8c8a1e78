/*
 * orc.h — the ORACLE: a plain, slow, double-precision CPU restatement of the
 * dfreproject method (arXiv 2505.03932, PAPER.md = /root/reference/PAPER.md).
 *
 * THIS IS TEST INFRASTRUCTURE. Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it. It shares no
 * code, header, table or helper with the CUDA library (include/dfr.h,
 * paper_2505_03932_b200/csrc/): the struct below is declared here on its own
 * and merely has the same field order so that one Python description of a WCS
 * can be packed for either side.
 *
 * Every routine follows the paper's equations literally, one pixel at a time,
 * IEEE double, libm trig, in the paper's order (steps O1..O13 of DESIGN.md §3,
 * each citing its PAPER.md line). OpenMP over output rows is used only so the
 * timed baseline can use all host cores; it does not change any arithmetic.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1..P16 of DESIGN.md §4.
 * Readings that no available source can pin against the real package
 * ("parity unpinned"): G3 SIP sign (+, Shupe 2005), G6 footprint edge
 * (half-open pixel-area union), G7 bicubic kernel (Keys a = -0.75),
 * G19 the literal zero-pad / identity rule. (G14, NaN pixels in the source, is
 * pinned by the S6 stack pin and the interpolation pins.) See DESIGN.md §3.
 */
#ifndef ORC_H
#define ORC_H

#include <stdint.h>

#define ORC_SIP_DIM 10          /* orders 0..9 (Shupe 2005) */

typedef struct orc_wcs {
    double  crpix[2];           /* CRPIX1, CRPIX2, FITS 1-based */
    double  crval[2];           /* ra0, dec0 in degrees    */
    double  cd[4];              /* CD1_1 CD1_2 CD2_1 CD2_2, deg/px   */
    int32_t a_order, b_order, ap_order, bp_order;   /* 0 = absent */
    double  a [ORC_SIP_DIM * ORC_SIP_DIM];   /* coefficient of u^p v^q at [p*10+q] */
    double  b [ORC_SIP_DIM * ORC_SIP_DIM];
    double  ap[ORC_SIP_DIM * ORC_SIP_DIM];
    double  bp[ORC_SIP_DIM * ORC_SIP_DIM];
} orc_wcs;

enum { ORC_NEAREST = 0, ORC_BILINEAR = 1, ORC_BICUBIC = 3 };

/* O1-O5: pixel -> (ra, dec) in degrees, RA reduced to [0,360). */
void orc_pix2world(const orc_wcs *w, const double *x, const double *y, int64_t n,
                   double *ra_deg, double *dec_deg);

/* O6-O10: (ra, dec) degrees -> pixel; NaN when sin(theta) <= 0. */
void orc_world2pix(const orc_wcs *w, const double *ra_deg, const double *dec_deg, int64_t n,
                   double *x, double *y);

/* O1-O10 for every pixel of an out_ny x out_nx target grid: x, y are
 * double[out_ny*out_nx] source-pixel coordinates (NaN when invalid in O7). */
void orc_src_coords(const orc_wcs *tgt, const orc_wcs *src, int32_t out_ny, int32_t out_nx,
                    double *x, double *y);

/* O11-O12 at given coordinates: val[k] = interpolated src at (x[k], y[k]) as a
 * double (NaN outside the footprint). `a` is the Keys parameter for bicubic. */
void orc_interp(const float *src, int32_t ny, int32_t nx, const double *x, const double *y,
                int64_t n, int32_t order, double a, double *val);

/* The paper's literal footprint normalisation ("simultaneously projecting an
 * identity tensor called the footprint. The final reprojected frame is normalized by this
 * footprint"; reading G19 of DESIGN.md): the image AND an all-ones image
 * are interpolated with ZERO padding (a tap outside the image contributes nothing to
 * either), val = interp(image) / interp(ones) where interp(ones) > 0, NaN elsewhere.
 * Defined for nearest and bilinear (order 0, 1); for bicubic the projected identity
 * changes sign near the rim, so the ratio is not a footprint: returns -1.
 * foot (optional) receives interp(ones). Pins: tests/test_oracle_interp.py (F1-F4). */
int orc_interp_paper(const float *src, int32_t ny, int32_t nx, const double *x, const double *y,
                     int64_t n, int32_t order, double *val, double *foot);

/* O1-O13, the whole path: out[e][j][i] float32. Returns 0, or -1 on a bad order. */
int orc_reproject(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                  const orc_wcs *src_wcs, const orc_wcs *tgt_wcs,
                  int32_t out_ny, int32_t out_nx, int32_t order, float *out);

/* Stacking (the paper's stated purpose of reprojection, "combined
 * to produce a single, deeper image"; reading G17 of DESIGN.md):
 *   sum [j][i] = sum over exposures e of weight[e] * v_e(i, j)
 *   wsum[j][i] = sum over the same exposures of weight[e]
 * where v_e is the value O1-O12 give for exposure e (a double, NOT rounded to float32
 * first) and an exposure contributes to a pixel only where v_e is not NaN (outside its
 * footprint, or NaN source pixels under the taps). Accumulated in double in exposure
 * order, stored as float32. weight == NULL means 1 for every exposure.
 * Returns 0, or -1 on a bad order. Pins: tests/test_oracle_stack.py (S1-S6). */
int orc_stack(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
              const orc_wcs *src_wcs, const orc_wcs *tgt_wcs,
              int32_t out_ny, int32_t out_nx, int32_t order, const double *weight,
              float *sum, float *wsum);

/* CD_ij = CDELT_i * PC_ij. */
void orc_cd_from_pc_cdelt(const double pc[4], const double cdelt[2], double cd[4]);

/* OpenMP control for the timed baseline (no effect on results). */
void orc_set_threads(int n);
int  orc_get_max_threads(void);

#endif
