// dfr_internal.h — private declarations shared by the translation units of libdfr.
// Not part of the C ABI (include/dfr.h). No torch types, no oracle code.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "dfr.h"

namespace dfr {

constexpr int kTriMax = 55;                 // T(9) = (9+1)(9+2)/2 packed coefficients

// Packed bivariate polynomial sum_{p+q<=order} c[p][q] u^p v^q. Row p holds
// q = 0..order-p contiguously at c[off(p)], off(p) = p*(order+1) - p*(p-1)/2.
struct Poly {
    int32_t order;                          // 0 = absent
    int32_t pad_;
    double  c[kTriMax];
};

// Target-side constants (steps a1-a3 of SURVEY.md §8(a)); passed by value as a
// __grid_constant__ kernel parameter.
struct TargetDev {
    double c1, c2;                          // crpix - 1
    Poly   a, b;                            // SIP_A, SIP_B
};

// Per-exposure constants (steps a4-a6), one entry per exposure in device memory.
//   (a, b, c) = M (U, V, 1)^T ; u_s = a/c, v_s = b/c ; valid iff c > 0
// M = diag(CD_s^-1 / k, 1) . B_s^T . B_t . diag-block(k CD_t, 1), k = pi/180, B = [e n k]
// triads at the two tangent points. Composed on the host in fp64.
struct SourceDev {
    double m[9];
    double c1, c2;                          // crpix_s - 1
    Poly   ap, bp;                          // SIP_INV_A, SIP_INV_B; inv_exact: SIP_A, SIP_B
    int32_t inv_exact;                      // DFR_SIP_INVERSE_EXACT: invert ap/bp (= A/B) by iteration
    int32_t pad_;
};

// Full WCS for the literal-trig kernels (dfr_pix2world / dfr_world2pix).
struct SkyDev {
    double c1, c2, ra0, dec0;               // radians
    double cd[4], cdi[4];                   // CD and its inverse (deg/px, px/deg)
    Poly   a, b, ap, bp;
    int32_t inv_exact;                      // DFR_SIP_INVERSE_EXACT: world2pix inverts a/b by iteration
    int32_t pad_;
};

// ---- host side (dfr_host.cpp) ---------------------------------------------
int  validate_wcs(const dfr_wcs *w);                        // DFR_OK or an error code
void pack_poly(const double *c10x10, int order, Poly *out);
void make_target(const dfr_wcs *t, TargetDev *out);
void make_source(const dfr_wcs *t, const dfr_wcs *s, SourceDev *out);
void make_sky(const dfr_wcs *w, SkyDev *out);
int  fit_inverse_sip(dfr_wcs *w, int order, int nx, int ny, double *max_resid);
void set_error(const char *fmt, ...);
int  cuda_fail(cudaError_t e, const char *what);            // records text, returns DFR_ERR_CUDA

// ---- launchers (one per .cu) -----------------------------------------------
// exact per-pixel path
cudaError_t launch_exact_reproject(const float *src, int n, int sny, int snx,
                                   const TargetDev &tgt, const SourceDev *srcdev,
                                   int ony, int onx, int order, float *out, cudaStream_t st,
                                   int edge = DFR_EDGE_AREA, float *foot = nullptr);
cudaError_t launch_exact_coords(int n, const TargetDev &tgt, const SourceDev *srcdev,
                                int ony, int onx, double *x, double *y, cudaStream_t st);
// literal sky kernels
cudaError_t launch_pix2world(const SkyDev *w, const double *x, const double *y, int64_t npts,
                             double *ra, double *dec, cudaStream_t st);
cudaError_t launch_world2pix(const SkyDev *w, const double *ra, const double *dec, int64_t npts,
                             double *x, double *y, cudaStream_t st);

}  // namespace dfr
