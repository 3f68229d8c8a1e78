// dfr_kernels_sky.cu — dfr_pix2world / dfr_world2pix: the LITERAL formulas of
// PAPER.md §3.2.1 (:87-95) and §3.2.2 (:101-121) in fp64 with CUDA libm trig,
// one thread per point. These are the testing entry points north_star names;
// the hot path uses the algebraically equal projective form (dfr_host.cu).
#include "dfr_device.cuh"

namespace dfr {

constexpr double kPi = 3.14159265358979323846264338327950288;

__device__ __forceinline__ double clamp1(double s) { return fmin(1.0, fmax(-1.0, s)); }

__global__ void __launch_bounds__(256)
pix2world_kernel(const SkyDev *__restrict__ wp, const double *__restrict__ x,
                 const double *__restrict__ y, int64_t npts,
                 double *__restrict__ ra_deg, double *__restrict__ dec_deg)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= npts) return;
    const SkyDev &w = *wp;
    double u = x[k] - w.c1, v = y[k] - w.c2;
    const double f = poly_eval(w.a, u, v), g = poly_eval(w.b, u, v);
    u += f;                                                      // PAPER.md:89 (sign: G3)
    v += g;
    const double up = w.cd[0] * u + w.cd[1] * v;
    const double vp = w.cd[2] * u + w.cd[3] * v;
    const double r = sqrt(up * up + vp * vp);
    const double phi = atan2(-up, vp);
    const double theta = atan2(180.0 / kPi, r);
    double st, ct, sp, cp, sd0, cd0;
    sincos(theta, &st, &ct);
    sincos(phi, &sp, &cp);
    sincos(w.dec0, &sd0, &cd0);
    const double dec = asin(clamp1(st * sd0 + ct * cd0 * cp));
    const double ra = w.ra0 + atan2(-ct * sp, st * cd0 - ct * sd0 * cp);
    double rd = fmod(ra * (180.0 / kPi), 360.0);                 // RA in [0, 360)
    if (rd < 0.0) rd += 360.0;
    if (rd >= 360.0) rd -= 360.0;
    ra_deg[k] = rd;
    dec_deg[k] = dec * (180.0 / kPi);
}

__global__ void __launch_bounds__(256)
world2pix_kernel(const SkyDev *__restrict__ wp, const double *__restrict__ ra_deg,
                 const double *__restrict__ dec_deg, int64_t npts,
                 double *__restrict__ x, double *__restrict__ y)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= npts) return;
    const SkyDev &w = *wp;
    const double ra = ra_deg[k] * (kPi / 180.0), dec = dec_deg[k] * (kPi / 180.0);
    const double dra = ra - w.ra0;
    double sd, cd, sd0, cd0, sa, ca;
    sincos(dec, &sd, &cd);
    sincos(w.dec0, &sd0, &cd0);
    sincos(dra, &sa, &ca);
    const double phi = atan2(-cd * sa, sd * cd0 - cd * sd0 * ca);
    const double theta = asin(clamp1(sd * sd0 + cd * cd0 * ca));
    double st, ct, sp, cp;
    sincos(theta, &st, &ct);
    if (!(st > 0.0)) {                                           // >= 90 deg away (G12)
        x[k] = y[k] = __longlong_as_double(0x7ff8000000000000ULL);
        return;
    }
    sincos(phi, &sp, &cp);
    const double r = (180.0 / kPi) * ct / st;
    const double up = -r * sp, vp = r * cp;
    double u = w.cdi[0] * up + w.cdi[1] * vp;
    double v = w.cdi[2] * up + w.cdi[3] * vp;
    if (w.inv_exact) {                                           // DFR_SIP_INVERSE_EXACT: invert A/B
        const double U = u, V = v;
        invert_sip([&](double p, double q) { return poly_eval(w.a, p, q); },
                   [&](double p, double q) { return poly_eval(w.b, p, q); }, U, V, u, v);
    } else {
        const double f = poly_eval(w.ap, u, v), g = poly_eval(w.bp, u, v);
        u += f;
        v += g;
    }
    x[k] = u + w.c1;
    y[k] = v + w.c2;
}

cudaError_t launch_pix2world(const SkyDev *w, const double *x, const double *y, int64_t npts,
                             double *ra, double *dec, cudaStream_t st)
{
    if (npts == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((npts + 255) / 256);
    pix2world_kernel<<<blocks, 256, 0, st>>>(w, x, y, npts, ra, dec);
    return cudaGetLastError();
}

cudaError_t launch_world2pix(const SkyDev *w, const double *ra, const double *dec, int64_t npts,
                             double *x, double *y, cudaStream_t st)
{
    if (npts == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((npts + 255) / 256);
    world2pix_kernel<<<blocks, 256, 0, st>>>(w, ra, dec, npts, x, y);
    return cudaGetLastError();
}

}  // namespace dfr
