/*
 * orc_closed.c — a SECOND, independent statement of the gnomonic step, used
 * only to pin orc.c (pin P2 of DESIGN.md §4). Test infrastructure; shares no
 * code with orc.c or with the CUDA path.
 *
 * These are the textbook gnomonic (tangent-plane) formulas in standard
 * coordinates (xi, eta), e.g. Calabretta & Greisen 2002 §5.1.3
 * specialised to LONPOLE = 180 deg; the paper's phi/theta chain
 * must agree with them to rounding.
 *
 *   forward:  ra  = ra0 + atan2(xi, cos dec0 - eta sin dec0)
 *             dec = atan2(sin dec0 + eta cos dec0, hypot(xi, cos dec0 - eta sin dec0))
 *   inverse:  D   = sin dec0 sin dec + cos dec0 cos dec cos(ra - ra0)
 *             xi  = cos dec sin(ra - ra0) / D
 *             eta = (cos dec0 sin dec - sin dec0 cos dec cos(ra - ra0)) / D
 * with xi = u' pi/180, eta = v' pi/180 (u', v' = CD (u, v) in degrees).
 */
#include <math.h>
#include <stdint.h>

static const double CPI = 3.14159265358979323846264338327950288;

/* intermediate world coordinates (degrees) -> sky (degrees, RA not reduced) */
void orc_closed_iwc2sky(const double crval[2], const double *up, const double *vp, int64_t n,
                        double *ra_deg, double *dec_deg)
{
    double ra0 = crval[0] * CPI / 180.0, dec0 = crval[1] * CPI / 180.0;
    for (int64_t k = 0; k < n; ++k) {
        double xi = up[k] * CPI / 180.0, eta = vp[k] * CPI / 180.0;
        double den = cos(dec0) - eta * sin(dec0);
        double ra = ra0 + atan2(xi, den);
        double dec = atan2(sin(dec0) + eta * cos(dec0), hypot(xi, den));
        ra_deg[k] = ra * 180.0 / CPI;
        dec_deg[k] = dec * 180.0 / CPI;
    }
}

/* sky (degrees) -> intermediate world coordinates (degrees); NaN when D <= 0 */
void orc_closed_sky2iwc(const double crval[2], const double *ra_deg, const double *dec_deg,
                        int64_t n, double *up, double *vp)
{
    double ra0 = crval[0] * CPI / 180.0, dec0 = crval[1] * CPI / 180.0;
    for (int64_t k = 0; k < n; ++k) {
        double ra = ra_deg[k] * CPI / 180.0, dec = dec_deg[k] * CPI / 180.0;
        double dra = ra - ra0;
        double D = sin(dec0) * sin(dec) + cos(dec0) * cos(dec) * cos(dra);
        if (!(D > 0.0)) { up[k] = NAN; vp[k] = NAN; continue; }
        double xi = cos(dec) * sin(dra) / D;
        double eta = (cos(dec0) * sin(dec) - sin(dec0) * cos(dec) * cos(dra)) / D;
        up[k] = xi * 180.0 / CPI;
        vp[k] = eta * 180.0 / CPI;
    }
}
