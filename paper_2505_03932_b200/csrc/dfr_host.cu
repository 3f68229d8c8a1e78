// dfr_host.cu — host-side WCS validation and fp64 pre-composition (no kernels).
//
// The per-pixel spherical trigonometry of PAPER.md:91-95 and :101-111 is
// algebraically a fixed projective map between the two tangent planes
// (DESIGN.md §6): with the orthonormal triad at a tangent point (ra, dec)
//   e = (-sin ra, cos ra, 0)             east
//   n = (-sin dec cos ra, -sin dec sin ra, cos dec)   north
//   k = ( cos dec cos ra,  cos dec sin ra, sin dec)   towards the tangent point
// a target-plane point (xi, eta) [radians] is the direction p = k_t + xi e_t + eta n_t
// and its source-plane coordinates are xi_s = (p.e_s)/(p.k_s), eta_s = (p.n_s)/(p.k_s);
// p.k_s <= 0 <=> the paper's sin(theta) <= 0. Everything that
// depends only on the (target, exposure) pair is folded here, once, in double.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "dfr_internal.h"

namespace dfr {

static thread_local std::string g_err;

void set_error(const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
}

const char *last_error_cstr() { return g_err.c_str(); }

int cuda_fail(cudaError_t e, const char *what)
{
    set_error("%s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
    return DFR_ERR_CUDA;
}

static bool poly_finite(const double *c, int order)
{
    for (int p = 0; p <= order; ++p)
        for (int q = 0; p + q <= order; ++q)
            if (!std::isfinite(c[p * DFR_SIP_DIM + q])) return false;
    return true;
}

int validate_wcs(const dfr_wcs *w)
{
    const bool inv_exact = w->ap_order == DFR_SIP_INVERSE_EXACT && w->bp_order == DFR_SIP_INVERSE_EXACT;
    const int32_t ords[4] = {w->a_order, w->b_order, inv_exact ? 0 : w->ap_order, inv_exact ? 0 : w->bp_order};
    for (int k = 0; k < 4; ++k)
        if (ords[k] < 0 || ords[k] > DFR_SIP_MAX_ORDER) {
            set_error("SIP order %d outside [0, %d]", ords[k], DFR_SIP_MAX_ORDER);
            return DFR_ERR_SIP_ORDER;
        }
    for (int k = 0; k < 2; ++k)
        if (!std::isfinite(w->crpix[k]) || !std::isfinite(w->crval[k])) {
            set_error("non-finite CRPIX/CRVAL");
            return DFR_ERR_NONFINITE_WCS;
        }
    for (int k = 0; k < 4; ++k)
        if (!std::isfinite(w->cd[k])) {
            set_error("non-finite CD");
            return DFR_ERR_NONFINITE_WCS;
        }
    if (!poly_finite(w->a, w->a_order) || !poly_finite(w->b, w->b_order) ||
        !poly_finite(w->ap, ords[2]) || !poly_finite(w->bp, ords[3])) {
        set_error("non-finite SIP coefficient");
        return DFR_ERR_NONFINITE_WCS;
    }
    const double det = w->cd[0] * w->cd[3] - w->cd[1] * w->cd[2];
    if (!(std::fabs(det) > 0.0) || !std::isfinite(det)) {
        set_error("singular CD matrix (det = %g)", det);
        return DFR_ERR_SINGULAR_CD;
    }
    return DFR_OK;
}

void pack_poly(const double *c, int order, Poly *out)
{
    std::memset(out, 0, sizeof *out);
    out->order = order;
    if (order <= 0) { out->order = 0; return; }
    int k = 0;
    for (int p = 0; p <= order; ++p)
        for (int q = 0; p + q <= order; ++q) out->c[k++] = c[p * DFR_SIP_DIM + q];
}

void make_target(const dfr_wcs *t, TargetDev *out)
{
    out->c1 = t->crpix[0] - 1.0;
    out->c2 = t->crpix[1] - 1.0;
    pack_poly(t->a, t->a_order, &out->a);
    pack_poly(t->b, t->b_order, &out->b);
}

static void triad(double ra_deg, double dec_deg, double B[9] /* columns e, n, k */)
{
    const double d2r = 3.14159265358979323846264338327950288 / 180.0;
    const double sa = std::sin(ra_deg * d2r), ca = std::cos(ra_deg * d2r);
    const double sd = std::sin(dec_deg * d2r), cdc = std::cos(dec_deg * d2r);
    // row-major 3x3, column 0 = e, column 1 = n, column 2 = k
    B[0] = -sa;  B[1] = -sd * ca;  B[2] = cdc * ca;
    B[3] = ca;   B[4] = -sd * sa;  B[5] = cdc * sa;
    B[6] = 0.0;  B[7] = cdc;       B[8] = sd;
}

static void mat3(const double *A, const double *B, double *C)   // C = A B
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0.0;
            for (int k = 0; k < 3; ++k) s += A[3 * i + k] * B[3 * k + j];
            C[3 * i + j] = s;
        }
}

void make_source(const dfr_wcs *t, const dfr_wcs *s, SourceDev *out)
{
    const double kk = 3.14159265358979323846264338327950288 / 180.0;
    double Bt[9], Bs[9], BsT[9], R[9], Dt[9], Es[9], T1[9];
    triad(t->crval[0], t->crval[1], Bt);
    triad(s->crval[0], s->crval[1], Bs);
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) BsT[3 * i + j] = Bs[3 * j + i];
    mat3(BsT, Bt, R);                                   // rotation target frame -> source frame
    // (xi, eta, 1) = Dt (U, V, 1): CD_t and degrees -> radians
    const double dt[9] = {kk * t->cd[0], kk * t->cd[1], 0, kk * t->cd[2], kk * t->cd[3], 0, 0, 0, 1};
    std::memcpy(Dt, dt, sizeof dt);
    // (u_s c, v_s c, c) = Es (p.e_s, p.n_s, p.k_s): radians -> degrees and CD_s^-1
    const double det = s->cd[0] * s->cd[3] - s->cd[1] * s->cd[2];
    const double es[9] = {s->cd[3] / det / kk, -s->cd[1] / det / kk, 0,
                          -s->cd[2] / det / kk, s->cd[0] / det / kk, 0, 0, 0, 1};
    std::memcpy(Es, es, sizeof es);
    mat3(R, Dt, T1);
    mat3(Es, T1, out->m);
    out->c1 = s->crpix[0] - 1.0;
    out->c2 = s->crpix[1] - 1.0;
    out->inv_exact = (s->ap_order == DFR_SIP_INVERSE_EXACT) ? 1 : 0;
    out->pad_ = 0;
    if (out->inv_exact) {                               // the forward polynomials, inverted on the device
        pack_poly(s->a, s->a_order, &out->ap);
        pack_poly(s->b, s->b_order, &out->bp);
    } else {
        pack_poly(s->ap, s->ap_order, &out->ap);
        pack_poly(s->bp, s->bp_order, &out->bp);
    }
}

void make_sky(const dfr_wcs *w, SkyDev *out)
{
    const double kk = 3.14159265358979323846264338327950288 / 180.0;
    out->c1 = w->crpix[0] - 1.0;
    out->c2 = w->crpix[1] - 1.0;
    out->ra0 = w->crval[0] * kk;
    out->dec0 = w->crval[1] * kk;
    const double det = w->cd[0] * w->cd[3] - w->cd[1] * w->cd[2];
    for (int k = 0; k < 4; ++k) out->cd[k] = w->cd[k];
    out->cdi[0] = w->cd[3] / det;
    out->cdi[1] = -w->cd[1] / det;
    out->cdi[2] = -w->cd[2] / det;
    out->cdi[3] = w->cd[0] / det;
    pack_poly(w->a, w->a_order, &out->a);
    pack_poly(w->b, w->b_order, &out->b);
    out->inv_exact = (w->ap_order == DFR_SIP_INVERSE_EXACT) ? 1 : 0;
    out->pad_ = 0;
    pack_poly(w->ap, out->inv_exact ? 0 : w->ap_order, &out->ap);
    pack_poly(w->bp, out->inv_exact ? 0 : w->bp_order, &out->bp);
}

// ---- inverse SIP fit ---------------------------------------
// Least squares by Householder QR (the scaled-monomial Gram matrix of order 9 is far too
// ill-conditioned for normal equations). A is m x n column-major, overwritten; b1, b2 are
// the two right-hand sides, overwritten; the solutions come back in x1, x2.
static void qr_solve2(std::vector<double> &A, int m, int n, std::vector<double> &b1,
                      std::vector<double> &b2, std::vector<double> &x1, std::vector<double> &x2)
{
    for (int k = 0; k < n; ++k) {
        double *col = &A[(size_t)k * m];
        double norm = 0.0;
        for (int i = k; i < m; ++i) norm += col[i] * col[i];
        norm = std::sqrt(norm);
        if (norm == 0.0) continue;
        const double alpha = col[k] > 0.0 ? -norm : norm;
        col[k] -= alpha;                              // v = x - alpha e_k, stored in place
        double vnorm2 = 0.0;
        for (int i = k; i < m; ++i) vnorm2 += col[i] * col[i];
        if (vnorm2 > 0.0) {
            auto reflect = [&](double *y) {
                double dot = 0.0;
                for (int i = k; i < m; ++i) dot += col[i] * y[i];
                const double f = 2.0 * dot / vnorm2;
                for (int i = k; i < m; ++i) y[i] -= f * col[i];
            };
            for (int j = k + 1; j < n; ++j) reflect(&A[(size_t)j * m]);
            reflect(b1.data());
            reflect(b2.data());
        }
        col[k] = alpha;                               // R_kk (the rest of v is no longer needed)
    }
    x1.assign((size_t)n, 0.0);
    x2.assign((size_t)n, 0.0);
    for (int k = n - 1; k >= 0; --k) {
        double s1 = b1[k], s2 = b2[k];
        for (int j = k + 1; j < n; ++j) {
            s1 -= A[(size_t)j * m + k] * x1[j];
            s2 -= A[(size_t)j * m + k] * x2[j];
        }
        const double r = A[(size_t)k * m + k];
        x1[k] = r != 0.0 ? s1 / r : 0.0;
        x2[k] = r != 0.0 ? s2 / r : 0.0;
    }
}

static double sip_sum(const double *c, int order, double u, double v)
{
    double r = 0.0;
    for (int p = order; p >= 0; --p) {
        double inner = 0.0;
        for (int q = order - p; q >= 0; --q) inner = inner * v + c[p * DFR_SIP_DIM + q];
        r = r * u + inner;
    }
    return r;
}

int fit_inverse_sip(dfr_wcs *w, int order, int nx, int ny, double *max_resid)
{
    constexpr int G = 64;
    const int m = G * G, n = (order + 1) * (order + 2) / 2;
    std::vector<double> U((size_t)m), V((size_t)m), du((size_t)m), dv((size_t)m);
    double hx = 0.0, hy = 0.0;
    for (int j = 0; j < G; ++j)
        for (int i = 0; i < G; ++i) {
            const double x = (nx - 1.0) * i / (G - 1.0), y = (ny - 1.0) * j / (G - 1.0);
            const double u = x - (w->crpix[0] - 1.0), v = y - (w->crpix[1] - 1.0);
            const int k = j * G + i;
            U[k] = u + (w->a_order > 0 ? sip_sum(w->a, w->a_order, u, v) : 0.0);
            V[k] = v + (w->b_order > 0 ? sip_sum(w->b, w->b_order, u, v) : 0.0);
            du[k] = u - U[k];
            dv[k] = v - V[k];
            hx = std::fmax(hx, std::fabs(U[k]));
            hy = std::fmax(hy, std::fabs(V[k]));
        }
    if (!(hx > 0.0)) hx = 1.0;
    if (!(hy > 0.0)) hy = 1.0;
    std::vector<double> A((size_t)m * n), x1, x2, b1 = du, b2 = dv;
    int col = 0;
    for (int p = 0; p <= order; ++p)
        for (int q = 0; p + q <= order; ++q, ++col)
            for (int k = 0; k < m; ++k) A[(size_t)col * m + k] = std::pow(U[k] / hx, p) * std::pow(V[k] / hy, q);
    qr_solve2(A, m, n, b1, b2, x1, x2);
    std::memset(w->ap, 0, sizeof w->ap);
    std::memset(w->bp, 0, sizeof w->bp);
    col = 0;
    for (int p = 0; p <= order; ++p)
        for (int q = 0; p + q <= order; ++q, ++col) {
            const double s = std::pow(hx, p) * std::pow(hy, q);
            w->ap[p * DFR_SIP_DIM + q] = x1[col] / s;
            w->bp[p * DFR_SIP_DIM + q] = x2[col] / s;
        }
    w->ap_order = w->bp_order = order;
    double res = 0.0;
    for (int k = 0; k < m; ++k) {
        res = std::fmax(res, std::fabs(sip_sum(w->ap, order, U[k], V[k]) - du[k]));
        res = std::fmax(res, std::fabs(sip_sum(w->bp, order, U[k], V[k]) - dv[k]));
    }
    if (max_resid) *max_resid = res;
    return DFR_OK;
}

}  // namespace dfr
