// Host utility, off the hot path: smallest eigenvalue of the
// symmetric tridiagonal T_m by bisection on the Sturm count.
#include <cmath>
#include <cstdint>
#include <limits>
#include <new>

#include "../../include/hubbard.h"

namespace {

// number of eigenvalues of T strictly below x (LDL^T pivot signs)
int sturm_count(const double *a, const double *b, int m, double x)
{
    int cnt = 0;
    double d = 1.0;
    const double tiny = std::numeric_limits<double>::min();
    for (int i = 0; i < m; ++i) {
        double off = (i == 0) ? 0.0 : b[i - 1] * b[i - 1];
        d = (a[i] - x) - (i == 0 ? 0.0 : off / d);
        if (d == 0.0) d = -tiny;  // treat an exact zero pivot as negative
        if (d < 0.0) ++cnt;
    }
    return cnt;
}

}  // namespace

extern "C" int lanczos_ground_energy(const double *alpha, const double *beta, int m, double *e0)
{
    if (!alpha || !e0 || m < 1 || (m > 1 && !beta)) return HUBBARD_ERR_INVALID;
    for (int i = 0; i < m; ++i)
        if (!std::isfinite(alpha[i]) || (i + 1 < m && !std::isfinite(beta[i]))) return HUBBARD_ERR_INVALID;
    // Gershgorin bounds
    double lo = std::numeric_limits<double>::infinity(), hi = -lo;
    for (int i = 0; i < m; ++i) {
        double r = (i > 0 ? std::fabs(beta[i - 1]) : 0.0) + (i + 1 < m ? std::fabs(beta[i]) : 0.0);
        lo = std::fmin(lo, alpha[i] - r);
        hi = std::fmax(hi, alpha[i] + r);
    }
    double span = std::fmax(hi - lo, 1.0);
    lo -= 1e-12 * span;
    hi += 1e-12 * span;
    // invariant: count(lo) == 0, count(hi) >= 1
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (mid <= lo || mid >= hi) break;
        if (sturm_count(alpha, beta, m, mid) >= 1) hi = mid; else lo = mid;
    }
    *e0 = 0.5 * (lo + hi);
    return HUBBARD_OK;
}

// Eigenvector of T_m for its smallest eigenvalue ("the
// eigenvalues and eigenvectors of T can be computed with standard methods"):
// inverse iteration on (T - sigma I) with sigma just below the bisection value,
// tridiagonal LU with partial pivoting, three sweeps.  y has unit norm and
// y[0] >= 0.
extern "C" int lanczos_ground_vector(const double *alpha, const double *beta, int m, double *e0, double *y)
{
    if (!y) return HUBBARD_ERR_INVALID;
    double lam = 0.0;
    int rc = lanczos_ground_energy(alpha, beta, m, &lam);
    if (rc) return rc;
    if (e0) *e0 = lam;
    if (m == 1) { y[0] = 1.0; return HUBBARD_OK; }
    double scale = 0.0;
    for (int i = 0; i < m; ++i) scale = std::fmax(scale, std::fabs(alpha[i]) + (i + 1 < m ? std::fabs(beta[i]) : 0.0));
    const double sigma = lam - 1e-13 * std::fmax(scale, 1.0);
    double *buf = new (std::nothrow) double[5 * (size_t)m];
    if (!buf) return HUBBARD_ERR_HOST_OOM;
    double *d = buf, *u1 = buf + m, *u2 = buf + 2 * m, *l = buf + 3 * m, *rhs = buf + 4 * m;
    int *piv = new (std::nothrow) int[(size_t)m];
    if (!piv) { delete[] buf; return HUBBARD_ERR_HOST_OOM; }
    // LU of the shifted matrix: rows are (sub, diag, super); after elimination row i holds d[i], u1[i], u2[i]
    for (int i = 0; i < m; ++i) { d[i] = alpha[i] - sigma; u1[i] = (i + 1 < m) ? beta[i] : 0.0; u2[i] = 0.0; }
    const double tiny = 1e-300 + 1e-16 * std::fmax(scale, 1.0);
    for (int i = 0; i + 1 < m; ++i) {
        const double sub = beta[i];                 // element (i+1, i)
        if (std::fabs(sub) > std::fabs(d[i])) {     // swap rows i and i+1
            piv[i] = 1;
            const double di = d[i], ui = u1[i];
            d[i] = sub; u1[i] = d[i + 1]; u2[i] = u1[i + 1];
            l[i] = di / sub;
            d[i + 1] = ui - l[i] * u1[i];
            u1[i + 1] = -l[i] * u2[i];
        } else {
            piv[i] = 0;
            if (d[i] == 0.0) d[i] = tiny;
            l[i] = sub / d[i];
            d[i + 1] -= l[i] * u1[i];
        }
    }
    if (d[m - 1] == 0.0) d[m - 1] = tiny;
    for (int i = 0; i < m; ++i) y[i] = 1.0 / std::sqrt((double)m) * (1.0 + 0.01 * ((i * 7) % 5));
    for (int sweep = 0; sweep < 3; ++sweep) {
        for (int i = 0; i < m; ++i) rhs[i] = y[i];
        for (int i = 0; i + 1 < m; ++i) {           // forward: apply the row operations
            if (piv[i]) { const double t = rhs[i]; rhs[i] = rhs[i + 1]; rhs[i + 1] = t; }
            rhs[i + 1] -= l[i] * rhs[i];
        }
        for (int i = m - 1; i >= 0; --i) {          // back substitution
            double s = rhs[i];
            if (i + 1 < m) s -= u1[i] * y[i + 1];
            if (i + 2 < m) s -= u2[i] * y[i + 2];
            y[i] = s / d[i];
        }
        double nrm = 0.0;
        for (int i = 0; i < m; ++i) nrm = std::fmax(nrm, std::fabs(y[i]));
        if (!(nrm > 0.0) || !std::isfinite(nrm)) { delete[] buf; delete[] piv; return HUBBARD_ERR_INVALID; }
        for (int i = 0; i < m; ++i) y[i] /= nrm;
    }
    double n2 = 0.0;
    for (int i = 0; i < m; ++i) n2 += y[i] * y[i];
    const double s = (y[0] < 0.0 ? -1.0 : 1.0) / std::sqrt(n2);
    for (int i = 0; i < m; ++i) y[i] *= s;
    delete[] buf;
    delete[] piv;
    return HUBBARD_OK;
}

namespace {

// All eigenvalues d[] and eigenvectors Z (row-major m x m, column k = vector k) of the symmetric tridiagonal
// (d, e): implicit QL iteration with Wilkinson shifts (the classical EISPACK scheme restated), O(m^3) with the
// eigenvector accumulation; m is at most a few hundred here.  e has m entries, e[m-1] unused.
bool tridiag_eigh(int m, double *d, double *e, double *Z)
{
    for (int i = 0; i < m; ++i)
        for (int k = 0; k < m; ++k) Z[(size_t)i * m + k] = (i == k) ? 1.0 : 0.0;
    e[m - 1] = 0.0;
    for (int l = 0; l < m; ++l) {
        int iter = 0, mm;
        do {
            for (mm = l; mm < m - 1; ++mm) {
                const double dd = std::fabs(d[mm]) + std::fabs(d[mm + 1]);
                if (std::fabs(e[mm]) <= std::numeric_limits<double>::epsilon() * dd) break;
            }
            if (mm != l) {
                if (iter++ == 200) return false;
                double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
                double r = std::hypot(g, 1.0);
                g = d[mm] - d[l] + e[l] / (g + (g >= 0.0 ? std::fabs(r) : -std::fabs(r)));
                double s = 1.0, c = 1.0, p = 0.0;
                int i;
                for (i = mm - 1; i >= l; --i) {
                    double f = s * e[i];
                    const double b = c * e[i];
                    r = std::hypot(f, g);
                    e[i + 1] = r;
                    if (r == 0.0) {
                        d[i + 1] -= p;
                        e[mm] = 0.0;
                        break;
                    }
                    s = f / r;
                    c = g / r;
                    g = d[i + 1] - p;
                    r = (d[i] - g) * s + 2.0 * c * b;
                    p = s * r;
                    d[i + 1] = g + p;
                    g = c * r - b;
                    for (int k = 0; k < m; ++k) {
                        f = Z[(size_t)k * m + i + 1];
                        Z[(size_t)k * m + i + 1] = s * Z[(size_t)k * m + i] + c * f;
                        Z[(size_t)k * m + i] = c * Z[(size_t)k * m + i] - s * f;
                    }
                }
                if (r == 0.0 && i >= l) continue;
                d[l] -= p;
                e[l] = g;
                e[mm] = 0.0;
            }
        } while (mm != l);
    }
    return true;
}

}  // namespace

// y = exp(-(tau + i t) T_m) e_1 (host utility for lanczos_propagate; "time propagation"):
// T_m = Q diag(lambda) Q^T, y_j = sum_k Q[j][k] exp(-(tau + i t) lambda_k) Q[0][k].
extern "C" int lanczos_expm_e1(const double *alpha, const double *beta, int m, double tau, double t, double *y_re,
                               double *y_im)
{
    if (!alpha || m < 1 || (m > 1 && !beta) || !y_re || !y_im || !std::isfinite(tau) || !std::isfinite(t))
        return HUBBARD_ERR_INVALID;
    for (int i = 0; i < m; ++i)
        if (!std::isfinite(alpha[i]) || (i + 1 < m && !std::isfinite(beta[i]))) return HUBBARD_ERR_INVALID;
    double *buf = new (std::nothrow) double[(size_t)m * m + 2 * (size_t)m];
    if (!buf) return HUBBARD_ERR_HOST_OOM;
    double *Z = buf, *d = buf + (size_t)m * m, *e = d + m;
    for (int i = 0; i < m; ++i) { d[i] = alpha[i]; e[i] = (i + 1 < m) ? beta[i] : 0.0; }
    if (!tridiag_eigh(m, d, e, Z)) { delete[] buf; return HUBBARD_ERR_INVALID; }
    for (int j = 0; j < m; ++j) y_re[j] = y_im[j] = 0.0;
    for (int k = 0; k < m; ++k) {
        const double w = std::exp(-tau * d[k]) * Z[k];            // Z[0][k]
        const double cr = w * std::cos(t * d[k]), ci = -w * std::sin(t * d[k]);
        for (int j = 0; j < m; ++j) {
            y_re[j] += Z[(size_t)j * m + k] * cr;
            y_im[j] += Z[(size_t)j * m + k] * ci;
        }
    }
    delete[] buf;
    return HUBBARD_OK;
}
