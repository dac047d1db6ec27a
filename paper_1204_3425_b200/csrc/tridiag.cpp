// Host utility, off the hot path: smallest eigenvalue of the
// symmetric tridiagonal T_m by bisection on the Sturm count.
#include <cmath>
#include <cstdint>
#include <limits>

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
