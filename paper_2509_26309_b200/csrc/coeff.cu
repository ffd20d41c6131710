// coeff.cu -- step a1 of the path (host only): Chebyshev coefficients of exp(-i tau x) on [-1, 1].
//
//   c_k = (2 - delta_k0) (-i)^k J_k(tau)
//
// PAPER.md:434 (section 2.2.1): "the imaginary factor ... has been merged into the Chebyshev coefficients, and amxpy
// becomes amxsy defined as y = aMx - y with a being a real number" -- so the recursion T_{k+1} = 2H'T_k - T_{k-1} stays
// real-scaled and all powers of -i live here.  The paper prints no formula; formula, tau = pi and the truncation
// |J_k(tau)| < 1e-15 are BASELINE.json:configs[0] (SURVEY.md 8(c) readings #1-#3).
//
// J_k by downward recurrence (J_{k-1} = (2k/x) J_k - J_{k+1}) from an order well above max(k, x), normalised by
// Neumann's identity 1 = J_0 + 2 J_2 + 2 J_4 + ...; long double throughout.  Written independently of oracle/.
#include <cmath>
#include <vector>

#include "tbpm_internal.h"

namespace {

// J_0..J_kmax at x > 0
std::vector<long double> bessel_down(long double x, int kmax)
{
    int start = 2 * ((std::max(kmax, (int)std::ceil((double)x)) + 80 + (int)std::sqrt(40.0 * (double)(kmax + x))) / 2 + 1);
    std::vector<long double> f((size_t)start + 2, 0.0L);
    long double fp1 = 0.0L, fk = 1.0L;          // f_{k+1}, f_k at k = start
    long double neumann = 0.0L;
    f[start] = fk;
    for (int k = start; k >= 1; --k) {
        long double fm1 = (2.0L * k / x) * fk - fp1;
        fp1 = fk;
        fk = fm1;
        f[k - 1] = fk;
        if (std::fabs(fk) > 1e2000L) {          // keep the un-normalised sequence in range
            const long double sc = 1e-2000L;
            for (int m = k - 1; m <= start; ++m) f[m] *= sc;
            fk *= sc;
            fp1 *= sc;
        }
    }
    neumann = f[0];
    for (int k = 2; k <= start; k += 2) neumann += 2.0L * f[k];
    std::vector<long double> J((size_t)kmax + 1);
    for (int k = 0; k <= kmax; ++k) J[k] = f[k] / neumann;
    return J;
}

}  // namespace

extern "C" int tbpm_cheb_coeff(double tau, double tol, int kcap, int *K, double *coeff)
{
    if (!K || !coeff || kcap < 1 || !(tau >= 0.0) || !std::isfinite(tau) || !(tol > 0.0)) return TBPM_EINVAL;
    if (tau == 0.0) {                            // exp(0) = 1: only c_0 = J_0(0) = 1 survives
        *K = 1;
        coeff[0] = 1.0;
        coeff[1] = 0.0;
        return TBPM_OK;
    }
    const int k0 = (int)std::ceil(tau);
    const int kmax = k0 + 96 + (int)(10.0 * std::cbrt(tau));
    std::vector<long double> J = bessel_down((long double)tau, kmax);
    int Kf = -1;
    for (int k = k0; k <= kmax; ++k) {           // the k >= ceil(tau) guard avoids stopping at an early zero crossing
        if (std::fabs((double)J[k]) < tol) { Kf = k; break; }
    }
    if (Kf < 1) return TBPM_EINVAL;
    *K = Kf;
    if (Kf > kcap) return TBPM_ENOMEM;
    for (int k = 0; k < Kf; ++k) {
        const double m = (double)((k == 0 ? 1.0L : 2.0L) * J[k]);
        double re = 0.0, im = 0.0;               // (-i)^k cycles 1, -i, -1, +i
        switch (k % 4) {
        case 0: re = m; break;
        case 1: im = -m; break;
        case 2: re = -m; break;
        case 3: im = m; break;
        }
        coeff[2 * k] = re;
        coeff[2 * k + 1] = im;
    }
    return TBPM_OK;
}

// NEXT-4: Chebyshev coefficients of the Fermi operator f(E) = 1 / (exp(beta (E - mu)) + 1) on [-s, s] (or of 1 - f):
//     c_k = (2 - delta_k0) / pi * integral_0^pi f(s cos t) cos(k t) dt,
// evaluated by the midpoint rule on M = 16384 points (exact for the truncated series: Gauss-Chebyshev), k ascending until 64
// consecutive coefficients are below tol; the coefficients after the last one >= tol are dropped.  Real coefficients, written as
// (re, 0) pairs so that the series goes through the same fused kernels as the time step.  DESIGN.md reading #30.
extern "C" int tbpm_fermi_coeff(double beta, double mu, double rescale, int one_minus, double tol, int kcap, int *K, double *coeff)
{
    if (!K || !coeff || kcap < 1 || !(beta >= 0.0) || !std::isfinite(beta) || !std::isfinite(mu) || !(rescale > 0.0) || !(tol > 0.0)) return TBPM_EINVAL;
    constexpr int M = 16384;
    const double pi = 3.14159265358979323846;
    std::vector<double> f(M), th(M);
    for (int m = 0; m < M; ++m) {
        th[m] = pi * (m + 0.5) / M;
        const double x = beta * (rescale * std::cos(th[m]) - mu);
        const double e = std::exp(-std::fabs(x));
        f[m] = x > 0.0 ? e / (1.0 + e) : 1.0 / (1.0 + e);
    }
    std::vector<double> c;
    int last_big = 0, quiet = 0;
    for (int k = 0; k < M / 4 && quiet < 64; ++k) {
        long double acc = 0.0L;
        for (int m = 0; m < M; ++m) acc += (long double)f[m] * (long double)std::cos(k * th[m]);
        const double ck = (double)((k == 0 ? 1.0L : 2.0L) * acc / M);
        c.push_back(ck);
        if (std::fabs(ck) >= tol) { last_big = k; quiet = 0; } else ++quiet;
    }
    const int Kf = last_big + 1;
    *K = Kf;
    if (Kf > kcap) return TBPM_ENOMEM;
    for (int k = 0; k < Kf; ++k) {
        coeff[2 * k] = one_minus ? (k == 0 ? 1.0 - c[k] : -c[k]) : c[k];
        coeff[2 * k + 1] = 0.0;
    }
    return TBPM_OK;
}
