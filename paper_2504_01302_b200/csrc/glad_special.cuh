// fp64 special functions shared by the fp64 prep kernels of libglad (lens_prep_kernel, mge1d_kernel).
#pragma once
#include <math.h>

// ------------------------------------------------------------------------------------------------
// regularised incomplete gamma and the Sersic b_n root
// ------------------------------------------------------------------------------------------------
// Regularised lower incomplete gamma P(a,x) (series / Lentz continued fraction).
__device__ static double gamma_p(double a, double x) {
    if (x <= 0.0) return 0.0;
    double lg = lgamma(a);
    if (x < a + 1.0) {
        double ap = a, del = 1.0 / a, sum = del;
        for (int n = 0; n < 2000; ++n) {
            ap += 1.0;
            del *= x / ap;
            sum += del;
            if (fabs(del) < fabs(sum) * 1e-16) break;
        }
        return sum * exp(-x + a * log(x) - lg);
    }
    const double FPMIN = 1e-290;
    double b = x + 1.0 - a, c = 1.0 / FPMIN, d = 1.0 / b, h = d;
    for (int i = 1; i < 2000; ++i) {
        double an = -(double)i * ((double)i - a);
        b += 2.0;
        d = an * d + b;
        if (fabs(d) < FPMIN) d = FPMIN;
        c = b + an / c;
        if (fabs(c) < FPMIN) c = FPMIN;
        d = 1.0 / d;
        double del = d * c;
        h *= del;
        if (fabs(del - 1.0) < 1e-15) break;
    }
    return 1.0 - exp(-x + a * log(x) - lg) * h;
}

// Sersic b_n: root of P(2n, b) = 1/2 by safeguarded Newton (reading R-L7), started from the asymptotic
// expansion b ~ 2n - 1/3 + 4/(405 n) + 46/(25515 n^2) + 131/(1148175 n^3) - 2194697/(30690717750 n^4)
// (Ciotti & Bertin 1999) so that two steps reach fp64 round-off.
// The series of gamma_p without its prefactor, sum_k x^k / (a (a+1) .. (a+k)), x < a + 1: the same terms in the same order, but the
// quotients x / (a + k) of eight terms are formed before the dependent chain of products (the chain of fp64 divisions was most
// of lens_prep_kernel's 148 us on C2).
__device__ static double gamma_series_sum(double a, double x) {
    double ap = a, del = 1.0 / a, sum = del;
    for (int n = 0; n < 2000; n += 8) {
        double r[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) r[i] = x / (ap + (double)(i + 1));
        bool done = false;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (!done) {
                del *= r[i];
                sum += del;
                done = fabs(del) < fabs(sum) * 1e-16;
            }
        }
        if (done) break;
        ap += 8.0;
    }
    return sum;
}

__device__ static double sersic_bn(double n) {
    double a = 2.0 * n;
    double lo = 0.0, hi = a + 25.0;
    const double rn = 1.0 / n;
    double b = a - 1.0 / 3.0 + rn * (4.0 / 405.0 + rn * (46.0 / 25515.0 + rn * (131.0 / 1148175.0 - rn * (2194697.0 / 30690717750.0))));
    if (!(b > 0.0 && b < hi) || n < 0.36) b = (a > 1.0 / 3.0) ? a - 1.0 / 3.0 : 0.5 * a;
    double lg = lgamma(a);
    for (int it = 0; it < 60; ++it) {
        const double pref = exp(-b + a * log(b) - lg);               // x^a e^-x / Gamma(a): P = pref * series, dP/dx = pref / x
        double f = (b < a + 1.0 ? pref * gamma_series_sum(a, b) : gamma_p(a, b)) - 0.5;
        if (f > 0.0) hi = b; else lo = b;
        double fp = pref / b;
        double nb = b - f / fp;
        if (!(nb > lo && nb < hi)) nb = 0.5 * (lo + hi);
        if (fabs(nb - b) < 1e-10 * b) { b = nb; break; }      // Newton is quadratic: nb is then at round-off
        b = nb;
    }
    return b;
}

