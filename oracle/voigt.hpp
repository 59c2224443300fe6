// ORACLE — TEST INFRASTRUCTURE ONLY (see constants.hpp).
//
// Voigt function H(a,x) = (a/pi) Int_{-inf}^{inf} exp(-y^2) / ((x-y)^2 + a^2) dy = Re w(x + i a), with w the
// Faddeeva function.  This is the normalisation that makes Eq. 6 integrate to one.  The paper uses
// fast approximations (S15 by default, A.3) and takes the MIT Faddeeva package as the truth
// (PAPER.md:1098); reading A1: the oracle evaluates the exact function to <= 1e-10 relative in fp64, and is
// pinned in tests against scipy.special.wofz, H(a,0) = exp(a^2) erfc(a), Int H dx = sqrt(pi), the wing limit and a
// direct quadrature of the defining integral.
//
// Method (textbook identities, restated):
//   |x| <  X_SWITCH: Taylor expansion of w about the real axis, w(x+ia) = Sum_n (ia)^n w^(n)(x) / n!, with
//                    w(x) = exp(-x^2) + (2i/sqrt(pi)) F(x)  (F = Dawson's integral) and the derivative recurrence
//                    w' = -2 z w + 2i/sqrt(pi),  w^(n+1) = -2 z w^(n) - 2 n w^(n-1).
//   |x| >= X_SWITCH: the asymptotic series w(z) ~ (i / (sqrt(pi) z)) Sum_k (2k-1)!! / (2 z^2)^k, in complex
//                    arithmetic, summed until the terms stop decreasing or fall below 1e-17.
// Dawson's integral: Rybicki's sampling formula F(x) = lim (1/sqrt(pi)) Sum_{n odd} exp(-(x-nh)^2)/n
// (Rybicki 1989), h = 0.25 (error ~ exp(-(pi/2h)^2) ~ 1e-17), Maclaurin series for |x| < 0.2.
// Valid for 0 <= a <= ~0.05 (Lyα above 1 K has a <= 0.047).
#pragma once
#include <cmath>
#include <complex>
#include "constants.hpp"

namespace orc {

inline double dawson(double x) {
    const double ax = std::fabs(x);
    if (ax < 0.2) {
        // F(x) = x (1 - 2/3 x^2 + 4/15 x^4 - 8/105 x^6 + 16/945 x^8 - 32/10395 x^10 + ...)
        const double x2 = x * x;
        double term = 1.0, sum = 1.0;
        for (int n = 1; n < 12; ++n) { term *= -2.0 * x2 / (2.0 * n + 1.0); sum += term; }
        return x * sum;
    }
    const double h = 0.25;
    const int NT = 14;                       // ((2*13+1) h)^2 = 45.6
    static double ctab[NT];                  // exp(-((2i+1)h)^2), filled on first use
    static bool have_tab = false;
    if (!have_tab) {
        for (int i = 0; i < NT; ++i) ctab[i] = std::exp(-((2.0 * i + 1.0) * h) * ((2.0 * i + 1.0) * h));
        have_tab = true;
    }
    const int n0 = 2 * (int)std::lround(0.5 * ax / h);
    const double xp = ax - n0 * h;
    double e1 = std::exp(2.0 * xp * h);
    const double e2 = e1 * e1;
    double d1 = n0 + 1.0, d2 = d1 - 2.0, sum = 0.0;
    for (int i = 0; i < NT; ++i) {
        sum += ctab[i] * (e1 / d1 + 1.0 / (d2 * e1));
        d1 += 2.0; d2 -= 2.0; e1 *= e2;
    }
    const double r = std::exp(-xp * xp) * sum / SQRT_PI;
    return x < 0 ? -r : r;
}

inline double voigt_H(double a, double x) {
    const double X_SWITCH = 8.0;
    const double ax = std::fabs(x);
    if (ax >= X_SWITCH) {
        const std::complex<double> z(ax, a);
        const std::complex<double> iz2 = 1.0 / (2.0 * z * z);
        std::complex<double> term(1.0, 0.0), sum(1.0, 0.0);
        double prev = 1.0;
        for (int k = 1; k < 60; ++k) {
            term *= (2.0 * k - 1.0) * iz2;
            const double mag = std::abs(term);
            if (mag > prev) break;           // asymptotic series: stop at the smallest term
            sum += term;
            prev = mag;
            if (mag < 1e-17) break;
        }
        const std::complex<double> w = std::complex<double>(0.0, 1.0 / SQRT_PI) / z * sum;
        return w.real();
    }
    // Taylor about the real axis.  d_n = w^(n)(x)/n!:  d_1 = -2x d_0 + 2i/sqrt(pi),
    // d_{n+1} = (-2x d_n - 2 d_{n-1}) / (n+1).  Real coefficients: real and imaginary parts decouple.
    double re_prev = std::exp(-ax * ax);
    double im_prev = 2.0 / SQRT_PI * dawson(ax);
    double re_cur = -2.0 * ax * re_prev;
    double im_cur = -2.0 * ax * im_prev + 2.0 / SQRT_PI;
    // (ia)^n: n=0 -> 1, n=1 -> i a, n=2 -> -a^2, n=3 -> -i a^3, ...; Re[(ia)^n d_n] alternates re / -im parts.
    double H = re_prev;                      // n = 0
    double an = a;                           // a^n
    H += -an * im_cur;                       // n = 1: Re[i a (re + i im)] = -a im
    for (int n = 1; n < 40; ++n) {
        const double re_next = (-2.0 * ax * re_cur - 2.0 * re_prev) / (n + 1.0);
        const double im_next = (-2.0 * ax * im_cur - 2.0 * im_prev) / (n + 1.0);
        re_prev = re_cur; im_prev = im_cur; re_cur = re_next; im_cur = im_next;
        an *= a;
        const int m = n + 1;                 // order of the term being added
        double contrib;
        switch (m & 3) {
            case 0: contrib = an * re_cur; break;    // (ia)^m = a^m
            case 1: contrib = -an * im_cur; break;   // i a^m
            case 2: contrib = -an * re_cur; break;   // -a^m
            default: contrib = an * im_cur; break;   // -i a^m
        }
        H += contrib;
        if (std::fabs(an) * (std::fabs(re_cur) + std::fabs(im_cur)) < 1e-18 * std::fabs(H)) break;
    }
    return H;
}

// Core-to-wing transition x_cw(a): root of exp(-x^2) = a / (sqrt(pi) x^2) (A.2), by bisection.
inline double x_cw_exact(double a) {
    double lo = 1.0, hi = 8.0;               // f(x) = exp(-x^2) sqrt(pi) x^2 - a: >0 at 1, <0 at 8 for a in (1e-12, 0.6)
    for (int it = 0; it < 80; ++it) {
        const double mid = 0.5 * (lo + hi);
        const double f = std::exp(-mid * mid) * SQRT_PI * mid * mid - a;
        if (f > 0) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

// The paper's "B25" approximation: 4th-order polynomial in ln a (coefficients printed at PAPER.md:1078).
inline double x_cw_b25(double a) {
    const double c0 = 1.03489162, c1 = -6.17680644e-1, c2 = -8.73073343e-2, c3 = -7.91384757e-3, c4 = -2.76037084e-4;
    const double L = std::log(a);
    return c0 + L * (c1 + L * (c2 + L * (c3 + L * c4)));
}

}  // namespace orc
