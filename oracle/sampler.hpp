// ORACLE — TEST INFRASTRUCTURE ONLY (see constants.hpp).
//
// Random variates of the scattering event (§2.3.1, §3.4):
//   u_par  : Eq. 6 by rejection with the piecewise comparison function of Eq. 10
//            (Zheng & Miralda-Escude 2002).
//   u_perp : Eq. 5, f ∝ exp(-u^2) per component, i.e. variance 1/2 (reading A5), with the
//            left-truncated magnitude for core-skipping (reading A7).
//   mu     : isotropic or dipole phase function.
// Each function takes its uniforms from a DrawStream, one draw per uniform, in the order written here.
#pragma once
#include <cmath>
#include "constants.hpp"
#include "philox.hpp"
#include "voigt.hpp"

namespace orc {

// u0(a, x) for Eq. 10, x >= 0.  The paper uses the rule of Seon & Kim (2020), which it does not print
// (PAPER.md:232); reading A2: Eq. 6 is sampled exactly for ANY u0, so the oracle takes a simple rule of its own:
// minimise the envelope mass  M(u0) = 1/(x-u0) + (pi/a) exp(-u0^2)  approximately.
//   core:  delta = sqrt(a exp(x^2) / (2 pi x))  (stationary point of M for delta << x), capped at 0.45;
//   wing:  u0 <= u_w = sqrt(ln(pi/a)) + 0.4     (keeps the peak piece's envelope mass below the tail piece's).
// u0 < x always, which keeps the acceptance away from the H(a,x) ~ 1e-5 collapse.
inline double upar_u0(double a, double x) {
    if (x <= 0.0) return 0.0;
    double delta = std::sqrt(a * std::exp(std::fmin(x * x, 50.0)) / (2.0 * PI * x));
    if (delta > 0.45) delta = 0.45;
    if (delta > x) delta = x;
    const double u_w = std::sqrt(std::log(PI / a)) + 0.4;
    return std::fmin(x - delta, u_w);
}

// Eq. 10 rejection loop (Zheng & Miralda-Escude 2002), x >= 0 handled by symmetry f(u; -x) = f(-u; x).
//   g1 = 1/(a^2 + (x-u)^2) on u <= u0, g2 = exp(-u0^2)/(a^2 + (x-u)^2) on u > u0.
//   theta0 = atan((u0 - x)/a);  P(piece 1) = (theta0 + pi/2) / ((1 - e^{-u0^2}) theta0 + (1 + e^{-u0^2}) pi/2).
//   piece 1: theta ~ U[-pi/2, theta0], u = a tan(theta) + x, accept with exp(-u^2);
//   piece 2: theta ~ U[theta0, pi/2],  u = a tan(theta) + x, accept with exp(-u^2) / exp(-u0^2).
// Three draws per iteration.  *iters is incremented once per iteration.
inline double upar_zm02(double a, double x, DrawStream& rng, uint64_t* iters) {
    const double sgn = x < 0 ? -1.0 : 1.0;
    const double xa = std::fabs(x);
    const double u0 = upar_u0(a, xa);
    const double e0 = std::exp(-u0 * u0);
    const double theta0 = std::atan((u0 - xa) / a);
    const double p1 = (theta0 + 0.5 * PI) / ((1.0 - e0) * theta0 + (1.0 + e0) * 0.5 * PI);
    for (;;) {
        if (iters) ++*iters;
        const double r1 = rng.uniform(), r2 = rng.uniform(), r3 = rng.uniform();
        double theta, u;
        if (r1 <= p1) {
            theta = -0.5 * PI + r2 * (theta0 + 0.5 * PI);
            u = a * std::tan(theta) + xa;
            if (r3 <= std::exp(-u * u)) return sgn * u;
        } else {
            theta = theta0 + r2 * (0.5 * PI - theta0);
            u = a * std::tan(theta) + xa;
            if (r3 <= std::exp(u0 * u0 - u * u)) return sgn * u;
        }
    }
}

// Far wing (x >= X_FAR): the paper switches to a Gaussian APPROXIMATION for x > 8.  The oracle
// stays exact (reading A2) with a second two-piece envelope, with L(u) = 1/(a^2 + (x-u)^2):
//   piece A, u <= u0: exp(-u^2) L(u0)   -> u ~ N(0, 1/2) (Box-Muller), rejected if u > u0, else accept L(u)/L(u0)
//   piece B, u >  u0: exp(-u0^2) L(u)   -> Lorentzian as in piece 2 above, accept exp(u0^2 - u^2)
//   Piece A is sampled from the untruncated Gaussian and a draw above u0 is counted as a rejection, so the
//   envelope masses are  M_A = sqrt(pi) L(u0)  and  M_B = exp(-u0^2) (pi/2 - theta0)/a.
//   u0 = min(x/2, sqrt(ln(pi x^2 / a) + 3)): M_B <= 0.05/x^2, acceptance -> ((x-u0)/x)^2.
// Four draws per iteration.
inline double upar_far(double a, double x, DrawStream& rng, uint64_t* iters) {
    const double sgn = x < 0 ? -1.0 : 1.0;
    const double xa = std::fabs(x);
    const double u0 = std::fmin(0.5 * xa, std::sqrt(std::log(PI * xa * xa / a) + 3.0));
    const double L0 = 1.0 / (a * a + (xa - u0) * (xa - u0));
    const double theta0 = std::atan((u0 - xa) / a);
    const double MA = SQRT_PI * L0;
    const double MB = std::exp(-u0 * u0) * (0.5 * PI - theta0) / a;
    const double pA = MA / (MA + MB);
    for (;;) {
        if (iters) ++*iters;
        const double r1 = rng.uniform(), r2 = rng.uniform(), r3 = rng.uniform(), r4 = rng.uniform();
        if (r1 <= pA) {
            const double u = std::sqrt(-std::log(r2)) * std::cos(2.0 * PI * r3);   // N(0, 1/2), Eq. 5 form
            if (u > u0) continue;
            const double L = 1.0 / (a * a + (xa - u) * (xa - u));
            if (r4 * L0 <= L) return sgn * u;
        } else {
            const double theta = theta0 + r2 * (0.5 * PI - theta0);
            const double u = a * std::tan(theta) + xa;
            if (r3 <= std::exp(u0 * u0 - u * u)) return sgn * u;
        }
    }
}

constexpr double UPAR_X_FAR = 8.0;

inline double sample_upar(double a, double x, DrawStream& rng, uint64_t* iters) {
    return std::fabs(x) < UPAR_X_FAR ? upar_zm02(a, x, rng, iters) : upar_far(a, x, rng, iters);
}

// Eq. 6 itself, for tests: pdf of u_par.
inline double upar_pdf(double a, double x, double u) {
    return (a / PI) * std::exp(-u * u) / ((x - u) * (x - u) + a * a) / voigt_H(a, x);
}

// Eq. 5: two perpendicular components, each ∝ exp(-u^2) (variance 1/2).  Box-Muller in polar
// form: magnitude m = sqrt(-ln r1), angle 2 pi r2.  Core-skipping: when |x_in| < x_crit the
// magnitude is drawn from the Gaussian left-truncated at x_crit:  m = sqrt(x_crit^2 - ln r1).
inline void sample_uperp(double x_in, double x_crit, DrawStream& rng, double& up1, double& up2) {
    const double r1 = rng.uniform(), r2 = rng.uniform();
    const double shift = (std::fabs(x_in) < x_crit) ? x_crit * x_crit : 0.0;
    const double m = std::sqrt(shift - std::log(r1));
    up1 = m * std::cos(2.0 * PI * r2);
    up2 = m * std::sin(2.0 * PI * r2);
}

enum Phase { PHASE_ISOTROPIC = 0, PHASE_DIPOLE = 1, PHASE_MIX = 2 };

// mu = cos(scattering angle).  Isotropic: p(mu) = 1/2.  Dipole: p(mu) = 3/8 (1 + mu^2), inverted in closed form:
// the CDF (3 mu + mu^3 + 4)/8 = r gives mu^3 + 3 mu - 2B = 0 with B = 4r - 2, whose real root (Cardano) is
// mu = cbrt(B + sqrt(B^2 + 1)) + cbrt(B - sqrt(B^2 + 1)).
inline double dipole_mu(double r) {
    const double half_B = 4.0 * r - 2.0;
    const double s = std::sqrt(half_B * half_B + 1.0);
    return std::cbrt(half_B + s) + std::cbrt(half_B - s);
}

// "1-to-2 isotropic-dipole mix": with probability 1/3 isotropic, 2/3 dipole; one extra draw.
inline double sample_mu(int phase, DrawStream& rng, int* used_dipole) {
    int ph = phase;
    if (phase == PHASE_MIX) ph = (rng.uniform() < 1.0 / 3.0) ? PHASE_ISOTROPIC : PHASE_DIPOLE;
    if (used_dipole) *used_dipole = (ph == PHASE_DIPOLE);
    const double r = rng.uniform();
    return ph == PHASE_DIPOLE ? dipole_mu(r) : 2.0 * r - 1.0;
}

// Henyey-Greenstein phase function of dust scattering, Eq. 9: P_HG(mu) = (1/2)(1 - g^2)/(1 + g^2 - 2 g mu)^(3/2),
// g = <mu>.  Its CDF inverts in closed form: mu = (1 + g^2 - ((1 - g^2)/(1 - g + 2 g r))^2) / (2 g); isotropic for g = 0.
inline double hg_mu(double g, double r) {
    if (std::fabs(g) < 1e-6) return 2.0 * r - 1.0;
    const double q = (1.0 - g * g) / (1.0 - g + 2.0 * g * r);
    return (1.0 + g * g - q * q) / (2.0 * g);
}
// 2 P_HG(mu): the phase function normalised so that isotropic scattering gives 1 (the convention of phase_value below).
inline double hg_value(double g, double mu) { return (1.0 - g * g) / std::pow(1.0 + g * g - 2.0 * g * mu, 1.5); }

// Normalised phase function toward a fixed direction, for peel-off: P^(mu) = 1 or 3/4 (1 + mu^2).
inline double phase_value(int resolved_dipole, double mu) { return resolved_dipole ? 0.75 * (1.0 + mu * mu) : 1.0; }

}  // namespace orc
