// ORACLE — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded fp64 CPU statement of the method of
// arXiv 2507.11603 (THOR).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may build, load or run anything in this directory.  It shares no code with the CUDA path.
//
// Lyα atomic constants (CGS).  The paper prints none of them except t ~ 1/A ~ 1 ns; they are the
// textbook values listed in SURVEY.md §8(c) "Constants".  Definitions of x, u and v_th: PAPER.md:107 (§2.3.1).
#pragma once
#include <cmath>

namespace orc {

constexpr double PI = 3.14159265358979323846;
constexpr double SQRT_PI = 1.77245385090551602730;

constexpr double K_BOLTZ = 1.380649e-16;       // erg / K
constexpr double M_HYDROGEN = 1.6735575e-24;   // g, mass of the hydrogen atom (the scattering atom)
constexpr double C_LIGHT = 2.99792458e10;      // cm / s
constexpr double E_CHARGE = 4.80320471e-10;    // esu
constexpr double M_ELECTRON = 9.1093837e-28;   // g
constexpr double LAMBDA0 = 1215.67e-8;         // cm, Lyα line centre
constexpr double F12 = 0.4162;                 // oscillator strength
constexpr double A21 = 6.265e8;                // 1/s, Einstein A

// v_th = sqrt(2 k_B T / m), returned in km/s.
inline double vth_kms(double T) { return std::sqrt(2.0 * K_BOLTZ * T / M_HYDROGEN) * 1e-5; }

// Doppler width in Hz.
inline double dnu_doppler(double T) { return vth_kms(T) * 1e5 / LAMBDA0; }

// Voigt parameter a = A21 / (4 pi dnu_D).
inline double voigt_a(double T) { return A21 / (4.0 * PI * dnu_doppler(T)); }

// Line-centre cross-section sigma_0 in cm^2, so that sigma(x) = sigma_0 H(a, x) with H normalised as in Eq. 6
// (PAPER.md:116): H(a,x) = (a/pi) Int exp(-y^2) / ((x-y)^2 + a^2) dy.
inline double sigma0_cm2(double T) {
    return F12 * SQRT_PI * E_CHARGE * E_CHARGE / (M_ELECTRON * C_LIGHT * dnu_doppler(T));
}

}  // namespace orc
