// a8-a10: random variates of one scattering event (§2.3.1, §3.4).
//   u_par  : Eq. 6, f(u) ∝ e^{-u^2} / ((x-u)^2 + a^2), by rejection.
//   u_perp : Eq. 5, each component ∝ e^{-u^2} (variance 1/2, reading A5), with the
//            left-truncated magnitude of core-skipping (reading A7).
//   mu     : isotropic or dipole phase function.
//
// u_par envelope (own design).  Eq. 10 splits the u axis once, at u0, and
// bounds e^{-u^2} by a constant on each side; Eq. 6 is sampled exactly for any split (reading A2).  Here the axis
// is split up to twice, 0 <= u1 <= u0 < x (x >= 0 by the symmetry f(u;-x) = f(-u;x)), with w = x - u:
//   A  u <= u1      bound e^{-u^2} L(u1),       L(u) = 1/((x-u)^2 + a^2);  propose u ~ N(0,1/2), a draw above u1 is a
//                   rejection; accept with L(u)/L(u1).                     mass sqrt(pi) L(u1)
//   B  u1 < u <= u0 bound e^{-u1^2} / w^2;  propose 1/w uniform in (1/w1, 1/w0); accept with
//                   e^{u1^2 - u^2} w^2/(w^2 + a^2).                        mass e^{-u1^2} (1/w0 - 1/w1)
//   C  u > u0       bound e^{-u0^2} L(u);   propose psi = atan2(a, w) uniform in (psi0, pi), u = x - a cot(psi);
//                   accept with e^{u0^2 - u^2}.                            mass e^{-u0^2} (pi - psi0)/a
// Piece A (the Gaussian bulk of non-resonant atoms) exists for x >= 1.5; below that B runs from u = -inf with
// u1^2 := 0 (that is Eq. 10's left piece with a 1/w^2 proposal); for x < 0.3 only C is left (plain Lorentzian,
// acceptance H(a,x) >= 0.9, and no envelope to set up in the line centre where most scatterings happen).
// B is written in w, not in the angle, because atan((u-x)/a) + pi/2 cancels catastrophically in fp32 when w >> a.
// Split rules (any value is exact; these are within ~10 % of the acceptance optimum, 0.2 worst case near x_cw,
// -> 0.9 in the far wing where Eq. 10 alone falls below 0.1):
//   u1 = min(1.9 + 0.03 x, x - 0.45),  delta0 = sqrt(a e^{x^2 - u1^2} / (2 pi x)),  delta = delta0/(1 + x delta0),
//   u0 = min(x - delta, sqrt(ln(pi x^2 / a) + 2)).
// Piece A's bound is exponentially tilted (see upar_envelope): the proposal is N(beta, 1/2), not N(0, 1/2).
#pragma once
#include "philox.cuh"

namespace thor {

constexpr float PI_F = 3.14159265358979323846f;
constexpr float SQRT_PI_F = 1.77245385090551602730f;

// The envelope of one scattering, kept in registers while the packet is in its rejection trials (walk_kernel runs
// ONE trial per loop iteration for every lane that still needs one, instead of an inner loop the whole warp waits on).
struct UparEnvelope {
    float xa;                 // |x_in|
    float u1, u0sq, beta;
    float inv_w0, inv_w1;     // 1/(x-u0), 1/(x-u1) (0 when B starts at -inf)
    float psi0pi;             // atan(a / (x-u0)) / pi
    float mA, mAB, mTot;      // cumulative masses
};

#ifndef THOR_UPAR_X_LORENTZ
#define THOR_UPAR_X_LORENTZ 0.7f
#endif
constexpr float UPAR_X_LORENTZ = THOR_UPAR_X_LORENTZ;   // below this a plain Lorentzian proposal accepts with H(a,x) >= e^{-x^2}
constexpr float UPAR_U_MIN = -4.5f;       // left end of piece A (see below)
constexpr float TWO_PI_F = 6.28318530717958647692f;
constexpr float LN2_F = 0.693147180559945309f;

// All arithmetic of the path is written with explicit fmaf / rounded operations and the library is compiled with
// -fmad=false: a value never depends on how the compiler happened to contract the expression around it, so every code
// variant that walks a packet (staged loop, cooperative drain, unit kernels) produces the same bits.

__device__ __forceinline__ float dot3(float ax, float ay, float az, float bx, float by, float bz) {
    return fmaf(az, bz, fmaf(ay, by, ax * bx));
}

// -ln r for a uniform r in (0,1): one MUFU.LG2 and one multiply.
__device__ __forceinline__ float neg_log(float r) { return __log2f(r) * -LN2_F; }

// sin / cos of the uniform random angle 2 pi r, r in (0,1): MUFU.SIN/COS on the reduced argument 2 pi (r - 1/2) in
// (-pi, pi), negated (a half-turn); absolute error ~5e-7, far below the 2^-23 grain of r.
__device__ __forceinline__ void sincos_uniform(float r, float& s, float& c) {
    const float t = TWO_PI_F * (r - 0.5f);
    s = -__sinf(t); c = -__cosf(t);
}
__device__ __forceinline__ float cos_uniform(float r) { return -__cosf(TWO_PI_F * (r - 0.5f)); }

// atan(y) for 0 <= y <= 0.5 (4.7e-8 relative): y P(y^2), minimax fit; atanf beyond (a / w0 > 0.5 needs a > 0.02).
__device__ __forceinline__ float atan_small(float y) {
    if (y > 0.5f) return atanf(y);
    const float z = y * y;
    const float pz = fmaf(z, fmaf(z, fmaf(z, fmaf(z, fmaf(z, -5.201264606e-02f, 1.019391841e-01f), -1.418004712e-01f),
                                          1.999438943e-01f), -3.333322389e-01f), 9.999999966e-01f);
    return y * pz;
}

// Piece A with an exponentially tilted bound.  On u <= u1 the Lorentzian factor L(u) = 1/((x-u)^2 + a^2) grows with
// u; Eq. 10's constant bound L(u1) wastes a factor (x/(x-u1))^2 on the bulk of the Gaussian.  ln L is convex in u,
// so with s = u1 - u, f(s) = ln(L(u1)/L(u)) is concave with f(0) = 0 and f(s) >= s f(s_max)/s_max on [0, s_max]:
//     L(u) <= L(u1) exp(2 beta (u - u1)),   beta = f(s_max) / (2 s_max),   u in [UPAR_U_MIN, u1],  s_max = u1 - UPAR_U_MIN.
// e^{-u^2} e^{2 beta u} is a Gaussian of mean beta: propose u ~ N(beta, 1/2), reject outside [UPAR_U_MIN, u1], accept
// with L(u) / (L(u1) e^{2 beta (u - u1)}).  Mass sqrt(pi) L(u1) e^{beta^2 - 2 beta u1}.  Acceptance in the wings rises
// from 0.25-0.55 to 0.5-0.8 (x = 4 ... 8).  The Gaussian mass left of UPAR_U_MIN is < 1e-9 of the piece: below the
// 2^-23 grain of the uniform that picks the piece, so no separate piece can ever be selected for it.
__device__ __forceinline__ UparEnvelope upar_envelope(float a, float xa) {
    UparEnvelope e;
    e.xa = xa;
    if (xa < UPAR_X_LORENTZ) {              // C only, u0 = 0: no set-up cost in the line centre
        e.u1 = 0.f; e.u0sq = 0.f; e.beta = 0.f; e.inv_w0 = 0.f; e.inv_w1 = 0.f;
        e.psi0pi = 0.f; e.mA = 0.f; e.mAB = 0.f; e.mTot = 1.f;
        return e;
    }
    const bool useA = xa >= 1.5f;
    const float a2 = a * a;
    float u1 = useA ? fminf(fmaf(0.03f, xa, 1.9f), xa - 0.45f) : 0.f;
    const float q = a * __expf(fminf(fmaf(xa, xa, -(u1 * u1)), 40.f)) / (TWO_PI_F * xa);
    const float d0 = sqrtf(q);
    const float delta = d0 / fmaf(xa, d0, 1.f);
    float u0 = xa - delta;
    if (useA) u0 = fminf(u0, sqrtf(__logf(PI_F * xa * xa / a) + 2.f));   // the cap never binds below x = 1.5
    u0 = fmaxf(u0, 0.f);
    u1 = fminf(u1, u0);
    e.u0sq = u0 * u0;
    e.u1 = u1;
    const float w0 = xa - u0, w1 = xa - u1;
    e.inv_w0 = 1.f / w0;
    e.psi0pi = atan_small(a * e.inv_w0) * (1.f / PI_F);
    const float mC = __expf(-e.u0sq) * (PI_F * (1.f - e.psi0pi)) / a;
    if (useA) {
        const float smax = u1 - UPAR_U_MIN, ws = w1 + smax;
        const float L1inv = fmaf(w1, w1, a2);
        e.inv_w1 = 1.f / w1;
        e.beta = __logf(fmaf(ws, ws, a2) / L1inv) / (2.f * smax);
        e.mA = SQRT_PI_F * __expf(e.beta * fmaf(-2.f, u1, e.beta)) / L1inv;
        e.mAB = fmaf(__expf(-(u1 * u1)), e.inv_w0 - e.inv_w1, e.mA);
    } else {
        e.inv_w1 = 0.f; e.beta = 0.f; e.mA = 0.f;
        e.mAB = e.inv_w0;
    }
    e.mTot = e.mAB + mC;
    return e;
}

// One proposal + accept test from four uniforms.  Returns true and sets u (for x >= 0) on acceptance.  PRE: (sC, cC) =
// sincospif(r.y) was computed ahead by a helper lane (cooperative drain); it is the angle of piece C exactly when
// psi0pi == 0, because then t = fmaf(r.y, 1, 0) = r.y.
template <bool PRE>
__device__ __forceinline__ bool upar_try(const UparEnvelope& e, float a, const float4 r, float sC, float cC, float& u) {
    const float r1 = r.x * e.mTot;
    const float a2 = a * a;
    if (r1 >= e.mAB) {                                   // C: Lorentzian peak and beyond
        float s, c;
        if (PRE && e.psi0pi == 0.f) { s = sC; c = cC; }
        else sincospif(fmaf(r.y, 1.f - e.psi0pi, e.psi0pi), &s, &c);
        const float uu = fmaf(-a, c / s, e.xa);
        u = uu;
        return r.z <= __expf(fmaf(-uu, uu, e.u0sq));
    } else if (r1 >= e.mA) {                             // B
        const float iw = fmaf(r.y, e.inv_w0 - e.inv_w1, e.inv_w1);
        const float w = 1.f / iw;
        const float uu = e.xa - w;
        const float w2 = w * w;
        u = uu;
        return r.z * (w2 + a2) <= __expf(fmaf(e.u1, e.u1, -(uu * uu))) * w2;
    } else {                                             // A: Gaussian bulk, tilted bound
        const float uu = fmaf(sqrtf(neg_log(r.y)), cos_uniform(r.z), e.beta);
        const float w = e.xa - uu, w1 = e.xa - e.u1;
        u = uu;
        return uu >= UPAR_U_MIN && uu <= e.u1 &&
               r.w * fmaf(w, w, a2) * __expf(2.f * e.beta * (uu - e.u1)) <= fmaf(w1, w1, a2);
    }
}

// Whole rejection loop for one variate (unit kernel); one counter block per trial.
__device__ __forceinline__ float sample_upar(float a, float x, BlockRng& rng, uint32_t k0, uint32_t k1,
                                             uint32_t& iters) {
    const UparEnvelope e = upar_envelope(a, fabsf(x));
    float u;
    uint32_t guard = 0;                      // fail-safe: acceptance is >= ~0.2 everywhere, 2^20 rejections cannot
    bool ok;                                 // happen unless x is NaN; never hang the GPU
    do {
        ++iters;
        ok = upar_try<false>(e, a, rng.next4(k0, k1), 0.f, 0.f, u);
    } while (!ok && ++guard < (1u << 20));
    return x < 0.f ? -u : u;
}

// Eq. 5 in polar form: magnitude m = sqrt(-ln r1) (or sqrt(x_crit^2 - ln r1) when |x_in| < x_crit),
// angle 2 pi r2; nl1 = -ln r1 and (s2, c2) = sincos(2 pi r2) arrive precomputed (neg_log, sincos_uniform).
__device__ __forceinline__ void uperp_from(float x_in, float x_crit, float nl1, float s2, float c2, float& up1, float& up2) {
    const float shift = fabsf(x_in) < x_crit ? x_crit * x_crit : 0.f;
    const float m = sqrtf(shift + nl1);
    up1 = m * c2; up2 = m * s2;
}
__device__ __forceinline__ void sample_uperp(float x_in, float x_crit, float r1, float r2, float& up1, float& up2) {
    float s, c;
    sincos_uniform(r2, s, c);
    uperp_from(x_in, x_crit, neg_log(r1), s, c, up1, up2);
}

// Dipole p(mu) = 3/8 (1 + mu^2): the CDF (mu^3 + 3 mu + 4)/8 = r gives mu^3 + 3 mu - 2B = 0, B = 4r - 2, with the
// real root mu = cbrt(B + sqrt(B^2+1)) - cbrt(sqrt(B^2+1) - B)  (Cardano).
__device__ __forceinline__ float dipole_mu(float r) {
    const float B = fmaf(4.f, r, -2.f);
    const float s = sqrtf(fmaf(B, B, 1.f));
    // cancellation-free: with p = cbrt(s + |B|), mu = sign(B) (p - 1/p)
    const float p = cbrtf(s + fabsf(B));
    const float m = p - 1.f / p;
    return B < 0.f ? -m : m;
}

// phase: 0 isotropic, 1 dipole, 2 = 1/3 isotropic + 2/3 dipole; r_mix decides the mix, r gives mu.
// PRE: mu_dip = dipole_mu(r) was computed ahead by a helper lane.
template <bool PRE>
__device__ __forceinline__ float sample_mu(int phase, float r_mix, float r, float mu_dip, bool& is_dipole) {
    int ph = phase;
    if (phase == 2) ph = r_mix < (1.f / 3.f) ? 0 : 1;
    is_dipole = ph == 1;
    const float mu = is_dipole ? (PRE ? mu_dip : dipole_mu(r)) : fmaf(2.f, r, -1.f);
    return fminf(fmaxf(mu, -1.f), 1.f);
}

// Henyey-Greenstein phase function of dust scattering, Eq. 9, by closed-form inversion of its CDF:
// mu = (1 + g^2 - ((1 - g^2) / (1 - g + 2 g r))^2) / (2 g); isotropic for g = 0.  hg_value = 2 P_HG (isotropic -> 1).
__device__ __forceinline__ float hg_mu(float g, float r) {
    if (fabsf(g) < 1e-6f) return fmaf(2.f, r, -1.f);
    const float q = fmaf(-g, g, 1.f) / fmaf(2.f * g, r, 1.f - g);
    return fminf(fmaxf(fmaf(-q, q, fmaf(g, g, 1.f)) / (2.f * g), -1.f), 1.f);
}
__device__ __forceinline__ float hg_value(float g, float mu) {
    const float d = fmaf(-2.f * g, mu, fmaf(g, g, 1.f));
    return fmaf(-g, g, 1.f) * rsqrtf(d) / d;
}

// Orthonormal basis (e1, e2) perpendicular to the unit vector k, branch-free (Duff et al. 2017 construction: with
// sg = sign(kz), a = -1/(sg + kz), b = kx ky a:  e1 = (1 + sg kx^2 a, sg b, -sg kx),  e2 = (b, sg + ky^2 a, -ky)).
// Any right-handed choice gives the same distribution of k' because the azimuth is uniform.
__device__ __forceinline__ void ortho_basis(float kx, float ky, float kz, float e1[3], float e2[3]) {
    const float sg = copysignf(1.f, kz);
    const float a = -1.f / (sg + kz);
    const float b = kx * ky * a;
    e1[0] = fmaf(sg * kx, kx * a, 1.f); e1[1] = sg * b; e1[2] = -sg * kx;
    e2[0] = b; e2[1] = fmaf(ky, ky * a, sg); e2[2] = -ky;
}

}  // namespace thor
