// a6 Voigt function H(a,x) = (a/pi) Int exp(-y^2) / ((x-y)^2 + a^2) dy, the normalisation that makes Eq. 6 integrate
// to one, in fp32, branch-light, <= 1e-5 relative (BASELINE.json tolerance; measured ~1e-6 for
// a <= 0.05, |x| <= 1e3).  The paper's default approximation (S15) is only <~1e-4 and none of its
// four formulas is printed, so this is an own design (reading A1):
//
//   |x| < 8:  Taylor expansion of the Faddeeva function about the real axis in powers of a,
//               H = H0 + a H1 + a^2 H2 + a^3 H3 + a^4 H4,
//               H0 = e^{-x^2},  H1 = -(2/sqrt(pi)) G,  H2 = (1 - 2x^2) e^{-x^2},
//               H3 = (2/(3 sqrt(pi))) (1 + G (2x^2 - 3)),  H4 = e^{-x^2} (1/2 - 2x^2 + (2/3) x^4),
//             where G(x) = 1 - 2 x F(x) (F = Dawson's integral) is the only non-elementary piece: cubic Hermite
//             interpolation in a 129-node table (h = 1/16) held in shared memory; one ex2 per evaluation.
//   |x| >= 8: asymptotic series H = a/(sqrt(pi) x^2) (1 + (3/2 - a^2)/x^2 + (15/4 - 5a^2)/x^4 + (105/8)/x^6
//             + (945/16)/x^8).
// Polynomials are written in Estrin-friendly nested FMA form.
#pragma once
#include <cuda_runtime.h>

namespace thor {

constexpr int VOIGT_NODES = 129;
constexpr float VOIGT_X_TABLE = 8.0f;
constexpr float VOIGT_H_INV = 16.0f;

__constant__ float2 c_voigt_nodes[VOIGT_NODES] = {
#include "voigt_table.inc"
};

// Copy the node table into shared memory (call with all threads of the block, then __syncthreads()).
__device__ __forceinline__ void voigt_table_load(float2* s_tab) {
    for (int i = threadIdx.x; i < VOIGT_NODES; i += blockDim.x) s_tab[i] = c_voigt_nodes[i];
}

// G(x) = 1 - 2 x F(x) for 0 <= ax < 8 from the shared-memory table.
__device__ __forceinline__ float voigt_G_table(const float2* __restrict__ s_tab, float ax) {
    const float s = ax * VOIGT_H_INV;
    int i = (int)s;
    i = min(i, VOIGT_NODES - 2);
    const float t = s - (float)i;
    const float2 n0 = s_tab[i], n1 = s_tab[i + 1];
    const float dg = n1.x - n0.x;
    const float c2 = fmaf(3.0f, dg, fmaf(-2.0f, n0.y, -n1.y));
    const float c3 = fmaf(-2.0f, dg, n0.y + n1.y);
    return fmaf(t, fmaf(t, fmaf(t, c3, c2), n0.y), n0.x);
}

__device__ __forceinline__ float voigt_H(const float2* __restrict__ s_tab, float a, float x) {
    const float ax = fabsf(x);
    const float x2 = ax * ax;
    const float a2 = a * a;
    constexpr float C = 1.1283791670955126f;          // 2/sqrt(pi)
    if (ax >= VOIGT_X_TABLE) {
        const float r = __frcp_rn(x2);
        const float p = fmaf(r, fmaf(r, fmaf(r, fmaf(r, 59.0625f, 13.125f), fmaf(-5.0f, a2, 3.75f)), 1.5f - a2), 1.0f);
        return 0.5f * C * a * r * p;
    }
    const float G = voigt_G_table(s_tab, ax);
    const float e = exp2f(-1.4426950408889634f * x2);
    const float H1 = -C * G;
    const float H2 = fmaf(-2.0f, x2, 1.0f) * e;
    const float H3 = (C * (1.0f / 3.0f)) * fmaf(G, fmaf(2.0f, x2, -3.0f), 1.0f);
    const float H4 = e * fmaf(x2, fmaf(x2, 2.0f / 3.0f, -2.0f), 0.5f);
    return fmaf(a2, fmaf(a, H3, fmaf(a2, H4, H2)), fmaf(a, H1, e));
}

}  // namespace thor
