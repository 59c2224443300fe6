// Ray-tracing operators on the walk's DDA + gather + Voigt function (PAPER.md 3.5): projection, absorption
// spectra (Eq. 11) with periodic wrap-around and Hubble sub-sampling, volume rendering (Eq. 12), slices.
#include <cuda_runtime.h>
#include <math_constants.h>
#include "walk.cuh"

namespace thor {

// (n_HI, T) alone: 8 B of the cell's packed sector, or two SoA loads.
__device__ __forceinline__ void load_nT(const WalkParams& p, int64_t i, float& n, float& T) {
    if (p.packed) { const float2 q = __ldg(reinterpret_cast<const float2*>(p.packed + 2 * i)); n = q.x; T = q.y; }
    else { n = __ldg(p.nHI + i); T = __ldg(p.T + i); }
}

// One thread per ray.  Projection (PAPER.md 3.5.1): Q = Int q w ds with q = n_HI, w = 1 (column density, cm^-2) and q = T,
// w = n_HI (density-weighted temperature Q / Q^).  Absorption spectrum (PAPER.md 3.5.2, Eq. 11): tau(V_j) =
// Int n sigma(nu(s), T) ds with the gas seeing the sight-line frequency shifted by its line-of-sight velocity v.k and the
// Hubble term H s; piecewise-constant cells; each face-to-face segment cut into n_sub = ceil(|H len| / (eps v_th)) sub-steps
// (eps = 0: one), the Hubble term taken at each sub-step's midpoint (reading A12's rule).  WRAP: the ray
// re-enters at periodic faces and ends after max_len cell lengths; else it ends at the first box face.
template <bool WRAP>
__global__ void raytrace_kernel(const __grid_constant__ WalkParams p, long long n_rays, const float* __restrict__ org,
                                const float* __restrict__ dir, float hubble, float hubble_eps, float max_len, int n_v,
                                float v_lo, float dv, float* __restrict__ out_column, float* __restrict__ out_tmean,
                                float* __restrict__ out_tau) {
    __shared__ float2 s_tab[VOIGT_NODES];
    voigt_table_load(s_tab);
    __syncthreads();
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_rays) return;
    RayMarch r;
    const float kx = dir[3 * i], ky = dir[3 * i + 1], kz = dir[3 * i + 2];
    march_init(r, p.g, org[3 * i], org[3 * i + 1], org[3 * i + 2], kx, ky, kz);
    float col = 0.f, tn = 0.f, s_path = 0.f;
    float* tau = out_tau ? out_tau + i * n_v : nullptr;
    if (tau) for (int j = 0; j < n_v; ++j) tau[j] = 0.f;
    for (;;) {
        bool ex_x, ex_y;
        float len = march_next_face(r, ex_x, ex_y);
        if (!WRAP && !(len < CUDART_INF_F)) break;
        bool last = false;
        if (WRAP && s_path + len >= max_len) { len = max_len - s_path; last = true; }
        Cell c;
        if (tau) c = load_cell_raw(p, r.idx);
        else load_nT(p, r.idx, c.nsig, c.a);                  // projections need 8 B of the cell only
        const float n = c.nsig, T = c.a;
        col = fmaf(n, len, col);
        tn = fmaf(n * T, len, tn);
        if (tau && len > 0.f) {
            derive_cell(p, c);
            if (c.nsig > 0.f || c.kd > 0.f) {
                int nsub = 1;
                if (hubble_eps > 0.f && hubble != 0.f && c.nsig > 0.f) {
                    const float q = ceilf(fabsf(hubble * len) * c.inv_vth / hubble_eps);
                    nsub = q < 1.f ? 1 : (q > 1e6f ? 1000000 : (int)q);
                }
                const float ds = len / (float)nsub;
                const float vk = dot3(c.vx, c.vy, c.vz, kx, ky, kz);
                for (int m = 0; m < nsub; ++m) {
                    const float vgas = fmaf(hubble, fmaf((float)m + 0.5f, ds, s_path), vk);
                    for (int j = 0; j < n_v; ++j) {
                        const float V = fmaf((float)j + 0.5f, dv, v_lo);
                        const float kl = c.nsig > 0.f ? c.nsig * voigt_H(s_tab, c.a, (V - vgas) * c.inv_vth) : 0.f;
                        tau[j] = fmaf(kl + c.kd, ds, tau[j]);
                    }
                }
            }
        }
        s_path += len;
        if (last) break;
        if (WRAP ? !march_cross_wrap(r, p.g, ex_x, ex_y, len) : !march_cross(r, p.g, ex_x, ex_y, len)) break;
    }
    if (out_column) out_column[i] = col * p.cell_cm;
    if (out_tmean) out_tmean[i] = col > 0.f ? tn / col : 0.f;
}

cudaError_t launch_raytrace(const WalkParams& p, long long n_rays, const float* org, const float* dir, float hubble,
                            float hubble_eps, float max_len, int n_v, float v_lo, float dv, float* out_column,
                            float* out_tmean, float* out_tau, cudaStream_t stream) {
    const unsigned blocks = (unsigned)((n_rays + 127) / 128);
    if (max_len > 0.f)
        raytrace_kernel<true><<<blocks, 128, 0, stream>>>(p, n_rays, org, dir, hubble, hubble_eps, max_len, n_v, v_lo, dv,
                                                           out_column, out_tmean, out_tau);
    else
        raytrace_kernel<false><<<blocks, 128, 0, stream>>>(p, n_rays, org, dir, hubble, hubble_eps, max_len, n_v, v_lo, dv,
                                                            out_column, out_tmean, out_tau);
    return cudaGetLastError();
}

// Volume rendering (PAPER.md 3.5.3, Eq. 12) on the same march: front-to-back compositing with the exact integral of
// each piecewise-constant segment, C += Tr c (1 - e^{-mu l}), Tr *= e^{-mu l}.  The transfer function (Gaussian peaks
// in log10 T) arrives by value: per peak {centre in log2 T, -log2(e) / (2 s^2) in log2 units, R, G, B, A / n_ref}.
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__global__ void __launch_bounds__(128) volume_render_kernel(const __grid_constant__ WalkParams p, const __grid_constant__ TransferFn tf,
                                     long long n_rays, const float* __restrict__ org, const float* __restrict__ dir,
                                     float4* __restrict__ out_rgba) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_rays) return;
    RayMarch r;
    march_init(r, p.g, org[3 * i], org[3 * i + 1], org[3 * i + 2], dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]);
    float cr = 0.f, cg = 0.f, cb = 0.f, tr = 1.f, tau = 0.f;
    for (;;) {
        bool ex_x, ex_y;
        const float len = march_next_face(r, ex_x, ex_y);
        if (!(len < CUDART_INF_F)) break;
        float n, T;
        load_nT(p, r.idx, n, T);
        const float w = tf.weight_by_density ? n : 1.f;
        if (w > 0.f && T > 0.f) {
            const float lt = __log2f(T);
            float mu = 0.f, er = 0.f, eg = 0.f, eb = 0.f;
#pragma unroll
            for (int q = 0; q < MAX_TF_PEAKS; ++q) {
                if (q >= tf.n_peaks) break;                     // uniform: n_peaks is a kernel parameter
                const float z = lt - tf.centre[q];
                const float ag = tf.amp[q] * ex2_approx(tf.neg_inv_2s2[q] * z * z);
                mu += ag;
                er = fmaf(ag, tf.r[q], er);
                eg = fmaf(ag, tf.g[q], eg);
                eb = fmaf(ag, tf.b[q], eb);
            }
            mu *= w;
            if (mu > 0.f) {
                // 1 - e^{-y}: below y = 1e-2 the subtraction from an approximate exponential cancels (relative error
                // 1e-7 / y, zero contribution below 6e-8): the series y (1 - y/2 + y^2/6) is exact to 4e-9 there
                const float y = mu * len;
                const float em1 = y < 1e-2f ? y * fmaf(y, fmaf(y, 1.f / 6.f, -0.5f), 1.f) : 1.f - ex2_approx(-1.4426950408889634f * y);
                const float f = tr * em1 * w / mu;              // Tr (1 - e^{-mu l}) / mu, times w for the emission
                cr = fmaf(f, er, cr);
                cg = fmaf(f, eg, cg);
                cb = fmaf(f, eb, cb);
                tr = fmaf(-tr, em1, tr);                        // Tr e^{-mu l}
                tau += y;
            }
        }
        if (!march_cross(r, p.g, ex_x, ex_y, len)) break;
    }
    // opacity 1 - e^{-tau}: from the summed optical depth when thin (1 - Tr would cancel), else from the running product
    const float op = tau < 1e-2f ? tau * fmaf(tau, fmaf(tau, 1.f / 6.f, -0.5f), 1.f) : 1.f - tr;
    out_rgba[i] = make_float4(cr, cg, cb, op);
}

cudaError_t launch_volume_render(const WalkParams& p, const TransferFn& tf, long long n_rays, const float* org,
                                 const float* dir, float* out_rgba, cudaStream_t stream) {
    volume_render_kernel<<<(unsigned)((n_rays + 127) / 128), 128, 0, stream>>>(p, tf, n_rays, org, dir,
                                                                              reinterpret_cast<float4*>(out_rgba));
    return cudaGetLastError();
}

// Slice: the field value of the cell that holds each point.  field: 0 n_HI, 1 T, 2 vx, 3 vy, 4 vz, 5 kdust.
__global__ void slice_kernel(const __grid_constant__ WalkParams p, long long n, const float* __restrict__ pos, int field,
                             float* __restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Ray r;
    dda_locate(r, p.g, pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]);
    const int64_t idx = dda_linear(r, p.g);
    const Cell c = load_cell_raw(p, idx);                     // raw fields: n in nsig, T in a, kdust in kd
    out[i] = field == 0 ? c.nsig : field == 1 ? c.a : field == 2 ? c.vx : field == 3 ? c.vy : field == 4 ? c.vz : c.kd;
}

cudaError_t launch_slice(const WalkParams& p, long long n, const float* pos, int field, float* out, cudaStream_t stream) {
    slice_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(p, n, pos, field, out);
    return cudaGetLastError();
}

}  // namespace thor
