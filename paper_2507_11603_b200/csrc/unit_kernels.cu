// Single steps of the path as stand-alone kernels (thor_unit_* of include/thor.h) + the field validation scan.
#include <cuda_runtime.h>
#include <curand_kernel.h>
#include <string>
#include "../../include/thor.h"
#include "philox.cuh"
#include "dda.cuh"
#include "voigt.cuh"
#include "sampler.cuh"

namespace thor {

__global__ void validate_fields_kernel(const float* nHI, const float* T, const float* vx, const float* vy,
                                       const float* vz, const float* kdust, long long n, unsigned* flags) {
    unsigned f = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float a = nHI[i], t = T[i], x = vx[i], y = vy[i], z = vz[i], k = kdust ? kdust[i] : 0.f;
        if (!isfinite(a) || !isfinite(t) || !isfinite(x) || !isfinite(y) || !isfinite(z) || !isfinite(k)) f |= 1u;
        if (a < 0.f || k < 0.f) f |= 2u;
        if (a > 0.f && !(t > 0.f)) f |= 4u;
    }
    f = __reduce_or_sync(0xffffffffu, f);
    if ((threadIdx.x & 31) == 0 && f) atomicOr(flags, f);
}

cudaError_t launch_validate_fields(const float* nHI, const float* T, const float* vx, const float* vy, const float* vz,
                                   const float* kdust, long long n, unsigned* d_flags, cudaStream_t stream) {
    long long blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    validate_fields_kernel<<<(unsigned)blocks, 256, 0, stream>>>(nHI, T, vx, vy, vz, kdust, n, d_flags);
    return cudaGetLastError();
}

__global__ void pack_fields_kernel(const float* nHI, const float* T, const float* vx, const float* vy, const float* vz,
                                   const float* kdust, long long n, float4* out) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        out[2 * i] = make_float4(nHI[i], T[i], vx[i], vy[i]);
        out[2 * i + 1] = make_float4(vz[i], kdust ? kdust[i] : 0.f, 0.f, 0.f);
    }
}

cudaError_t launch_pack_fields(const float* nHI, const float* T, const float* vx, const float* vy, const float* vz,
                               const float* kdust, long long n, float4* out, cudaStream_t stream) {
    long long blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    pack_fields_kernel<<<(unsigned)blocks, 256, 0, stream>>>(nHI, T, vx, vy, vz, kdust, n, out);
    return cudaGetLastError();
}

__global__ void unit_philox_kernel(uint64_t seed, uint64_t id0, long long n_ids, int n_draws, uint32_t* out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_ids) return;
    Stream s;
    s.init(seed, id0 + (uint64_t)i);
    for (int d = 0; d < n_draws; ++d) out[i * n_draws + d] = s.next_u32();
}

// cuRAND's Philox4x32-10 on the same (seed, subsequence = photon id, offset = 0): test-only cross-check of the layout.
__global__ void unit_curand_kernel(uint64_t seed, uint64_t id0, long long n_ids, int n_draws, uint32_t* out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_ids) return;
    curandStatePhilox4_32_10_t st;
    curand_init((unsigned long long)seed, (unsigned long long)(id0 + (uint64_t)i), 0ull, &st);
    for (int d = 0; d < n_draws; d += 4) {
        const uint4 r = curand4(&st);
        const uint32_t w[4] = {r.x, r.y, r.z, r.w};
        for (int j = 0; j < 4 && d + j < n_draws; ++j) out[i * n_draws + d + j] = w[j];
    }
}

__device__ __forceinline__ uint64_t fnv_word(uint64_t h, uint64_t w) { return (h ^ w) * 0x100000001B3ull; }

__global__ void unit_dda_kernel(GridDims g, long long n, const float* org, const float* dir, long long max_steps,
                                uint64_t* hash_idx, uint64_t* hash_len, uint32_t* count, int64_t* seq_idx,
                                float* seq_len) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Ray r;
    dda_locate(r, g, org[3 * i], org[3 * i + 1], org[3 * i + 2]);
    ray_set_direction(r, dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]);
    uint64_t hi = 0xCBF29CE484222325ull, hl = 0xCBF29CE484222325ull;
    uint32_t cnt = 0;
    for (long long s = 0; s < max_steps; ++s) {
        float len;
        const int ex = dda_next_face(r, g, len);
        const int64_t lin = dda_linear(r, g);
        hi = fnv_word(hi, (uint64_t)lin);
        hl = fnv_word(hl, (uint64_t)__float_as_uint(len));
        if (seq_idx) seq_idx[cnt] = lin;
        if (seq_len) seq_len[cnt] = len;
        ++cnt;
        if (!dda_cross(r, g, ex, len)) break;
    }
    hash_idx[i] = hi; hash_len[i] = hl; count[i] = cnt;
}

__global__ void unit_voigt_kernel(long long n, const float* a, const float* x, float* out) {
    __shared__ float2 s_tab[VOIGT_NODES];
    voigt_table_load(s_tab);
    __syncthreads();
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        out[i] = voigt_H(s_tab, a[i], x[i]);
}

__global__ void unit_scatter_kernel(float a, float x_in, float x_crit, int phase, uint64_t seed, uint64_t id0,
                                    long long n, float* u_par, float* x_out, float* k_out, uint32_t* iters) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    BlockRng rng;
    rng.init(id0 + (uint64_t)i);
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    uint32_t it = 0;
    const float4 s1 = rng.next4(k0, k1), s2 = rng.next4(k0, k1);        // same draw layout as walk_kernel
    const float upar = sample_upar(a, x_in, rng, k0, k1, it);
    float up1, up2;
    sample_uperp(x_in, x_crit, s1.w, s2.x, up1, up2);
    bool dip;
    const float mu = sample_mu<false>(phase, s2.z, s1.y, 0.f, dip);
    float sph, cph;
    sincos_uniform(s1.z, sph, cph);
    float e1[3], e2[3];
    ortho_basis(0.f, 0.f, 1.f, e1, e2);
    const float st = sqrtf(fmaxf(0.f, fmaf(-mu, mu, 1.f)));
    if (u_par) u_par[i] = upar;
    if (x_out) x_out[i] = fmaf(st, fmaf(up1, cph, up2 * sph), fmaf(upar, mu, x_in - upar));
    if (k_out) {
        k_out[3 * i + 0] = st * fmaf(cph, e1[0], sph * e2[0]);
        k_out[3 * i + 1] = st * fmaf(cph, e1[1], sph * e2[1]);
        k_out[3 * i + 2] = fmaf(st, fmaf(cph, e1[2], sph * e2[2]), mu);
    }
    if (iters) iters[i] = it;
}

}  // namespace thor

static thread_local std::string g_unit_err;
static thor_status unit_done(cudaStream_t st, const char* what) {
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        g_unit_err = std::string(what) + ": " + cudaGetErrorString(e);
        return e == cudaErrorNoDevice || e == cudaErrorInsufficientDriver ? THOR_ERR_UNSUPPORTED : THOR_ERR_CUDA;
    }
    return THOR_OK;
}

extern "C" thor_status thor_unit_philox(uint64_t seed, uint64_t id0, long long n_ids, int n_draws, uint32_t* out,
                                        void* stream) {
    if (n_ids <= 0 || n_draws <= 0 || !out) return THOR_ERR_ARG;
    thor::unit_philox_kernel<<<(unsigned)((n_ids + 127) / 128), 128, 0, (cudaStream_t)stream>>>(seed, id0, n_ids, n_draws, out);
    return unit_done((cudaStream_t)stream, "thor_unit_philox");
}

extern "C" thor_status thor_unit_curand_philox(uint64_t seed, uint64_t id0, long long n_ids, int n_draws, uint32_t* out,
                                               void* stream) {
    if (n_ids <= 0 || n_draws <= 0 || !out) return THOR_ERR_ARG;
    thor::unit_curand_kernel<<<(unsigned)((n_ids + 127) / 128), 128, 0, (cudaStream_t)stream>>>(seed, id0, n_ids, n_draws, out);
    return unit_done((cudaStream_t)stream, "thor_unit_curand_philox");
}

extern "C" thor_status thor_unit_dda_trace(int nx, int ny, int nz, unsigned periodic_flags, long long n,
                                           const float* org, const float* dir, long long max_steps, uint64_t* hash_idx,
                                           uint64_t* hash_len, uint32_t* count, int64_t* seq_idx, float* seq_len,
                                           void* stream) {
    if (nx <= 0 || ny <= 0 || nz <= 0 || n <= 0 || !org || !dir || max_steps <= 0 || !hash_idx || !hash_len || !count)
        return THOR_ERR_ARG;
    if ((seq_idx || seq_len) && n != 1) return THOR_ERR_ARG;
    thor::GridDims g;
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.periodic = ((periodic_flags & THOR_PERIODIC_X) ? 1u : 0u) | ((periodic_flags & THOR_PERIODIC_Y) ? 2u : 0u) |
                 ((periodic_flags & THOR_PERIODIC_Z) ? 4u : 0u);
    g.frozen = ((g.periodic & 1u) && nx == 1 ? 1u : 0u) | ((g.periodic & 2u) && ny == 1 ? 2u : 0u) |
               ((g.periodic & 4u) && nz == 1 ? 4u : 0u);
    thor::unit_dda_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(g, n, org, dir, max_steps, hash_idx,
                                                                                      hash_len, count, seq_idx, seq_len);
    return unit_done((cudaStream_t)stream, "thor_unit_dda_trace");
}

extern "C" thor_status thor_unit_voigt(long long n, const float* a, const float* x, float* out, void* stream) {
    if (n <= 0 || !a || !x || !out) return THOR_ERR_ARG;
    long long blocks = (n + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    thor::unit_voigt_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(n, a, x, out);
    return unit_done((cudaStream_t)stream, "thor_unit_voigt");
}

extern "C" thor_status thor_unit_scatter(float a, float x_in, float x_crit, int phase, uint64_t seed, uint64_t id0,
                                         long long n, float* u_par, float* x_out, float* k_out, uint32_t* iters,
                                         void* stream) {
    if (n <= 0 || !(a > 0.f) || phase < 0 || phase > 2) return THOR_ERR_ARG;
    thor::unit_scatter_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(a, x_in, x_crit, phase, seed, id0, n,
                                                                                          u_par, x_out, k_out, iters);
    return unit_done((cudaStream_t)stream, "thor_unit_scatter");
}
