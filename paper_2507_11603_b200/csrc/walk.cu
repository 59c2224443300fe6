// Persistent-thread walk kernel + its launcher.  See walk.cuh for the step functions.
#include <cuda_runtime.h>
#include "walk.cuh"

namespace thor {

constexpr int WALK_THREADS = 256;
constexpr int MAX_SPEC_BINS = 4096;

struct BlockTallies {
    float2 voigt[VOIGT_NODES];
    unsigned long long counters[N_COUNTERS];
    unsigned int nscat_hist[64];
    unsigned int spectrum[MAX_SPEC_BINS + 2];
};

// a13: tallies of a finished packet into the block's shared-memory histograms.
__device__ __forceinline__ void tally_finish(const WalkParams& p, BlockTallies& sh, int status, float V,
                                             uint32_t nscat, uint32_t crossings, uint32_t rej_iters,
                                             unsigned long long id, float kx, float ky, float kz) {
    atomicAdd(&sh.counters[status], 1ull);
    atomicAdd(&sh.counters[CT_SCATTERINGS], (unsigned long long)nscat);
    atomicAdd(&sh.counters[CT_CROSSINGS], (unsigned long long)crossings);
    atomicAdd(&sh.counters[CT_REJ_ITERS], (unsigned long long)rej_iters);
    const int hb = nscat == 0 ? 0 : 32 - __clz(nscat);       // bin b: 2^(b-1) <= nscat < 2^b
    atomicAdd(&sh.nscat_hist[hb], 1u);
    if ((status == CT_ESCAPED || status == CT_TERMINATED) && p.spec_bins > 0) {
        const float val = p.spec_mode == 0 ? V * p.spec_inv_vth_ref : -V;
        const float b = floorf((val - p.spec_lo) * p.spec_inv_width);
        const int bin = b < 0.f ? p.spec_bins : (b >= (float)p.spec_bins ? p.spec_bins + 1 : (int)b);
        atomicAdd(&sh.spectrum[bin], 1u);
    }
    if (p.raw) p.raw[id - p.id_offset] = RawRecord{V, nscat, status, kx, ky, kz};
}

__global__ void __launch_bounds__(WALK_THREADS, 2) walk_kernel(const __grid_constant__ WalkParams p) {
    __shared__ BlockTallies sh;
    voigt_table_load(sh.voigt);
    for (int i = threadIdx.x; i < N_COUNTERS; i += blockDim.x) sh.counters[i] = 0ull;
    for (int i = threadIdx.x; i < 64; i += blockDim.x) sh.nscat_hist[i] = 0u;
    for (int i = threadIdx.x; i < p.spec_bins + 2; i += blockDim.x) sh.spectrum[i] = 0u;
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u;
    int state = LS_IDLE;
    Ray ray;
    Stream rng;
    float V = 0.f, tau_rem = 0.f;
    unsigned long long id = 0;
    uint32_t nscat = 0, crossings = 0, rej_iters = 0, peel_rays = 0, peel_cells = 0;
    // properties of the cell in which the interaction happens (set at the hit, used by the scatter phase)
    float h_a = 0.f, h_vth = 1.f, h_vx = 0.f, h_vy = 0.f, h_vz = 0.f, h_xcrit = 0.f;
    bool more = true;                                         // warp-uniform: photon counter not yet exhausted

    for (;;) {
        // ---- a14 + a2/a3: refill idle lanes from the global photon counter, emit ----
        const unsigned idle = __ballot_sync(0xffffffffu, state == LS_IDLE);
        if (idle && more) {
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(p.next_photon, (unsigned long long)__popc(idle));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (state == LS_IDLE) {
                const unsigned long long i = base + __popc(idle & ((1u << lane) - 1u));
                if (i >= p.n_photons) {
                    state = LS_OUT;
                } else {
                    id = p.id_offset + i;
                    rng.init(p.seed, id);
                    const double us = (double)rng.uniform();
                    long long lo = 0, hi = p.n_src - 1;           // smallest j with us < cdf[j]
                    while (lo < hi) { const long long mid = (lo + hi) >> 1; if (us < p.src_cdf[mid]) hi = mid; else lo = mid + 1; }
                    const float mu0 = fmaf(2.f, rng.uniform(), -1.f);   // isotropic direction (reading A22)
                    float sp, cp;
                    sincospif(2.f * rng.uniform(), &sp, &cp);
                    const float st0 = sqrtf(fmaxf(0.f, 1.f - mu0 * mu0));
                    const float g1 = rng.uniform(), g2 = rng.uniform();
                    const float gauss = sqrtf(-2.f * logf(g1)) * cospif(2.f * g2);
                    dda_locate(ray, p.g, p.src_pos[3 * lo], p.src_pos[3 * lo + 1], p.src_pos[3 * lo + 2]);
                    ray_set_direction(ray, st0 * cp, st0 * sp, mu0);
                    const CellProps c = fetch_cell(p, dda_linear(ray, p.g));
                    const float dV = p.src_sigma[lo] * gauss;     // Gaussian line in the gas frame (reading A10)
                    V = c.vx * ray.kx + c.vy * ray.ky + c.vz * ray.kz + dV;
                    nscat = 0; crossings = 0; rej_iters = 0;
                    if (p.peel_on) {
                        ++peel_rays;
                        peel_ray(p, sh.voigt, ray, c.vx * p.kobs[0] + c.vy * p.kobs[1] + c.vz * p.kobs[2] + dV, 1.f,
                                 peel_cells);
                    }
                    tau_rem = -logf(rng.uniform());               // a3 (Eq. 3)
                    state = LS_MARCH;
                }
            }
            if (__any_sync(0xffffffffu, state == LS_OUT)) more = false;
        }
        const unsigned marching = __ballot_sync(0xffffffffu, state == LS_MARCH);
        const unsigned scattering = __ballot_sync(0xffffffffu, state == LS_SCATTER);
        if (!(marching | scattering)) {
            if (!more) break;
            continue;
        }

        // ---- a4-a7: one cell step for every marching lane ----
        if (state == LS_MARCH) {
            float len;
            const int ex = dda_next_face(ray, p.g, len);
            const CellProps c = fetch_cell(p, dda_linear(ray, p.g));
            const CellDerived d = derive_cell(p, c);
            const float vk = c.vx * ray.kx + c.vy * ray.ky + c.vz * ray.kz;
            float dtau, s_hit, kl, kt;
            const bool hit = integrate_segment(p, sh.voigt, c, d, V, vk, len, tau_rem, dtau, s_hit, kl, kt);
            if (hit) {
                dda_advance_within(ray, p.g, s_hit);
                if (p.hubble != 0.f) V -= p.hubble * s_hit;
                // a7 interaction kind: dust with probability kappa_dust / kappa_total
                bool absorbed = false;
                if (p.kdust) absorbed = rng.uniform() * kt < c.kd;
                if (absorbed) {
                    tally_finish(p, sh, CT_ABSORBED, V, nscat, crossings, rej_iters, id, ray.kx, ray.ky, ray.kz);
                    state = LS_IDLE;
                } else {
                    h_a = d.a; h_vth = d.vth; h_vx = c.vx; h_vy = c.vy; h_vz = c.vz;
                    h_xcrit = 0.f;
                    if (p.core_skip_mode == 1) h_xcrit = p.x_crit;
                    else if (p.core_skip_mode == 2) {              // local: a tau_0 over half a cell (reading A7)
                        const float atau = d.a * d.nsig * 0.5f;
                        h_xcrit = atau >= 1.f ? 0.2f * cbrtf(atau) : 0.f;
                    }
                    state = LS_SCATTER;
                }
            } else if (!(len < CUDART_INF_F)) {
                // reading A24: infinite segment (ray parallel to every non-frozen axis) without interaction: the
                // packet can neither leave nor be followed -> capped
                tally_finish(p, sh, CT_CAPPED, V, nscat, crossings, rej_iters, id, ray.kx, ray.ky, ray.kz);
                state = LS_IDLE;
            } else {
                tau_rem -= dtau;
                V -= p.hubble * len;
                ++crossings;
                if (!dda_cross(ray, p.g, ex, len)) {
                    tally_finish(p, sh, CT_ESCAPED, V, nscat, crossings, rej_iters, id, ray.kx, ray.ky, ray.kz);
                    state = LS_IDLE;
                } else if (p.v_max > 0.f && fabsf(V) > p.v_max) {
                    tally_finish(p, sh, CT_TERMINATED, V, nscat, crossings, rej_iters, id, ray.kx, ray.ky, ray.kz);
                    state = LS_IDLE;
                }
            }
        }

        // ---- a8-a11: scatter.  Deferred while most lanes are still marching, so that scatterers run together ----
        const unsigned want = __ballot_sync(0xffffffffu, state == LS_SCATTER);
        const unsigned still = __ballot_sync(0xffffffffu, state == LS_MARCH);
        if (want && (__popc(want) >= __popc(still) || __popc(want) >= 8)) {
            if (state == LS_SCATTER) {
                const float kx = ray.kx, ky = ray.ky, kz = ray.kz;
                const float x_in = (V - (h_vx * kx + h_vy * ky + h_vz * kz)) / h_vth;
                const float upar = sample_upar(h_a, x_in, rng, rej_iters);
                float up1, up2;
                sample_uperp(x_in, h_xcrit, rng, up1, up2);
                const float xsel = p.phase_frame == 0 ? fabsf(x_in - upar) : fabsf(x_in);
                const int phase = xsel > p.phase_split_x ? p.phase_wing : p.phase_core;
                bool is_dipole;
                const float mu = sample_mu(phase, rng, is_dipole);
                float sph, cph;
                sincospif(2.f * rng.uniform(), &sph, &cph);
                float e1[3], e2[3];
                ortho_basis(kx, ky, kz, e1, e2);
                if (p.peel_on) {                                  // a12, before adopting k'
                    const float mu_o = kx * p.kobs[0] + ky * p.kobs[1] + kz * p.kobs[2];
                    const float e1o = e1[0] * p.kobs[0] + e1[1] * p.kobs[1] + e1[2] * p.kobs[2];
                    const float e2o = e2[0] * p.kobs[0] + e2[1] * p.kobs[1] + e2[2] * p.kobs[2];
                    const float x_o = x_in - upar + upar * mu_o + up1 * e1o + up2 * e2o;
                    const float V_o = x_o * h_vth + h_vx * p.kobs[0] + h_vy * p.kobs[1] + h_vz * p.kobs[2];
                    ++peel_rays;
                    peel_ray(p, sh.voigt, ray, V_o, is_dipole ? 0.75f * (1.f + mu_o * mu_o) : 1.f, peel_cells);
                }
                const float st = sqrtf(fmaxf(0.f, 1.f - mu * mu));
                float nx = mu * kx + st * (cph * e1[0] + sph * e2[0]);
                float ny = mu * ky + st * (cph * e1[1] + sph * e2[1]);
                float nz = mu * kz + st * (cph * e1[2] + sph * e2[2]);
                const float inv = rsqrtf(nx * nx + ny * ny + nz * nz);
                nx *= inv; ny *= inv; nz *= inv;
                // a11, Eq. 7, recoil dropped: x_out = x_in + u.(k_out - k_in)
                const float x_out = x_in - upar + upar * mu + st * (up1 * cph + up2 * sph);
                ray_set_direction(ray, nx, ny, nz);
                V = x_out * h_vth + h_vx * nx + h_vy * ny + h_vz * nz;
                ++nscat;
                if (p.v_max > 0.f && fabsf(V) > p.v_max) {
                    tally_finish(p, sh, CT_TERMINATED, V, nscat, crossings, rej_iters, id, nx, ny, nz);
                    state = LS_IDLE;
                } else if ((p.max_scatter && nscat >= p.max_scatter) || !(fabsf(V) <= 3.0e38f)) {   // cap, or fail-safe: non-finite V
                    tally_finish(p, sh, CT_CAPPED, V, nscat, crossings, rej_iters, id, nx, ny, nz);
                    state = LS_IDLE;
                } else {
                    tau_rem = -logf(rng.uniform());
                    state = LS_MARCH;
                }
            }
        }
    }

    // ---- flush the block's tallies with global atomics ----
    atomicAdd(&sh.counters[CT_PEEL_RAYS], (unsigned long long)peel_rays);
    atomicAdd(&sh.counters[CT_PEEL_CELLS], (unsigned long long)peel_cells);
    __syncthreads();
    for (int i = threadIdx.x; i < N_COUNTERS; i += blockDim.x)
        if (sh.counters[i]) atomicAdd(p.counters + i, sh.counters[i]);
    for (int i = threadIdx.x; i < 64; i += blockDim.x)
        if (sh.nscat_hist[i]) atomicAdd(p.nscat_hist + i, (unsigned long long)sh.nscat_hist[i]);
    for (int i = threadIdx.x; i < p.spec_bins + 2; i += blockDim.x)
        if (sh.spectrum[i]) atomicAdd(p.spectrum + i, (unsigned long long)sh.spectrum[i]);
}

// Launch configuration: one persistent grid, blocks = SMs x resident blocks per SM.
cudaError_t launch_walk(const WalkParams& p, int n_sm, cudaStream_t stream, int* blocks_out) {
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, walk_kernel, WALK_THREADS, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long blocks = (long long)n_sm * per_sm;
    const long long need = (long long)((p.n_photons + 31) / 32);   // few packets: spread the warps over the SMs
    if (need < blocks) blocks = need < 1 ? 1 : need;
    if (blocks_out) *blocks_out = (int)blocks;
    walk_kernel<<<(unsigned)blocks, WALK_THREADS, 0, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace thor
