// Persistent-thread walk kernel + its launcher.  See walk.cuh for the step functions.
#include <cuda_runtime.h>
#include <math_constants.h>
#include "walk.cuh"

namespace thor {

__device__ __forceinline__ unsigned long long global_timer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

#ifndef THOR_WALK_THREADS
#define THOR_WALK_THREADS 256
#endif
#ifndef THOR_WALK_MIN_CTAS
#define THOR_WALK_MIN_CTAS 3
#endif
#ifndef THOR_FINISH_MIN_LANES
#define THOR_FINISH_MIN_LANES 24
#endif
constexpr int WALK_THREADS = THOR_WALK_THREADS;
constexpr int MAX_SPEC_BINS = 4096;
constexpr int FINISH_MIN_LANES = THOR_FINISH_MIN_LANES;
#ifndef THOR_REFILL_MIN_LANES
#define THOR_REFILL_MIN_LANES 8
#endif
constexpr int REFILL_MIN_LANES = THOR_REFILL_MIN_LANES;

struct BlockTallies {
    float2 voigt[VOIGT_NODES];
    unsigned long long counters[N_COUNTERS];
    unsigned int nscat_hist[64];
    unsigned int max_nscat;
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
    atomicMax(&sh.max_nscat, nscat);
    if ((status == CT_ESCAPED || status == CT_TERMINATED) && p.spec_bins > 0) {
        const float val = p.spec_mode == 0 ? V * p.spec_inv_vth_ref : -V;
        const float b = floorf((val - p.spec_lo) * p.spec_inv_width);
        const int bin = b < 0.f ? p.spec_bins : (b >= (float)p.spec_bins ? p.spec_bins + 1 : (int)b);
        atomicAdd(&sh.spectrum[bin], 1u);
    }
    if (p.raw) p.raw[id - p.id_offset] = RawRecord{V, nscat, status, kx, ky, kz};
}

template <bool HUBBLE, bool PEEL, int MIN_CTAS>
__global__ void __launch_bounds__(WALK_THREADS, MIN_CTAS) walk_kernel(const __grid_constant__ WalkParams p) {
    __shared__ BlockTallies sh;
    if (threadIdx.x == 0) atomicMin(p.t_start, global_timer_ns());
    voigt_table_load(sh.voigt);
    for (int i = threadIdx.x; i < N_COUNTERS; i += blockDim.x) sh.counters[i] = 0ull;
    for (int i = threadIdx.x; i < 64; i += blockDim.x) sh.nscat_hist[i] = 0u;
    if (threadIdx.x == 0) sh.max_nscat = 0u;
    for (int i = threadIdx.x; i < p.spec_bins + 2; i += blockDim.x) sh.spectrum[i] = 0u;
    __syncthreads();

    constexpr bool EARLY_GATHER = MIN_CTAS >= 4;              // the variant launched for grids beyond L2
    const unsigned lane = threadIdx.x & 31u;
    const uint32_t k0 = (uint32_t)p.seed, k1 = (uint32_t)(p.seed >> 32);   // Philox key = seed (reading A16)
    int state = LS_IDLE;
    Ray ray;
    BlockRng rng;
    Cell cell;                                                // the cell the packet is in (valid unless `stale`)
    bool stale = true, inv_ok = false;                        // inv_ok: 1/k of the current direction is in `ray`
    float V = 0.f, tau_rem = 0.f, hit_kt = 0.f, x_in = 0.f, upar = 0.f;
    UparEnvelope env;
    env.mTot = -1.f;
    uint32_t trials = 0;
    uint32_t nscat = 0, crossings = 0, rej_iters = 0, peel_rays = 0, peel_cells = 0;
    bool more = true;                                         // warp-uniform: photon counter not yet exhausted

    for (;;) {
        // ---- a14 + a2/a3: refill idle lanes from the global photon counter, emit ----
        // Refills are batched: emission is a chain of dependent loads (binary search of the source CDF, source cell
        // gather) that stalls the whole warp, so it waits until REFILL_MIN_LANES lanes are idle (or nothing else runs).
        const unsigned idle = __ballot_sync(0xffffffffu, state == LS_IDLE);
        if (more && idle && (__popc(idle) >= REFILL_MIN_LANES || idle == __ballot_sync(0xffffffffu, state == LS_IDLE || state == LS_OUT))) {
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(p.next_photon, (unsigned long long)__popc(idle));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (state == LS_IDLE) {
                const unsigned long long i = base + __popc(idle & ((1u << lane) - 1u));
                if (i >= p.n_photons) {
                    state = LS_OUT;
                } else {
                    rng.init(p.id_offset + i);
                    const float4 e1 = rng.next4(k0, k1), e2 = rng.next4(k0, k1);   // (src, mu, phi, g1), (g2, tau, -, -)
                    const double us = (double)e1.x;
                    long long lo = 0, hi = p.n_src - 1;           // smallest j with us < cdf[j]
                    while (lo < hi) { const long long mid = (lo + hi) >> 1; if (us < p.src_cdf[mid]) hi = mid; else lo = mid + 1; }
                    const float mu0 = fmaf(2.f, e1.y, -1.f);      // isotropic direction (reading A22)
                    float sp, cp;
                    sincos_uniform(e1.z, sp, cp);
                    const float st0 = sqrtf(fmaxf(0.f, 1.f - mu0 * mu0));
                    const float gauss = sqrtf(-2.f * __logf(e1.w)) * cos_uniform(e2.x);
                    dda_locate(ray, p.g, p.src_pos[3 * lo], p.src_pos[3 * lo + 1], p.src_pos[3 * lo + 2]);
                    ray_set_k(ray, st0 * cp, st0 * sp, mu0);
                    inv_ok = false;
                    cell = load_cell(p, dda_linear(ray, p.g));
                    stale = false;
                    const float dV = p.src_sigma[lo] * gauss;     // Gaussian line in the gas frame (reading A10)
                    V = cell.vx * ray.kx + cell.vy * ray.ky + cell.vz * ray.kz + dV;
                    nscat = 0; crossings = 0; rej_iters = 0;
                    if (PEEL) {
                        ++peel_rays;
                        peel_ray<HUBBLE>(p, sh.voigt, ray,
                                         cell.vx * p.kobs[0] + cell.vy * p.kobs[1] + cell.vz * p.kobs[2] + dV, 1.f, peel_cells);
                    }
                    tau_rem = -__logf(e2.y);                      // a3 (Eq. 3)
                    state = LS_MARCH;
                }
            }
            if (__any_sync(0xffffffffu, state == LS_OUT)) {
                // the queue is empty: from here on the launch only drains the packets in flight
                if (more && lane == 0) atomicMin(p.t_dry, global_timer_ns());
                more = false;
            }
        }

        // ---- a4-a7: one cell step for every marching lane ----
        if (state == LS_MARCH) {
            if (stale) {
                if (EARLY_GATHER) derive_cell(p, cell);           // raw fields gathered at the last face crossing
                else cell = load_cell(p, dda_linear(ray, p.g));
                stale = false;
            }
            const float vk = cell.vx * ray.kx + cell.vy * ray.ky + cell.vz * ray.kz;
            bool hit = false;
            float len = 0.f, dtau = 0.f, s_hit = 0.f, kt = 0.f;
            int ex = 0;
            if (!HUBBLE) {
                // Piecewise-constant cell: the interaction lies at s = tau / kappa if that is inside the
                // cell.  Deep in an optically thick cell s is far smaller than the distance to the nearest face, which
                // bounds the segment length from below: no DDA step and no reciprocals of k are needed at all.
                kt = cell_opacity(sh.voigt, cell, V, vk);
                const float s = kt > 0.f ? tau_rem / kt : CUDART_INF_F;
                if (kt > 0.f && s <= dda_min_face_distance(ray, p.g)) {
                    hit = true; s_hit = s;
                } else {
                    if (!inv_ok) { ray_set_inv(ray); inv_ok = true; }
                    ex = dda_next_face(ray, p.g, len);
                    hit = kt > 0.f && s <= len;
                    s_hit = s;
                    dtau = kt * len;
                }
            } else {
                if (!inv_ok) { ray_set_inv(ray); inv_ok = true; }
                ex = dda_next_face(ray, p.g, len);
                hit = integrate_segment<true>(p, sh.voigt, cell, V, vk, len, tau_rem, dtau, s_hit, kt);
            }
            if (hit) {
                dda_advance_within(ray, p.g, s_hit);
                if (HUBBLE) { if (p.hubble != 0.f) V -= p.hubble * s_hit; }
                hit_kt = kt;
                x_in = (V - vk) * cell.inv_vth;
                env.mTot = -1.f;                                  // envelope not built yet
                trials = 0u;
                state = LS_TRIAL;
            } else if (!(len < CUDART_INF_F)) {
                // reading A24: infinite segment (ray parallel to every non-frozen axis) without interaction: the
                // packet can neither leave nor be followed -> capped
                tally_finish(p, sh, CT_CAPPED, V, nscat, crossings, rej_iters, rng.id(), ray.kx, ray.ky, ray.kz);
                state = LS_IDLE;
            } else {
                tau_rem -= dtau;
                if (HUBBLE) V -= p.hubble * len;
                ++crossings;
                if (!dda_cross(ray, p.g, ex, len)) {
                    tally_finish(p, sh, CT_ESCAPED, V, nscat, crossings, rej_iters, rng.id(), ray.kx, ray.ky, ray.kz);
                    state = LS_IDLE;
                } else if (p.v_max > 0.f && fabsf(V) > p.v_max) {
                    tally_finish(p, sh, CT_TERMINATED, V, nscat, crossings, rej_iters, rng.id(), ray.kx, ray.ky, ray.kz);
                    state = LS_IDLE;
                } else if (crossings >= p.max_crossings) {        // reading A26: a packet nothing else would ever end
                    tally_finish(p, sh, CT_CAPPED, V, nscat, crossings, rej_iters, rng.id(), ray.kx, ray.ky, ray.kz);
                    state = LS_IDLE;
                } else {
                    // a5: beyond L2 the gather is issued now and used next iteration, hiding the loop control and the
                    // other stage sections in its shadow; a cache-resident grid gathers at first use (fewer live values)
                    if (EARLY_GATHER) cell = load_cell_raw(p, dda_linear(ray, p.g));
                    stale = true;
                }
            }
        }

        // ---- a8: ONE rejection trial of u_par for every lane that needs one.  No inner loop: a
        // lane whose trial is rejected tries again in the next iteration, alongside the lanes that arrive from the
        // march, instead of the whole warp waiting for its slowest lane (the paper's "largest source of thread
        // divergence"; E[max of 32 iterations]/E[iterations] = 2.1-4.2) ----
        if (state == LS_TRIAL) {
            if (env.mTot < 0.f) env = upar_envelope(cell.a, fabsf(x_in));
            ++rej_iters;
            float u;
            const bool ok = upar_try(env, cell.a, rng.next4(k0, k1), u);
            // fail-safe: acceptance is >= ~0.2 everywhere; 2^20 rejections cannot happen unless x is NaN
            if (ok || ++trials >= (1u << 20)) { upar = x_in < 0.f ? -u : u; state = LS_FINISH; }
        }

        // ---- a7, a9-a12: finish the interaction.  The most expensive section: deferred until enough lanes want it ----
        const unsigned fin = __ballot_sync(0xffffffffu, state == LS_FINISH);
        const unsigned busy = __ballot_sync(0xffffffffu, state == LS_MARCH || state == LS_TRIAL);
        if (!(fin | busy)) {
            if (!more) break;
            continue;
        }
        if (fin && (__popc(fin) >= __popc(busy) || __popc(fin) >= FINISH_MIN_LANES)) {
            if (state == LS_FINISH) {
                // draws of this event: (tau, mu, phi, perp1), (perp2, dust, mix, -)
                const float4 s1 = rng.next4(k0, k1), s2 = rng.next4(k0, k1);
                // a7 interaction kind: dust with probability kappa_dust / kappa_total
                if (p.has_dust && s2.y * hit_kt < cell.kd) {
                    tally_finish(p, sh, CT_ABSORBED, V, nscat, crossings, rej_iters, rng.id(), ray.kx, ray.ky, ray.kz);
                    state = LS_IDLE;
                } else {
                    const float kx = ray.kx, ky = ray.ky, kz = ray.kz;
                    float x_crit = 0.f;
                    if (p.core_skip_mode == 1) x_crit = p.x_crit;
                    else if (p.core_skip_mode == 2) {              // local: a tau_0 over half a cell (reading A7)
                        const float atau = cell.a * cell.nsig * 0.5f;
                        x_crit = atau >= 1.f ? 0.2f * cbrtf(atau) : 0.f;
                    }
                    float up1, up2;
                    sample_uperp(x_in, x_crit, s1.w, s2.x, up1, up2);
                    const float xsel = p.phase_frame == 0 ? fabsf(x_in - upar) : fabsf(x_in);
                    const int phase = xsel > p.phase_split_x ? p.phase_wing : p.phase_core;
                    bool is_dipole;
                    const float mu = sample_mu(phase, s2.z, s1.y, is_dipole);
                    float sph, cph;
                    sincos_uniform(s1.z, sph, cph);
                    float e1[3], e2[3];
                    ortho_basis(kx, ky, kz, e1, e2);
                    if (PEEL) {                                   // a12, before adopting k'
                        const float mu_o = kx * p.kobs[0] + ky * p.kobs[1] + kz * p.kobs[2];
                        const float e1o = e1[0] * p.kobs[0] + e1[1] * p.kobs[1] + e1[2] * p.kobs[2];
                        const float e2o = e2[0] * p.kobs[0] + e2[1] * p.kobs[1] + e2[2] * p.kobs[2];
                        const float x_o = x_in - upar + upar * mu_o + up1 * e1o + up2 * e2o;
                        const float V_o = x_o * cell.vth + cell.vx * p.kobs[0] + cell.vy * p.kobs[1] + cell.vz * p.kobs[2];
                        ++peel_rays;
                        peel_ray<HUBBLE>(p, sh.voigt, ray, V_o, is_dipole ? 0.75f * (1.f + mu_o * mu_o) : 1.f, peel_cells);
                    }
                    const float st = sqrtf(fmaxf(0.f, 1.f - mu * mu));
                    float nx = mu * kx + st * (cph * e1[0] + sph * e2[0]);
                    float ny = mu * ky + st * (cph * e1[1] + sph * e2[1]);
                    float nz = mu * kz + st * (cph * e1[2] + sph * e2[2]);
                    const float inv = rsqrtf(nx * nx + ny * ny + nz * nz);
                    nx *= inv; ny *= inv; nz *= inv;
                    // a11, Eq. 7, recoil dropped: x_out = x_in + u.(k_out - k_in)
                    const float x_out = x_in - upar + upar * mu + st * (up1 * cph + up2 * sph);
                    ray_set_k(ray, nx, ny, nz);
                    inv_ok = false;
                    V = x_out * cell.vth + cell.vx * nx + cell.vy * ny + cell.vz * nz;
                    ++nscat;
                    if (p.v_max > 0.f && fabsf(V) > p.v_max) {
                        tally_finish(p, sh, CT_TERMINATED, V, nscat, crossings, rej_iters, rng.id(), nx, ny, nz);
                        state = LS_IDLE;
                    } else if ((p.max_scatter && nscat >= p.max_scatter) || !(fabsf(V) <= 3.0e38f)) {   // cap, or fail-safe: non-finite V
                        tally_finish(p, sh, CT_CAPPED, V, nscat, crossings, rej_iters, rng.id(), nx, ny, nz);
                        state = LS_IDLE;
                    } else {
                        tau_rem = -__logf(s1.x);
                        state = LS_MARCH;
                    }
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
    if (threadIdx.x == 0 && sh.max_nscat) atomicMax(p.max_nscat, (unsigned long long)sh.max_nscat);
    for (int i = threadIdx.x; i < p.spec_bins + 2; i += blockDim.x)
        if (sh.spectrum[i]) atomicAdd(p.spectrum + i, (unsigned long long)sh.spectrum[i]);
}

// (n_HI, T) alone: 8 B of the cell's packed sector, or two SoA loads.
__device__ __forceinline__ void load_nT(const WalkParams& p, int64_t i, float& n, float& T) {
    if (p.packed) { const float2 q = __ldg(reinterpret_cast<const float2*>(p.packed + 2 * i)); n = q.x; T = q.y; }
    else { n = __ldg(p.nHI + i); T = __ldg(p.T + i); }
}

// ---- ray-tracing operators on the same DDA + gather + Voigt (PAPER.md 3.5) ----
// One thread per ray, marched from its origin to the first box face.  Projection (PAPER.md 3.5.1): Q = Int q w ds with
// q = n_HI, w = 1 (column density, cm^-2) and q = T, w = n_HI (density-weighted temperature Q / Q^).  Absorption
// spectrum (PAPER.md 3.5.2, Eq. 11): tau(V_j) = Int n sigma(nu(s), T) ds with the gas seeing the sight-line
// frequency shifted by its line-of-sight velocity v.k and the Hubble term H s; piecewise-constant cells, midpoint of
// each segment for the Hubble term.
__global__ void raytrace_kernel(const __grid_constant__ WalkParams p, long long n_rays, const float* __restrict__ org,
                                const float* __restrict__ dir, float hubble, int n_v, float v_lo, float dv,
                                float* __restrict__ out_column, float* __restrict__ out_tmean, float* __restrict__ out_tau) {
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
        const float len = march_next_face(r, ex_x, ex_y);
        if (!(len < CUDART_INF_F)) break;
        Cell c;
        if (tau) c = load_cell_raw(p, r.idx);
        else load_nT(p, r.idx, c.nsig, c.a);                  // projections need 8 B of the cell only
        const float n = c.nsig, T = c.a;
        col += n * len;
        tn += n * T * len;
        if (tau) {
            derive_cell(p, c);
            const float vgas = c.vx * kx + c.vy * ky + c.vz * kz + hubble * (s_path + 0.5f * len);
            if (c.nsig > 0.f || c.kd > 0.f)
                for (int j = 0; j < n_v; ++j) {
                    const float V = v_lo + ((float)j + 0.5f) * dv;
                    const float kl = c.nsig > 0.f ? c.nsig * voigt_H(s_tab, c.a, (V - vgas) * c.inv_vth) : 0.f;
                    tau[j] += (kl + c.kd) * len;
                }
        }
        s_path += len;
        if (!march_cross(r, p.g, ex_x, ex_y, len)) break;     // rays end at the first box face, periodic or not
    }
    if (out_column) out_column[i] = col * p.cell_cm;
    if (out_tmean) out_tmean[i] = col > 0.f ? tn / col : 0.f;
}

cudaError_t launch_raytrace(const WalkParams& p, long long n_rays, const float* org, const float* dir, float hubble,
                            int n_v, float v_lo, float dv, float* out_column, float* out_tmean, float* out_tau,
                            cudaStream_t stream) {
    raytrace_kernel<<<(unsigned)((n_rays + 127) / 128), 128, 0, stream>>>(p, n_rays, org, dir, hubble, n_v, v_lo, dv,
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
    float cr = 0.f, cg = 0.f, cb = 0.f, tr = 1.f;
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
                const float att = ex2_approx(-1.4426950408889634f * mu * len);
                const float f = tr * (1.f - att) * w / mu;      // Tr (1 - e^{-mu l}) / mu, times w for the emission
                cr = fmaf(f, er, cr);
                cg = fmaf(f, eg, cg);
                cb = fmaf(f, eb, cb);
                tr *= att;
            }
        }
        if (!march_cross(r, p.g, ex_x, ex_y, len)) break;
    }
    out_rgba[i] = make_float4(cr, cg, cb, 1.f - tr);
}

cudaError_t launch_volume_render(const WalkParams& p, const TransferFn& tf, long long n_rays, const float* org,
                                 const float* dir, float* out_rgba, cudaStream_t stream) {
    volume_render_kernel<<<(unsigned)((n_rays + 127) / 128), 128, 0, stream>>>(p, tf, n_rays, org, dir,
                                                                              reinterpret_cast<float4*>(out_rgba));
    return cudaGetLastError();
}

// Launch configuration: one persistent grid, blocks = SMs x resident blocks per SM.  The kernel is specialised at
// compile time on (Hubble drift, peel-off) so that the common static, no-peel walk carries neither, and on the
// register budget: 3 CTAs of 256 threads per SM (<= 80 registers) when the grid fits the 126 MB L2 and the walk is
// issue-bound, 4 CTAs (64 registers, 32 warps) when it does not and the walk needs more gathers in flight
// (+18 % on the 512^3 gather workload, -6 % on the cache-resident sphere); 2 CTAs with peel-off (<= 128 registers).
template <bool HUBBLE, bool PEEL, int MIN_CTAS>
static cudaError_t launch_variant(const WalkParams& p, int n_sm, cudaStream_t stream, int* blocks_out) {
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, walk_kernel<HUBBLE, PEEL, MIN_CTAS>, WALK_THREADS, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long blocks = (long long)n_sm * per_sm;
    const long long need = (long long)((p.n_photons + 31) / 32);   // few packets: spread the warps over the SMs
    if (need < blocks) blocks = need < 1 ? 1 : need;
    if (blocks_out) *blocks_out = (int)blocks;
    walk_kernel<HUBBLE, PEEL, MIN_CTAS><<<(unsigned)blocks, WALK_THREADS, 0, stream>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_walk(const WalkParams& p, int n_sm, cudaStream_t stream, int* blocks_out) {
    const bool hub = p.hubble != 0.f, peel = p.peel_on != 0;
    const double cells = (double)p.g.nx * p.g.ny * p.g.nz;
    const double grid_bytes = cells * (p.packed ? 32.0 : (p.has_dust ? 24.0 : 20.0));
    const bool beyond_l2 = grid_bytes > 96.0e6;
    if (peel) return hub ? launch_variant<true, true, 2>(p, n_sm, stream, blocks_out)
                         : launch_variant<false, true, 2>(p, n_sm, stream, blocks_out);
    if (beyond_l2) return hub ? launch_variant<true, false, 4>(p, n_sm, stream, blocks_out)
                              : launch_variant<false, false, 4>(p, n_sm, stream, blocks_out);
    return hub ? launch_variant<true, false, THOR_WALK_MIN_CTAS>(p, n_sm, stream, blocks_out)
               : launch_variant<false, false, THOR_WALK_MIN_CTAS>(p, n_sm, stream, blocks_out);
}

}  // namespace thor
