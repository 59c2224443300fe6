// The walk kernel: steps a1-a14 of DESIGN.md §Path (§3.4, Fig. 1) in one persistent
// launch.  One lane = one photon packet; finished lanes are refilled from a global atomic photon counter
// (warp-aggregated, a14); the warp alternates between a MARCH phase (one DDA cell step + gather + Voigt optical
// depth for every marching lane) and a SCATTER phase (u_par rejection, u_perp, phase function, Eq. 7 for every lane
// that reached its interaction site), so that lanes execute the same phase together.
// Escape tallies go to shared-memory histograms flushed once per block with global atomics (a13).
#pragma once
#include "params.cuh"
#include "philox.cuh"
#include "voigt.cuh"
#include "sampler.cuh"

namespace thor {

enum : int { LS_IDLE = 0, LS_MARCH = 1, LS_TRIAL = 2, LS_FINISH = 3, LS_OUT = 4, LS_SELECT = 5 };

// a5 cell gather + derived per-cell quantities (one MUFU.RSQ): SoA fp32 fields through the read-only path.  A packet
// keeps the Cell of the cell it is in (registers) until it crosses a face: in optically thick cells a packet
// scatters thousands of times between crossings and re-gathers nothing.
struct Cell {
    float a;         // Voigt parameter
    float vth;       // km/s
    float inv_vth;
    float nsig;      // n sigma_0(T) cell_cm: line-centre optical depth per cell length (0 in empty cells)
    float kd;        // dust absorption optical depth per cell length
    float vx, vy, vz;
};

// The gather is issued as soon as the packet knows its next cell (right after the face crossing) and consumed one
// loop iteration later: load_cell_raw leaves the raw fields in the Cell's own registers (n in nsig, T in a, kdust in
// kd) and derive_cell turns them into the derived quantities at first use, so the loop control and the other stage
// sections run in the shadow of the load.
__device__ __forceinline__ Cell load_cell_raw(const WalkParams& p, int64_t i) {
    Cell c;
    if (p.packed) {                     // one 32-byte sector per cell instead of five or six
        const float4 q0 = __ldg(p.packed + 2 * i), q1 = __ldg(p.packed + 2 * i + 1);
        c.nsig = q0.x; c.a = q0.y; c.vx = q0.z; c.vy = q0.w; c.vz = q1.x; c.kd = q1.y;
    } else {
        c.nsig = __ldg(p.nHI + i); c.a = __ldg(p.T + i);
        c.vx = __ldg(p.vx + i); c.vy = __ldg(p.vy + i); c.vz = __ldg(p.vz + i);
        c.kd = p.kdust ? __ldg(p.kdust + i) : 0.f;
    }
    c.vth = 0.f; c.inv_vth = 0.f;
    return c;
}

__device__ __forceinline__ void derive_cell(const WalkParams& p, Cell& c) {
    const float n = c.nsig, T = c.a;
    const float rs = rsqrtf(T);
    c.kd = c.kd * p.cell_cm;
    c.a = p.c_a * rs;
    c.inv_vth = p.inv_c_vth * rs;
    c.vth = p.c_vth * (T * rs);
    c.nsig = n > 0.f ? n * p.sig_cell * rs : 0.f;
}

__device__ __forceinline__ Cell load_cell(const WalkParams& p, int64_t i) {
    Cell c = load_cell_raw(p, i);
    derive_cell(p, c);
    return c;
}

// Line opacity per cell length at gas-frame frequency x of line 1: n sigma_0 [H(a, x) + rs H(a ra, x - dv / v_th)]
// (the cross-sections of a doublet's transitions add); k2 = the second line's share.
// DB = false: instantiated for runs without a doublet (drain kernel): the tests of that run constant — a uniform-register
// load, compare and branch of ~45 cycles each on the serial chain of a lone packet — are compiled out.
template <bool DB = true>
__device__ __forceinline__ float line_opacity(const WalkParams& p, const float2* s_tab, const Cell& c, float x, float& k2) {
    k2 = 0.f;
    if (!(c.nsig > 0.f)) return 0.f;
    const float k1 = c.nsig * voigt_H(s_tab, c.a, x);
    if (DB && p.doublet_on) k2 = c.nsig * p.db_rs * voigt_H(s_tab, c.a * p.db_ra, fmaf(-p.db_dv, c.inv_vth, x));
    return k1 + k2;
}

// a6/a7: optical depth of one segment of length len (cell units) starting at velocity offset V0, or the distance
// s_hit at which tau_need is reached (linear within the step).  Without Hubble drift: kappa len.
// With drift Hc (km/s per cell length): sub-steps per reading A12 — n_sub = 1 if min|x| over the segment > 6 else
// ceil(|dV| / (eps v_th)), midpoint rule.  Returns true on interaction; k_tot is the opacity there.
template <bool HUBBLE, bool DB = true>
__device__ __forceinline__ bool integrate_segment(const WalkParams& p, const float2* s_tab, const Cell& c, float V0,
                                                  float vk, float len, float tau_need, float& tau_out, float& s_hit,
                                                  float& k_tot, float& k2) {
    tau_out = 0.f; s_hit = 0.f; k_tot = 0.f; k2 = 0.f;
    if (c.nsig <= 0.f && c.kd <= 0.f) return false;
    if (!HUBBLE) {
        const float kl = line_opacity<DB>(p, s_tab, c, (V0 - vk) * c.inv_vth, k2);
        const float kt = kl + c.kd;
        const float dtau = kt * len;
        if (dtau >= tau_need && kt > 0.f) {
            s_hit = fminf(tau_need / kt, len);
            k_tot = kt;
            tau_out = tau_need;
            return true;
        }
        tau_out = dtau;
        return false;
    }
    const float Hc = p.hubble;
    int nsub = 1;
    if (Hc != 0.f && c.nsig > 0.f && len > 0.f) {
        const float xa = (V0 - vk) * c.inv_vth, xb = (fmaf(-Hc, len, V0) - vk) * c.inv_vth;
        const float minabs = xa * xb <= 0.f ? 0.f : fminf(fabsf(xa), fabsf(xb));
        if (minabs <= 6.f) {
            const float q = ceilf(fabsf(Hc * len) * c.inv_vth / p.hubble_eps);
            nsub = q < 1.f ? 1 : (q > 1e6f ? 1000000 : (int)q);
        }
    }
    const float ds = len / (float)nsub;
    float tau = 0.f;
    for (int j = 0; j < nsub; ++j) {
        const float Vmid = Hc != 0.f ? fmaf(-Hc, ((float)j + 0.5f) * ds, V0) : V0;   // no 0 * inf when ds = +inf (A24)
        const float kl = line_opacity<DB>(p, s_tab, c, (Vmid - vk) * c.inv_vth, k2);
        const float kt = kl + c.kd;
        const float dtau = kt * ds;
        if (tau + dtau >= tau_need && kt > 0.f) {
            s_hit = fminf((j ? (float)j * ds : 0.f) + (tau_need - tau) / kt, len);
            k_tot = kt;
            tau_out = tau_need;
            return true;
        }
        tau += dtau;
    }
    tau_out = tau;
    return false;
}

// Total opacity per cell length at velocity offset V for direction cosine-weighted bulk velocity vk (no drift).
template <bool DB = true>
__device__ __forceinline__ float cell_opacity(const WalkParams& p, const float2* s_tab, const Cell& c, float V, float vk, float& k2) {
    return line_opacity<DB>(p, s_tab, c, (V - vk) * c.inv_vth, k2) + c.kd;
}

// a12 peel-off: w = P^ exp(-tau_obs), tau_obs integrated from `at` along k_obs to the box face at
// velocity offset V_o by the same march (a4-a6), dropped beyond tau_peel_max (reading A13); added to
// (pixel of the starting point projected perpendicular to k_obs, spectral bin of dv = -V at the box face).  `add` is
// false on the lanes that only shadow a packet in the cooperative drain (one lane tallies).
// The ray is written as three steps shared by the two ways it is run: whole (peel_ray_body: the drain kernel and the
// emission of a lone packet) and deferred (walk kernel: the first cell in place, the rest queued).

// Pixel of the ray's starting point; -1 if it projects outside the image.
__device__ __forceinline__ int peel_pixel(const WalkParams& p, const Ray& at) {
    const float px0 = (float)at.cx + at.fx - 0.5f * (float)p.g.nx;
    const float py0 = (float)at.cy + at.fy - 0.5f * (float)p.g.ny;
    const float pz0 = (float)at.cz + at.fz - 0.5f * (float)p.g.nz;
    const float px = fmaf(dot3(px0, py0, pz0, p.img1[0], p.img1[1], p.img1[2]), p.peel_inv_width, 0.5f) * (float)p.peel_nx;
    const float py = fmaf(dot3(px0, py0, pz0, p.img2[0], p.img2[1], p.img2[2]), p.peel_inv_width, 0.5f) * (float)p.peel_ny;
    if (!(px >= 0.f && px < (float)p.peel_nx && py >= 0.f && py < (float)p.peel_ny)) return -1;
    return (int)py * p.peel_nx + (int)px;
}

enum : int { PEEL_DROPPED = 0, PEEL_LEFT = 1, PEEL_NEXT = 2 };

// One cell of the ray (r along k_obs, c = the gas of r's cell): PEEL_DROPPED beyond tau_peel_max (or a ray that never
// meets a face, reading A24), PEEL_LEFT at the box face (tau, V final), PEEL_NEXT after stepping into the next cell.
template <bool HUBBLE>
__device__ __forceinline__ int peel_cell(const WalkParams& p, const float2* s_tab, Ray& r, const Cell& c, float& tau, float& V,
                                         uint32_t& n_cells) {
    float len;
    const int ex = dda_next_face(r, p.g, len);
    if (!(len < CUDART_INF_F)) return PEEL_DROPPED;
    const float vk = dot3(c.vx, c.vy, c.vz, r.kx, r.ky, r.kz);
    float dtau, s_hit, kt;
    // the ray is dropped beyond tau_peel_max (reading A13): asking the segment for no more than what is left to the
    // cap lets it stop at the sub-step that reaches it instead of integrating the whole cell
    ++n_cells;
    float k2;
    if (integrate_segment<HUBBLE>(p, s_tab, c, V, vk, len, fmaf(p.tau_peel_max - tau, 1.0000002f, 1e-30f), dtau, s_hit, kt, k2)) return PEEL_DROPPED;
    tau += dtau;
    if (HUBBLE) V = fmaf(-p.hubble, len, V);
    if (tau > p.tau_peel_max) return PEEL_DROPPED;
    // peel rays leave through the first box face they meet, periodic or not
    const float ke = ex == 0 ? r.kx : ex == 1 ? r.ky : r.kz;
    const int cn = (ex == 0 ? r.cx : ex == 1 ? r.cy : r.cz) + (ke > 0.f ? 1 : -1);
    const int nn = ex == 0 ? p.g.nx : ex == 1 ? p.g.ny : p.g.nz;
    if (cn < 0 || cn >= nn) return PEEL_LEFT;
    dda_cross(r, p.g, ex, len);
    return PEEL_NEXT;
}

__device__ __forceinline__ void peel_deposit(const WalkParams& p, int pix, float V, float tau, float phat, bool add) {
    const int iv = (int)floorf((-V - p.peel_v_lo) * p.peel_inv_dv);
    if (iv < 0 || iv >= p.peel_nv) return;
    const float w = phat * __expf(-tau);
    const unsigned long long q = (unsigned long long)__float2ull_rn(w * (float)CUBE_FIXED_SCALE);
    if (q && add) atomicAdd(p.cube + (size_t)pix * p.peel_nv + iv, q);
}

__device__ __forceinline__ void peel_ray_direction(const WalkParams& p, Ray& r) {
    r.kx = p.kobs[0]; r.ky = p.kobs[1]; r.kz = p.kobs[2];     // 1 / k_obs: IEEE quotients made once on the host
    r.ix = p.kobs_inv[0]; r.iy = p.kobs_inv[1]; r.iz = p.kobs_inv[2];
}

template <bool HUBBLE>
__device__ __forceinline__ void peel_ray_body(const WalkParams& p, const float2* s_tab, const Ray& at, const Cell& own, float V_o,
                                              float phat, uint32_t& n_cells, bool add) {
    const int pix = peel_pixel(p, at);
    if (pix < 0) return;
    Ray r = at;
    peel_ray_direction(p, r);
    float tau = 0.f, V = V_o;
    // the ray starts in the packet's own cell, whose derived properties the packet already holds (most rays end there)
    int st = peel_cell<HUBBLE>(p, s_tab, r, own, tau, V, n_cells);
    while (st == PEEL_NEXT) {
        const Cell c = load_cell(p, dda_linear(r, p.g));
        st = peel_cell<HUBBLE>(p, s_tab, r, c, tau, V, n_cells);
    }
    if (st == PEEL_LEFT) peel_deposit(p, pix, V, tau, phat, add);
}

// A peel ray that left its first cell, waiting in the walk kernel's per-warp queue for enough company.
struct PeelPend {
    int cx, cy, cz;
    float fx, fy, fz;
    float tau, V, phat;
    int pix;
    bool live;
};

// Deferred form: the first cell only; a ray that goes on is handed back in `pend` (live = true).
template <bool HUBBLE>
__device__ __forceinline__ void peel_ray_first(const WalkParams& p, const float2* s_tab, const Ray& at, const Cell& own, float V_o,
                                               float phat, uint32_t& n_cells, bool add, PeelPend& pend) {
    const int pix = peel_pixel(p, at);
    if (pix < 0) return;
    Ray r = at;
    peel_ray_direction(p, r);
    float tau = 0.f, V = V_o;
    const int st = peel_cell<HUBBLE>(p, s_tab, r, own, tau, V, n_cells);
    if (st == PEEL_LEFT) peel_deposit(p, pix, V, tau, phat, add);
    else if (st == PEEL_NEXT) {
        pend.cx = r.cx; pend.cy = r.cy; pend.cz = r.cz; pend.fx = r.fx; pend.fy = r.fy; pend.fz = r.fz;
        pend.tau = tau; pend.V = V; pend.phat = phat; pend.pix = pix; pend.live = true;
    }
}

// INLINE: the drain kernel has registers to spare and walks one packet per warp, where a call's spills are pure latency.

template <bool HUBBLE>
__device__ __noinline__ void peel_ray_call(const WalkParams& p, const float2* s_tab, const Ray& at, const Cell& own, float V_o,
                                           float phat, uint32_t& n_cells, bool add) {
    peel_ray_body<HUBBLE>(p, s_tab, at, own, V_o, phat, n_cells, add);
}

// How a caller runs the ray: PEEL_CALL / PEEL_INLINE = whole and in place (out of line / inlined), PEEL_FIRST = the first
// cell in place and the rest handed back in `pend` (walk kernel), PEEL_QUEUED = nothing in place, the whole ray handed back
// (drain kernel: the ray is off the packet's serial chain, and 32 of them are marched side by side).
enum : int { PEEL_CALL = 0, PEEL_INLINE = 1, PEEL_FIRST = 2, PEEL_QUEUED = 3 };
constexpr int PEEL_PIX_UNSET = -2;                     // a queued ray whose pixel is still to be found

template <bool HUBBLE, int MODE>
__device__ __forceinline__ void peel_ray(const WalkParams& p, const float2* s_tab, const Ray& at, const Cell& own, float V_o,
                                         float phat, uint32_t& n_cells, bool add, PeelPend* pend) {
    if (MODE == PEEL_QUEUED) {
        pend->cx = at.cx; pend->cy = at.cy; pend->cz = at.cz; pend->fx = at.fx; pend->fy = at.fy; pend->fz = at.fz;
        pend->tau = 0.f; pend->V = V_o; pend->phat = phat; pend->pix = PEEL_PIX_UNSET; pend->live = true;
    } else if (MODE == PEEL_FIRST) peel_ray_first<HUBBLE>(p, s_tab, at, own, V_o, phat, n_cells, add, *pend);
    else if (MODE == PEEL_INLINE) peel_ray_body<HUBBLE>(p, s_tab, at, own, V_o, phat, n_cells, add);
    else peel_ray_call<HUBBLE>(p, s_tab, at, own, V_o, phat, n_cells, add);
}

// ---- one packet, and the steps of its life as functions shared by every code variant that walks it ----
struct Packet {
    Ray ray;
    Cell cell;                   // the cell the packet is in (valid unless `stale`)
    BlockRng rng;
    float V;                     // lab-frame velocity offset from line centre, km/s
    float tau_rem;               // optical depth left to the next interaction
    float hit_kt, x_in, upar;    // at the interaction site: total opacity, gas-frame frequency (of the chosen line), accepted u_par
    float hit_k2;                // doublet: the second line's opacity there
    int line;                    // doublet: the interaction drawn at the site: 0 / 1 = line, -1 = dust
    uint32_t nscat, crossings, rej_iters, trials;
    bool stale;                  // cell must be (re)gathered / derived before use
    bool inv_ok;                 // 1/k of the current direction is in `ray`
    double gx, gy, gz;           // gridless datasets only: position in length units (fp64: a line-centre mean free path
                                 // is 1e-6 ... 1e-9 of the radius, below fp32 spacing); unused and optimised away on grids
};

enum : int { EV_CROSSED = 0, EV_HIT = 1, EV_ESCAPED = 2, EV_TERMINATED = 3, EV_CAPPED = 4, EV_ABSORBED = 5, EV_SCATTERED = 6, EV_DUST_SCATTERED = 7 };

// a2/a3: emission of photon `id`: source ∝ luminosity, isotropic k (reading A22), Gaussian line in the
// source cell's gas frame (A10), tau_target = -ln u.  dV_out: the line offset, for the peel of the unscattered packet.
__device__ __forceinline__ void emit_packet(const WalkParams& p, Packet& k, unsigned long long id, uint32_t k0, uint32_t k1,
                                            float& dV_out) {
    k.rng.init(id);
    const float4 e1 = k.rng.next4(k0, k1), e2 = k.rng.next4(k0, k1);   // (src, mu, phi, g1), (g2, tau, -, -)
    const double us = (double)e1.x;
    long long lo = 0, hi = p.n_src - 1;           // smallest j with us < cdf[j]
    while (lo < hi) { const long long mid = (lo + hi) >> 1; if (us < p.src_cdf[mid]) hi = mid; else lo = mid + 1; }
    const float mu0 = fmaf(2.f, e1.y, -1.f);
    float sp, cp;
    sincos_uniform(e1.z, sp, cp);
    const float st0 = sqrtf(fmaxf(0.f, fmaf(-mu0, mu0, 1.f)));
    const float gauss = sqrtf(2.f * neg_log(e1.w)) * cos_uniform(e2.x);
    dda_locate(k.ray, p.g, p.src_pos[3 * lo], p.src_pos[3 * lo + 1], p.src_pos[3 * lo + 2]);
    ray_set_k(k.ray, st0 * cp, st0 * sp, mu0);
    k.inv_ok = false;
    k.cell = load_cell(p, dda_linear(k.ray, p.g));
    k.stale = false;
    const float dV = p.src_sigma[lo] * gauss;
    k.V = dot3(k.cell.vx, k.cell.vy, k.cell.vz, k.ray.kx, k.ray.ky, k.ray.kz) + dV;
    k.nscat = 0; k.crossings = 0; k.rej_iters = 0; k.trials = 0;
    k.tau_rem = neg_log(e2.y);
    dV_out = dV;
}

// a4-a7: one cell step.  EV_HIT: the packet sits at its interaction site (hit_kt, x_in set); EV_CROSSED: it entered the
// next cell; else it ended (escaped / terminated / capped).  EARLY: the variant for grids beyond L2 issues the gather
// of the next cell at the face crossing and derives it at first use.
template <bool HUBBLE, bool EARLY, bool DB = true>
__device__ __forceinline__ int march_step(const WalkParams& p, const float2* s_tab, Packet& k) {
    if (k.stale) {
        if (EARLY) derive_cell(p, k.cell);
        else k.cell = load_cell(p, dda_linear(k.ray, p.g));
        k.stale = false;
    }
    const float vk = dot3(k.cell.vx, k.cell.vy, k.cell.vz, k.ray.kx, k.ray.ky, k.ray.kz);
    bool hit = false;
    float len = 0.f, dtau = 0.f, s_hit = 0.f, kt = 0.f;
    int ex = 0;
    if (!HUBBLE) {
        // Piecewise-constant cell: the interaction lies at s = tau / kappa if that is inside the cell.
        // Deep in an optically thick cell s is far smaller than the distance to the nearest face, which bounds the
        // segment length from below: no DDA step and no reciprocals of k are needed at all.
        kt = cell_opacity<DB>(p, s_tab, k.cell, k.V, vk, k.hit_k2);
        const float s = kt > 0.f ? k.tau_rem / kt : CUDART_INF_F;
        if (kt > 0.f && s <= dda_min_face_distance(k.ray, p.g)) {
            hit = true; s_hit = s;
        } else {
            if (!k.inv_ok) { ray_set_inv(k.ray); k.inv_ok = true; }
            ex = dda_next_face(k.ray, p.g, len);
            hit = kt > 0.f && s <= len;
            s_hit = s;
            dtau = kt * len;
        }
    } else {
        if (!k.inv_ok) { ray_set_inv(k.ray); k.inv_ok = true; }
        ex = dda_next_face(k.ray, p.g, len);
        hit = integrate_segment<true, DB>(p, s_tab, k.cell, k.V, vk, len, k.tau_rem, dtau, s_hit, kt, k.hit_k2);
    }
    if (hit) {
        dda_advance_within(k.ray, p.g, s_hit);
        if (HUBBLE) { if (p.hubble != 0.f) k.V = fmaf(-p.hubble, s_hit, k.V); }
        k.hit_kt = kt;
        k.x_in = (k.V - vk) * k.cell.inv_vth;
        k.trials = 0u;
        k.line = 0;
        return EV_HIT;
    }
    // reading A24: infinite segment (ray parallel to every non-frozen axis) without interaction: the packet can neither
    // leave nor be followed -> capped
    if (!(len < CUDART_INF_F)) return EV_CAPPED;
    k.tau_rem -= dtau;
    if (HUBBLE) k.V = fmaf(-p.hubble, len, k.V);
    ++k.crossings;
    if (!dda_cross(k.ray, p.g, ex, len)) return EV_ESCAPED;
    if (p.v_max > 0.f && fabsf(k.V) > p.v_max) return EV_TERMINATED;
    if (k.crossings >= p.max_crossings) return EV_CAPPED;     // reading A26
    // a5: beyond L2 the gather is issued now and used next iteration, hiding the loop control and the other stage
    // sections in its shadow; a cache-resident grid gathers at first use (fewer live values)
    if (EARLY) k.cell = load_cell_raw(p, dda_linear(k.ray, p.g));
    k.stale = true;
    return EV_CROSSED;
}

// ---- gridless datasets (PAPER.md 3.3; readings A29-A31): analytic shell / sphere / slab ----
// Geometry in fp64 (positions, boundary distances), physics in fp32 as on grids.  B200's FP64 pipe makes the handful of
// double operations per step cheap; there is no cell to anchor an fp32 offset to.

// Gas of a step: the dataset's properties at position r (the step's midpoint, reading A30) into the packet's Cell.
__device__ __forceinline__ void gl_props(const WalkParams& p, double x, double y, double z, Cell& c) {
    c.a = p.gl_a; c.vth = p.gl_vth; c.inv_vth = p.gl_inv_vth;
    c.vx = 0.f; c.vy = 0.f; c.vz = 0.f;
    if (p.gl_geom == 1) {
        const bool in = fabs(z) <= p.gl_rout;
        c.nsig = in ? p.gl_nsig0 : 0.f;
        c.kd = in ? p.gl_kd0 : 0.f;
        if (in) c.vz = p.gl_vmax * (float)(z / p.gl_rout);
        return;
    }
    const double rr = sqrt(fma(z, z, fma(y, y, x * x)));
    if (rr < p.gl_rin || rr > p.gl_rout) { c.nsig = 0.f; c.kd = 0.f; return; }
    const float q = (float)(rr / p.gl_rout);
    const float w = p.gl_alpha_rho == 0.f ? 1.f : __powf(q, p.gl_alpha_rho);
    c.nsig = p.gl_nsig0 * w;
    c.kd = p.gl_kd0 * w;
    if (rr > 0.0 && p.gl_vmax != 0.f) {
        const float vm = p.gl_vmax * (p.gl_alpha_v == 1.f ? q : __powf(q, p.gl_alpha_v)) / (float)rr;
        c.vx = vm * (float)x; c.vy = vm * (float)y; c.vz = vm * (float)z;
    }
}

__device__ __forceinline__ void emit_packet_gridless(const WalkParams& p, Packet& k, unsigned long long id, uint32_t k0, uint32_t k1) {
    k.rng.init(id);
    const float4 e1 = k.rng.next4(k0, k1), e2 = k.rng.next4(k0, k1);   // (src, mu, phi, g1), (g2, tau, -, -)
    const double us = (double)e1.x;
    long long lo = 0, hi = p.n_src - 1;
    while (lo < hi) { const long long mid = (lo + hi) >> 1; if (us < p.src_cdf[mid]) hi = mid; else lo = mid + 1; }
    const float mu0 = fmaf(2.f, e1.y, -1.f);
    float sp, cp;
    sincos_uniform(e1.z, sp, cp);
    const float st0 = sqrtf(fmaxf(0.f, fmaf(-mu0, mu0, 1.f)));
    const float gauss = sqrtf(2.f * neg_log(e1.w)) * cos_uniform(e2.x);
    k.gx = (double)p.src_pos[3 * lo]; k.gy = (double)p.src_pos[3 * lo + 1]; k.gz = (double)p.src_pos[3 * lo + 2];
    ray_set_k(k.ray, st0 * cp, st0 * sp, mu0);
    k.inv_ok = false; k.stale = false;
    gl_props(p, k.gx, k.gy, k.gz, k.cell);
    k.V = dot3(k.cell.vx, k.cell.vy, k.cell.vz, k.ray.kx, k.ray.ky, k.ray.kz) + p.src_sigma[lo] * gauss;
    k.nscat = 0; k.crossings = 0; k.rej_iters = 0; k.trials = 0;
    k.tau_rem = neg_log(e2.y);
}

// One step (readings A29-A31): to the next boundary ahead but at most l_max; gas of the midpoint; interaction site linear
// within the step.  Same events as march_step; `crossings` counts steps.
__device__ __forceinline__ int march_step_gridless(const WalkParams& p, const float2* s_tab, Packet& k) {
    const double kx = (double)k.ray.kx, ky = (double)k.ray.ky, kz = (double)k.ray.kz;
    const double R = p.gl_rout;
    double db;
    bool in_gas = true;
    if (p.gl_geom == 1) {
        db = kz > 0.0 ? (R - k.gz) / kz : (kz < 0.0 ? (-R - k.gz) / kz : (double)CUDART_INF_F);
    } else {
        const double b = fma(k.gz, kz, fma(k.gy, ky, k.gx * kx));
        const double r2 = fma(k.gz, k.gz, fma(k.gy, k.gy, k.gx * k.gx));
        if (p.gl_rin == 0.0 && p.gl_lmax == CUDART_INF_F && p.gl_alpha_rho == 0.f && p.gl_vmax == 0.f) {
            // homogeneous static sphere: the gas does not depend on the step, so the interaction site s = tau / kappa is
            // known before the boundary is; (|r| + s)^2 <= R^2 is implied by r^2 + s^2 + 2 s R <= R^2: no square root
            gl_props(p, k.gx, k.gy, k.gz, k.cell);
            const float kt0 = cell_opacity(p, s_tab, k.cell, k.V, 0.f, k.hit_k2);
            if (kt0 > 0.f) {
                const double s = (double)(k.tau_rem / kt0);
                if (fma(s, s + 2.0 * R, r2) <= R * R) {
                    k.gx = fma(s, kx, k.gx); k.gy = fma(s, ky, k.gy); k.gz = fma(s, kz, k.gz);
                    k.hit_kt = kt0; k.x_in = k.V * k.cell.inv_vth; k.trials = 0u; k.line = 0;
                    return EV_HIT;
                }
            }
        }
        if (r2 < p.gl_rin * p.gl_rin) {
            in_gas = false;
            db = -b + sqrt(fmax(0.0, fma(b, b, -(r2 - p.gl_rin * p.gl_rin))));
        } else {
            db = -1.0;
            if (p.gl_rin > 0.0 && b < 0.0) {
                const double disc = fma(b, b, -(r2 - p.gl_rin * p.gl_rin));
                if (disc > 0.0) { const double t = -b - sqrt(disc); if (t >= 0.0) db = t; }
            }
            if (db < 0.0) db = -b + sqrt(fmax(0.0, fma(b, b, -(r2 - R * R))));
        }
    }
    const bool inf_step = !(db < (double)CUDART_INF_F) && p.gl_lmax == CUDART_INF_F;   // slab, k_z = 0, no limiter (A24)
    const double len = inf_step ? 0.0 : (in_gas ? fmin(db, (double)p.gl_lmax) : db);
    float kt = 0.f, vk = 0.f;
    if (in_gas) {
        gl_props(p, fma(0.5 * len, kx, k.gx), fma(0.5 * len, ky, k.gy), fma(0.5 * len, kz, k.gz), k.cell);
        vk = dot3(k.cell.vx, k.cell.vy, k.cell.vz, k.ray.kx, k.ray.ky, k.ray.kz);
        kt = cell_opacity(p, s_tab, k.cell, k.V, vk, k.hit_k2);
    }
    if (kt > 0.f && (inf_step || kt * (float)len >= k.tau_rem)) {
        const double s = (double)(k.tau_rem / kt);
        k.gx = fma(s, kx, k.gx); k.gy = fma(s, ky, k.gy); k.gz = fma(s, kz, k.gz);
        k.hit_kt = kt; k.x_in = (k.V - vk) * k.cell.inv_vth; k.trials = 0u; k.line = 0;
        return EV_HIT;
    }
    if (inf_step) return EV_CAPPED;
    k.tau_rem -= kt * (float)len;
    k.gx = fma(len, kx, k.gx); k.gy = fma(len, ky, k.gy); k.gz = fma(len, kz, k.gz);
    ++k.crossings;
    if (len >= db) {                                          // a boundary: leaving the dataset ends the packet (A31)
        if (p.gl_geom == 1) return EV_ESCAPED;
        const double rr = sqrt(fma(k.gz, k.gz, fma(k.gy, k.gy, k.gx * k.gx)));
        const double bb = fma(k.gz, kz, fma(k.gy, ky, k.gx * kx));
        const bool at_inner = p.gl_rin > 0.0 && rr < p.gl_rin * (1.0 + 1e-12);
        if (bb > 0.0 && rr >= R * (1.0 - 1e-12) && !at_inner) return EV_ESCAPED;
        const double nudge = 1e-12 * R;                       // step across the inner sphere
        k.gx = fma(nudge, kx, k.gx); k.gy = fma(nudge, ky, k.gy); k.gz = fma(nudge, kz, k.gz);
    }
    if (p.v_max > 0.f && fabsf(k.V) > p.v_max) return EV_TERMINATED;
    if (k.crossings >= p.max_crossings) return EV_CAPPED;
    return EV_CROSSED;
}

// The random numbers of one FINISH, turned into what the event needs.  Draws: (tau, mu, phi, perp1), (perp2, dust, mix, -).
struct FinDraws {
    float tau_next;              // -ln s1.x
    float r_mu, mu_dip;          // s1.y, and dipole_mu(s1.y) if computed ahead
    float sphi, cphi;            // azimuth of k'
    float nl_p1, spsi, cpsi;     // u_perp: -ln s1.w, angle 2 pi s2.x
    float u_dust, u_mix, u_alb;  // s2.y, s2.z, s2.w
};

__device__ __forceinline__ FinDraws fin_draws(const float4 s1, const float4 s2) {
    FinDraws d;
    d.tau_next = neg_log(s1.x);
    d.r_mu = s1.y; d.mu_dip = 0.f;
    sincos_uniform(s1.z, d.sphi, d.cphi);
    d.nl_p1 = neg_log(s1.w);
    sincos_uniform(s2.x, d.spsi, d.cpsi);
    d.u_dust = s2.y; d.u_mix = s2.z; d.u_alb = s2.w;
    return d;
}

// Doublet: the interaction is drawn at the site, before the u_par trials, because they need the line's own x and a
// (interaction i with probability tau_i / tau): u kappa < kappa_dust -> dust, < kappa_dust + kappa_1 -> line 1,
// else line 2, whose frequencies are measured from ITS centre.
__device__ __forceinline__ void select_line(const WalkParams& p, Packet& k, float u) {
    const float t = u * k.hit_kt;
    if (p.has_dust && t < k.cell.kd) { k.line = -1; return; }
    if (t >= k.hit_kt - k.hit_k2) { k.line = 1; k.x_in = fmaf(-p.db_dv, k.cell.inv_vth, k.x_in); }
    else k.line = 0;
}
template <bool DB = true>
__device__ __forceinline__ float line_a(const WalkParams& p, const Packet& k) { return (DB && k.line > 0) ? k.cell.a * p.db_ra : k.cell.a; }

// a7, a9-a12: the interaction itself (PAPER.md 2.3.1): dust or line, u_perp (Eq. 5, core-skipping
// PAPER.md:244), phase function, rotation, Eq. 7 with the recoil dropped, peel-off
// before k' is adopted, new tau_target.  Returns EV_ABSORBED / EV_TERMINATED / EV_CAPPED / EV_SCATTERED.
// FIN: the event compiled for the run's core-skipping mode and phase functions (run constants whose tests are uniform branches,
// a handful per scattering): 0 = generic (read from the options), 1 / 2 / 3 = isotropic scattering in core and wing with
// core-skipping mode 1 / 2 / 0, 4 = BASELINE.json config 3's combination: dipole core, isotropic wing, split on the atom-frame
// frequency, core-skipping mode 1.
template <bool HUBBLE, bool PEEL, bool PRE, int PMODE = PEEL_INLINE, bool DB = true, int FIN = 0>
__device__ __forceinline__ int finish_scatter(const WalkParams& p, const float2* s_tab, Packet& k, const FinDraws& d,
                                              uint32_t& peel_rays, uint32_t& peel_cells, bool add, PeelPend* pend = nullptr,
                                              float* xc_cache = nullptr) {
    const float kx = k.ray.kx, ky = k.ray.ky, kz = k.ray.kz;
    const Cell& c = k.cell;
    // (a run without dust has kd = 0 in every cell, and u kappa < 0 is never true: the has_dust flag need not be read)
    if ((DB && p.doublet_on) ? (p.has_dust && k.line < 0) : (d.u_dust * k.hit_kt < c.kd)) {
        // dust (PAPER.md 2.3.2): scattered with probability albedo (Eq. 8) into the Henyey-Greenstein phase function (Eq. 9),
        // coherently in the bulk frame of the cell (grains are heavy and move with the gas, reading A33); else destroyed
        if (!(p.dust_albedo > 0.f) || !(d.u_alb < p.dust_albedo)) return EV_ABSORBED;
        const float mu = hg_mu(p.dust_g, d.r_mu);
        float e1[3], e2[3];
        ortho_basis(kx, ky, kz, e1, e2);
        const float vk = dot3(c.vx, c.vy, c.vz, kx, ky, kz);
        if (PEEL) {
            const float mu_o = dot3(kx, ky, kz, p.kobs[0], p.kobs[1], p.kobs[2]);
            ++peel_rays;
            peel_ray<HUBBLE, PMODE>(p, s_tab, k.ray, c, k.V - vk + dot3(c.vx, c.vy, c.vz, p.kobs[0], p.kobs[1], p.kobs[2]),
                                  hg_value(p.dust_g, mu_o), peel_cells, add, pend);
        }
        const float st = sqrtf(fmaxf(0.f, fmaf(-mu, mu, 1.f)));
        float nx = fmaf(st, fmaf(d.cphi, e1[0], d.sphi * e2[0]), mu * kx);
        float ny = fmaf(st, fmaf(d.cphi, e1[1], d.sphi * e2[1]), mu * ky);
        float nz = fmaf(st, fmaf(d.cphi, e1[2], d.sphi * e2[2]), mu * kz);
        const float inv = rsqrtf(dot3(nx, ny, nz, nx, ny, nz));
        nx *= inv; ny *= inv; nz *= inv;
        ray_set_k(k.ray, nx, ny, nz);
        if (HUBBLE) { ray_set_inv(k.ray); k.inv_ok = true; } else k.inv_ok = false;
        k.V = k.V - vk + dot3(c.vx, c.vy, c.vz, nx, ny, nz);
        k.tau_rem = d.tau_next;
        return EV_DUST_SCATTERED;
    }
    const float dv_line = (DB && k.line > 0) ? p.db_dv : 0.f;             // frequencies of this event are relative to its line
    const float a_l = line_a<DB>(p, k);
    // x_crit depends on the run and, in local mode, on the cell (and the line of a doublet): the cooperative drain, whose
    // packet scatters ~1e5 times per cell, keeps it between scatterings (xc_cache < 0 = not yet known for this cell; the mode
    // tests and the cube root are ~200 cycles of a lone packet's serial chain)
    constexpr int CS = (FIN == 1 || FIN == 4) ? 1 : FIN == 2 ? 2 : FIN == 3 ? 0 : -1;
    constexpr bool ISO = FIN >= 1 && FIN <= 3;
    const int cs_mode = CS >= 0 ? CS : p.core_skip_mode;
    float x_crit = 0.f;
    if (!DB && xc_cache && *xc_cache >= 0.f) x_crit = *xc_cache;
    else {
        if (cs_mode == 1) x_crit = p.x_crit;
        else if (cs_mode == 2) {              // local: a tau_0 over half a cell (reading A7)
            const float atau = a_l * c.nsig * ((DB && k.line > 0) ? p.db_rs : 1.f) * 0.5f;
            x_crit = atau >= 1.f ? 0.2f * cbrtf(atau) : 0.f;
        }
        if (!DB && xc_cache) *xc_cache = x_crit;
    }
    float up1, up2;
    uperp_from(k.x_in, x_crit, d.nl_p1, d.spsi, d.cpsi, up1, up2);
    const float xsel = (FIN == 4 || p.phase_frame == 0) ? fabsf(k.x_in - k.upar) : fabsf(k.x_in);
    const int phase = ISO ? 0 : FIN == 4 ? (xsel > p.phase_split_x ? 0 : 1) : (xsel > p.phase_split_x ? p.phase_wing : p.phase_core);
    bool is_dipole;
    const float mu = sample_mu<PRE>(phase, d.u_mix, d.r_mu, d.mu_dip, is_dipole);
    float e1[3], e2[3];
    ortho_basis(kx, ky, kz, e1, e2);
    const float xa = k.x_in - k.upar;                 // atom-frame frequency
    if (PEEL) {                                       // a12, before adopting k'
        const float mu_o = dot3(kx, ky, kz, p.kobs[0], p.kobs[1], p.kobs[2]);
        const float e1o = dot3(e1[0], e1[1], e1[2], p.kobs[0], p.kobs[1], p.kobs[2]);
        const float e2o = dot3(e2[0], e2[1], e2[2], p.kobs[0], p.kobs[1], p.kobs[2]);
        const float x_o = fmaf(up2, e2o, fmaf(up1, e1o, fmaf(k.upar, mu_o, xa)));
        const float V_o = fmaf(x_o, c.vth, dot3(c.vx, c.vy, c.vz, p.kobs[0], p.kobs[1], p.kobs[2])) + dv_line;
        ++peel_rays;
        // mix: the sampled branch weights the ray (unbiased; reading A27)
        peel_ray<HUBBLE, PMODE>(p, s_tab, k.ray, c, V_o, is_dipole ? 0.75f * fmaf(mu_o, mu_o, 1.f) : 1.f, peel_cells, add, pend);
    }
    const float st = sqrtf(fmaxf(0.f, fmaf(-mu, mu, 1.f)));
    float nx = fmaf(st, fmaf(d.cphi, e1[0], d.sphi * e2[0]), mu * kx);
    float ny = fmaf(st, fmaf(d.cphi, e1[1], d.sphi * e2[1]), mu * ky);
    float nz = fmaf(st, fmaf(d.cphi, e1[2], d.sphi * e2[2]), mu * kz);
    const float inv = rsqrtf(dot3(nx, ny, nz, nx, ny, nz));
    nx *= inv; ny *= inv; nz *= inv;
    // a11, Eq. 7, recoil dropped: x_out = x_in + u.(k_out - k_in)
    const float x_out = fmaf(st, fmaf(up1, d.cphi, up2 * d.sphi), fmaf(k.upar, mu, xa));
    // With Hubble drift every march needs the DDA step, hence 1/k: made here, where the three reciprocals (~270 cycles of
    // MUFU + rounding fix-up) overlap the rest of the event instead of heading the next march; a static walk makes them
    // only when a segment actually reaches a face
    ray_set_k(k.ray, nx, ny, nz);
    if (HUBBLE) { ray_set_inv(k.ray); k.inv_ok = true; } else k.inv_ok = false;
    k.V = fmaf(x_out, c.vth, dot3(c.vx, c.vy, c.vz, nx, ny, nz)) + dv_line;
    ++k.nscat;
    if (fabsf(k.V) > p.v_max_or_inf) return EV_TERMINATED;     // +inf when there is no v_max
    if (k.nscat >= p.max_scatter_or_max || !(fabsf(k.V) <= 3.0e38f)) return EV_CAPPED;   // cap (2^32 - 1 when there is none), or fail-safe: non-finite V
    k.tau_rem = d.tau_next;
    return EV_SCATTERED;
}

}  // namespace thor
