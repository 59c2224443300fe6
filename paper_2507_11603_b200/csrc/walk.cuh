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

enum : int { LS_IDLE = 0, LS_MARCH = 1, LS_TRIAL = 2, LS_FINISH = 3, LS_OUT = 4 };

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

// a6/a7: optical depth of one segment of length len (cell units) starting at velocity offset V0, or the distance
// s_hit at which tau_need is reached (linear within the step).  Without Hubble drift: kappa len.
// With drift Hc (km/s per cell length): sub-steps per reading A12 — n_sub = 1 if min|x| over the segment > 6 else
// ceil(|dV| / (eps v_th)), midpoint rule.  Returns true on interaction; k_tot is the opacity there.
template <bool HUBBLE>
__device__ __forceinline__ bool integrate_segment(const WalkParams& p, const float2* s_tab, const Cell& c, float V0,
                                                  float vk, float len, float tau_need, float& tau_out, float& s_hit,
                                                  float& k_tot) {
    tau_out = 0.f; s_hit = 0.f; k_tot = 0.f;
    if (c.nsig <= 0.f && c.kd <= 0.f) return false;
    if (!HUBBLE) {
        const float kl = c.nsig > 0.f ? c.nsig * voigt_H(s_tab, c.a, (V0 - vk) * c.inv_vth) : 0.f;
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
        const float xa = (V0 - vk) * c.inv_vth, xb = (V0 - Hc * len - vk) * c.inv_vth;
        const float minabs = xa * xb <= 0.f ? 0.f : fminf(fabsf(xa), fabsf(xb));
        if (minabs <= 6.f) {
            const float q = ceilf(fabsf(Hc * len) * c.inv_vth / p.hubble_eps);
            nsub = q < 1.f ? 1 : (q > 1e6f ? 1000000 : (int)q);
        }
    }
    const float ds = len / (float)nsub;
    float tau = 0.f;
    for (int j = 0; j < nsub; ++j) {
        const float Vmid = Hc != 0.f ? V0 - Hc * ((float)j + 0.5f) * ds : V0;   // no 0 * inf when ds = +inf (A24)
        const float kl = c.nsig > 0.f ? c.nsig * voigt_H(s_tab, c.a, (Vmid - vk) * c.inv_vth) : 0.f;
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
__device__ __forceinline__ float cell_opacity(const float2* s_tab, const Cell& c, float V, float vk) {
    const float kl = c.nsig > 0.f ? c.nsig * voigt_H(s_tab, c.a, (V - vk) * c.inv_vth) : 0.f;
    return kl + c.kd;
}

// a12 peel-off: w = P^ exp(-tau_obs), tau_obs integrated from `at` along k_obs to the box face at
// velocity offset V_o by the same march (a4-a6), dropped beyond tau_peel_max (reading A13); added to
// (pixel of the starting point projected perpendicular to k_obs, spectral bin of dv = -V at the box face).
template <bool HUBBLE>
__device__ __noinline__ void peel_ray(const WalkParams& p, const float2* s_tab, const Ray& at, float V_o, float phat,
                                      uint32_t& n_cells) {
    const float px0 = (float)at.cx + at.fx - 0.5f * (float)p.g.nx;
    const float py0 = (float)at.cy + at.fy - 0.5f * (float)p.g.ny;
    const float pz0 = (float)at.cz + at.fz - 0.5f * (float)p.g.nz;
    const float px = ((px0 * p.img1[0] + py0 * p.img1[1] + pz0 * p.img1[2]) * p.peel_inv_width + 0.5f) * (float)p.peel_nx;
    const float py = ((px0 * p.img2[0] + py0 * p.img2[1] + pz0 * p.img2[2]) * p.peel_inv_width + 0.5f) * (float)p.peel_ny;
    if (!(px >= 0.f && px < (float)p.peel_nx && py >= 0.f && py < (float)p.peel_ny)) return;
    Ray r = at;
    ray_set_direction(r, p.kobs[0], p.kobs[1], p.kobs[2]);
    float tau = 0.f, V = V_o;
    for (;;) {
        float len;
        const int ex = dda_next_face(r, p.g, len);
        if (!(len < CUDART_INF_F)) return;                    // reading A24: never reaches a box face -> dropped
        const Cell c = load_cell(p, dda_linear(r, p.g));
        const float vk = c.vx * r.kx + c.vy * r.ky + c.vz * r.kz;
        float dtau, s_hit, kt;
        integrate_segment<HUBBLE>(p, s_tab, c, V, vk, len, 3.0e38f, dtau, s_hit, kt);
        tau += dtau;
        if (HUBBLE) V -= p.hubble * len;
        ++n_cells;
        if (tau > p.tau_peel_max) return;
        // peel rays leave through the first box face they meet, periodic or not
        const float ke = ex == 0 ? r.kx : ex == 1 ? r.ky : r.kz;
        const int cn = (ex == 0 ? r.cx : ex == 1 ? r.cy : r.cz) + (ke > 0.f ? 1 : -1);
        const int nn = ex == 0 ? p.g.nx : ex == 1 ? p.g.ny : p.g.nz;
        if (cn < 0 || cn >= nn) break;
        dda_cross(r, p.g, ex, len);
    }
    const int iv = (int)floorf((-V - p.peel_v_lo) * p.peel_inv_dv);
    if (iv < 0 || iv >= p.peel_nv) return;
    const float w = phat * __expf(-tau);
    const unsigned long long q = (unsigned long long)__float2ull_rn(w * (float)CUBE_FIXED_SCALE);
    if (q) atomicAdd(p.cube + ((size_t)(int)py * p.peel_nx + (int)px) * p.peel_nv + iv, q);
}

}  // namespace thor
