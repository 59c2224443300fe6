// ORACLE — TEST INFRASTRUCTURE ONLY (see constants.hpp).
// Flat C entry points so that tests/ (and bench.py's cpu_baseline leg) can call the oracle through ctypes.
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fPIC -shared capi.cpp -o liboracle.so   (oracle/build.py)
#include <cstring>
#include <chrono>
#include "walker.hpp"
#include "gridless.hpp"

using namespace orc;

static inline uint64_t fnv_word(uint64_t h, uint64_t w) { return (h ^ w) * 0x100000001B3ull; }

template <class Real>
static void trace_rays(const GridDims& g, int64_t n, const float* org, const float* dir, int64_t max_steps,
                       uint64_t* hash_idx, uint64_t* hash_len, uint32_t* count, int64_t* seq_idx, double* seq_len) {
    for (int64_t i = 0; i < n; ++i) {
        Ray<Real> r;
        const Real pos[3] = {(Real)org[3 * i], (Real)org[3 * i + 1], (Real)org[3 * i + 2]};
        const Real kk[3] = {(Real)dir[3 * i], (Real)dir[3 * i + 1], (Real)dir[3 * i + 2]};
        dda_locate(r, g, pos);
        r.set_direction(kk);
        uint64_t hi = 0xCBF29CE484222325ull, hl = 0xCBF29CE484222325ull;
        uint32_t cnt = 0;
        for (int64_t s = 0; s < max_steps; ++s) {
            Real len;
            const int ex = dda_next_face(r, g, len);
            const int64_t lin = g.linear(r.c);
            hi = fnv_word(hi, (uint64_t)lin);
            uint64_t bits = 0;
            if (sizeof(Real) == 4) { float fl = (float)len; uint32_t b; std::memcpy(&b, &fl, 4); bits = b; }
            else { double dl = (double)len; std::memcpy(&bits, &dl, 8); }
            hl = fnv_word(hl, bits);
            if (seq_idx) seq_idx[cnt] = lin;
            if (seq_len) seq_len[cnt] = (double)len;
            ++cnt;
            if (!dda_cross(r, g, ex, len)) break;
        }
        hash_idx[i] = hi; hash_len[i] = hl; count[i] = cnt;
    }
}

extern "C" {

// ---- constants ----
double orc_vth_kms(double T) { return vth_kms(T); }
double orc_voigt_a(double T) { return voigt_a(T); }
double orc_sigma0_cm2(double T) { return sigma0_cm2(T); }

// ---- Philox ----
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const Philox4 r = philox4x32_10(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1]);
    std::memcpy(out, r.v, sizeof r.v);
}
// first n u32 draws of packet `id` under `seed`
void orc_draws_u32(uint64_t seed, uint64_t id, int64_t n, uint32_t* out) {
    DrawStream s(seed, id);
    for (int64_t i = 0; i < n; ++i) out[i] = s.next_u32();
}
double orc_u32_to_uniform(uint32_t r) { return u32_to_uniform(r); }

// ---- Voigt ----
double orc_dawson(double x) { return dawson(x); }
double orc_voigt_H(double a, double x) { return voigt_H(a, x); }
void orc_voigt_H_array(int64_t n, const double* a, const double* x, double* out) {
    for (int64_t i = 0; i < n; ++i) out[i] = voigt_H(a[i], x[i]);
}
double orc_x_cw_exact(double a) { return x_cw_exact(a); }
double orc_x_cw_b25(double a) { return x_cw_b25(a); }

// ---- samplers ----
// n draws of u_par at fixed (a, x), one packet stream per call; iters_out receives the total iteration count.
// which: 0 = sample_upar (production choice), 1 = force Eq. 10 loop, 2 = force far-wing scheme.
void orc_sample_upar(double a, double x, uint64_t seed, uint64_t id, int64_t n, int which, double* out,
                     uint64_t* iters_out) {
    DrawStream s(seed, id);
    uint64_t it = 0;
    for (int64_t i = 0; i < n; ++i)
        out[i] = which == 1 ? upar_zm02(a, x, s, &it) : which == 2 ? upar_far(a, x, s, &it) : sample_upar(a, x, s, &it);
    if (iters_out) *iters_out = it;
}
double orc_upar_pdf(double a, double x, double u) { return upar_pdf(a, x, u); }
double orc_upar_u0(double a, double x) { return upar_u0(a, x); }
void orc_sample_uperp(double x_in, double x_crit, uint64_t seed, uint64_t id, int64_t n, double* out1, double* out2) {
    DrawStream s(seed, id);
    for (int64_t i = 0; i < n; ++i) sample_uperp(x_in, x_crit, s, out1[i], out2[i]);
}
void orc_sample_mu(int phase, uint64_t seed, uint64_t id, int64_t n, double* out) {
    DrawStream s(seed, id);
    for (int64_t i = 0; i < n; ++i) out[i] = sample_mu(phase, s, nullptr);
}
double orc_dipole_mu(double r) { return dipole_mu(r); }
double orc_hg_mu(double g, double r) { return hg_mu(g, r); }
double orc_hg_value(double g, double mu) { return hg_value(g, mu); }

// One full scattering at gas-frame x_in for direction k_in = +z: returns x_out and k_out (for pins P9/P10).
void orc_scatter_once(double a, double x_in, double x_crit, int phase, uint64_t seed, uint64_t id, int64_t n,
                      double* x_out, double* k_out /* [n][3] */) {
    DrawStream s(seed, id);
    for (int64_t i = 0; i < n; ++i) {
        const double k[3] = {0, 0, 1};
        const double upar = sample_upar(a, x_in, s, nullptr);
        double up1, up2;
        sample_uperp(x_in, x_crit, s, up1, up2);
        const double mu = sample_mu(phase, s, nullptr);
        const double phi = 2.0 * PI * s.uniform();
        double e1[3], e2[3];
        ortho_basis(k, e1, e2);
        const double st = std::sqrt(std::fmax(0.0, 1.0 - mu * mu));
        for (int c = 0; c < 3; ++c) k_out[3 * i + c] = mu * k[c] + st * (std::cos(phi) * e1[c] + std::sin(phi) * e2[c]);
        x_out[i] = x_in - upar + upar * mu + st * (up1 * std::cos(phi) + up2 * std::sin(phi));
    }
}

// ---- DDA ----
// Trace n rays through an (nx,ny,nz) grid.  Origins in cell units, directions as given (not renormalised).
// real32 != 0: the fp32 specification (bit-exact reference for the GPU); else the fp64 twin.
// Per ray: hash_idx = word-wise FNV-1a over the 64-bit linear indices of the visited cells (starting cell first),
// hash_len = the same over the bit patterns of the segment lengths, count = number of cells visited.
// Stops on leaving the grid or after max_steps cells.  If seq_out != NULL (n must be 1), the visited indices and
// lengths are written there (up to max_steps).
void orc_dda_trace(int nx, int ny, int nz, int px, int py, int pz, int64_t n, const float* org, const float* dir,
                   int64_t max_steps, int real32, uint64_t* hash_idx, uint64_t* hash_len, uint32_t* count,
                   int64_t* seq_idx, double* seq_len) {
    GridDims g{{nx, ny, nz}, {px != 0, py != 0, pz != 0}};
    if (real32) trace_rays<float>(g, n, org, dir, max_steps, hash_idx, hash_len, count, seq_idx, seq_len);
    else trace_rays<double>(g, n, org, dir, max_steps, hash_idx, hash_len, count, seq_idx, seq_len);
}

// ---- the walk ----
struct orc_opts_c {
    int32_t phase_core, phase_wing, phase_frame;
    double phase_split_x;
    int32_t core_skip_mode;
    double x_crit;
    int32_t spec_mode;
    double spec_T_ref;
    int32_t spec_bins;
    double spec_lo, spec_hi;
    double hubble_kms_per_cell, hubble_eps, v_max_kms;
    int32_t peel_on;
    double k_obs[3];
    int32_t peel_nx, peel_ny, peel_nv;
    double peel_v_lo, peel_v_hi, peel_width_cells, tau_peel_max;
    uint64_t photon_id_offset, max_scatter, max_crossings;
    double dust_albedo, dust_g;
    int32_t doublet_on;
    double doublet_dv_kms, doublet_sigma_ratio, doublet_a_ratio;
};

// Outputs (any may be NULL): spectrum u64[spec_bins+2], nscat_hist u64[64], counters u64[10],
// cube f64[peel_ny*peel_nx*peel_nv], raw: RawRecord[n_photons] (24 bytes each).  Returns seconds of wall time
// spent in the walk itself.
double orc_run(int nx, int ny, int nz, int px, int py, int pz, double cell_cm,
               const float* nHI, const float* T, const float* vx, const float* vy, const float* vz, const float* kdust,
               int64_t n_src, const float* src_pos, const float* src_lum, const float* src_sigma,
               const orc_opts_c* oc, uint64_t n_photons, uint64_t seed,
               uint64_t* spectrum, uint64_t* nscat_hist, uint64_t* counters, double* cube, void* raw) {
    Grid g{{{nx, ny, nz}, {px != 0, py != 0, pz != 0}}, cell_cm, nHI, T, vx, vy, vz, kdust};
    Sources s{n_src, src_pos, src_lum, src_sigma, {}};
    Opts o;
    o.phase_core = oc->phase_core; o.phase_wing = oc->phase_wing; o.phase_frame = oc->phase_frame;
    o.phase_split_x = oc->phase_split_x; o.core_skip_mode = oc->core_skip_mode; o.x_crit = oc->x_crit;
    o.spec_mode = oc->spec_mode; o.spec_T_ref = oc->spec_T_ref; o.spec_bins = oc->spec_bins;
    o.spec_lo = oc->spec_lo; o.spec_hi = oc->spec_hi;
    o.hubble_kms_per_cell = oc->hubble_kms_per_cell; o.hubble_eps = oc->hubble_eps; o.v_max_kms = oc->v_max_kms;
    o.peel_on = oc->peel_on;
    for (int i = 0; i < 3; ++i) o.k_obs[i] = oc->k_obs[i];
    o.peel_nx = oc->peel_nx; o.peel_ny = oc->peel_ny; o.peel_nv = oc->peel_nv;
    o.peel_v_lo = oc->peel_v_lo; o.peel_v_hi = oc->peel_v_hi; o.peel_width_cells = oc->peel_width_cells;
    o.tau_peel_max = oc->tau_peel_max;
    o.photon_id_offset = oc->photon_id_offset; o.max_scatter = oc->max_scatter; o.max_crossings = oc->max_crossings;
    o.dust_albedo = oc->dust_albedo; o.dust_g = oc->dust_g; o.doublet_on = oc->doublet_on;
    o.doublet_dv_kms = oc->doublet_dv_kms; o.doublet_sigma_ratio = oc->doublet_sigma_ratio; o.doublet_a_ratio = oc->doublet_a_ratio;
    Walker w(g, s, o);
    Result res;
    const auto t0 = std::chrono::steady_clock::now();
    w.run(n_photons, seed, res, raw != nullptr);
    const auto t1 = std::chrono::steady_clock::now();
    if (spectrum) std::memcpy(spectrum, res.spectrum.data(), res.spectrum.size() * 8);
    if (nscat_hist) std::memcpy(nscat_hist, res.nscat_hist, sizeof res.nscat_hist);
    if (counters) std::memcpy(counters, res.counters, sizeof res.counters);
    if (cube && !res.cube.empty()) std::memcpy(cube, res.cube.data(), res.cube.size() * 8);
    if (raw) std::memcpy(raw, res.raw.data(), res.raw.size() * sizeof(RawRecord));
    return std::chrono::duration<double>(t1 - t0).count();
}

// The same walk through a gridless dataset (gridless.hpp; PAPER.md 3.3): geometry 0 = shell / sphere, 1 = slab.
double orc_run_gridless(int geometry, double r_in, double r_out, double length_cm, double n0, double alpha_rho, double T,
                        double v_max, double alpha_v, double kdust0, double step_f,
                        int64_t n_src, const float* src_pos, const float* src_lum, const float* src_sigma,
                        const orc_opts_c* oc, uint64_t n_photons, uint64_t seed,
                        uint64_t* spectrum, uint64_t* nscat_hist, uint64_t* counters, void* raw) {
    Gridless d{geometry, r_in, r_out, length_cm, n0, alpha_rho, T, v_max, alpha_v, kdust0, step_f};
    Sources s{n_src, src_pos, src_lum, src_sigma, {}};
    Opts o;
    o.phase_core = oc->phase_core; o.phase_wing = oc->phase_wing; o.phase_frame = oc->phase_frame;
    o.phase_split_x = oc->phase_split_x; o.core_skip_mode = oc->core_skip_mode; o.x_crit = oc->x_crit;
    o.spec_mode = oc->spec_mode; o.spec_T_ref = oc->spec_T_ref; o.spec_bins = oc->spec_bins;
    o.spec_lo = oc->spec_lo; o.spec_hi = oc->spec_hi; o.v_max_kms = oc->v_max_kms;
    o.photon_id_offset = oc->photon_id_offset; o.max_scatter = oc->max_scatter; o.max_crossings = oc->max_crossings;
    o.dust_albedo = oc->dust_albedo; o.dust_g = oc->dust_g;
    GridlessWalker w(d, s, o);
    Result res;
    const auto t0 = std::chrono::steady_clock::now();
    w.run(n_photons, seed, res, raw != nullptr);
    const auto t1 = std::chrono::steady_clock::now();
    if (spectrum) std::memcpy(spectrum, res.spectrum.data(), res.spectrum.size() * 8);
    if (nscat_hist) std::memcpy(nscat_hist, res.nscat_hist, sizeof res.nscat_hist);
    if (counters) std::memcpy(counters, res.counters, sizeof res.counters);
    if (raw) std::memcpy(raw, res.raw.data(), res.raw.size() * sizeof(RawRecord));
    return std::chrono::duration<double>(t1 - t0).count();
}

// Ray-tracing operators (PAPER.md 3.5), one ray at a time in fp64 on the DDA's fp64 twin: projection Q = Int q w ds
// (PAPER.md 3.5.1: column density with q = n_HI, w = 1; weighted mean Q / Q^ with q = T, w = n_HI) and the absorption
// spectrum of Eq. 11 (PAPER.md 3.5.2): tau(V_j) = Int n sigma(nu(s), T) ds, the gas seeing the frequency shifted by
// its line-of-sight velocity and the Hubble term Hc * s (s in cells; midpoint of each face-to-face segment), with
// piecewise-constant cells.  Rays run from their origin to the first box face.
void orc_raytrace(int nx, int ny, int nz, double cell_cm, const float* nHI, const float* T, const float* vx,
                  const float* vy, const float* vz, const float* kdust, int64_t n_rays, const float* org,
                  const float* dir, double hubble, int n_v, double v_lo, double v_hi, double* out_column,
                  double* out_tmean, double* out_tau) {
    Grid g{{{nx, ny, nz}, {false, false, false}}, cell_cm, nHI, T, vx, vy, vz, kdust};
    for (int64_t i = 0; i < n_rays; ++i) {
        Ray<double> r;
        const double pos[3] = {org[3 * i], org[3 * i + 1], org[3 * i + 2]};
        dda_locate(r, g.dims, pos);
        const double k[3] = {dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]};
        r.set_direction(k);
        double col = 0, tn = 0, s_path = 0;
        if (out_tau) for (int j = 0; j < n_v; ++j) out_tau[i * n_v + j] = 0.0;
        for (;;) {
            double len;
            const int ex = dda_next_face(r, g.dims, len);
            if (std::isinf(len)) break;
            const CellProps cp = fetch_cell(g, r.c);
            col += cp.n * len;
            tn += cp.n * cp.T * len;
            if (out_tau && (cp.n > 0 || cp.kd > 0)) {
                const double vgas = dot3(cp.v, k) + hubble * (s_path + 0.5 * len);
                const double vth = vth_kms(cp.T), a = voigt_a(cp.T);
                for (int j = 0; j < n_v; ++j) {
                    const double V = v_lo + (j + 0.5) * (v_hi - v_lo) / n_v;
                    const double kl = cp.n > 0 ? cp.n * sigma0_cm2(cp.T) * voigt_H(a, (V - vgas) / vth) * cell_cm : 0.0;
                    out_tau[i * n_v + j] += (kl + cp.kd * cell_cm) * len;
                }
            }
            s_path += len;
            const int s = r.k[ex] > 0 ? 1 : -1;
            const int cn = r.c[ex] + s;
            if (cn < 0 || cn >= g.dims.n[ex]) break;
            dda_cross(r, g.dims, ex, len);
        }
        if (out_column) out_column[i] = col * cell_cm;
        if (out_tmean) out_tmean[i] = col > 0 ? tn / col : 0.0;
    }
}

// Sight lines as the paper draws them for the Lyα forest ("periodic boundary conditions", cells sub-sampled
// "such that each ray step corresponds to a Hubble induced velocity-shift much smaller than the line width"): the ray
// wraps at the periodic faces given and ends after max_len cell lengths (or at the first non-periodic face; max_len <= 0:
// first box face as orc_raytrace); with hubble_eps > 0 each face-to-face segment is cut into
// n_sub = ceil(|Hc len| / (hubble_eps v_th(T_cell))) sub-steps (the rule of reading A12), the gas frequency evaluated at
// each sub-step's midpoint.
void orc_raytrace_ex(int nx, int ny, int nz, int px, int py, int pz, double cell_cm, const float* nHI, const float* T,
                     const float* vx, const float* vy, const float* vz, const float* kdust, int64_t n_rays, const float* org,
                     const float* dir, double hubble, double hubble_eps, double max_len, int n_v, double v_lo, double v_hi,
                     double* out_column, double* out_tmean, double* out_tau) {
    const bool wrap = max_len > 0;
    Grid g{{{nx, ny, nz}, {wrap && px != 0, wrap && py != 0, wrap && pz != 0}}, cell_cm, nHI, T, vx, vy, vz, kdust};
    for (int64_t i = 0; i < n_rays; ++i) {
        Ray<double> r;
        const double pos[3] = {org[3 * i], org[3 * i + 1], org[3 * i + 2]};
        dda_locate(r, g.dims, pos);
        const double k[3] = {dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]};
        r.set_direction(k);
        double col = 0, tn = 0, s_path = 0;
        if (out_tau) for (int j = 0; j < n_v; ++j) out_tau[i * n_v + j] = 0.0;
        for (;;) {
            double len;
            const int ex = dda_next_face(r, g.dims, len);
            if (std::isinf(len) && !wrap) break;
            bool last = false;
            if (wrap && s_path + len >= max_len) { len = max_len - s_path; last = true; }
            const CellProps cp = fetch_cell(g, r.c);
            col += cp.n * len;
            tn += cp.n * cp.T * len;
            if (out_tau && (cp.n > 0 || cp.kd > 0) && len > 0) {
                const double vth = vth_kms(cp.T), a = voigt_a(cp.T);
                int nsub = 1;
                if (hubble_eps > 0 && hubble != 0 && cp.n > 0) {
                    const double q = std::ceil(std::fabs(hubble * len) / (hubble_eps * vth));
                    nsub = q < 1.0 ? 1 : (q > 1e6 ? 1000000 : (int)q);
                }
                const double ds = len / nsub;
                for (int m = 0; m < nsub; ++m) {
                    const double vgas = dot3(cp.v, k) + hubble * (s_path + (m + 0.5) * ds);
                    for (int j = 0; j < n_v; ++j) {
                        const double V = v_lo + (j + 0.5) * (v_hi - v_lo) / n_v;
                        const double kl = cp.n > 0 ? cp.n * sigma0_cm2(cp.T) * voigt_H(a, (V - vgas) / vth) * cell_cm : 0.0;
                        out_tau[i * n_v + j] += (kl + cp.kd * cell_cm) * ds;
                    }
                }
            }
            s_path += len;
            if (last) break;
            if (!dda_cross(r, g.dims, ex, len)) break;     // left through a non-periodic face
        }
        if (out_column) out_column[i] = col * cell_cm;
        if (out_tmean) out_tmean[i] = col > 0 ? tn / col : 0.0;
    }
}

// Pins of orc_raytrace and orc_volume_render (tests/test_oracle_raytrace.py), none through this file's DDA or Voigt:
// density x analytic chord, two-slab weighted mean, N sigma_0 H by scipy's Faddeeva function with a bulk-velocity shift,
// Hubble-swept line against adaptive quadrature; volume rendering: c (1 - e^{-mu L}) in a uniform medium, two slabs seen
// from either end (order of attenuation), nested adaptive quadrature of Eq. 12 on a random 6^3 grid with fields looked
// up by floor(position).  The transfer function itself is the caller's and is restated in the test.
//
// Volume rendering (PAPER.md 3.5.3, Eq. 12): C = Int_0^L c(s) mu(s) exp(-Int_0^s mu dt) ds along each ray, observer at
// the ray origin.  Transfer function as in PAPER.md:510 (Gaussian peaks in log10 T, brightness weighted by density):
// g_p = exp(-(log10 T - c_p)^2 / (2 s_p^2)); mu = w Sum_p A_p g_p per cell length, c mu = w Sum_p A_p g_p (R,G,B)_p,
// w = n_HI / n_ref (n_ref > 0) or 1 (n_ref = 0).  Cells are piecewise constant, so each face-to-face
// segment of length l integrates exactly: C += Tr c (1 - e^{-mu l}), Tr *= e^{-mu l} (reading A25).  Output per ray:
// (C_R, C_G, C_B, 1 - Tr).  peaks: double[n_peaks][6] = {c_p, s_p, R, G, B, A}.
void orc_volume_render(int nx, int ny, int nz, const float* nHI, const float* T, int64_t n_rays, const float* org,
                       const float* dir, int n_peaks, const double* peaks, double n_ref, double* out_rgba) {
    Grid g{{{nx, ny, nz}, {false, false, false}}, 1.0, nHI, T, nullptr, nullptr, nullptr, nullptr};
    for (int64_t i = 0; i < n_rays; ++i) {
        Ray<double> r;
        const double pos[3] = {org[3 * i], org[3 * i + 1], org[3 * i + 2]};
        dda_locate(r, g.dims, pos);
        const double k[3] = {dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]};
        r.set_direction(k);
        double C[3] = {0, 0, 0}, Tr = 1.0;
        for (;;) {
            double len;
            const int ex = dda_next_face(r, g.dims, len);
            if (std::isinf(len)) break;
            const int64_t idx = ((int64_t)r.c[2] * ny + r.c[1]) * nx + r.c[0];
            const double n = nHI[idx], Tc = T[idx];
            const double w = n_ref > 0 ? n / n_ref : 1.0;
            if (w > 0 && Tc > 0) {
                const double lt = std::log10(Tc);
                double mu = 0, e[3] = {0, 0, 0};
                for (int p = 0; p < n_peaks; ++p) {
                    const double* q = peaks + 6 * p;
                    const double z = (lt - q[0]) / q[1];
                    const double ag = w * q[5] * std::exp(-0.5 * z * z);
                    mu += ag;
                    for (int c = 0; c < 3; ++c) e[c] += ag * q[2 + c];
                }
                if (mu > 0) {
                    const double att = std::exp(-mu * len);
                    for (int c = 0; c < 3; ++c) C[c] += Tr * (e[c] / mu) * (1.0 - att);
                    Tr *= att;
                }
            }
            const int s = r.k[ex] > 0 ? 1 : -1;
            const int cn = r.c[ex] + s;
            if (cn < 0 || cn >= g.dims.n[ex]) break;
            dda_cross(r, g.dims, ex, len);
        }
        for (int c = 0; c < 3; ++c) out_rgba[4 * i + c] = C[c];
        out_rgba[4 * i + 3] = 1.0 - Tr;
    }
}

}  // extern "C"
