// ORACLE — TEST INFRASTRUCTURE ONLY (see constants.hpp).
//
// The Monte Carlo resonant-scattering random walk of PAPER.md §3.4 (Fig. 1), step by step, in
// fp64, one packet at a time.  Numbered steps follow DESIGN.md §"Algorithm"; each cites the
// passage it restates.  Readings of silent/ambiguous points are the A-numbers of DESIGN.md.
//
// Pins (tests/test_oracle_walk.py, tests/test_oracle_walk_pins2.py): Neufeld slab and Dijkstra sphere escape CDFs, E_2
// unscattered fraction, thin limit, dust-only escape fraction, interaction-kind probability, core-skip and Galilean
// invariance, Gunn-Peterson depth under Hubble drift, peel-off (thin limit + pixel mapping, next-event-estimator
// identity, dipole weight ratio), infinite segments, photon-number conservation; local core-skipping (mode 2 == mode 1
// with the cell's hand-computed x_crit, record for record, and spectrum invariance), source selection (every packet's V
// and direction recomputed from its Philox draws through the luminosity CDF), peel rays under Hubble drift (exp(-tau) by
// quadrature of scipy's Faddeeva function along the swept line), the crossing cap (reading A26).
// PARITY UNPINNED: the scattering COUNT of a walk has no closed form in the paper or the literature quoted by it
// (only "N_scat ∝ tau_0" at high tau_0), so the absolute number of scatterings per packet is checked
// only for order of magnitude; and the paper's outflow-sphere, MgII and cosmological results (PAPER.md:326 right,
// 358, Figs. 7-10) are figures without printed values.
#pragma once
#include <cstdint>
#include <cmath>
#include <vector>
#include "constants.hpp"
#include "philox.hpp"
#include "voigt.hpp"
#include "sampler.hpp"
#include "dda.hpp"

namespace orc {

struct Grid {
    GridDims dims;
    double cell_cm;
    const float* nHI;      // cm^-3,   [nz][ny][nx], x fastest
    const float* T;        // K
    const float* vx;       // km/s
    const float* vy;
    const float* vz;
    const float* kdust;    // cm^-1 absorption coefficient, or nullptr
};

struct Sources {
    int64_t n;
    const float* pos;      // [n][3], cell units
    const float* lum;      // [n], relative weights
    const float* sigma;    // [n], km/s
    std::vector<double> cdf;   // normalised cumulative luminosity, built by prepare()
    void prepare() {
        cdf.resize(n);
        double tot = 0;
        for (int64_t i = 0; i < n; ++i) tot += lum[i];
        double acc = 0;
        for (int64_t i = 0; i < n; ++i) { acc += lum[i]; cdf[i] = acc / tot; }
        cdf[n - 1] = 1.0;
    }
};

enum Status { ST_ESCAPED = 0, ST_ABSORBED = 1, ST_TERMINATED = 2, ST_CAPPED = 3 };
enum Counter { CT_ESCAPED = 0, CT_ABSORBED, CT_TERMINATED, CT_CAPPED, CT_SCATTERINGS, CT_CROSSINGS, CT_REJ_ITERS,
               CT_PEEL_RAYS, CT_PEEL_CELLS, CT_DUST_SCATTERINGS, CT_COUNT };

struct Opts {
    int phase_core = PHASE_ISOTROPIC, phase_wing = PHASE_ISOTROPIC;
    int phase_frame = 0;            // 0: atom frame |x_in - u_par| (reading A3 default), 1: gas frame |x_in|
    double phase_split_x = 0.2;
    int core_skip_mode = 0;         // 0 off, 1 global x_crit, 2 local per cell (reading A7)
    double x_crit = 0.0;
    int spec_mode = 0;              // 0: x = V / v_th(T_ref); 1: dv = -V in km/s (reading A14)
    double spec_T_ref = 1e4;
    int spec_bins = 0;
    double spec_lo = 0, spec_hi = 1;
    double hubble_kms_per_cell = 0; // reading A12/A15
    double hubble_eps = 0.25;
    double v_max_kms = 0;           // 0 = off
    int peel_on = 0;
    double k_obs[3] = {0, 0, 1};
    int peel_nx = 0, peel_ny = 0, peel_nv = 0;
    double peel_v_lo = 0, peel_v_hi = 1;
    double peel_width_cells = 0;    // image side in cell units, centred on the grid centre
    double tau_peel_max = 30.0;     // reading A13
    uint64_t photon_id_offset = 0;
    uint64_t max_scatter = 0;       // 0 = no cap
    uint64_t max_crossings = 0;     // cap on cell crossings per packet; 0 = the built-in limit 2^32 - 1 (reading A26)
    // dust scattering (PAPER.md 2.3.2, Eq. 8-9): with albedo > 0 kdust is the dust EXTINCTION coefficient; an interaction
    // with dust scatters with probability albedo (Henyey-Greenstein, asymmetry g), else absorbs (reading A32)
    double dust_albedo = 0.0, dust_g = 0.0;
    // doublet: a second transition of the same species, its line centre dv km/s from the first, with
    // sigma_0 and a scaled by the two ratios; cross-sections add, a scattering happens in ONE line (reading A34)
    int doublet_on = 0;
    double doublet_dv_kms = 0.0, doublet_sigma_ratio = 0.0, doublet_a_ratio = 1.0;
};

struct RawRecord { float V; uint32_t nscat; int32_t status; float kx, ky, kz; };

struct Result {
    std::vector<uint64_t> spectrum;     // [bins] + underflow + overflow
    uint64_t nscat_hist[64] = {0};      // bin 0: nscat = 0; bin b: 2^(b-1) <= nscat < 2^b
    uint64_t counters[CT_COUNT] = {0};
    std::vector<double> cube;           // [peel_ny][peel_nx][peel_nv]
    std::vector<RawRecord> raw;
};

struct CellProps { double n, T, v[3], kd; };

inline CellProps fetch_cell(const Grid& g, const int c[3]) {
    const int64_t i = g.dims.linear(c);
    CellProps p;
    p.n = g.nHI[i]; p.T = g.T[i]; p.v[0] = g.vx[i]; p.v[1] = g.vy[i]; p.v[2] = g.vz[i];
    p.kd = g.kdust ? (double)g.kdust[i] : 0.0;
    return p;
}

inline double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

// Opacity per cell length at lab-frame velocity offset V for direction k: Eq. 4, with sigma
// evaluated in the gas frame, x = (V - v.k)/v_th.  Returns line part; dust part is p.kd * cell_cm.
inline double kappa_line(const Grid& g, const CellProps& p, double V, const double k[3]) {
    if (p.n <= 0.0) return 0.0;                          // reading A19
    const double vth = vth_kms(p.T);
    const double x = (V - dot3(p.v, k)) / vth;
    return p.n * sigma0_cm2(p.T) * voigt_H(voigt_a(p.T), x) * g.cell_cm;
}

// The doublet's second line (reading A34): centre at dv, sigma_0 and a scaled by the ratios.
struct Doublet { bool on; double dv, rs, ra; };
inline double kappa_line2(const Grid& g, const CellProps& p, double V, const double k[3], const Doublet& d) {
    if (!d.on || p.n <= 0.0) return 0.0;
    const double vth = vth_kms(p.T);
    const double x = (V - d.dv - dot3(p.v, k)) / vth;
    return p.n * sigma0_cm2(p.T) * d.rs * voigt_H(voigt_a(p.T) * d.ra, x) * g.cell_cm;
}

// Optical depth of one segment of length len (cell units) starting at velocity offset V0, or the distance at
// which tau_need is reached.  Without Hubble drift this is kappa * len (piecewise-constant cells).
// With drift (V falls by Hc per cell length), sub-cell stepping per reading A12: n_sub = 1 if
// min|x| over the segment > 6, else ceil(|dV| / (eps v_th)); midpoint rule; interaction site linear in the
// sub-step.  Returns true on interaction; then s_hit = distance, kappa_hit_* = opacities at the site.
struct SegmentOut { double tau; bool hit; double s_hit; double k_line, k_dust, k_line2; };

inline SegmentOut integrate_segment(const Grid& g, const CellProps& p, double V0, const double k[3], double len,
                                    double tau_need, double Hc, double eps, const Doublet& db = Doublet{false, 0, 0, 1}) {
    SegmentOut o{0.0, false, 0.0, 0.0, 0.0, 0.0};
    const double kdust = p.kd * g.cell_cm;
    o.k_dust = kdust;
    if (p.n <= 0.0 && kdust <= 0.0) return o;
    int nsub = 1;
    if (Hc != 0.0 && p.n > 0.0 && len > 0.0) {
        const double vth = vth_kms(p.T);
        const double vk = dot3(p.v, k);
        const double xa = (V0 - vk) / vth, xb = (V0 - Hc * len - vk) / vth;
        const double minabs = (xa * xb <= 0.0) ? 0.0 : std::fmin(std::fabs(xa), std::fabs(xb));
        if (minabs <= 6.0) {
            const double q = std::ceil(std::fabs(Hc * len) / (eps * vth));
            nsub = q < 1.0 ? 1 : (q > 1e6 ? 1000000 : (int)q);
        }
    }
    const double ds = len / nsub;
    for (int j = 0; j < nsub; ++j) {
        const double Vmid = Hc != 0.0 ? V0 - Hc * (j + 0.5) * ds : V0;   // no 0 * inf when ds = +inf (reading A24)
        const double kl = kappa_line(g, p, Vmid, k);
        const double kl2 = kappa_line2(g, p, Vmid, k, db);
        const double kt = kl + kl2 + kdust;
        const double dtau = kt * ds;
        if (o.tau + dtau >= tau_need && kt > 0.0) {
            o.hit = true;
            o.s_hit = (j ? j * ds : 0.0) + (tau_need - o.tau) / kt;       // linear within the step
            if (o.s_hit > len) o.s_hit = len;
            o.k_line = kl;
            o.k_line2 = kl2;
            o.tau = tau_need;
            return o;
        }
        o.tau += dtau;
    }
    return o;
}

// Deterministic orthonormal basis (e1, e2) perpendicular to k (any fixed rule is valid: the azimuth is uniform).
inline void ortho_basis(const double k[3], double e1[3], double e2[3]) {
    double h[3] = {0, 0, 0};
    if (std::fabs(k[0]) <= std::fabs(k[1]) && std::fabs(k[0]) <= std::fabs(k[2])) h[0] = 1;
    else if (std::fabs(k[1]) <= std::fabs(k[2])) h[1] = 1;
    else h[2] = 1;
    const double hk = dot3(h, k);
    double n2 = 0;
    for (int i = 0; i < 3; ++i) { e1[i] = h[i] - hk * k[i]; n2 += e1[i] * e1[i]; }
    const double inv = 1.0 / std::sqrt(n2);
    for (int i = 0; i < 3; ++i) e1[i] *= inv;
    e2[0] = k[1] * e1[2] - k[2] * e1[1];
    e2[1] = k[2] * e1[0] - k[0] * e1[2];
    e2[2] = k[0] * e1[1] - k[1] * e1[0];
}

class Walker {
public:
    Walker(const Grid& g, Sources& s, const Opts& o) : g_(g), s_(s), o_(o),
        db_{o.doublet_on != 0, o.doublet_dv_kms, o.doublet_sigma_ratio, o.doublet_a_ratio} {
        s_.prepare();
        if (o_.peel_on) {
            double n2 = dot3(o_.k_obs, o_.k_obs);
            for (int i = 0; i < 3; ++i) kobs_[i] = o_.k_obs[i] / std::sqrt(n2);
            // Image-plane basis: helper axis = x unless k_obs is closest to x, then y.
            double h[3] = {1, 0, 0};
            if (std::fabs(kobs_[0]) > std::fabs(kobs_[1]) && std::fabs(kobs_[0]) > std::fabs(kobs_[2])) { h[0] = 0; h[1] = 1; }
            const double hk = dot3(h, kobs_);
            double m2 = 0;
            for (int i = 0; i < 3; ++i) { img1_[i] = h[i] - hk * kobs_[i]; m2 += img1_[i] * img1_[i]; }
            for (int i = 0; i < 3; ++i) img1_[i] /= std::sqrt(m2);
            img2_[0] = kobs_[1] * img1_[2] - kobs_[2] * img1_[1];
            img2_[1] = kobs_[2] * img1_[0] - kobs_[0] * img1_[2];
            img2_[2] = kobs_[0] * img1_[1] - kobs_[1] * img1_[0];
        }
    }

    void run(uint64_t n_photons, uint64_t seed, Result& res, bool want_raw) {
        res.spectrum.assign(o_.spec_bins + 2, 0);
        if (o_.peel_on) res.cube.assign((size_t)o_.peel_nx * o_.peel_ny * o_.peel_nv, 0.0);
        if (want_raw) res.raw.resize(n_photons);
        for (uint64_t i = 0; i < n_photons; ++i) {
            RawRecord rec = walk_one(seed, o_.photon_id_offset + i, res);
            if (want_raw) res.raw[i] = rec;
        }
    }

private:
    const Grid& g_;
    Sources& s_;
    Opts o_;
    double kobs_[3], img1_[3], img2_[3];
    Doublet db_;

    // Step 6: contribution escaping toward the observer from position (ray cell/offset) at
    // velocity offset V_o with phase weight P^:  w = P^ exp(-tau_obs), tau_obs integrated along k_obs to the box
    // face by the same march (steps a4-a6), cut at tau_peel_max (reading A13).
    void peel(const Ray<double>& at, double V_o, double phat, Result& res) {
        Ray<double> r = at;
        r.set_direction(kobs_);
        res.counters[CT_PEEL_RAYS]++;
        double tau = 0, V = V_o;
        // pixel of the starting point
        double p[3];
        for (int ax = 0; ax < 3; ++ax) p[ax] = (at.c[ax] + at.f[ax]) - 0.5 * g_.dims.n[ax];
        const double W = o_.peel_width_cells;
        const double px = (dot3(p, img1_) / W + 0.5) * o_.peel_nx;
        const double py = (dot3(p, img2_) / W + 0.5) * o_.peel_ny;
        if (!(px >= 0 && px < o_.peel_nx && py >= 0 && py < o_.peel_ny)) return;
        for (;;) {
            double len;
            const int ex = dda_next_face(r, g_.dims, len);
            if (std::isinf(len)) return;                      // reading A24: never reaches a box face -> dropped
            const CellProps cp = fetch_cell(g_, r.c);
            const SegmentOut so = integrate_segment(g_, cp, V, kobs_, len, 1e300, o_.hubble_kms_per_cell, o_.hubble_eps, db_);
            tau += so.tau;
            V -= o_.hubble_kms_per_cell * len;
            res.counters[CT_PEEL_CELLS]++;
            if (tau > o_.tau_peel_max) return;
            // a periodic axis would never end the ray: peel rays leave through the first box face they meet
            const int s = r.k[ex] > 0 ? 1 : -1;
            const int cn = r.c[ex] + s;
            if (cn < 0 || cn >= g_.dims.n[ex]) break;
            dda_cross(r, g_.dims, ex, len);
        }
        const double dv = -V;
        const int iv = (int)std::floor((dv - o_.peel_v_lo) / (o_.peel_v_hi - o_.peel_v_lo) * o_.peel_nv);
        if (iv < 0 || iv >= o_.peel_nv) return;
        res.cube[((size_t)(int)py * o_.peel_nx + (int)px) * o_.peel_nv + iv] += phat * std::exp(-tau);
    }

    RawRecord walk_one(uint64_t seed, uint64_t id, Result& res) {
        DrawStream rng(seed, id);
        // ---- Step 1: emission.  Draws 0..4.
        const double us = rng.uniform();
        int64_t j = 0;
        { int64_t lo = 0, hi = s_.n - 1;                 // smallest j with us < cdf[j]
          while (lo < hi) { const int64_t mid = (lo + hi) / 2; if (us < s_.cdf[mid]) hi = mid; else lo = mid + 1; }
          j = lo; }
        const double mu0 = 2.0 * rng.uniform() - 1.0;    // isotropic direction, direct (mu, phi) (reading A22)
        const double phi0 = 2.0 * PI * rng.uniform();
        const double st0 = std::sqrt(std::fmax(0.0, 1.0 - mu0 * mu0));
        double k[3] = {st0 * std::cos(phi0), st0 * std::sin(phi0), mu0};
        const double g1 = rng.uniform(), g2 = rng.uniform();
        const double gauss = std::sqrt(-2.0 * std::log(g1)) * std::cos(2.0 * PI * g2);   // N(0,1), Box-Muller
        Ray<double> ray;
        const double pos[3] = {s_.pos[3 * j], s_.pos[3 * j + 1], s_.pos[3 * j + 2]};
        dda_locate(ray, g_.dims, pos);
        ray.set_direction(k);
        CellProps cp = fetch_cell(g_, ray.c);
        // Gaussian line in the source cell's gas frame, then into the lab frame (reading A10).
        const double dV = (double)s_.sigma[j] * gauss;
        double V = dot3(cp.v, k) + dV;
        if (o_.peel_on) peel(ray, dot3(cp.v, kobs_) + dV, 1.0, res);
        uint64_t nscat = 0, ncross = 0;
        // Reading A26: a packet that can neither escape nor be destroyed (periodic box, empty gas) would never end;
        // it is finished as capped after max_crossings cell crossings (built-in limit 2^32 - 1).
        const uint64_t cross_cap = (o_.max_crossings && o_.max_crossings < 0xffffffffull) ? o_.max_crossings : 0xffffffffull;
        int status = ST_ESCAPED;
        const double Hc = o_.hubble_kms_per_cell;
        for (;;) {
            // ---- Step 2: tau_target = -ln u (Eq. 3).
            const double tau_target = -std::log(rng.uniform());
            double tau_acc = 0.0;
            SegmentOut so;
            bool done = false;
            // ---- Step 3: march face to face.
            for (;;) {
                double len;
                const int ex = dda_next_face(ray, g_.dims, len);
                cp = fetch_cell(g_, ray.c);
                so = integrate_segment(g_, cp, V, k, len, tau_target - tau_acc, Hc, o_.hubble_eps, db_);
                if (so.hit) {
                    dda_advance_within(ray, g_.dims, so.s_hit);
                    if (Hc != 0.0) V -= Hc * so.s_hit;
                    break;
                }
                // Reading A24: a ray parallel to every non-frozen axis has an infinite segment; if it did not
                // interact there (empty cell, or a drifting frequency) it can neither leave nor be followed: capped.
                if (std::isinf(len)) { status = ST_CAPPED; done = true; break; }
                tau_acc += so.tau;
                V -= Hc * len;
                res.counters[CT_CROSSINGS]++;
                if (!dda_cross(ray, g_.dims, ex, len)) { status = ST_ESCAPED; done = true; break; }
                if (o_.v_max_kms > 0 && std::fabs(V) > o_.v_max_kms) { status = ST_TERMINATED; done = true; break; }
                if (++ncross >= cross_cap) { status = ST_CAPPED; done = true; break; }
            }
            if (done) break;
            // ---- Step 4: which interaction: interaction i with probability tau_i / tau — dust, line 1, line 2.
            int line = 0;
            if (g_.kdust || db_.on) {
                const double r = rng.uniform();
                const double kt = so.k_line + so.k_line2 + so.k_dust;
                if (r * kt < so.k_dust) {
                    // dust (PAPER.md 2.3.2): scattered with probability albedo (Eq. 8), else destroyed
                    if (!(o_.dust_albedo > 0.0) || !(rng.uniform() < o_.dust_albedo)) { status = ST_ABSORBED; break; }
                    const double mu = hg_mu(o_.dust_g, rng.uniform());          // Eq. 9
                    const double phi = 2.0 * PI * rng.uniform();
                    double e1[3], e2[3];
                    ortho_basis(k, e1, e2);
                    const double vk = dot3(cp.v, k);
                    // grains move with the gas and are heavy: the frequency is unchanged in the cell's bulk frame (A33)
                    if (o_.peel_on) peel(ray, V - vk + dot3(cp.v, kobs_), hg_value(o_.dust_g, dot3(k, kobs_)), res);
                    const double st = std::sqrt(std::fmax(0.0, 1.0 - mu * mu));
                    double kn[3];
                    for (int i = 0; i < 3; ++i) kn[i] = mu * k[i] + st * (std::cos(phi) * e1[i] + std::sin(phi) * e2[i]);
                    const double nrm = 1.0 / std::sqrt(dot3(kn, kn));
                    for (int i = 0; i < 3; ++i) k[i] = kn[i] * nrm;
                    ray.set_direction(k);
                    V = V - vk + dot3(cp.v, k);
                    res.counters[CT_DUST_SCATTERINGS]++;
                    continue;
                }
                if (db_.on && r * kt >= so.k_dust + so.k_line) line = 1;
            }
            // ---- Step 5: resonant scattering (§2.3.1) in the chosen line: frequencies relative to ITS centre.
            const double dv_line = line ? db_.dv : 0.0;
            const double vth = vth_kms(cp.T);
            const double a = voigt_a(cp.T) * (line ? db_.ra : 1.0);
            const double vk = dot3(cp.v, k);
            const double x_in = (V - dv_line - vk) / vth;
            const double upar = sample_upar(a, x_in, rng, &res.counters[CT_REJ_ITERS]);
            double x_crit = 0.0;
            if (o_.core_skip_mode == 1) x_crit = o_.x_crit;
            else if (o_.core_skip_mode == 2) {
                const double atau = a * cp.n * sigma0_cm2(cp.T) * (line ? db_.rs : 1.0) * g_.cell_cm * 0.5;
                x_crit = atau >= 1.0 ? 0.2 * std::cbrt(atau) : 0.0;
            }
            double up1, up2;
            sample_uperp(x_in, x_crit, rng, up1, up2);
            const double xsel = o_.phase_frame == 0 ? std::fabs(x_in - upar) : std::fabs(x_in);
            const int phase = xsel > o_.phase_split_x ? o_.phase_wing : o_.phase_core;
            int is_dipole = 0;
            const double mu = sample_mu(phase, rng, &is_dipole);
            const double phi = 2.0 * PI * rng.uniform();
            double e1[3], e2[3];
            ortho_basis(k, e1, e2);
            if (o_.peel_on) {
                const double mu_o = dot3(k, kobs_);
                const double x_o = x_in - upar + upar * mu_o + up1 * dot3(e1, kobs_) + up2 * dot3(e2, kobs_);
                peel(ray, x_o * vth + dot3(cp.v, kobs_) + dv_line, phase_value(is_dipole, mu_o), res);
            }
            const double st = std::sqrt(std::fmax(0.0, 1.0 - mu * mu));
            const double cph = std::cos(phi), sph = std::sin(phi);
            double kn[3];
            for (int i = 0; i < 3; ++i) kn[i] = mu * k[i] + st * (cph * e1[i] + sph * e2[i]);
            const double nrm = 1.0 / std::sqrt(dot3(kn, kn));
            for (int i = 0; i < 3; ++i) kn[i] *= nrm;
            // Eq. 7, recoil dropped: x_out = x_in + u.(k_out - k_in).
            const double x_out = x_in - upar + upar * mu + st * (up1 * cph + up2 * sph);
            for (int i = 0; i < 3; ++i) k[i] = kn[i];
            ray.set_direction(k);
            V = x_out * vth + dot3(cp.v, k) + dv_line;
            ++nscat;
            res.counters[CT_SCATTERINGS]++;
            if (o_.v_max_kms > 0 && std::fabs(V) > o_.v_max_kms) { status = ST_TERMINATED; break; }
            if (o_.max_scatter && nscat >= o_.max_scatter) { status = ST_CAPPED; break; }
        }
        // ---- Step 7: tallies.
        res.counters[status]++;
        int hb = 0;
        if (nscat > 0) { hb = 1; uint64_t t = nscat; while (t >>= 1) ++hb; if (hb > 63) hb = 63; }
        res.nscat_hist[hb]++;
        if ((status == ST_ESCAPED || status == ST_TERMINATED) && o_.spec_bins > 0) {
            const double val = o_.spec_mode == 0 ? V / vth_kms(o_.spec_T_ref) : -V;
            const double b = std::floor((val - o_.spec_lo) / (o_.spec_hi - o_.spec_lo) * o_.spec_bins);
            if (b < 0) res.spectrum[o_.spec_bins]++;
            else if (b >= o_.spec_bins) res.spectrum[o_.spec_bins + 1]++;
            else res.spectrum[(int)b]++;
        }
        return RawRecord{(float)V, (uint32_t)(nscat > 0xffffffffull ? 0xffffffffull : nscat), status,
                         (float)k[0], (float)k[1], (float)k[2]};
    }
};

}  // namespace orc
