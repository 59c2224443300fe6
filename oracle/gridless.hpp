// ORACLE — TEST INFRASTRUCTURE ONLY (see constants.hpp).
//
// The random walk of walker.hpp through the paper's GRIDLESS datasets (PAPER.md 3.3): a spherical shell
// r_in <= r <= r_out (r_in = 0: a sphere) and an infinite slab |z| <= r_out, with the power-law density and velocity of
// PAPER.md:380 and the global step limiter of PAPER.md:382.  Nothing is voxelised: boundaries are the analytic sphere /
// planes (the paper validates on these).  fp64, one packet at a time, in the paper's order.
//
//   shell:  n_HI(r) = n0 (r / r_out)^alpha_rho,  v(r) = v_max (r / r_out)^alpha_v r^,  kappa_dust(r) = kdust0 (r / r_out)^alpha_rho
//   slab:   n_HI = n0,  v = (0, 0, v_max z / r_out),  kappa_dust = kdust0
// Lengths are in the dataset's own unit (length_cm centimetres each); positions are relative to the centre / midplane.
//
// Readings (A29-A31; the paper prints no algorithm for `query` on these datasets):
//   A29  a step runs from the current position to the next boundary (outer sphere, inner sphere, slab face) but never
//        farther than l_max = f min(l_v, l_rho), l_v = v_th / max|dv/dr|, l_rho = max[rho / |d rho/dr|] over the gas
//        (f = 0.01; a static homogeneous medium has l_max = inf);
//   A30  within a step the gas is constant, with the properties of the step's MIDPOINT; the interaction site
//        is linear within the step and the scattering happens in the gas of that step;
//   A31  the cavity r < r_in and the outside are empty; a packet ends (escapes) when it leaves r_out (|z| > r_out).
// Pins (tests/test_oracle_gridless.py): exp(-tau) / E_2 unscattered fractions, Neufeld slab and Dijkstra sphere CDFs with
// NO voxelisation error, dust-only escape e^{-tau_d}, the swept line of a linearly expanding sphere against quadrature of
// scipy's Faddeeva function, convergence in the step limiter, agreement with the voxelised walker on a fine grid.
#pragma once
#include "walker.hpp"

namespace orc {

struct Gridless {
    int geometry;            // 0 shell / sphere, 1 slab
    double r_in, r_out, length_cm;
    double n0, alpha_rho, T, v_max, alpha_v, kdust0, step_f;
};

struct GridlessStep { double n, kd, v[3]; };

inline double gl_radius(const double r[3]) { return std::sqrt(dot3(r, r)); }

// Gas properties at a point (reading A30 evaluates them at step midpoints).
inline GridlessStep gl_props(const Gridless& d, const double r[3]) {
    GridlessStep s{0, 0, {0, 0, 0}};
    if (d.geometry == 1) {
        if (std::fabs(r[2]) > d.r_out) return s;
        s.n = d.n0; s.kd = d.kdust0;
        s.v[2] = d.v_max * r[2] / d.r_out;
        return s;
    }
    const double rr = gl_radius(r);
    if (rr < d.r_in || rr > d.r_out) return s;
    const double q = rr / d.r_out;
    const double w = d.alpha_rho == 0.0 ? 1.0 : std::pow(q, d.alpha_rho);
    s.n = d.n0 * w; s.kd = d.kdust0 * w;
    if (rr > 0.0 && d.v_max != 0.0) {
        const double vm = d.v_max * (d.alpha_v == 1.0 ? q : std::pow(q, d.alpha_v)) / rr;
        for (int i = 0; i < 3; ++i) s.v[i] = vm * r[i];
    }
    return s;
}

// Global step limiter l_max (reading A29), in length units; +inf without gradients or with step_f = 0.
inline double gl_step_limit(const Gridless& d) {
    if (!(d.step_f > 0.0)) return INFINITY;
    const double vth = vth_kms(d.T);
    double lv = INFINITY, lrho = INFINITY;
    if (d.geometry == 1) {
        if (d.v_max != 0.0) lv = vth * d.r_out / std::fabs(d.v_max);
    } else {
        if (d.v_max != 0.0 && d.alpha_v != 0.0) {
            // |dv/dr| = |alpha_v v_max| r^(alpha_v - 1) / r_out^alpha_v: largest at r_out (alpha_v >= 1) or at r_in
            const double rm = d.alpha_v >= 1.0 ? d.r_out : std::fmax(d.r_in, 1e-300);
            lv = vth / (std::fabs(d.alpha_v * d.v_max) * std::pow(rm / d.r_out, d.alpha_v - 1.0) / d.r_out);
        }
        if (d.alpha_rho != 0.0) lrho = d.r_out / std::fabs(d.alpha_rho);   // rho / |d rho/dr| = r / |alpha_rho|, largest at r_out
    }
    const double m = std::fmin(lv, lrho);
    return std::isinf(m) ? INFINITY : d.step_f * m;
}

// Distance along k from r to the next boundary ahead, and whether the path up to it lies in gas.
//   shell: inside the cavity -> to the inner sphere (empty); in the gas -> to the inner sphere if the ray meets it, else
//   to the outer sphere; slab: to the face ahead (infinite if k_z = 0).
inline double gl_to_boundary(const Gridless& d, const double r[3], const double k[3], bool& in_gas) {
    if (d.geometry == 1) {
        in_gas = true;
        if (k[2] > 0) return (d.r_out - r[2]) / k[2];
        if (k[2] < 0) return (-d.r_out - r[2]) / k[2];
        return INFINITY;
    }
    const double b = dot3(r, k), r2 = dot3(r, r);
    const double rr = std::sqrt(r2);
    if (rr < d.r_in) {                                   // in the cavity: forward root of the inner sphere
        in_gas = false;
        return -b + std::sqrt(std::fmax(0.0, b * b - (r2 - d.r_in * d.r_in)));
    }
    in_gas = true;
    if (d.r_in > 0.0 && b < 0.0) {                       // heading inward: does the ray meet the inner sphere?
        const double disc = b * b - (r2 - d.r_in * d.r_in);
        if (disc > 0.0) {
            const double t = -b - std::sqrt(disc);
            if (t >= 0.0) return t;
        }
    }
    return -b + std::sqrt(std::fmax(0.0, b * b - (r2 - d.r_out * d.r_out)));
}

class GridlessWalker {
public:
    GridlessWalker(const Gridless& d, Sources& s, const Opts& o) : d_(d), s_(s), o_(o), lmax_(gl_step_limit(d)) { s_.prepare(); }

    void run(uint64_t n_photons, uint64_t seed, Result& res, bool want_raw) {
        res.spectrum.assign(o_.spec_bins + 2, 0);
        if (want_raw) res.raw.resize(n_photons);
        for (uint64_t i = 0; i < n_photons; ++i) {
            RawRecord rec = walk_one(seed, o_.photon_id_offset + i, res);
            if (want_raw) res.raw[i] = rec;
        }
    }

private:
    const Gridless& d_;
    Sources& s_;
    Opts o_;
    double lmax_;

    RawRecord walk_one(uint64_t seed, uint64_t id, Result& res) {
        DrawStream rng(seed, id);
        // ---- emission, the same draws as the grid walker: source, mu, phi, g1, g2
        const double us = rng.uniform();
        int64_t j = 0;
        { int64_t lo = 0, hi = s_.n - 1;
          while (lo < hi) { const int64_t mid = (lo + hi) / 2; if (us < s_.cdf[mid]) hi = mid; else lo = mid + 1; }
          j = lo; }
        const double mu0 = 2.0 * rng.uniform() - 1.0;
        const double phi0 = 2.0 * PI * rng.uniform();
        const double st0 = std::sqrt(std::fmax(0.0, 1.0 - mu0 * mu0));
        double k[3] = {st0 * std::cos(phi0), st0 * std::sin(phi0), mu0};
        const double g1 = rng.uniform(), g2 = rng.uniform();
        const double gauss = std::sqrt(-2.0 * std::log(g1)) * std::cos(2.0 * PI * g2);
        double r[3] = {s_.pos[3 * j], s_.pos[3 * j + 1], s_.pos[3 * j + 2]};
        const GridlessStep g0 = gl_props(d_, r);
        double V = dot3(g0.v, k) + (double)s_.sigma[j] * gauss;        // Gaussian line in the gas frame at the source (A10)
        const double vth = vth_kms(d_.T), a = voigt_a(d_.T), sig = sigma0_cm2(d_.T) * d_.length_cm;
        uint64_t nscat = 0, nstep = 0;
        const uint64_t step_cap = (o_.max_crossings && o_.max_crossings < 0xffffffffull) ? o_.max_crossings : 0xffffffffull;
        int status = ST_ESCAPED;
        for (;;) {
            const double tau_target = -std::log(rng.uniform());
            double tau_acc = 0.0, k_line = 0.0, k_dust = 0.0;
            GridlessStep gs{};
            bool done = false;
            for (;;) {                                           // steps to the interaction site (reading A29)
                bool in_gas;
                const double db = gl_to_boundary(d_, r, k, in_gas);
                if (std::isinf(db) && std::isinf(lmax_)) {      // slab, k_z = 0, no limiter: one infinite step (reading A24)
                    gs = gl_props(d_, r);
                    k_dust = gs.kd * d_.length_cm;
                    k_line = gs.n > 0 ? gs.n * sig * voigt_H(a, (V - dot3(gs.v, k)) / vth) : 0.0;
                    if (k_line + k_dust > 0) {
                        const double l = (tau_target - tau_acc) / (k_line + k_dust);
                        for (int i = 0; i < 3; ++i) r[i] += l * k[i];
                        break;
                    }
                    status = ST_CAPPED; done = true; break;
                }
                const double len = in_gas ? std::fmin(db, lmax_) : db;
                double kt = 0.0;
                if (in_gas) {
                    double rm[3];
                    for (int i = 0; i < 3; ++i) rm[i] = r[i] + 0.5 * len * k[i];
                    gs = gl_props(d_, rm);                       // reading A30: the step's gas is that of its midpoint
                    k_dust = gs.kd * d_.length_cm;
                    k_line = gs.n > 0 ? gs.n * sig * voigt_H(a, (V - dot3(gs.v, k)) / vth) : 0.0;
                    kt = k_line + k_dust;
                }
                if (kt > 0.0 && tau_acc + kt * len >= tau_target) {
                    const double l = (tau_target - tau_acc) / kt;      // linear within the step
                    for (int i = 0; i < 3; ++i) r[i] += l * k[i];
                    break;
                }
                tau_acc += kt * len;
                for (int i = 0; i < 3; ++i) r[i] += len * k[i];
                res.counters[CT_CROSSINGS]++;
                if (len >= db) {                                 // reached a boundary: leaving the dataset ends the packet (A31)
                    const bool out = d_.geometry == 1 ? true : (dot3(r, k) > 0.0 && gl_radius(r) >= d_.r_out * (1.0 - 1e-12));
                    if (out && (d_.geometry == 1 || !(gl_radius(r) < d_.r_in * (1.0 + 1e-12) && d_.r_in > 0))) {
                        status = ST_ESCAPED; done = true; break;
                    }
                    // inner sphere reached (from either side): nudge across it so the next step starts on the far side
                    for (int i = 0; i < 3; ++i) r[i] += 1e-12 * d_.r_out * k[i];
                }
                if (o_.v_max_kms > 0 && std::fabs(V) > o_.v_max_kms) { status = ST_TERMINATED; done = true; break; }
                if (++nstep >= step_cap) { status = ST_CAPPED; done = true; break; }
            }
            if (done) break;
            if (d_.kdust0 > 0.0) {                               // dust with probability kappa_dust / kappa_total
                const double rr = rng.uniform();
                if (rr * (k_line + k_dust) < k_dust) {
                    // PAPER.md 2.3.2: scattered with probability albedo (Eq. 8; Henyey-Greenstein, Eq. 9), else destroyed
                    if (!(o_.dust_albedo > 0.0) || !(rng.uniform() < o_.dust_albedo)) { status = ST_ABSORBED; break; }
                    const double mu = hg_mu(o_.dust_g, rng.uniform());
                    const double phi = 2.0 * PI * rng.uniform();
                    double e1[3], e2[3];
                    ortho_basis(k, e1, e2);
                    const double vk0 = dot3(gs.v, k);
                    const double st = std::sqrt(std::fmax(0.0, 1.0 - mu * mu));
                    double kn[3];
                    for (int i = 0; i < 3; ++i) kn[i] = mu * k[i] + st * (std::cos(phi) * e1[i] + std::sin(phi) * e2[i]);
                    const double nrm = 1.0 / std::sqrt(dot3(kn, kn));
                    for (int i = 0; i < 3; ++i) k[i] = kn[i] * nrm;
                    V = V - vk0 + dot3(gs.v, k);                 // coherent in the bulk frame of the step's gas (A33)
                    res.counters[CT_DUST_SCATTERINGS]++;
                    continue;
                }
            }
            // ---- resonant scattering in the gas of the step (PAPER.md 2.3.1), as in walker.hpp step 5
            const double vk = dot3(gs.v, k);
            const double x_in = (V - vk) / vth;
            const double upar = sample_upar(a, x_in, rng, &res.counters[CT_REJ_ITERS]);
            const double x_crit = o_.core_skip_mode == 1 ? o_.x_crit : 0.0;       // no local mode: there are no cells
            double up1, up2;
            sample_uperp(x_in, x_crit, rng, up1, up2);
            const double xsel = o_.phase_frame == 0 ? std::fabs(x_in - upar) : std::fabs(x_in);
            const int phase = xsel > o_.phase_split_x ? o_.phase_wing : o_.phase_core;
            const double mu = sample_mu(phase, rng, nullptr);
            const double phi = 2.0 * PI * rng.uniform();
            double e1[3], e2[3];
            ortho_basis(k, e1, e2);
            const double st = std::sqrt(std::fmax(0.0, 1.0 - mu * mu));
            const double cph = std::cos(phi), sph = std::sin(phi);
            double kn[3];
            for (int i = 0; i < 3; ++i) kn[i] = mu * k[i] + st * (cph * e1[i] + sph * e2[i]);
            const double nrm = 1.0 / std::sqrt(dot3(kn, kn));
            for (int i = 0; i < 3; ++i) kn[i] *= nrm;
            const double x_out = x_in - upar + upar * mu + st * (up1 * cph + up2 * sph);   // Eq. 7, recoil dropped
            for (int i = 0; i < 3; ++i) k[i] = kn[i];
            V = x_out * vth + dot3(gs.v, k);
            ++nscat;
            res.counters[CT_SCATTERINGS]++;
            if (o_.v_max_kms > 0 && std::fabs(V) > o_.v_max_kms) { status = ST_TERMINATED; break; }
            if (o_.max_scatter && nscat >= o_.max_scatter) { status = ST_CAPPED; break; }
        }
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
