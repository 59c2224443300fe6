// Kernel-side parameter block of the walk (filled by api.cu from thor_grid_create / thor_sources_set / thor_opts).
#pragma once
#include <cstdint>
#include "dda.cuh"

namespace thor {

// Lyα atomic constants, CGS (textbook values; the paper prints none of them).
// Definitions of x, u, v_th: PAPER.md:107.
struct LyaConstants {
    double c_vth;   // v_th [km/s]      = c_vth sqrt(T)        (sqrt(2 k_B / m_H) 1e-5)
    double c_a;     // a                = c_a / sqrt(T)        (A21 lambda0 / (4 pi sqrt(2 k_B / m_H)))
    double c_sig;   // sigma_0 [cm^2]   = c_sig / sqrt(T)      (f12 sqrt(pi) e^2 lambda0 / (m_e c sqrt(2 k_B / m_H)))
};

inline LyaConstants lya_constants() {
    const double kB = 1.380649e-16, mH = 1.6735575e-24, c = 2.99792458e10, e = 4.80320471e-10, me = 9.1093837e-28;
    const double lambda0 = 1215.67e-8, f12 = 0.4162, A21 = 6.265e8, pi = 3.14159265358979323846;
    const double s = __builtin_sqrt(2.0 * kB / mH);          // cm/s per sqrt(K)
    LyaConstants k;
    k.c_vth = s * 1e-5;
    k.c_a = A21 * lambda0 / (4.0 * pi * s);
    k.c_sig = f12 * __builtin_sqrt(pi) * e * e * lambda0 / (me * c * s);
    return k;
}

enum : int { CT_ESCAPED = 0, CT_ABSORBED, CT_TERMINATED, CT_CAPPED, CT_SCATTERINGS, CT_CROSSINGS, CT_REJ_ITERS,
             CT_PEEL_RAYS, CT_PEEL_CELLS, CT_DUST_SCATTERINGS, N_COUNTERS };

struct RawRecord { float V; uint32_t nscat; int32_t status; float kx, ky, kz; };

constexpr double CUBE_FIXED_SCALE = 4294967296.0;   // peel weights are summed as round(w 2^32) in uint64

constexpr int MAX_TF_PEAKS = 8;                    // THOR_MAX_TF_PEAKS

// Transfer function of the volume renderer, prepared on the host in log2 units.
struct TransferFn {
    int n_peaks;
    int weight_by_density;           // w = n_HI (1 / n_ref folded into amp) or w = 1
    float centre[MAX_TF_PEAKS];      // log2 T of the peak
    float neg_inv_2s2[MAX_TF_PEAKS]; // -log2(e) / (2 s^2), s in log2 T
    float amp[MAX_TF_PEAKS];         // A_p (/ n_ref)
    float r[MAX_TF_PEAKS], g[MAX_TF_PEAKS], b[MAX_TF_PEAKS];
};

struct WalkParams {
    GridDims g;
    const float* __restrict__ nHI;
    const float* __restrict__ T;
    const float* __restrict__ vx;
    const float* __restrict__ vy;
    const float* __restrict__ vz;
    const float* __restrict__ kdust;     // nullptr = no dust
    const float4* __restrict__ packed;   // THOR_GRID_PACK: [cell][2] = {nHI, T, vx, vy}, {vz, kdust, 0, 0}: one 32-byte sector
    int has_dust;                        // kdust was given (packed or not)
    float sig_cell;      // c_sig * cell_cm: kappa_line per cell length = n * sig_cell * rsqrt(T) * H(a,x)
    float c_a, c_vth, inv_c_vth;
    float cell_cm;
    // sources
    long long n_src;
    const float* __restrict__ src_pos;   // [n][3]
    const float* __restrict__ src_sigma; // [n]
    const double* __restrict__ src_cdf;  // [n], normalised cumulative luminosity, last = 1
    // opts
    int phase_core, phase_wing, phase_frame;
    float phase_split_x;
    int core_skip_mode;
    float x_crit;
    int spec_mode, spec_bins;
    float spec_inv_vth_ref;              // 1 / v_th(spec_T_ref)
    float spec_lo, spec_inv_width;       // bin = floor((val - lo) * inv_width), inv_width = bins / (hi - lo)
    float hubble, hubble_eps, v_max;
    float v_max_or_inf;                  // v_max, or +inf when there is none: one compare on a lone packet's serial chain
    int peel_on;
    float kobs[3], kobs_inv[3], img1[3], img2[3];   // kobs_inv = 1 / kobs (IEEE single-precision quotients; +-inf for 0)
    int peel_nx, peel_ny, peel_nv;
    float peel_v_lo, peel_inv_dv;        // iv = floor((dv - lo) * inv_dv)
    float peel_inv_width;                // 1 / peel_width_cells
    float tau_peel_max;
    unsigned long long id_offset, n_photons, seed, max_scatter;
    unsigned int max_scatter_or_max;     // max_scatter clamped to 32 bits (the per-packet counter's width); 2^32 - 1 = none
    unsigned int max_crossings;          // per-packet cap on cell crossings (reading A26); 2^32 - 1 = the built-in limit
    // work distribution + tallies (device)
    unsigned long long* next_photon;     // a14: global atomic photon counter
    unsigned long long* max_nscat;       // max over packets of the scattering count (the longest dependent chain)
    unsigned long long* t_start;         // min over CTAs of %globaltimer at kernel entry (ns)
    unsigned long long* t_dry;           // min over warps of %globaltimer when the photon counter was found exhausted
    unsigned long long* spectrum;        // [spec_bins + 2]
    unsigned long long* nscat_hist;      // [64]
    unsigned long long* counters;        // [N_COUNTERS]
    unsigned long long* cube;            // [ny][nx][nv] fixed point, or nullptr
    RawRecord* raw;                      // [n_photons] or nullptr
    // cooperative drain: packets parked by walk_kernel for drain_kernel
    uint32_t* pool;                      // [slots][PK_WORDS] parked packet states, or nullptr = no drain kernel
    unsigned long long* pool_count;      // packets parked
    unsigned long long* pool_next;       // next slot to pop
    unsigned int* pool_order;            // [slots]: pool slots by decreasing scattering count (longest first)
    // the tail in passes: a walk launch parks a warp's packets into pool_mid once the counter is dry and at
    // most half its lanes are live; the next launch of the walk kernel re-packs them into full warps and walks on
    uint32_t* pool_mid;                  // two halves the passes alternate between; nullptr = single pass
    unsigned long long* pool_mid_count;  // [2]
    // per launch of the walk kernel (set by the launcher):
    int resume;                          // 1: no photon counter; lanes start from the packets of resume_in
    const uint32_t* resume_in; const unsigned long long* resume_count;
    uint32_t* park_out; unsigned long long* park_count; int park_lanes;   // where, and at how many live lanes, a warp parks
    // gridless dataset (PAPER.md 3.3: spherical shell / infinite slab with power-law density and velocity); gl_geom < 0 = grid
    int gl_geom;                         // -1 grid, 0 shell / sphere, 1 slab
    double gl_rin, gl_rout;              // length units
    float gl_lmax;                       // step limiter l_max, +inf = none
    float gl_nsig0, gl_kd0;              // n0 sigma_0(T) length_cm and kdust0 length_cm: optical depths per length unit at r_out
    float gl_alpha_rho, gl_vmax, gl_alpha_v;
    float gl_a, gl_vth, gl_inv_vth;      // the one temperature of the dataset
    // dust scattering (Eq. 8-9) and the doublet's second line
    float dust_albedo, dust_g;
    int doublet_on;
    float db_dv, db_rs, db_ra;           // line 2: centre offset [km/s], sigma_0 ratio, a ratio
    int walk_variant;                    // 0 = by grid size, 3 / 4 = force the cache-resident / beyond-L2 kernel; + 16 = the generic kernels (tests)
};

}  // namespace thor
