/* thor.h — C-ABI of the B200-native hot path of THOR (arXiv 2507.11603): the Monte Carlo resonant-scattering random
 * walk of Lyα photon packets through a 3D Cartesian gas grid (§3.4, Fig. 1).
 *
 * Implemented by libthor_b200.so (paper_2507_11603_b200/csrc, CUDA, sm_100a only).  Every step of the path runs in
 * CUDA kernels; there is no CPU fallback.  Nothing here throws or aborts: every call returns a thor_status and the
 * reason is available from thor_last_error().  "DEVICE" / "HOST" say where a pointer must live.
 *
 * Entry points of the path (BASELINE.json north_star): thor_grid_create, thor_sources_set, thor_run, thor_tally_get.
 * The thor_unit_* calls run single steps of the path (RNG, DDA, Voigt, samplers) in isolation for parity tests.
 */
#ifndef THOR_B200_H
#define THOR_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct thor_ctx thor_ctx; /* opaque; one per grid.  One context must not be used from two host threads at once;
                                     different contexts are independent — they may run at once, from different threads or
                                     through thor_run_async, and may borrow the same device fields */

typedef enum {
    THOR_OK = 0,
    THOR_ERR_ARG = 1,         /* bad argument (NULL, size, NaN/negative field, source outside grid, ...) */
    THOR_ERR_STATE = 2,       /* call order (run before sources_set, tally not produced by the last run, ...) */
    THOR_ERR_OOM = 3,         /* device or host allocation failed */
    THOR_ERR_CUDA = 4,        /* a CUDA runtime call or kernel failed; text in thor_last_error */
    THOR_ERR_UNSUPPORTED = 5  /* no CUDA device / device is not sm_100 */
} thor_status;

/* ---- grid flags ---- */
#define THOR_GRID_BORROW 0x0u     /* default: field arrays are DEVICE pointers the caller keeps alive and unmodified
                                     until thor_grid_destroy; nothing is copied (the 72 GB grid of config 5) */
#define THOR_GRID_HOST 0x1u       /* field arrays are HOST pointers; the library copies them to the device */
#define THOR_PERIODIC_X 0x10u
#define THOR_PERIODIC_Y 0x20u
#define THOR_PERIODIC_Z 0x40u
#define THOR_GRID_NO_VALIDATE 0x100u /* skip the device-side scan for NaN / negative fields */
#define THOR_GRID_PACK 0x200u     /* the library makes its OWN copy, re-laid-out as one 32-byte record per cell
                                     {nHI, T, vx, vy, vz, kdust, 0, 0}: one DRAM sector per cell gather instead of
                                     five or six.  Costs 32 B per cell of device memory; the caller's
                                     arrays are not referenced after thor_grid_create returns.  Results are
                                     bit-identical to the borrowed SoA layout. */

#define THOR_GRID_L2_PERSIST 0x400u /* with THOR_GRID_PACK: thor_sources_set puts an L2 access-policy window (persisting
                                     lines) on the contiguous z-slabs of the packed grid that hold the most source
                                     luminosity, as large as the device allows (BASELINE.json north_star; measured in
                                     DESIGN.md 5).  Results do not depend on it */
#define THOR_GRID_L2_FETCH32 0x800u /* cudaLimitMaxL2FetchGranularity = 32 B for this process: a cell gather needs one
                                     32-byte sector; the default granularity pulls its neighbours as well */

/* The dataset (uniform Cartesian grid, fields constant per cell).  Six SoA fp32 arrays, dense
 * row-major [nz][ny][nx] (x fastest): nHI [cm^-3], T [K], vx, vy, vz [km/s], and kdust [cm^-1], the dust ABSORPTION
 * coefficient (NULL = no dust; reading A21).  cell_cm = cell edge in cm.  A periodic axis of extent 1 is
 * treated as infinite (DDA).  stream = cudaStream_t as void* (NULL = default stream); all later work
 * of this context is issued on it.  Errors: THOR_ERR_ARG for n<=0, NULL arrays, cell_cm<=0, n>0 with T<=0 or any
 * NaN (reading A19); THOR_ERR_UNSUPPORTED without a CUDA sm_100 device. */
thor_status thor_grid_create(thor_ctx **out, int nx, int ny, int nz, double cell_cm,
                             const float *nHI, const float *T, const float *vx, const float *vy, const float *vz,
                             const float *kdust, unsigned flags, void *stream);
void thor_grid_destroy(thor_ctx *ctx);

/* The paper's GRIDLESS datasets (PAPER.md 3.3; power laws PAPER.md:380; step limiter PAPER.md:382):
 * nothing is voxelised, boundaries are the analytic sphere(s) / planes.  Lengths are in the dataset's own unit of
 * length_cm centimetres, relative to the centre (shell) or the midplane (slab).
 *   THOR_GEOM_SHELL: gas in r_in <= r <= r_out (r_in = 0: a sphere), n_HI(r) = n0 (r/r_out)^alpha_rho [cm^-3],
 *                    v(r) = v_max (r/r_out)^alpha_v radially outward [km/s], dust absorption kdust0 (r/r_out)^alpha_rho
 *                    [cm^-1]; the cavity and the outside are empty; a packet ends when it leaves r_out.
 *   THOR_GEOM_SLAB:  gas in |z| <= r_out, n_HI = n0, v_z = v_max z / r_out, dust kdust0; infinite in x and y.
 * T [K] is uniform.  step_f: no step is longer than step_f * min(v_th / max|dv/dr|, max[rho / |d rho/dr|]) (0.01 in the
 * paper; 0 = no limiter; a static homogeneous medium has none anyway); the gas of a step is that of its midpoint and the
 * interaction site is linear within it (readings A29-A31).  The context then works with thor_sources_set
 * (positions in length units, inside r_out), thor_run and thor_tally_get as a grid context does; thor_run refuses
 * peel-off, Hubble drift and local core-skipping on it (THOR_ERR_UNSUPPORTED); the ray operators need a grid.
 * THOR_ERR_ARG for a bad geometry, r_out <= r_in, T <= 0, negative n0 / kdust0, non-finite values. */
#define THOR_GEOM_SHELL 0
#define THOR_GEOM_SLAB 1
typedef struct thor_gridless {
    uint32_t struct_size;     /* = sizeof(thor_gridless) */
    int32_t geometry;         /* THOR_GEOM_* */
    double r_in, r_out;       /* length units; slab: r_out = half thickness, r_in ignored */
    double length_cm;
    double n0, alpha_rho;
    double T;
    double v_max, alpha_v;
    double kdust0;
    double step_f;
} thor_gridless;
thor_status thor_dataset_create_gridless(thor_ctx **out, const thor_gridless *dataset, void *stream);

/* The generator: a list of point sources.  HOST arrays, copied: pos_xyz [n_src][3] in cell units
 * (grid spans [0,nx) x [0,ny) x [0,nz)), lum [n_src] >= 0 relative luminosities (a packet picks source j with
 * probability lum_j / sum, reading A18), sigma_kms [n_src] Gaussian line width in the source cell's gas frame
 * (0 = line centre, reading A10).  Replaces any earlier list.  THOR_ERR_ARG if a source lies outside the grid,
 * a luminosity is negative/NaN, or the total is zero. */
thor_status thor_sources_set(thor_ctx *ctx, long long n_src, const float *pos_xyz, const float *lum,
                             const float *sigma_kms);

/* phase functions */
#define THOR_PHASE_ISOTROPIC 0
#define THOR_PHASE_DIPOLE 1
#define THOR_PHASE_MIX 2 /* 1/3 isotropic + 2/3 dipole */

/* Run options.  Set struct_size = sizeof(thor_opts); use thor_opts_default() for the defaults. */
typedef struct thor_opts {
    uint32_t struct_size;
    int32_t phase_core, phase_wing;   /* THOR_PHASE_*; default isotropic / isotropic, which is what BASELINE.json's configs
                                         state; the paper's own assignment is MIX in the core and DIPOLE in
                                         the wings and has to be asked for */
    int32_t phase_frame;              /* 0: split on atom-frame |x_in - u_par| (default), 1: gas-frame |x_in| (A3) */
    double phase_split_x;             /* 0.2 */
    int32_t core_skip_mode;           /* 0 off, 1 global x_crit, 2 local per cell (reading A7) */
    double x_crit;
    int32_t spec_mode;                /* escape spectrum axis: 0: x = V / v_th(spec_T_ref); 1: dv = -V km/s (A14) */
    double spec_T_ref;
    int32_t spec_bins;                /* 0 = no spectrum; <= 4096 */
    double spec_lo, spec_hi;
    double hubble_kms_per_cell;       /* frequency drift per cell length travelled (A12, A15); 0 = off */
    double hubble_eps;                /* sub-step size in units of v_th (0.25) */
    double v_max_kms;                 /* stop when |V| exceeds this; 0 = off */
    int32_t peel_on;                  /* peel-off toward k_obs at emission and at every scattering */
    double k_obs[3];
    int32_t peel_nx, peel_ny, peel_nv;/* image pixels and spectral bins of the IFU cube [ny][nx][nv] */
    double peel_v_lo, peel_v_hi;      /* spectral axis dv = -V (km/s) at the box face */
    double peel_width_cells;          /* image side in cell units, centred on the grid centre */
    double tau_peel_max;              /* peel rays are dropped beyond this optical depth (30; A13) */
    uint64_t photon_id_offset;        /* the run covers photon ids [offset, offset + n_photons) */
    uint64_t max_scatter;             /* safety cap per packet (0 = none); capped packets are counted, not tallied */
    int32_t raw_output;               /* keep one thor_raw_record per packet (THOR_TALLY_RAW) */
    int32_t accumulate;               /* do not zero the tallies before this run; the spectrum axis and the peel geometry must
                                         be those of the run it adds to (THOR_ERR_ARG otherwise) */
    uint64_t max_crossings;           /* cap on cell crossings per packet (capped packets are counted, not tallied);
                                         0 = the built-in limit 2^32 - 1 (reading A26).  Required (> 0) on a
                                         grid that is periodic on all three axes: no packet can ever leave it */
    int32_t walk_variant;             /* 0 (default): kernel variant chosen by grid size; 3 / 4: force the cache-resident /
                                         beyond-L2 variant of the walk kernel; + 16: the generic kernels instead of the ones compiled
                                         for the run's doublet / core-skipping / phase-function options.  Results do not
                                         depend on it (tests, tuning) */
    int32_t drain_mode;               /* how the tail of a run is walked once the photon counter is dry.  0 (default): in
                                         passes — a warp down to half its lanes parks its packets, the next launch of the
                                         walk kernel re-packs them into full warps — and warps left with
                                         <= 4 packets hand them to the cooperative drain kernel; 2: one pass,
                                         then the drain kernel; 1: the walk kernel finishes every packet itself.  Results do
                                         not depend on it */
    double dust_albedo;               /* PAPER.md 2.3.2, Eq. 8: with albedo > 0 kdust is the dust EXTINCTION coefficient and an
                                         interaction with dust scatters with this probability, else destroys (0: absorption
                                         only, as before; the paper's fiducial value is 0.32) */
    double dust_g;                    /* asymmetry g = <mu> of the Henyey-Greenstein phase function, Eq. 9 (fiducial 0.73) */
    int32_t doublet_on;               /* a second transition of the same species: cross-sections add, each
                                         scattering happens in one line, chosen with probability tau_i / tau */
    double doublet_dv_kms;            /* its line centre, km/s from the first line's */
    double doublet_sigma_ratio;       /* sigma_0 of line 2 / sigma_0 of line 1 (the ratio of oscillator strengths) */
    double doublet_a_ratio;           /* Voigt parameter of line 2 / that of line 1 */
} thor_opts;

void thor_opts_default(thor_opts *o);

/* Walks photon ids [photon_id_offset, +n_photons) under `seed` (Philox4x32-10 keyed on (seed, photon id, draw
 * index), reading A16): emit, draw tau = -ln u, DDA march with Voigt optical depth in each cell's gas frame, scatter
 * (u_par by rejection from Eq. 6, u_perp Gaussian, phase function, Eq. 7), until escape / dust absorption, tallying
 * into the context's spectrum / cube / counters.  One persistent kernel launch; synchronous: returns after the
 * stream has drained.  opts == NULL -> defaults.  Errors: THOR_ERR_STATE without sources; THOR_ERR_ARG for
 * inconsistent opts, and for a grid periodic on all three axes (with at least one of extent > 1) when max_crossings
 * is 0 — nothing could end a packet in empty gas there, and thor_run never hangs; THOR_ERR_OOM if tallies cannot be
 * allocated; THOR_ERR_CUDA. */
thor_status thor_run(thor_ctx *ctx, unsigned long long n_photons, unsigned long long seed, const thor_opts *opts);

/* thor_run in two halves, so that ONE host thread can keep several contexts busy (consecutive batches overlap: the tail of
 * one run — a few long packets, DESIGN.md 5 — with the feed phase of the next; contexts may borrow the same device fields).
 * thor_run_async validates, allocates what the run needs and enqueues the kernels on the context's stream, then returns;
 * thor_wait blocks until that run has finished and publishes its tallies and timings (no-op if nothing is pending).
 * thor_run == thor_run_async + thor_wait.  While a run is pending, every other call on the SAME context that uses the
 * run's state (thor_run*, thor_sources_set, thor_tally_get, thor_grid_destroy) completes it first; thor_last_run_* return
 * THOR_ERR_STATE.  Arguments, results and errors as thor_run; a kernel fault surfaces in thor_wait. */
thor_status thor_run_async(thor_ctx *ctx, unsigned long long n_photons, unsigned long long seed, const thor_opts *opts);
thor_status thor_wait(thor_ctx *ctx);

/* thor_run for callers that cannot allocate device memory at run time (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the same walk (same kernels, same packets: tallies equal thor_run's bit for bit),
 * but this call makes NO cudaMalloc / cudaFree and no allocating library call.  thor_run allocates its parked-packet pool,
 * its cube and its raw records on first use; here the kernels' scratch — photon counter, timers, pool counters, the pool
 * of parked packets and its ordering — lives in ONE file-scope `static __device__` array of
 * THOR_NOALLOC_SCRATCH_BYTES (4.0 MB) that every GPU which loads the library holds until exit, and the tallies go straight
 * into buffers the caller owns:
 *   spectrum_out   DEVICE uint64[opts->spec_bins + 2]   (layout of THOR_TALLY_SPECTRUM; may be NULL if spec_bins == 0)
 *   counters_out   DEVICE uint64[THOR_N_COUNTERS]
 *   nscat_hist_out DEVICE uint64[64]                    (layout of THOR_TALLY_NSCAT_HIST)
 * all three overwritten (cleared, then filled).  ctx is a grid context with its sources set (that set-up allocates; do
 * it beforehand).  Asynchronous: the clears and kernels are enqueued on the context's stream and the call returns; the
 * outputs are valid once that stream has drained.  The context's own tallies, thor_tally_get and thor_last_run_* are not
 * touched.
 * Limits: the pool is sized for GPUs of up to THOR_NOALLOC_MAX_SM multiprocessors — a larger GPU is refused with
 * THOR_ERR_ARG and a message saying so; peel-off (its cube would have to be allocated), raw_output, accumulate and
 * gridless datasets are refused with THOR_ERR_UNSUPPORTED.  Other errors as thor_run.
 * Every call on a GPU shares the one array, which keeps the last call's contents (each call clears the words that must
 * start at zero).  Calls on the same context are ordered by its stream; calls that OVERLAP on the GPU — two contexts on
 * different streams of one device — race on the scratch and give wrong tallies: serialise them.  The first call on a
 * device looks the array's device address up (cudaGetSymbolAddress: no allocation): make it outside a capture. */
#define THOR_NOALLOC_MAX_SM 160
#define THOR_NOALLOC_SCRATCH_BYTES (256 + 160 * 128 * 4 + 160 * 128 * 192)
thor_status thor_run_noalloc(thor_ctx *ctx, unsigned long long n_photons, unsigned long long seed, const thor_opts *opts,
                             unsigned long long *spectrum_out, unsigned long long *counters_out,
                             unsigned long long *nscat_hist_out);

/* Duration of the walk kernel of the last thor_run in milliseconds, from CUDA events on the context's stream. */
thor_status thor_last_run_ms(const thor_ctx *ctx, float *ms);

/* Time, in milliseconds from kernel entry (device %globaltimer), at which the photon counter of the last thor_run was
 * first found exhausted: until then the walk is fed (throughput phase); the rest of thor_last_run_ms is the drain of
 * the packets in flight, whose length is set by the longest single packet. */
thor_status thor_last_run_feed_ms(const thor_ctx *ctx, float *ms);

/* Largest scattering count of any single packet of the last thor_run: the longest dependent chain, which bounds the
 * drain phase from below. */
thor_status thor_last_run_max_nscat(const thor_ctx *ctx, unsigned long long *n);

/* tallies */
#define THOR_TALLY_SPECTRUM 0   /* uint64[spec_bins + 2]: bins, then underflow, overflow */
#define THOR_TALLY_NSCAT_HIST 1 /* uint64[64]: bin 0: nscat = 0; bin b: 2^(b-1) <= nscat < 2^b */
#define THOR_TALLY_COUNTERS 2   /* uint64[THOR_N_COUNTERS] */
#define THOR_TALLY_CUBE 3       /* double[peel_ny][peel_nx][peel_nv] (kept as 2^-32 fixed point on the device) */
#define THOR_TALLY_RAW 4        /* thor_raw_record[n_photons] of the last run */
#define THOR_TALLY_DEVICE_DST 0x100 /* OR into kind: dst is a DEVICE pointer (CUBE then yields uint64 fixed point) */

enum { THOR_CT_ESCAPED = 0, THOR_CT_ABSORBED, THOR_CT_TERMINATED, THOR_CT_CAPPED, THOR_CT_SCATTERINGS,
       THOR_CT_CROSSINGS, THOR_CT_REJ_ITERS, THOR_CT_PEEL_RAYS, THOR_CT_PEEL_CELLS, THOR_CT_DUST_SCATTERINGS,
       THOR_N_COUNTERS };

typedef struct thor_raw_record {
    float V;          /* lab-frame velocity offset from line centre at the end, km/s */
    uint32_t nscat;   /* saturates at 2^32-1 */
    int32_t status;   /* THOR_CT_ESCAPED .. THOR_CT_CAPPED */
    float kx, ky, kz; /* final direction */
} thor_raw_record;

/* Copies tally `kind` into dst (HOST unless THOR_TALLY_DEVICE_DST).  *needed (may be NULL) receives the size in
 * bytes; THOR_ERR_ARG if dst_bytes is smaller (nothing is written); dst == NULL just queries the size.
 * THOR_ERR_STATE if the last run did not produce that tally. */
thor_status thor_tally_get(thor_ctx *ctx, int kind, void *dst, size_t dst_bytes, size_t *needed);

/* Ray-tracing operators on the context's grid (PAPER.md 3.5; the same DDA, gather and Voigt function as the walk).
 * org_xyz, dir_xyz: DEVICE float[n_rays][3], origins in cell units inside the grid and unit directions; each ray is
 * marched to the first box face.  Outputs are DEVICE arrays, any may be NULL:
 *   out_column[n_rays]     Int n_HI ds [cm^-2]                         (projection, PAPER.md 3.5.1 with q = n_HI, w = 1)
 *   out_tmean[n_rays]      Int T n_HI ds / Int n_HI ds [K]              (weighted average Q / Q^, w = n_HI)
 *   out_tau[n_rays][n_v]   tau(V_j), V_j = v_lo + (j + 1/2)(v_hi - v_lo)/n_v [km/s offset from line centre at the
 *                          ray origin]: Eq. 11 (PAPER.md 3.5.2) with the gas frequency shifted by its line-of-sight
 *                          velocity and the Hubble term hubble_kms_per_cell * s (s = path length in cells), dust
 *                          absorption included.
 * One kernel launch; synchronous.  THOR_ERR_ARG for NULL / empty inputs or a bad velocity axis. */
thor_status thor_raytrace(thor_ctx *ctx, long long n_rays, const float *org_xyz, const float *dir_xyz,
                          double hubble_kms_per_cell, int n_v, double v_lo, double v_hi, float *out_column,
                          float *out_tmean, float *out_tau);

/* Volume rendering (PAPER.md 3.5.3, Eq. 12): C = Int_0^L c(s) mu(s) exp(-Int_0^s mu dt) ds along each ray, the observer
 * at the ray origin, rays as in thor_raytrace.  Transfer function as in PAPER.md:510 (Gaussian peaks in log10 T,
 * brightness weighted by density): peaks = HOST float[n_peaks][6] rows {log10 T centre, width [dex] > 0, R, G, B, A >= 0},
 * 1 <= n_peaks <= THOR_MAX_TF_PEAKS (copied); g_p = exp(-(log10 T - c_p)^2 / (2 s_p^2)); absorption coefficient per
 * cell length mu = w Sum_p A_p g_p, emission c mu = w Sum_p A_p g_p (R,G,B)_p, w = n_HI / n_ref, or 1 if n_ref == 0.
 * Cells are piecewise constant, each face-to-face segment is integrated exactly (reading A25).
 * out_rgba: DEVICE float[n_rays][4] = (C_R, C_G, C_B, 1 - exp(-Int mu)).  One kernel launch; synchronous.
 * THOR_ERR_ARG for NULL / empty inputs, n_peaks out of range, a non-positive width, negative A or n_ref. */
#define THOR_MAX_TF_PEAKS 8
thor_status thor_volume_render(thor_ctx *ctx, long long n_rays, const float *org_xyz, const float *dir_xyz,
                               int n_peaks, const float *peaks, double n_ref, float *out_rgba);

/* The same operators with the sight lines of the paper's Lyα-forest application and with HOST buffers.
 *   max_length_cells > 0: the ray wraps at the faces the grid was declared periodic on and ends after that path length
 *                         (in cell lengths), or at the first non-periodic face; 0: ends at the first box face.
 *   hubble_eps > 0:       Eq. 11 is sub-sampled: each face-to-face segment is cut into ceil(|H len| / (hubble_eps v_th))
 *                         sub-steps with the Hubble term at each sub-step's midpoint ("each ray step ... much smaller than
 *                         the line width"; the rule of reading A12); 0: one midpoint per segment, as thor_raytrace.
 *   flags & THOR_RAYS_HOST: org_xyz, dir_xyz and every output are HOST pointers; the library stages them through device
 *                         buffers of its own inside the call (else DEVICE pointers, as thor_raytrace). */
#define THOR_RAYS_HOST 0x1u
typedef struct thor_ray_opts {
    uint32_t struct_size;             /* = sizeof(thor_ray_opts) */
    uint32_t flags;                   /* THOR_RAYS_HOST */
    double hubble_kms_per_cell, hubble_eps;
    double max_length_cells;
    int32_t n_v;
    double v_lo, v_hi;
} thor_ray_opts;
thor_status thor_raytrace_ex(thor_ctx *ctx, long long n_rays, const float *org_xyz, const float *dir_xyz,
                             const thor_ray_opts *opts, float *out_column, float *out_tmean, float *out_tau);
thor_status thor_volume_render_ex(thor_ctx *ctx, long long n_rays, const float *org_xyz, const float *dir_xyz,
                                  int n_peaks, const float *peaks, double n_ref, float *out_rgba, unsigned flags);

/* Slice operator: out[i] = the value of one field in the cell that holds point pos_xyz[i] (cell units,
 * clamped into the grid).  field: THOR_FIELD_*.  pos_xyz / out are DEVICE pointers, or HOST with THOR_RAYS_HOST.
 * THOR_ERR_ARG for NULL / empty input, an unknown field, or kdust on a grid without dust. */
#define THOR_FIELD_NHI 0
#define THOR_FIELD_T 1
#define THOR_FIELD_VX 2
#define THOR_FIELD_VY 3
#define THOR_FIELD_VZ 4
#define THOR_FIELD_KDUST 5
thor_status thor_slice(thor_ctx *ctx, long long n_points, const float *pos_xyz, int field, float *out, unsigned flags);

/* Static-lifetime or context-owned text of the last error (ctx may be NULL for create-time errors). */
const char *thor_last_error(const thor_ctx *ctx);

/* ---- single steps of the path, for parity tests and micro-benchmarks.  All arrays are DEVICE pointers; `stream`
 * as above.  Each call launches one kernel and synchronises. ---- */

/* a1 RNG: out[i*n_draws + d] = draw d of photon (id0 + i) under seed — Philox4x32-10, counter = (d>>2 lo, d>>2 hi,
 * id lo, id hi), key = (seed lo, seed hi), word d&3 (reading A16; cuRAND's curand_init(seed, id, 0) layout). */
thor_status thor_unit_philox(uint64_t seed, uint64_t id0, long long n_ids, int n_draws, uint32_t *out, void *stream);

/* The same draws through cuRAND's own device API — curand_init(seed, id0 + i, 0) on a curandStatePhilox4_32_10_t, then
 * curand4() word by word — to pin reading A16's counter / key layout against the library that defines it. */
thor_status thor_unit_curand_philox(uint64_t seed, uint64_t id0, long long n_ids, int n_draws, uint32_t *out, void *stream);

/* a4 DDA: traces n rays (org, dir: float[n][3], cell units) through an (nx,ny,nz) grid with `periodic_flags`
 * (THOR_PERIODIC_*), at most max_steps cells each.  Per ray: hash_idx = word-wise FNV-1a (offset 0xCBF29CE484222325,
 * prime 0x100000001B3, h = (h ^ w) * prime) over the 64-bit linear indices of the visited cells, hash_len = the same
 * over the fp32 bit patterns of the segment lengths, count = cells visited.  If seq_idx/seq_len are non-NULL (n must
 * be 1) the visited indices / lengths are written there (max_steps entries). */
thor_status thor_unit_dda_trace(int nx, int ny, int nz, unsigned periodic_flags, long long n, const float *org,
                                const float *dir, long long max_steps, uint64_t *hash_idx, uint64_t *hash_len,
                                uint32_t *count, int64_t *seq_idx, float *seq_len, void *stream);

/* a6 Voigt: out[i] = H(a[i], x[i]) (normalisation of Eq. 6). */
thor_status thor_unit_voigt(long long n, const float *a, const float *x, float *out, void *stream);

/* a8-a11: n independent scatterings at gas-frame x_in with Voigt parameter a, incoming direction +z, photon stream
 * (seed, id0 + i): writes u_par[n], x_out[n], k_out[n][3], iters[n] (rejection iterations).  Any output may be NULL. */
thor_status thor_unit_scatter(float a, float x_in, float x_crit, int phase, uint64_t seed, uint64_t id0, long long n,
                              float *u_par, float *x_out, float *k_out, uint32_t *iters, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* THOR_B200_H */
