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
#ifndef THOR_PEEL_MIN_CTAS
#define THOR_PEEL_MIN_CTAS 2
#endif
#ifndef THOR_FINISH_MIN_LANES
#define THOR_FINISH_MIN_LANES 24
#endif
constexpr int WALK_THREADS = THOR_WALK_THREADS;
constexpr int MAX_SPEC_BINS = 4096;
constexpr int FINISH_MIN_LANES = THOR_FINISH_MIN_LANES;
#ifndef THOR_REFILL_MIN_LANES
#define THOR_REFILL_MIN_LANES 1
#endif
constexpr int REFILL_MIN_LANES = THOR_REFILL_MIN_LANES;
#ifndef THOR_COOP_MAX_LANES
#define THOR_COOP_MAX_LANES 4
#endif
#ifndef THOR_PARK1_LANES
#define THOR_PARK1_LANES 16
#endif
constexpr int PARK1_LANES = THOR_PARK1_LANES;           // every pass of the tail but the last: a warp parks at this many live lanes
#ifndef THOR_TAIL_PASSES
#define THOR_TAIL_PASSES 3
#endif
constexpr int TAIL_PASSES = THOR_TAIL_PASSES;           // launches of the walk kernel per run (1 feed + re-packed passes of the tail)
constexpr int COOP_MAX_LANES = THOR_COOP_MAX_LANES;     // cooperative drain when a warp has at most this many packets left
constexpr int WIN_STRIDE = 20;                          // floats per window slot (16 used; 80 B keeps STS.128 conflict-free)
constexpr int PK_WORDS = 48;                            // 32-bit words of a parked packet

struct BlockTallies {
    float2 voigt[VOIGT_NODES];
    unsigned long long counters[N_COUNTERS];
    unsigned int nscat_hist[64];
    unsigned int max_nscat;
    unsigned int spectrum[MAX_SPEC_BINS + 2];
};

constexpr int DRAIN_THREADS = 128;                     // drain kernel: 4 warps per CTA, one per SM sub-partition
constexpr int DRAIN_WARPS = DRAIN_THREADS / 32;

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

__device__ __forceinline__ void tally_packet(const WalkParams& p, BlockTallies& sh, int ev, const Packet& k) {
    const int status = ev == EV_ESCAPED ? CT_ESCAPED : ev == EV_ABSORBED ? CT_ABSORBED : ev == EV_TERMINATED ? CT_TERMINATED : CT_CAPPED;
    tally_finish(p, sh, status, k.V, k.nscat, k.crossings, k.rej_iters, k.rng.id(), k.ray.kx, k.ray.ky, k.ray.kz);
}

// ---- cooperative drain --------------------------------------------------------------------------
// When the photon counter is dry and a warp is down to a few packets, every further scattering is a serial chain of
// ~590 dependent instructions issued for one live lane (measured: 1.29 us per scattering).  Most of that chain does not
// depend on the packet's state at all: the Philox blocks (3 per scattering, ~45 instructions each) and everything
// computed from uniforms alone (-ln r, sin/cos of random angles, the dipole inversion, the Lorentzian angle of a
// line-centre trial).  So the warp's 32 lanes turn to ONE packet at a time: lane i generates counter block b + i of that
// packet and works out those quantities (a window of 32 blocks, ~10 scatterings' worth, in shared memory), then all
// lanes step the packet redundantly — same instructions, same operands, warp-uniform control flow — reading the window
// instead of computing.  Blocks are consumed in the packet's own order (trial, trial, ..., finish, finish), so the walk
// is bit-identical to the staged loop's.  Packets of the warp take turns, one window each.
template <bool GL>
__device__ __forceinline__ void park_store(uint32_t* w, const Packet& k, int state) {
    w[0] = (uint32_t)k.ray.cx; w[1] = (uint32_t)k.ray.cy; w[2] = (uint32_t)k.ray.cz;
    w[3] = __float_as_uint(k.ray.fx); w[4] = __float_as_uint(k.ray.fy); w[5] = __float_as_uint(k.ray.fz);
    w[6] = __float_as_uint(k.ray.kx); w[7] = __float_as_uint(k.ray.ky); w[8] = __float_as_uint(k.ray.kz);
    w[9] = __float_as_uint(k.ray.ix); w[10] = __float_as_uint(k.ray.iy); w[11] = __float_as_uint(k.ray.iz);
    w[12] = __float_as_uint(k.cell.a); w[13] = __float_as_uint(k.cell.vth); w[14] = __float_as_uint(k.cell.inv_vth);
    w[15] = __float_as_uint(k.cell.nsig); w[16] = __float_as_uint(k.cell.kd);
    w[17] = __float_as_uint(k.cell.vx); w[18] = __float_as_uint(k.cell.vy); w[19] = __float_as_uint(k.cell.vz);
    w[20] = k.rng.id_lo; w[21] = k.rng.id_hi; w[22] = k.rng.b_lo; w[23] = k.rng.b_hi;
    w[24] = __float_as_uint(k.V); w[25] = __float_as_uint(k.tau_rem); w[26] = __float_as_uint(k.hit_kt);
    w[27] = __float_as_uint(k.x_in); w[28] = __float_as_uint(k.upar);
    w[29] = k.nscat; w[30] = k.crossings; w[31] = k.rej_iters; w[32] = k.trials;
    w[33] = (k.stale ? 1u : 0u) | (k.inv_ok ? 2u : 0u); w[34] = (uint32_t)state;
    w[35] = __float_as_uint(k.hit_k2); w[42] = (uint32_t)k.line;
    if (GL) {
        const unsigned long long x = (unsigned long long)__double_as_longlong(k.gx), y = (unsigned long long)__double_as_longlong(k.gy),
                                 z = (unsigned long long)__double_as_longlong(k.gz);
        w[36] = (uint32_t)x; w[37] = (uint32_t)(x >> 32); w[38] = (uint32_t)y; w[39] = (uint32_t)(y >> 32);
        w[40] = (uint32_t)z; w[41] = (uint32_t)(z >> 32);
    }
}

template <bool GL>
__device__ __forceinline__ int park_load(const uint32_t* w, Packet& k) {
    k.ray.cx = (int)w[0]; k.ray.cy = (int)w[1]; k.ray.cz = (int)w[2];
    k.ray.fx = __uint_as_float(w[3]); k.ray.fy = __uint_as_float(w[4]); k.ray.fz = __uint_as_float(w[5]);
    k.ray.kx = __uint_as_float(w[6]); k.ray.ky = __uint_as_float(w[7]); k.ray.kz = __uint_as_float(w[8]);
    k.ray.ix = __uint_as_float(w[9]); k.ray.iy = __uint_as_float(w[10]); k.ray.iz = __uint_as_float(w[11]);
    k.cell.a = __uint_as_float(w[12]); k.cell.vth = __uint_as_float(w[13]); k.cell.inv_vth = __uint_as_float(w[14]);
    k.cell.nsig = __uint_as_float(w[15]); k.cell.kd = __uint_as_float(w[16]);
    k.cell.vx = __uint_as_float(w[17]); k.cell.vy = __uint_as_float(w[18]); k.cell.vz = __uint_as_float(w[19]);
    k.rng.id_lo = w[20]; k.rng.id_hi = w[21]; k.rng.b_lo = w[22]; k.rng.b_hi = w[23];
    k.V = __uint_as_float(w[24]); k.tau_rem = __uint_as_float(w[25]); k.hit_kt = __uint_as_float(w[26]);
    k.x_in = __uint_as_float(w[27]); k.upar = __uint_as_float(w[28]);
    k.nscat = w[29]; k.crossings = w[30]; k.rej_iters = w[31]; k.trials = w[32];
    k.stale = (w[33] & 1u) != 0u; k.inv_ok = (w[33] & 2u) != 0u;
    k.hit_k2 = __uint_as_float(w[35]); k.line = (int)w[42];
    if (GL) {
        k.gx = __longlong_as_double((long long)(((unsigned long long)w[37] << 32) | w[36]));
        k.gy = __longlong_as_double((long long)(((unsigned long long)w[39] << 32) | w[38]));
        k.gz = __longlong_as_double((long long)(((unsigned long long)w[41] << 32) | w[40]));
    }
    return (int)w[34];
}

// Lane i of the warp generates counter block (b + i) of packet `k` and stores, per block, the uniforms and what the
// event code would compute from them alone, for each role the block can end up in:
//   q0 = (u.x, u.y, u.z, u.w)                           any role
//   q1 = (sin, cos of pi u.y; -ln u.x; dipole_mu(u.y))  trial: Lorentzian angle when psi0 = 0 | first FINISH block: tau', mu
//   q2 = (sin, cos of 2 pi u.z; -ln u.w; 0)             first FINISH block: azimuth of k', |u_perp|^2
//   q3 = (sin, cos of 2 pi u.x; 0; 0)                   second FINISH block: angle of u_perp
__device__ __forceinline__ void coop_fill_window(float4* win, const BlockRng& rng, uint32_t k0, uint32_t k1, unsigned lane,
                                                 float4& my_u, float& my_sC, float& my_cC) {
    const uint32_t lo = rng.b_lo + lane, hi = rng.b_hi + (lo < rng.b_lo ? 1u : 0u);
    const U4 r = philox4x32_10(lo, hi, rng.id_lo, rng.id_hi, k0, k1);
    const float4 u = make_float4(u01(r.x), u01(r.y), u01(r.z), u01(r.w));
    float4 q1, q2, q3;
    sincospif(u.y, &q1.x, &q1.y);
    q1.z = neg_log(u.x);
    q1.w = dipole_mu(u.y);
    sincos_uniform(u.z, q2.x, q2.y);
    q2.z = neg_log(u.w); q2.w = 0.f;
    sincos_uniform(u.x, q3.x, q3.y);
    q3.z = 0.f; q3.w = 0.f;
    float4* slot = win + 5 * lane;
    slot[0] = u; slot[1] = q1; slot[2] = q2; slot[3] = q3;
    my_u = u; my_sC = q1.x; my_cC = q1.y;
}

// Longest first: a packet that has already scattered the most is the one most likely to go on the longest (the
// scattering counts are heavy-tailed), and the launch ends when its longest packet does.  order[r] = the pool slot with the
// r-th largest scattering count so far (ties by slot); one thread per slot, a scan of the pool's counts each.
__global__ void pool_order_kernel(const __grid_constant__ WalkParams p) {
    const unsigned long long n = *p.pool_count;
    const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t mine = p.pool[i * PK_WORDS + 29];          // word 29 = nscat (park_store)
    unsigned int rank = 0;
    for (unsigned long long j = 0; j < n; ++j) {
        const uint32_t o = __ldg(p.pool + j * PK_WORDS + 29);
        rank += (o > mine || (o == mine && j < i)) ? 1u : 0u;
    }
    p.pool_order[rank] = (unsigned int)i;
}

// ---- deferred peel rays --------------------------------------------------------------------------
// Most peel rays end in the packet's own cell (optically thick: tau > tau_peel_max) and the few that go on cross tens to
// thousands of cells.  Marched in place they hold the warp at ONE active lane: 43 % of the walk kernel's issued
// instructions on config 5 (profiles/r02_lanes.md).  So the walk kernel marches only the first cell in place and puts a
// ray that goes on into a per-warp queue in shared memory (10 words: cell, offset, tau, V, weight, pixel); when 32 have
// gathered the warp serves them, one ray per lane and one cell per turn, topping idle lanes up from the queue and putting
// the unfinished rays back once fewer than PEEL_MIN_ACTIVE are left.  The cube is fixed point, so the order of its
// additions changes nothing: tallies stay bit-identical to the in-place march.
constexpr int PEELQ_CAP = 64;                           // entries per warp (at most PEEL_MIN_ACTIVE - 1 + 32 are ever queued)
constexpr int PEELQ_WORDS = 10;
constexpr int PEELQ_SERVE = 32;                         // serve when this many are queued
#ifndef THOR_PEEL_MIN_ACTIVE
#define THOR_PEEL_MIN_ACTIVE 16
#endif
constexpr int PEEL_MIN_ACTIVE = THOR_PEEL_MIN_ACTIVE;

// Queue layout: word w of entry e at q[w * PEELQ_CAP + e] (consecutive lanes, consecutive banks).
__device__ __forceinline__ void peelq_put(uint32_t* q, int e, const PeelPend& d) {
    q[0 * PEELQ_CAP + e] = (uint32_t)d.cx; q[1 * PEELQ_CAP + e] = (uint32_t)d.cy; q[2 * PEELQ_CAP + e] = (uint32_t)d.cz;
    q[3 * PEELQ_CAP + e] = __float_as_uint(d.fx); q[4 * PEELQ_CAP + e] = __float_as_uint(d.fy); q[5 * PEELQ_CAP + e] = __float_as_uint(d.fz);
    q[6 * PEELQ_CAP + e] = __float_as_uint(d.tau); q[7 * PEELQ_CAP + e] = __float_as_uint(d.V);
    q[8 * PEELQ_CAP + e] = __float_as_uint(d.phat); q[9 * PEELQ_CAP + e] = (uint32_t)d.pix;
}
__device__ __forceinline__ void peelq_get(const uint32_t* q, int e, PeelPend& d) {
    d.cx = (int)q[0 * PEELQ_CAP + e]; d.cy = (int)q[1 * PEELQ_CAP + e]; d.cz = (int)q[2 * PEELQ_CAP + e];
    d.fx = __uint_as_float(q[3 * PEELQ_CAP + e]); d.fy = __uint_as_float(q[4 * PEELQ_CAP + e]); d.fz = __uint_as_float(q[5 * PEELQ_CAP + e]);
    d.tau = __uint_as_float(q[6 * PEELQ_CAP + e]); d.V = __uint_as_float(q[7 * PEELQ_CAP + e]);
    d.phat = __uint_as_float(q[8 * PEELQ_CAP + e]); d.pix = (int)q[9 * PEELQ_CAP + e];
}

// The lanes whose `pend` is live append it to the warp's queue (whole warp calls; cnt is warp-uniform).
__device__ __forceinline__ void peelq_push(uint32_t* q, int& cnt, PeelPend& pend, unsigned lane) {
    const unsigned m = __ballot_sync(0xffffffffu, pend.live);
    if (!m) return;
    if (pend.live) peelq_put(q, cnt + __popc(m & ((1u << lane) - 1u)), pend);
    pend.live = false;
    cnt += __popc(m);
    __syncwarp();
}

// Serve the queue (whole warp calls).  flush: to the last ray (before the warp leaves the kernel).
template <bool HUBBLE>
__device__ __noinline__ void peelq_serve(const WalkParams& p, const float2* s_tab, uint32_t* q, int& cnt, uint32_t& n_cells,
                                        bool flush, unsigned lane) {
    PeelPend d;
    d.live = false;
    Ray r;
    peel_ray_direction(p, r);
    for (;;) {
        const unsigned idle = __ballot_sync(0xffffffffu, !d.live);
        if (idle && cnt > 0) {                                // top idle lanes up from the back of the queue
            const int take = min(__popc(idle), cnt);
            const int rank = __popc(idle & ((1u << lane) - 1u));
            if (!d.live && rank < take) {
                peelq_get(q, cnt - 1 - rank, d);
                r.cx = d.cx; r.cy = d.cy; r.cz = d.cz; r.fx = d.fx; r.fy = d.fy; r.fz = d.fz;
                if (d.pix == PEEL_PIX_UNSET) d.pix = peel_pixel(p, r);      // a ray queued whole (drain kernel) starts here
                d.live = d.pix >= 0;
            }
            cnt -= take;
            __syncwarp();
        }
        const unsigned act = __ballot_sync(0xffffffffu, d.live);
        if (!act) return;
        if (!flush && __popc(act) < PEEL_MIN_ACTIVE) {        // too few left (the queue is empty): back they go
            if (d.live) {
                d.cx = r.cx; d.cy = r.cy; d.cz = r.cz; d.fx = r.fx; d.fy = r.fy; d.fz = r.fz;
                peelq_put(q, cnt + __popc(act & ((1u << lane) - 1u)), d);
            }
            cnt += __popc(act);
            __syncwarp();
            return;
        }
        if (d.live) {
            const Cell c = load_cell(p, dda_linear(r, p.g));
            const int st = peel_cell<HUBBLE>(p, s_tab, r, c, d.tau, d.V, n_cells);
            if (st != PEEL_NEXT) {
                if (st == PEEL_LEFT) peel_deposit(p, d.pix, d.V, d.tau, d.phat, true);
                d.live = false;
            }
        }
    }
}

// The drain kernel: launched behind walk_kernel on the same stream.  Each warp pops one parked packet at a time from the
// global pool and walks it to its end, all 32 lanes on that one packet (see above).  4 warps per CTA — one per SM
// sub-partition — and a register budget of its own (the walk kernel is held to 80 registers by its occupancy).
template <bool HUBBLE, bool PEEL, bool GL, bool DB, int FIN>
__global__ void __launch_bounds__(DRAIN_THREADS, 4) drain_kernel(const __grid_constant__ WalkParams p) {
    __shared__ BlockTallies sh;
    __shared__ float4 s_win[DRAIN_WARPS][32 * WIN_STRIDE / 4];
    __shared__ uint32_t sh_peelq[PEEL ? DRAIN_WARPS * PEELQ_CAP * PEELQ_WORDS : 1];
    voigt_table_load(sh.voigt);
    for (int i = threadIdx.x; i < N_COUNTERS; i += blockDim.x) sh.counters[i] = 0ull;
    for (int i = threadIdx.x; i < 64; i += blockDim.x) sh.nscat_hist[i] = 0u;
    if (threadIdx.x == 0) sh.max_nscat = 0u;
    for (int i = threadIdx.x; i < p.spec_bins + 2; i += blockDim.x) sh.spectrum[i] = 0u;
    __syncthreads();
    const unsigned lane = threadIdx.x & 31u;
    const uint32_t k0 = (uint32_t)p.seed, k1 = (uint32_t)(p.seed >> 32);
    float4* win = s_win[threadIdx.x >> 5];
    const unsigned long long n_pool = *p.pool_count;
    uint32_t pr = 0, pc = 0, ds = 0;
    // Peel rays are queued whole and served 32 at a time, one per lane: a ray is ~230 of the ~900 dependent
    // instructions of a scattering but nothing in the packet's walk waits for it — the one place where this warp's lanes do
    // different work.
    uint32_t* const peelq = sh_peelq + (PEEL ? (threadIdx.x >> 5) * PEELQ_CAP * PEELQ_WORDS : 0);
    int peelq_cnt = 0;
    PeelPend pend;
    pend.live = false;
    const int need0 = (DB && p.doublet_on) ? 4 : 3;                   // blocks one scattering takes at least: [select,] trial, 2 x finish
    Packet k;
    for (;;) {
        unsigned long long slot = 0;
        if (lane == 0) slot = atomicAdd(p.pool_next, 1ull);
        slot = __shfl_sync(0xffffffffu, slot, 0);
        if (slot >= n_pool) break;
        slot = p.pool_order[slot];
        int st = park_load<GL>(p.pool + slot * PK_WORDS, k);      // every lane reads the same words: one broadcast per load
        int c = 32;                                           // first unconsumed block of the window (32 = none left)
        float4 my_u = make_float4(0.f, 0.f, 0.f, 0.f);        // this lane's own block of the window
        float my_sC = 0.f, my_cC = 0.f;
        UparEnvelope env;
        env.mTot = -1.f;
        float xc = -1.f;                                      // x_crit of the packet's present cell, once known (finish_scatter)
        for (;;) {
            if (st == LS_MARCH) {
                const int ev = GL ? march_step_gridless(p, sh.voigt, k) : march_step<HUBBLE, false, DB>(p, sh.voigt, k);
                if (ev == EV_CROSSED) { xc = -1.f; continue; }
                if (ev != EV_HIT) { if (lane == 0) tally_packet(p, sh, ev, k); break; }
                st = (DB && p.doublet_on) ? LS_SELECT : LS_TRIAL;
                env.mTot = -1.f;
            }
            if (c + need0 > 32) {                                 // fewer than a trial + a FINISH left: a new window
                __syncwarp();
                coop_fill_window(win, k.rng, k0, k1, lane, my_u, my_sC, my_cC);
                __syncwarp();
                c = 0;
            }
            if (DB && st == LS_SELECT) {                      // doublet: which interaction, from one more block
                const float4 u = win[5 * c];
                ++c;
                k.rng.b_lo += 1u; k.rng.b_hi += (k.rng.b_lo == 0u);
                select_line(p, k, u.x);
                st = k.line < 0 ? LS_FINISH : LS_TRIAL;
            }
            if (st == LS_TRIAL) {
                // every lane tries its OWN block; the packet takes the first acceptance at or after block c — exactly the
                // trial the sequential rejection loop would have accepted, found in one step however many it rejects
                if (env.mTot < 0.f) env = upar_envelope(line_a<DB>(p, k), fabsf(k.x_in));
                float uu;
                const bool ok = upar_try<true>(env, line_a<DB>(p, k), my_u, my_sC, my_cC, uu);
                const unsigned acc = __ballot_sync(0xffffffffu, ok) & ~((1u << c) - 1u);
                const uint32_t nrej = (uint32_t)((acc ? __ffs(acc) - 1 : 32) - c);   // rejections before the first acceptance
                uint32_t ntr;                                 // blocks this step consumes
                bool done_trial;
                if (k.trials + nrej >= (1u << 20)) {          // fail-safe of the sequential loop: its 2^20-th rejection is taken
                    ntr = (1u << 20) - k.trials;
                    k.trials = 1u << 20;
                    done_trial = true;
                } else {
                    k.trials += nrej;
                    done_trial = acc != 0u;
                    ntr = nrej + (done_trial ? 1u : 0u);
                }
                const int jj = c + (int)ntr - 1;              // the block whose u is taken, if any
                k.rej_iters += ntr;
                const uint32_t lo = k.rng.b_lo;
                k.rng.b_lo += ntr; k.rng.b_hi += (k.rng.b_lo < lo);
                c += (int)ntr;
                if (!done_trial) continue;                    // the whole window rejected: refill, keep trying
                uu = __shfl_sync(0xffffffffu, uu, jj);
                k.upar = k.x_in < 0.f ? -uu : uu;
                st = LS_FINISH;
                if (c + 2 > 32) continue;                     // FINISH needs two more blocks: refill first
            }
            {   // LS_FINISH: blocks c, c + 1
                const float4 u1 = win[5 * c], a1 = win[5 * c + 1], a2 = win[5 * c + 2];
                const float4 u2 = win[5 * c + 5], b3 = win[5 * c + 8];
                c += 2;
                k.rng.b_lo += 2u; k.rng.b_hi += (k.rng.b_lo < 2u);
                FinDraws d;
                d.tau_next = a1.z; d.r_mu = u1.y; d.mu_dip = a1.w;
                d.sphi = a2.x; d.cphi = a2.y; d.nl_p1 = a2.z;
                d.spsi = b3.x; d.cpsi = b3.y; d.u_dust = u2.y; d.u_mix = u2.z; d.u_alb = u2.w;
                uint32_t none = 0;
                const int ev = finish_scatter<HUBBLE, PEEL, true, PEEL_QUEUED, DB, FIN>(p, sh.voigt, k, d, pr, none, lane == 0, &pend, &xc);
                if (PEEL && pend.live) {                      // warp-uniform: every lane holds the same ray
                    if (lane == 0) peelq_put(peelq, peelq_cnt, pend);
                    pend.live = false;
                    ++peelq_cnt;
                    __syncwarp();
                    if (peelq_cnt >= PEELQ_SERVE) peelq_serve<HUBBLE>(p, sh.voigt, peelq, peelq_cnt, pc, false, lane);
                }
                if (ev == EV_DUST_SCATTERED) ++ds;
                else if (ev != EV_SCATTERED) { if (lane == 0) tally_packet(p, sh, ev, k); break; }
                st = LS_MARCH;
            }
        }
    }
    if (PEEL) {
        if (peelq_cnt > 0) peelq_serve<HUBBLE>(p, sh.voigt, peelq, peelq_cnt, pc, true, lane);
        pc = __reduce_add_sync(0xffffffffu, pc);               // cells are counted by the lane that marched them
    }
    if (lane == 0) {
        atomicAdd(&sh.counters[CT_PEEL_RAYS], (unsigned long long)pr);
        atomicAdd(&sh.counters[CT_PEEL_CELLS], (unsigned long long)pc);
        if (ds) atomicAdd(&sh.counters[CT_DUST_SCATTERINGS], (unsigned long long)ds);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < N_COUNTERS; i += blockDim.x)
        if (sh.counters[i]) atomicAdd(p.counters + i, sh.counters[i]);
    for (int i = threadIdx.x; i < 64; i += blockDim.x)
        if (sh.nscat_hist[i]) atomicAdd(p.nscat_hist + i, (unsigned long long)sh.nscat_hist[i]);
    if (threadIdx.x == 0 && sh.max_nscat) atomicMax(p.max_nscat, (unsigned long long)sh.max_nscat);
    for (int i = threadIdx.x; i < p.spec_bins + 2; i += blockDim.x)
        if (sh.spectrum[i]) atomicAdd(p.spectrum + i, (unsigned long long)sh.spectrum[i]);
}

template <bool HUBBLE, bool PEEL, int MIN_CTAS, bool GL, bool DB, int FIN>
__global__ void __launch_bounds__(WALK_THREADS, MIN_CTAS) walk_kernel(const __grid_constant__ WalkParams p) {
    __shared__ BlockTallies sh;
    __shared__ uint32_t sh_peelq[PEEL ? (WALK_THREADS / 32) * PEELQ_CAP * PEELQ_WORDS : 1];
    if (threadIdx.x == 0) atomicMin(p.t_start, global_timer_ns());
    voigt_table_load(sh.voigt);
    for (int i = threadIdx.x; i < N_COUNTERS; i += blockDim.x) sh.counters[i] = 0ull;
    for (int i = threadIdx.x; i < 64; i += blockDim.x) sh.nscat_hist[i] = 0u;
    if (threadIdx.x == 0) sh.max_nscat = 0u;
    for (int i = threadIdx.x; i < p.spec_bins + 2; i += blockDim.x) sh.spectrum[i] = 0u;
    __syncthreads();

    uint32_t* const peelq = sh_peelq + (PEEL ? (threadIdx.x >> 5) * PEELQ_CAP * PEELQ_WORDS : 0);   // this warp's queue
    int peelq_cnt = 0;                                        // warp-uniform
    PeelPend pend;
    pend.live = false;
    constexpr bool EARLY = MIN_CTAS >= 4;                     // the variant launched for grids beyond L2
    const unsigned lane = threadIdx.x & 31u;
    const uint32_t k0 = (uint32_t)p.seed, k1 = (uint32_t)(p.seed >> 32);   // Philox key = seed (reading A16)
    int state = LS_IDLE;
    Packet k;
    k.stale = true; k.inv_ok = false;
    UparEnvelope env;
    env.mTot = -1.f;
    uint32_t peel_rays = 0, peel_cells = 0, dust_scat = 0;
    bool more = !p.resume;                                    // warp-uniform: photon counter not yet exhausted
    if (p.resume) {                                           // second pass of the tail: 32 parked packets per warp, densely
        const unsigned long long n_in = *p.resume_count;
        const unsigned long long idx = ((unsigned long long)blockIdx.x * (WALK_THREADS / 32) + (threadIdx.x >> 5)) * 32ull + lane;
        state = idx < n_in ? park_load<GL>(p.resume_in + idx * PK_WORDS, k) : LS_OUT;
    }

    for (;;) {
        // ---- a14 + a2/a3: refill idle lanes from the global photon counter, emit ----
        // A lane is refilled as soon as it is idle (REFILL_MIN_LANES = 1).  Emission is a chain of dependent loads (binary
        // search of the source CDF, source cell gather) run by the few lanes that need it, but waiting for 4 / 8 / 16 idle
        // lanes before paying for it was measured slower on every workload (feed phase +7 / +16 / +36 % on config 3, +100 % on
        // config 4 at 512^3: the idle lanes cost more than the emission's poor lane count).
        const unsigned idle = __ballot_sync(0xffffffffu, state == LS_IDLE);
        if (more && idle && (__popc(idle) >= REFILL_MIN_LANES || __ballot_sync(0xffffffffu, state == LS_IDLE || state == LS_OUT) == 0xffffffffu)) {
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(p.next_photon, (unsigned long long)__popc(idle));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (state == LS_IDLE) {
                const unsigned long long i = base + __popc(idle & ((1u << lane) - 1u));
                if (i >= p.n_photons) {
                    state = LS_OUT;
                } else {
                    float dV = 0.f;
                    if (GL) emit_packet_gridless(p, k, p.id_offset + i, k0, k1);
                    else emit_packet(p, k, p.id_offset + i, k0, k1, dV);
                    if (PEEL) {
                        ++peel_rays;
                        peel_ray<HUBBLE, PEEL_FIRST>(p, sh.voigt, k.ray, k.cell,
                                         dot3(k.cell.vx, k.cell.vy, k.cell.vz, p.kobs[0], p.kobs[1], p.kobs[2]) + dV, 1.f,
                                         peel_cells, true, &pend);
                    }
                    state = LS_MARCH;
                }
            }
            if (PEEL) {
                peelq_push(peelq, peelq_cnt, pend, lane);
                if (peelq_cnt >= PEELQ_SERVE) peelq_serve<HUBBLE>(p, sh.voigt, peelq, peelq_cnt, peel_cells, false, lane);
            }
            if (__any_sync(0xffffffffu, state == LS_OUT)) {
                // the queue is empty: from here on the launch only drains the packets in flight
                if (more && lane == 0) atomicMin(p.t_dry, global_timer_ns());
                more = false;
            }
        }
        if (!more && p.park_out) {
            // the counter is dry and this warp is down to a few packets: park them in the global pool for the drain
            // kernel (one warp per packet there) and leave
            const bool act = state == LS_MARCH || state == LS_TRIAL || state == LS_FINISH;
            const unsigned live = __ballot_sync(0xffffffffu, act);
            if (live && __popc(live) <= p.park_lanes) {
                unsigned long long base = 0;
                if (lane == 0) base = atomicAdd(p.park_count, (unsigned long long)__popc(live));
                base = __shfl_sync(0xffffffffu, base, 0);
                if (act) park_store<GL>(p.park_out + (base + __popc(live & ((1u << lane) - 1u))) * PK_WORDS, k, state);
                break;
            }
        }

        // ---- a4-a7: one cell step for every marching lane ----
        if (state == LS_MARCH) {
            const int ev = GL ? march_step_gridless(p, sh.voigt, k) : march_step<HUBBLE, EARLY, DB>(p, sh.voigt, k);
            if (ev == EV_HIT) {
                env.mTot = -1.f;                                  // envelope not built yet
                state = LS_TRIAL;
                if (DB && p.doublet_on) {                         // which interaction: one more counter block
                    select_line(p, k, k.rng.next4(k0, k1).x);
                    if (k.line < 0) state = LS_FINISH;            // dust: no atom velocity to draw
                }
            } else if (ev != EV_CROSSED) { tally_packet(p, sh, ev, k); state = LS_IDLE; }
        }

        // ---- a8: ONE rejection trial of u_par for every lane that needs one.  No inner loop: a
        // lane whose trial is rejected tries again in the next iteration, alongside the lanes that arrive from the
        // march, instead of the whole warp waiting for its slowest lane (the paper's "largest source of thread
        // divergence"; E[max of 32 iterations]/E[iterations] = 2.1-4.2) ----
        if (state == LS_TRIAL) {
            if (env.mTot < 0.f) env = upar_envelope(line_a<DB>(p, k), fabsf(k.x_in));
            ++k.rej_iters;
            float u;
            const bool ok = upar_try<false>(env, line_a<DB>(p, k), k.rng.next4(k0, k1), 0.f, 0.f, u);
            // fail-safe: acceptance is >= ~0.2 everywhere; 2^20 rejections cannot happen unless x is NaN
            if (ok || ++k.trials >= (1u << 20)) { k.upar = k.x_in < 0.f ? -u : u; state = LS_FINISH; }
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
                const float4 s1 = k.rng.next4(k0, k1), s2 = k.rng.next4(k0, k1);
                const FinDraws d = fin_draws(s1, s2);
                const int ev = finish_scatter<HUBBLE, PEEL, false, PEEL_FIRST, DB, FIN>(p, sh.voigt, k, d, peel_rays, peel_cells, true, &pend);
                if (ev == EV_SCATTERED) state = LS_MARCH;
                else if (ev == EV_DUST_SCATTERED) { state = LS_MARCH; ++dust_scat; }
                else { tally_packet(p, sh, ev, k); state = LS_IDLE; }
            }
            if (PEEL) {
                peelq_push(peelq, peelq_cnt, pend, lane);
                if (peelq_cnt >= PEELQ_SERVE) peelq_serve<HUBBLE>(p, sh.voigt, peelq, peelq_cnt, peel_cells, false, lane);
            }
        }
    }
    if (PEEL && peelq_cnt > 0) peelq_serve<HUBBLE>(p, sh.voigt, peelq, peelq_cnt, peel_cells, true, lane);

    // ---- flush the block's tallies with global atomics ----
    atomicAdd(&sh.counters[CT_PEEL_RAYS], (unsigned long long)peel_rays);
    atomicAdd(&sh.counters[CT_PEEL_CELLS], (unsigned long long)peel_cells);
    if (dust_scat) atomicAdd(&sh.counters[CT_DUST_SCATTERINGS], (unsigned long long)dust_scat);
    __syncthreads();
    for (int i = threadIdx.x; i < N_COUNTERS; i += blockDim.x)
        if (sh.counters[i]) atomicAdd(p.counters + i, sh.counters[i]);
    for (int i = threadIdx.x; i < 64; i += blockDim.x)
        if (sh.nscat_hist[i]) atomicAdd(p.nscat_hist + i, (unsigned long long)sh.nscat_hist[i]);
    if (threadIdx.x == 0 && sh.max_nscat) atomicMax(p.max_nscat, (unsigned long long)sh.max_nscat);
    for (int i = threadIdx.x; i < p.spec_bins + 2; i += blockDim.x)
        if (sh.spectrum[i]) atomicAdd(p.spectrum + i, (unsigned long long)sh.spectrum[i]);
}


// Launch configuration: one persistent grid, blocks = SMs x resident blocks per SM.  The kernel is specialised at
// compile time on (Hubble drift, peel-off) so that the common static, no-peel walk carries neither, and on the
// register budget: 3 CTAs of 256 threads per SM (<= 80 registers) when the grid fits the 126 MB L2 and the walk is
// issue-bound, 4 CTAs (64 registers, 32 warps) when it does not and the walk needs more gathers in flight
// (+18 % on the 512^3 gather workload, -6 % on the cache-resident sphere); 2 CTAs with peel-off (<= 128 registers).
// The drain kernel follows on the same stream: a persistent grid of 4-warp CTAs whose warps pop parked packets.
// Slots of ONE half of pool_mid (the packets a pass can park).
long long walk_pool_mid_slots(int n_sm) { return (long long)n_sm * 4 * (WALK_THREADS / 32) * PARK1_LANES; }

template <bool HUBBLE, bool PEEL, int MIN_CTAS, bool GL, bool DB, int FIN>
static cudaError_t launch_pair(const WalkParams& p, int n_sm, cudaStream_t stream, int* blocks_out) {
    int per_sm = 0;
    const auto walk = walk_kernel<HUBBLE, PEEL, MIN_CTAS, GL, DB, FIN>;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, walk, WALK_THREADS, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long blocks = (long long)n_sm * per_sm;
    const long long need = (long long)((p.n_photons + 31) / 32);   // few packets: spread the warps over the SMs
    if (need < blocks) blocks = need < 1 ? 1 : need;
    if (blocks_out) *blocks_out = (int)blocks;
    // The tail in passes: once the counter is dry a warp parks its packets as soon as at most PARK1_LANES are
    // live; the next launch of the same kernel re-packs them, 32 to a warp, and walks on; the warps of the last pass park at
    // COOP_MAX_LANES packets, which go to the cooperative drain.  Half-empty warps cost what full ones do, and every pass halves
    // the packets that reach the drain kernel, where a scattering costs a whole warp.  The passes alternate between the two
    // halves of pool_mid.
    const int passes = (p.pool != nullptr && p.pool_mid != nullptr) ? TAIL_PASSES : 1;
    const long long mid_slots = walk_pool_mid_slots(n_sm);
    uint32_t* const mid[2] = {p.pool_mid, p.pool_mid ? p.pool_mid + mid_slots * PK_WORDS : nullptr};
    for (int pass = 0; pass < passes; ++pass) {
        const bool last = pass == passes - 1;
        WalkParams q = p;
        q.resume = pass > 0 ? 1 : 0;
        q.resume_in = pass > 0 ? mid[(pass - 1) & 1] : nullptr;
        q.resume_count = pass > 0 ? p.pool_mid_count + ((pass - 1) & 1) : nullptr;
        q.park_out = last ? p.pool : mid[pass & 1];
        q.park_count = last ? p.pool_count : p.pool_mid_count + (pass & 1);
        q.park_lanes = last ? COOP_MAX_LANES : PARK1_LANES;
        if (pass >= 2 && !last) {                             // a half of pool_mid is used again: its count restarts
            e = cudaMemsetAsync(p.pool_mid_count + (pass & 1), 0, sizeof(unsigned long long), stream);
            if (e != cudaSuccess) return e;
        }
        walk<<<(unsigned)blocks, WALK_THREADS, 0, stream>>>(q);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        if (!last) blocks = (blocks * PARK1_LANES + 31) / 32;  // 32 parked packets per warp cover everything this pass can park
    }
    if (!p.pool) return cudaSuccess;
    const auto drain = drain_kernel<HUBBLE, PEEL, GL, DB, FIN>;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, drain, DRAIN_THREADS, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    const long long slots = blocks * (WALK_THREADS / 32) * COOP_MAX_LANES;      // most the walk kernel can have parked
    pool_order_kernel<<<(unsigned)((slots + 255) / 256), 256, 0, stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    long long dblocks = (long long)n_sm * per_sm;
    const long long cap = (slots + DRAIN_WARPS - 1) / DRAIN_WARPS;               // one warp per slot at most
    if (cap < dblocks) dblocks = cap;
    drain<<<(unsigned)dblocks, DRAIN_THREADS, 0, stream>>>(p);
    return cudaGetLastError();
}

// Both kernels are also compiled for the run constants whose tests would otherwise be uniform branches in every scattering:
// without the doublet (DB = false) for the runs that have none, and for the common case of isotropic scattering in core and
// wing with each core-skipping mode (FIN = 1 / 2 / 3; finish_scatter) and for config 3's dipole core / isotropic wing (FIN = 4).  Everything else takes the generic kernels.
template <bool HUBBLE, bool PEEL, int MIN_CTAS, bool GL = false>
static cudaError_t launch_variant(const WalkParams& p, int n_sm, cudaStream_t stream, int* blocks_out) {
    if (p.doublet_on || (p.walk_variant & 16)) return launch_pair<HUBBLE, PEEL, MIN_CTAS, GL, true, 0>(p, n_sm, stream, blocks_out);   // 16: generic kernels (tests)
    if (p.phase_core == 1 && p.phase_wing == 0 && p.phase_frame == 0 && p.core_skip_mode == 1)
        return launch_pair<HUBBLE, PEEL, MIN_CTAS, GL, false, 4>(p, n_sm, stream, blocks_out);
    if (p.phase_core != 0 || p.phase_wing != 0) return launch_pair<HUBBLE, PEEL, MIN_CTAS, GL, false, 0>(p, n_sm, stream, blocks_out);
    if (p.core_skip_mode == 1) return launch_pair<HUBBLE, PEEL, MIN_CTAS, GL, false, 1>(p, n_sm, stream, blocks_out);
    if (p.core_skip_mode == 2) return launch_pair<HUBBLE, PEEL, MIN_CTAS, GL, false, 2>(p, n_sm, stream, blocks_out);
    return launch_pair<HUBBLE, PEEL, MIN_CTAS, GL, false, 3>(p, n_sm, stream, blocks_out);
}

// Slots the pool must hold for a launch of `blocks` walk CTAs.
long long walk_pool_slots(int n_sm) { return (long long)n_sm * 4 * (WALK_THREADS / 32) * COOP_MAX_LANES; }

int walk_pool_words() { return PK_WORDS; }

cudaError_t launch_walk(const WalkParams& p, int n_sm, cudaStream_t stream, int* blocks_out) {
    if (p.gl_geom >= 0) return launch_variant<false, false, THOR_WALK_MIN_CTAS, true>(p, n_sm, stream, blocks_out);
    const bool hub = p.hubble != 0.f, peel = p.peel_on != 0;
    const double cells = (double)p.g.nx * p.g.ny * p.g.nz;
    const double grid_bytes = cells * (p.packed ? 32.0 : (p.has_dust ? 24.0 : 20.0));
    const bool beyond_l2 = (p.walk_variant & ~16) ? (p.walk_variant & ~16) == 4 : grid_bytes > 96.0e6;
    if (peel) return hub ? launch_variant<true, true, THOR_PEEL_MIN_CTAS>(p, n_sm, stream, blocks_out)
                         : launch_variant<false, true, THOR_PEEL_MIN_CTAS>(p, n_sm, stream, blocks_out);
    if (beyond_l2) return hub ? launch_variant<true, false, 4>(p, n_sm, stream, blocks_out)
                              : launch_variant<false, false, 4>(p, n_sm, stream, blocks_out);
    return hub ? launch_variant<true, false, THOR_WALK_MIN_CTAS>(p, n_sm, stream, blocks_out)
               : launch_variant<false, false, THOR_WALK_MIN_CTAS>(p, n_sm, stream, blocks_out);
}

}  // namespace thor
