// C-ABI of include/thor.h: context, argument validation, tally storage, kernel launches.  Host logic only; every
// step of the path runs in the kernels of walk.cu / unit_kernels.cu.
#include <cuda_runtime.h>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/thor.h"
#include "params.cuh"

namespace thor {
cudaError_t launch_walk(const WalkParams& p, int n_sm, cudaStream_t stream, int* blocks_out);
long long walk_pool_slots(int n_sm);
long long walk_pool_mid_slots(int n_sm);
int walk_pool_words();
cudaError_t launch_volume_render(const WalkParams& p, const TransferFn& tf, long long n_rays, const float* org,
                                 const float* dir, float* out_rgba, cudaStream_t stream);
cudaError_t launch_raytrace(const WalkParams& p, long long n_rays, const float* org, const float* dir, float hubble,
                            float hubble_eps, float max_len, int n_v, float v_lo, float dv, float* out_column,
                            float* out_tmean, float* out_tau, cudaStream_t stream);
cudaError_t launch_slice(const WalkParams& p, long long n, const float* pos, int field, float* out, cudaStream_t stream);
cudaError_t launch_pack_fields(const float* nHI, const float* T, const float* vx, const float* vy, const float* vz,
                               const float* kdust, long long n, float4* out, cudaStream_t stream);
cudaError_t launch_validate_fields(const float* nHI, const float* T, const float* vx, const float* vy, const float* vz,
                                   const float* kdust, long long n, unsigned* d_flags, cudaStream_t stream);
}  // namespace thor

struct thor_ctx {
    cudaStream_t stream = nullptr;
    int device = 0, n_sm = 0;
    thor::GridDims g{};
    double cell_cm = 0;
    long long n_cells = 0;
    const float* f[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // nHI, T, vx, vy, vz, kdust
    float* owned[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    float4* d_packed = nullptr;                 // THOR_GRID_PACK: the library's own one-sector-per-cell copy
    bool has_dust = false;
    bool l2_persist = false;
    bool gridless = false;
    thor_gridless gl{};
    size_t l2_window_max = 0;
    // sources
    long long n_src = 0;
    float* d_src_pos = nullptr;
    float* d_src_sigma = nullptr;
    double* d_src_cdf = nullptr;
    // tallies
    unsigned long long* d_small = nullptr;      // [1 next_photon][N_COUNTERS][64 hist][4098 spectrum]
    unsigned long long* d_cube = nullptr;
    size_t cube_elems = 0;
    thor::RawRecord* d_raw = nullptr;
    size_t raw_cap = 0;
    uint32_t* d_pool = nullptr;                 // parked packets for the drain kernel
    uint32_t* d_pool_mid = nullptr;             // parked packets between the passes of the tail (two halves)
    unsigned int* d_pool_order = nullptr;
    // last run
    bool have_run = false;
    bool pending = false;                       // thor_run_async launched, thor_wait not yet called
    unsigned long long pending_n = 0;
    thor_opts last{};
    unsigned long long last_n = 0;
    float last_ms = 0.f, last_feed_ms = 0.f;
    unsigned long long last_max_nscat = 0;
    int last_blocks = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    std::string err;
};

static thread_local std::string g_err;

// Every entry point works on the context's device and leaves the caller's current device as it found it.
struct DevGuard {
    int prev = -1;
    bool switched = false;
    explicit DevGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DevGuard() { if (switched) cudaSetDevice(prev); }
};

static constexpr size_t SMALL_NEXT = 0, SMALL_COUNTERS = 1, SMALL_HIST = SMALL_COUNTERS + thor::N_COUNTERS,
                        SMALL_SPEC = SMALL_HIST + 64, SMALL_TIMES = SMALL_SPEC + 4096 + 2, SMALL_MAXN = SMALL_TIMES + 2, SMALL_POOL = SMALL_MAXN + 1, SMALL_TOTAL = SMALL_POOL + 4;

static thor_status fail(thor_ctx* c, thor_status s, const std::string& msg) {
    if (c) c->err = msg;
    g_err = msg;
    return s;
}

static thor_status cuda_fail(thor_ctx* c, cudaError_t e, const char* what) {
    return fail(c, e == cudaErrorMemoryAllocation ? THOR_ERR_OOM : THOR_ERR_CUDA,
                std::string(what) + ": " + cudaGetErrorString(e));
}

#define CU(call)                                                   \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);   \
    } while (0)

static thor_status run_finish(thor_ctx* ctx);          // completes a pending thor_run_async (defined beside it)

extern "C" const char* thor_last_error(const thor_ctx* ctx) { return ctx ? ctx->err.c_str() : g_err.c_str(); }

extern "C" void thor_opts_default(thor_opts* o) {
    if (!o) return;
    std::memset(o, 0, sizeof *o);
    o->struct_size = (uint32_t)sizeof *o;
    o->phase_split_x = 0.2;
    o->spec_T_ref = 1e4;
    o->spec_hi = 1.0;
    o->hubble_eps = 0.25;
    o->k_obs[2] = 1.0;
    o->peel_v_hi = 1.0;
    o->tau_peel_max = 30.0;
    o->doublet_a_ratio = 1.0;
}

extern "C" void thor_grid_destroy(thor_ctx* ctx) {
    if (!ctx) return;
    run_finish(ctx);                                       // a pending run still reads what is freed below
    DevGuard dev_guard(ctx->device);
    for (float* p : ctx->owned) if (p) cudaFree(p);
    if (ctx->d_packed) cudaFree(ctx->d_packed);
    if (ctx->d_src_pos) cudaFree(ctx->d_src_pos);
    if (ctx->d_src_sigma) cudaFree(ctx->d_src_sigma);
    if (ctx->d_src_cdf) cudaFree(ctx->d_src_cdf);
    if (ctx->d_small) cudaFree(ctx->d_small);
    if (ctx->d_cube) cudaFree(ctx->d_cube);
    if (ctx->d_raw) cudaFree(ctx->d_raw);
    if (ctx->d_pool) cudaFree(ctx->d_pool);
    if (ctx->d_pool_mid) cudaFree(ctx->d_pool_mid);
    if (ctx->d_pool_order) cudaFree(ctx->d_pool_order);
    if (ctx->l2_persist) {                        // drop the access-policy window of the caller's stream
        cudaStreamAttrValue av{};
        cudaStreamSetAttribute(ctx->stream, cudaStreamAttributeAccessPolicyWindow, &av);
        cudaCtxResetPersistingL2Cache();
    }
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    delete ctx;
}

extern "C" thor_status thor_grid_create(thor_ctx** out, int nx, int ny, int nz, double cell_cm, const float* nHI,
                                        const float* T, const float* vx, const float* vy, const float* vz,
                                        const float* kdust, unsigned flags, void* stream) {
    if (!out) return fail(nullptr, THOR_ERR_ARG, "thor_grid_create: out is NULL");
    *out = nullptr;
    if (nx <= 0 || ny <= 0 || nz <= 0) return fail(nullptr, THOR_ERR_ARG, "thor_grid_create: grid extents must be > 0");
    if (!(cell_cm > 0) || !std::isfinite(cell_cm)) return fail(nullptr, THOR_ERR_ARG, "thor_grid_create: cell_cm must be > 0");
    if (!nHI || !T || !vx || !vy || !vz) return fail(nullptr, THOR_ERR_ARG, "thor_grid_create: a field array is NULL");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, THOR_ERR_UNSUPPORTED, "thor_grid_create: no CUDA device (this library has no CPU fallback)");
    }
    thor_ctx* ctx = new (std::nothrow) thor_ctx;
    if (!ctx) return fail(nullptr, THOR_ERR_OOM, "thor_grid_create: host allocation failed");
    struct Guard { thor_ctx* c; ~Guard() { if (c) thor_grid_destroy(c); } } guard{ctx};
    CU(cudaGetDevice(&ctx->device));
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, ctx->device));
    if (prop.major != 10) {
        return fail(nullptr, THOR_ERR_UNSUPPORTED,
                    std::string("thor_grid_create: device '") + prop.name + "' is not sm_100 (built for sm_100a only)");
    }
    ctx->n_sm = prop.multiProcessorCount;
    ctx->stream = (cudaStream_t)stream;
    ctx->g.nx = nx; ctx->g.ny = ny; ctx->g.nz = nz;
    ctx->g.periodic = ((flags & THOR_PERIODIC_X) ? 1u : 0u) | ((flags & THOR_PERIODIC_Y) ? 2u : 0u) |
                      ((flags & THOR_PERIODIC_Z) ? 4u : 0u);
    ctx->g.frozen = ((ctx->g.periodic & 1u) && nx == 1 ? 1u : 0u) | ((ctx->g.periodic & 2u) && ny == 1 ? 2u : 0u) |
                    ((ctx->g.periodic & 4u) && nz == 1 ? 4u : 0u);
    ctx->cell_cm = cell_cm;
    ctx->n_cells = (long long)nx * ny * nz;
    const float* src[6] = {nHI, T, vx, vy, vz, kdust};
    const size_t bytes = (size_t)ctx->n_cells * sizeof(float);
    for (int i = 0; i < 6; ++i) {
        if (!src[i]) continue;
        if (flags & THOR_GRID_HOST) {
            CU(cudaMalloc(&ctx->owned[i], bytes));
            CU(cudaMemcpyAsync(ctx->owned[i], src[i], bytes, cudaMemcpyHostToDevice, ctx->stream));
            ctx->f[i] = ctx->owned[i];
        } else {
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, src[i]) != cudaSuccess ||
                (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)) {
                cudaGetLastError();
                return fail(nullptr, THOR_ERR_ARG, "thor_grid_create: field array is not a device pointer (pass THOR_GRID_HOST for host arrays)");
            }
            ctx->f[i] = src[i];
        }
    }
    CU(cudaMalloc(&ctx->d_small, SMALL_TOTAL * sizeof(unsigned long long)));
    CU(cudaEventCreate(&ctx->ev0));
    CU(cudaEventCreate(&ctx->ev1));
    if (!(flags & THOR_GRID_NO_VALIDATE)) {
        // reading A19: NaN anywhere, negative n or kdust, or T <= 0 where n > 0 -> THOR_ERR_ARG
        unsigned* d_flags = reinterpret_cast<unsigned*>(ctx->d_small);
        CU(cudaMemsetAsync(d_flags, 0, sizeof(unsigned), ctx->stream));
        CU(thor::launch_validate_fields(ctx->f[0], ctx->f[1], ctx->f[2], ctx->f[3], ctx->f[4], ctx->f[5], ctx->n_cells,
                                        d_flags, ctx->stream));
        unsigned h_flags = 0;
        CU(cudaMemcpyAsync(&h_flags, d_flags, sizeof h_flags, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        if (h_flags) {
            std::string m = "thor_grid_create: invalid field values:";
            if (h_flags & 1u) m += " NaN/Inf";
            if (h_flags & 2u) m += " negative nHI or kdust";
            if (h_flags & 4u) m += " T <= 0 in a cell with nHI > 0";
            return fail(nullptr, THOR_ERR_ARG, m);
        }
    } else {
        CU(cudaStreamSynchronize(ctx->stream));
    }
    ctx->has_dust = kdust != nullptr;
    if (flags & THOR_GRID_L2_FETCH32) CU(cudaDeviceSetLimit(cudaLimitMaxL2FetchGranularity, 32));
    if ((flags & THOR_GRID_L2_PERSIST) && (flags & THOR_GRID_PACK) && prop.persistingL2CacheMaxSize > 0) {
        CU(cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, (size_t)prop.persistingL2CacheMaxSize));
        ctx->l2_persist = true;
        ctx->l2_window_max = (size_t)prop.accessPolicyMaxWindowSize;
    }
    if (flags & THOR_GRID_PACK) {
        CU(cudaMalloc(&ctx->d_packed, (size_t)ctx->n_cells * 2 * sizeof(float4)));
        CU(thor::launch_pack_fields(ctx->f[0], ctx->f[1], ctx->f[2], ctx->f[3], ctx->f[4], ctx->f[5], ctx->n_cells,
                                    ctx->d_packed, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        for (int i = 0; i < 6; ++i) {            // the SoA arrays are no longer read: drop our copies / the borrow
            if (ctx->owned[i]) { cudaFree(ctx->owned[i]); ctx->owned[i] = nullptr; }
            ctx->f[i] = nullptr;
        }
    }
    guard.c = nullptr;
    *out = ctx;
    return THOR_OK;
}

extern "C" thor_status thor_dataset_create_gridless(thor_ctx** out, const thor_gridless* d, void* stream) {
    if (!out) return fail(nullptr, THOR_ERR_ARG, "thor_dataset_create_gridless: out is NULL");
    *out = nullptr;
    if (!d || d->struct_size != sizeof(thor_gridless)) return fail(nullptr, THOR_ERR_ARG, "thor_dataset_create_gridless: struct_size is not set");
    if (d->geometry != THOR_GEOM_SHELL && d->geometry != THOR_GEOM_SLAB) return fail(nullptr, THOR_ERR_ARG, "thor_dataset_create_gridless: unknown geometry");
    const double vals[] = {d->r_in, d->r_out, d->length_cm, d->n0, d->alpha_rho, d->T, d->v_max, d->alpha_v, d->kdust0, d->step_f};
    for (double v : vals) if (!std::isfinite(v)) return fail(nullptr, THOR_ERR_ARG, "thor_dataset_create_gridless: non-finite value");
    const double r_in = d->geometry == THOR_GEOM_SLAB ? 0.0 : d->r_in;
    if (!(d->r_out > 0) || !(r_in >= 0) || !(d->r_out > r_in) || !(d->length_cm > 0) || !(d->T > 0) || !(d->n0 >= 0) ||
        !(d->kdust0 >= 0) || !(d->step_f >= 0))
        return fail(nullptr, THOR_ERR_ARG, "thor_dataset_create_gridless: need r_out > r_in >= 0, length_cm > 0, T > 0, n0 >= 0, kdust0 >= 0, step_f >= 0");
    if (d->geometry == THOR_GEOM_SHELL && r_in == 0.0 && (d->alpha_rho < 0 || (d->alpha_v < 0 && d->v_max != 0)))
        return fail(nullptr, THOR_ERR_ARG, "thor_dataset_create_gridless: a negative power law needs r_in > 0");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, THOR_ERR_UNSUPPORTED, "thor_dataset_create_gridless: no CUDA device (this library has no CPU fallback)");
    }
    thor_ctx* ctx = new (std::nothrow) thor_ctx;
    if (!ctx) return fail(nullptr, THOR_ERR_OOM, "thor_dataset_create_gridless: host allocation failed");
    struct Guard { thor_ctx* c; ~Guard() { if (c) thor_grid_destroy(c); } } guard{ctx};
    CU(cudaGetDevice(&ctx->device));
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, ctx->device));
    if (prop.major != 10)
        return fail(nullptr, THOR_ERR_UNSUPPORTED, std::string("thor_dataset_create_gridless: device '") + prop.name + "' is not sm_100");
    ctx->n_sm = prop.multiProcessorCount;
    ctx->stream = (cudaStream_t)stream;
    ctx->gridless = true;
    ctx->gl = *d;
    ctx->gl.r_in = r_in;
    ctx->g.nx = ctx->g.ny = ctx->g.nz = 1;
    ctx->cell_cm = d->length_cm;
    ctx->has_dust = d->kdust0 > 0;
    CU(cudaMalloc(&ctx->d_small, SMALL_TOTAL * sizeof(unsigned long long)));
    CU(cudaEventCreate(&ctx->ev0));
    CU(cudaEventCreate(&ctx->ev1));
    guard.c = nullptr;
    *out = ctx;
    return THOR_OK;
}

extern "C" thor_status thor_sources_set(thor_ctx* ctx, long long n_src, const float* pos_xyz, const float* lum,
                                        const float* sigma_kms) {
    if (!ctx) return fail(nullptr, THOR_ERR_ARG, "thor_sources_set: ctx is NULL");
    { const thor_status st = run_finish(ctx); if (st != THOR_OK) return st; }   // a pending run still reads the old list
    if (n_src <= 0 || !pos_xyz || !lum || !sigma_kms) return fail(ctx, THOR_ERR_ARG, "thor_sources_set: empty or NULL source list");
    const int n[3] = {ctx->g.nx, ctx->g.ny, ctx->g.nz};
    std::vector<double> cdf((size_t)n_src);
    double tot = 0;
    for (long long i = 0; i < n_src; ++i) {
        if (ctx->gridless) {
            const double x = pos_xyz[3 * i], y = pos_xyz[3 * i + 1], z = pos_xyz[3 * i + 2];
            const bool in = ctx->gl.geometry == THOR_GEOM_SLAB ? std::fabs(z) <= ctx->gl.r_out : x * x + y * y + z * z <= ctx->gl.r_out * ctx->gl.r_out;
            if (!in || !std::isfinite(x) || !std::isfinite(y)) return fail(ctx, THOR_ERR_ARG, "thor_sources_set: source " + std::to_string(i) + " lies outside the dataset");
        } else
        for (int ax = 0; ax < 3; ++ax) {
            const float p = pos_xyz[3 * i + ax];
            if (!(p >= 0.f && p <= (float)n[ax])) return fail(ctx, THOR_ERR_ARG, "thor_sources_set: source " + std::to_string(i) + " lies outside the grid");
        }
        if (!(lum[i] >= 0.f) || !std::isfinite(lum[i])) return fail(ctx, THOR_ERR_ARG, "thor_sources_set: luminosity " + std::to_string(i) + " is negative or not finite");
        if (!(sigma_kms[i] >= 0.f) || !std::isfinite(sigma_kms[i])) return fail(ctx, THOR_ERR_ARG, "thor_sources_set: sigma " + std::to_string(i) + " is negative or not finite");
        tot += lum[i];
    }
    if (!(tot > 0)) return fail(ctx, THOR_ERR_ARG, "thor_sources_set: total luminosity is zero");
    double acc = 0;
    for (long long i = 0; i < n_src; ++i) { acc += lum[i]; cdf[(size_t)i] = acc / tot; }
    cdf[(size_t)n_src - 1] = 1.0;
    DevGuard dev_guard(ctx->device);
    if (ctx->d_src_pos) { cudaFree(ctx->d_src_pos); ctx->d_src_pos = nullptr; }
    if (ctx->d_src_sigma) { cudaFree(ctx->d_src_sigma); ctx->d_src_sigma = nullptr; }
    if (ctx->d_src_cdf) { cudaFree(ctx->d_src_cdf); ctx->d_src_cdf = nullptr; }
    ctx->n_src = 0;
    CU(cudaMalloc(&ctx->d_src_pos, (size_t)n_src * 3 * sizeof(float)));
    CU(cudaMalloc(&ctx->d_src_sigma, (size_t)n_src * sizeof(float)));
    CU(cudaMalloc(&ctx->d_src_cdf, (size_t)n_src * sizeof(double)));
    CU(cudaMemcpyAsync(ctx->d_src_pos, pos_xyz, (size_t)n_src * 3 * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_src_sigma, sigma_kms, (size_t)n_src * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_src_cdf, cdf.data(), (size_t)n_src * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->n_src = n_src;
    if (ctx->l2_persist && ctx->d_packed) {
        // L2-persistence window (BASELINE.json north_star): the run of z-slabs of the packed grid, as long as the device's
        // window allows, that holds the most source luminosity — where packets are emitted and scatter first
        const size_t slab_bytes = (size_t)ctx->g.nx * ctx->g.ny * 2 * sizeof(float4);
        const size_t total = slab_bytes * (size_t)ctx->g.nz;
        long long S = (long long)(ctx->l2_window_max / slab_bytes);
        if (S > ctx->g.nz) S = ctx->g.nz;
        if (S >= 1) {
            std::vector<double> mass((size_t)ctx->g.nz, 0.0);
            for (long long i = 0; i < n_src; ++i) {
                int z = (int)pos_xyz[3 * i + 2];
                if (z >= ctx->g.nz) z = ctx->g.nz - 1;
                mass[(size_t)z] += lum[i];
            }
            double best = -1, run = 0;
            long long z0 = 0;
            for (long long z = 0; z < ctx->g.nz; ++z) {
                run += mass[(size_t)z];
                if (z >= S) run -= mass[(size_t)(z - S)];
                if (z >= S - 1 && run > best) { best = run; z0 = z - S + 1; }
            }
            cudaStreamAttrValue av{};
            av.accessPolicyWindow.base_ptr = reinterpret_cast<char*>(ctx->d_packed) + (size_t)z0 * slab_bytes;
            av.accessPolicyWindow.num_bytes = (size_t)S * slab_bytes < total ? (size_t)S * slab_bytes : total;
            av.accessPolicyWindow.hitRatio = 1.0f;
            av.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
            av.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
            CU(cudaStreamSetAttribute(ctx->stream, cudaStreamAttributeAccessPolicyWindow, &av));
        }
    }
    return THOR_OK;
}

static bool phase_ok(int p) { return p == THOR_PHASE_ISOTROPIC || p == THOR_PHASE_DIPOLE || p == THOR_PHASE_MIX; }

// Second half of a run: waits for the launch, reads its timers, publishes the tallies.  No-op when nothing is pending.
static thor_status run_finish(thor_ctx* ctx) {
    if (!ctx->pending) return THOR_OK;
    DevGuard dev_guard(ctx->device);
    ctx->pending = false;
    CU(cudaStreamSynchronize(ctx->stream));
    CU(cudaEventElapsedTime(&ctx->last_ms, ctx->ev0, ctx->ev1));
    ctx->last_feed_ms = 0.f;
    if (ctx->pending_n > 0) {
        unsigned long long t[3] = {0, 0, 0};                    // t_start, t_dry, max_nscat are adjacent
        CU(cudaMemcpyAsync(t, ctx->d_small + SMALL_TIMES, sizeof t, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        if (t[1] != ~0ull && t[1] >= t[0]) ctx->last_feed_ms = (float)((double)(t[1] - t[0]) * 1e-6);
        ctx->last_max_nscat = t[2];
    }
    ctx->last_n = ctx->pending_n; ctx->have_run = true;
    return THOR_OK;
}

extern "C" thor_status thor_wait(thor_ctx* ctx) {
    if (!ctx) return fail(nullptr, THOR_ERR_ARG, "thor_wait: ctx is NULL");
    return run_finish(ctx);
}

extern "C" thor_status thor_run_async(thor_ctx* ctx, unsigned long long n_photons, unsigned long long seed,
                                      const thor_opts* opts) {
    if (!ctx) return fail(nullptr, THOR_ERR_ARG, "thor_run: ctx is NULL");
    {
        const thor_status st = run_finish(ctx);                // a run still pending on this context is completed first
        if (st != THOR_OK) return st;
    }
    if (ctx->n_src <= 0) return fail(ctx, THOR_ERR_STATE, "thor_run: call thor_sources_set first");
    thor_opts o;
    thor_opts_default(&o);
    if (opts) {
        if (opts->struct_size == 0 || opts->struct_size > sizeof o) return fail(ctx, THOR_ERR_ARG, "thor_run: opts->struct_size is not set (use thor_opts_default)");
        std::memcpy(&o, opts, opts->struct_size);
        o.struct_size = (uint32_t)sizeof o;
    }
    if (!phase_ok(o.phase_core) || !phase_ok(o.phase_wing)) return fail(ctx, THOR_ERR_ARG, "thor_run: unknown phase function");
    if (o.core_skip_mode < 0 || o.core_skip_mode > 2 || !(o.x_crit >= 0)) return fail(ctx, THOR_ERR_ARG, "thor_run: bad core-skip options");
    if (o.spec_bins < 0 || o.spec_bins > 4096) return fail(ctx, THOR_ERR_ARG, "thor_run: spec_bins must be in [0, 4096]");
    if (o.spec_bins > 0 && !(o.spec_hi > o.spec_lo)) return fail(ctx, THOR_ERR_ARG, "thor_run: spec_hi must exceed spec_lo");
    if (o.spec_mode != 0 && o.spec_mode != 1) return fail(ctx, THOR_ERR_ARG, "thor_run: spec_mode must be 0 or 1");
    if (o.spec_mode == 0 && !(o.spec_T_ref > 0)) return fail(ctx, THOR_ERR_ARG, "thor_run: spec_T_ref must be > 0");
    if (((o.walk_variant & ~16) != 0 && (o.walk_variant & ~16) != 3 && (o.walk_variant & ~16) != 4) || (o.drain_mode < 0 || o.drain_mode > 2)) return fail(ctx, THOR_ERR_ARG, "thor_run: bad walk_variant / drain_mode");
    if (!(o.dust_albedo >= 0 && o.dust_albedo <= 1) || !(o.dust_g >= -1 && o.dust_g <= 1)) return fail(ctx, THOR_ERR_ARG, "thor_run: dust_albedo must be in [0, 1] and dust_g in [-1, 1]");
    if (o.doublet_on && (!std::isfinite(o.doublet_dv_kms) || !(o.doublet_sigma_ratio >= 0) || !(o.doublet_a_ratio > 0) || !std::isfinite(o.doublet_sigma_ratio) || !std::isfinite(o.doublet_a_ratio)))
        return fail(ctx, THOR_ERR_ARG, "thor_run: bad doublet options");
    if (!(o.hubble_eps > 0) || !(o.v_max_kms >= 0) || !std::isfinite(o.hubble_kms_per_cell)) return fail(ctx, THOR_ERR_ARG, "thor_run: bad Hubble / v_max options");
    // reading A26: on a grid periodic on all three axes nothing ends a packet in empty gas; without a crossing cap the
    // persistent kernel would never return (a fully frozen 1x1x1 grid has only infinite segments: reading A24 caps those)
    if (ctx->g.periodic == 7u && ctx->g.frozen != 7u && o.max_crossings == 0)
        return fail(ctx, THOR_ERR_ARG, "thor_run: the grid is periodic on all three axes (no packet can leave it): set opts.max_crossings");
    const thor::LyaConstants K = thor::lya_constants();
    thor::WalkParams p{};
    p.g = ctx->g;
    p.nHI = ctx->f[0]; p.T = ctx->f[1]; p.vx = ctx->f[2]; p.vy = ctx->f[3]; p.vz = ctx->f[4]; p.kdust = ctx->f[5];
    p.packed = ctx->d_packed; p.has_dust = ctx->has_dust ? 1 : 0;
    p.sig_cell = (float)(K.c_sig * ctx->cell_cm);
    p.c_a = (float)K.c_a; p.c_vth = (float)K.c_vth; p.inv_c_vth = (float)(1.0 / K.c_vth);
    p.cell_cm = (float)ctx->cell_cm;
    p.max_crossings = (o.max_crossings && o.max_crossings < 0xffffffffull) ? (unsigned)o.max_crossings : 0xffffffffu;
    p.gl_geom = -1;
    if (ctx->gridless) {
        const thor_gridless& d = ctx->gl;
        if (o.peel_on || o.hubble_kms_per_cell != 0 || o.core_skip_mode == 2 || o.doublet_on)
            return fail(ctx, THOR_ERR_UNSUPPORTED, "thor_run: peel-off, Hubble drift, local core-skipping and doublets need a grid dataset");
        const double vth = K.c_vth * std::sqrt(d.T);
        // step limiter l_max = f min(l_v, l_rho) (reading A29)
        double lv = INFINITY, lrho = INFINITY;
        if (d.geometry == THOR_GEOM_SLAB) {
            if (d.v_max != 0) lv = vth * d.r_out / std::fabs(d.v_max);
        } else {
            if (d.v_max != 0 && d.alpha_v != 0) {
                const double rm = d.alpha_v >= 1.0 ? d.r_out : std::fmax(d.r_in, 1e-300);
                lv = vth / (std::fabs(d.alpha_v * d.v_max) * std::pow(rm / d.r_out, d.alpha_v - 1.0) / d.r_out);
            }
            if (d.alpha_rho != 0) lrho = d.r_out / std::fabs(d.alpha_rho);
        }
        const double lm = std::fmin(lv, lrho);
        p.gl_geom = d.geometry;
        p.gl_rin = d.r_in; p.gl_rout = d.r_out;
        p.gl_lmax = (d.step_f > 0 && std::isfinite(lm)) ? (float)(d.step_f * lm) : INFINITY;
        p.gl_nsig0 = (float)(d.n0 * K.c_sig / std::sqrt(d.T) * d.length_cm);
        p.gl_kd0 = (float)(d.kdust0 * d.length_cm);
        p.gl_alpha_rho = (float)d.alpha_rho; p.gl_vmax = (float)d.v_max; p.gl_alpha_v = (float)d.alpha_v;
        p.gl_a = (float)(K.c_a / std::sqrt(d.T)); p.gl_vth = (float)vth; p.gl_inv_vth = (float)(1.0 / vth);
    }
    p.n_src = ctx->n_src; p.src_pos = ctx->d_src_pos; p.src_sigma = ctx->d_src_sigma; p.src_cdf = ctx->d_src_cdf;
    p.phase_core = o.phase_core; p.phase_wing = o.phase_wing; p.phase_frame = o.phase_frame;
    p.phase_split_x = (float)o.phase_split_x;
    p.core_skip_mode = o.core_skip_mode; p.x_crit = (float)o.x_crit;
    p.spec_mode = o.spec_mode; p.spec_bins = o.spec_bins;
    p.spec_inv_vth_ref = (float)(1.0 / (K.c_vth * std::sqrt(o.spec_T_ref)));
    p.spec_lo = (float)o.spec_lo;
    p.spec_inv_width = o.spec_bins > 0 ? (float)(o.spec_bins / (o.spec_hi - o.spec_lo)) : 0.f;
    p.hubble = (float)o.hubble_kms_per_cell; p.hubble_eps = (float)o.hubble_eps; p.v_max = (float)o.v_max_kms;
    p.v_max_or_inf = p.v_max > 0.f ? p.v_max : INFINITY;
    p.peel_on = o.peel_on ? 1 : 0;
    size_t cube_elems = 0;
    if (p.peel_on) {
        if (o.peel_nx <= 0 || o.peel_ny <= 0 || o.peel_nv <= 0 || !(o.peel_v_hi > o.peel_v_lo) || !(o.peel_width_cells > 0) || !(o.tau_peel_max > 0))
            return fail(ctx, THOR_ERR_ARG, "thor_run: bad peel options");
        const double n2 = o.k_obs[0] * o.k_obs[0] + o.k_obs[1] * o.k_obs[1] + o.k_obs[2] * o.k_obs[2];
        if (!(n2 > 0)) return fail(ctx, THOR_ERR_ARG, "thor_run: k_obs is zero");
        double k[3], h[3] = {1, 0, 0}, i1[3], i2[3];
        for (int i = 0; i < 3; ++i) k[i] = o.k_obs[i] / std::sqrt(n2);
        // image-plane basis: helper axis = x unless k_obs is closest to x, then y
        if (std::fabs(k[0]) > std::fabs(k[1]) && std::fabs(k[0]) > std::fabs(k[2])) { h[0] = 0; h[1] = 1; }
        const double hk = h[0] * k[0] + h[1] * k[1] + h[2] * k[2];
        double m2 = 0;
        for (int i = 0; i < 3; ++i) { i1[i] = h[i] - hk * k[i]; m2 += i1[i] * i1[i]; }
        for (int i = 0; i < 3; ++i) i1[i] /= std::sqrt(m2);
        i2[0] = k[1] * i1[2] - k[2] * i1[1]; i2[1] = k[2] * i1[0] - k[0] * i1[2]; i2[2] = k[0] * i1[1] - k[1] * i1[0];
        for (int i = 0; i < 3; ++i) {
            p.kobs[i] = (float)k[i]; p.img1[i] = (float)i1[i]; p.img2[i] = (float)i2[i];
            p.kobs_inv[i] = 1.0f / p.kobs[i];             // what __fdiv_rn(1, k) gives on the device
        }
        p.peel_nx = o.peel_nx; p.peel_ny = o.peel_ny; p.peel_nv = o.peel_nv;
        p.peel_v_lo = (float)o.peel_v_lo;
        p.peel_inv_dv = (float)(o.peel_nv / (o.peel_v_hi - o.peel_v_lo));
        p.peel_inv_width = (float)(1.0 / o.peel_width_cells);
        p.tau_peel_max = (float)o.tau_peel_max;
        cube_elems = (size_t)o.peel_nx * o.peel_ny * o.peel_nv;
    }
    p.id_offset = o.photon_id_offset; p.n_photons = n_photons; p.seed = seed; p.max_scatter = o.max_scatter;
    p.max_scatter_or_max = (o.max_scatter == 0 || o.max_scatter > 0xffffffffull) ? 0xffffffffu : (unsigned)o.max_scatter;
    p.walk_variant = o.walk_variant;
    p.dust_albedo = (float)o.dust_albedo; p.dust_g = (float)o.dust_g;
    p.doublet_on = o.doublet_on ? 1 : 0;
    p.db_dv = (float)o.doublet_dv_kms; p.db_rs = (float)o.doublet_sigma_ratio; p.db_ra = (float)o.doublet_a_ratio;
    DevGuard dev_guard(ctx->device);
    if (o.drain_mode != 1 && !ctx->d_pool)
        CU(cudaMalloc(&ctx->d_pool, (size_t)thor::walk_pool_slots(ctx->n_sm) * thor::walk_pool_words() * sizeof(uint32_t)));
    if (o.drain_mode != 1 && !ctx->d_pool_order)
        CU(cudaMalloc(&ctx->d_pool_order, (size_t)thor::walk_pool_slots(ctx->n_sm) * sizeof(unsigned int)));
    if (o.drain_mode == 0 && !ctx->d_pool_mid)
        CU(cudaMalloc(&ctx->d_pool_mid, 2 * (size_t)thor::walk_pool_mid_slots(ctx->n_sm) * thor::walk_pool_words() * sizeof(uint32_t)));   // two halves
    p.pool = o.drain_mode != 1 ? ctx->d_pool : nullptr;
    p.pool_mid = o.drain_mode == 0 ? ctx->d_pool_mid : nullptr;
    p.pool_order = ctx->d_pool_order;
    const bool keep = o.accumulate && ctx->have_run;
    if (keep) {
        const thor_opts& l = ctx->last;
        const bool same = l.spec_bins == o.spec_bins && l.spec_lo == o.spec_lo && l.spec_hi == o.spec_hi && l.spec_mode == o.spec_mode &&
                          l.spec_T_ref == o.spec_T_ref && l.peel_on == o.peel_on &&
                          (!o.peel_on || (l.peel_nx == o.peel_nx && l.peel_ny == o.peel_ny && l.peel_nv == o.peel_nv && l.peel_v_lo == o.peel_v_lo &&
                                          l.peel_v_hi == o.peel_v_hi && l.peel_width_cells == o.peel_width_cells && l.k_obs[0] == o.k_obs[0] &&
                                          l.k_obs[1] == o.k_obs[1] && l.k_obs[2] == o.k_obs[2]));
        if (!same) return fail(ctx, THOR_ERR_ARG, "thor_run: accumulate needs the spectrum axis and the peel geometry of the run it adds to");
    }
    ctx->have_run = false;                          // from here on the tallies are in flux: valid again only after a completed run
    if (cube_elems != ctx->cube_elems) {
        if (ctx->d_cube) { cudaFree(ctx->d_cube); ctx->d_cube = nullptr; }
        ctx->cube_elems = 0;
        if (cube_elems) {
            CU(cudaMalloc(&ctx->d_cube, cube_elems * sizeof(unsigned long long)));
            CU(cudaMemsetAsync(ctx->d_cube, 0, cube_elems * sizeof(unsigned long long), ctx->stream));
            ctx->cube_elems = cube_elems;
        }
    } else if (cube_elems && !keep) {
        CU(cudaMemsetAsync(ctx->d_cube, 0, cube_elems * sizeof(unsigned long long), ctx->stream));
    }
    if (o.raw_output && n_photons > 0) {
        if (ctx->raw_cap < n_photons) {
            if (ctx->d_raw) { cudaFree(ctx->d_raw); ctx->d_raw = nullptr; }
            ctx->raw_cap = 0;
            CU(cudaMalloc(&ctx->d_raw, (size_t)n_photons * sizeof(thor::RawRecord)));
            ctx->raw_cap = (size_t)n_photons;
        }
        p.raw = ctx->d_raw;
    }
    if (keep) CU(cudaMemsetAsync(ctx->d_small, 0, sizeof(unsigned long long), ctx->stream));
    else CU(cudaMemsetAsync(ctx->d_small, 0, SMALL_TOTAL * sizeof(unsigned long long), ctx->stream));
    CU(cudaMemsetAsync(ctx->d_small + SMALL_TIMES, 0xFF, 2 * sizeof(unsigned long long), ctx->stream));
    p.next_photon = ctx->d_small + SMALL_NEXT;
    p.t_start = ctx->d_small + SMALL_TIMES;
    p.max_nscat = ctx->d_small + SMALL_MAXN;
    CU(cudaMemsetAsync(ctx->d_small + SMALL_MAXN, 0, sizeof(unsigned long long), ctx->stream));
    p.t_dry = ctx->d_small + SMALL_TIMES + 1;
    p.pool_count = ctx->d_small + SMALL_POOL;
    p.pool_next = ctx->d_small + SMALL_POOL + 1;
    p.pool_mid_count = ctx->d_small + SMALL_POOL + 2;
    CU(cudaMemsetAsync(ctx->d_small + SMALL_POOL, 0, 4 * sizeof(unsigned long long), ctx->stream));
    p.counters = ctx->d_small + SMALL_COUNTERS;
    p.nscat_hist = ctx->d_small + SMALL_HIST;
    p.spectrum = ctx->d_small + SMALL_SPEC;
    p.cube = ctx->d_cube;
    CU(cudaEventRecord(ctx->ev0, ctx->stream));
    if (n_photons > 0) CU(thor::launch_walk(p, ctx->n_sm, ctx->stream, &ctx->last_blocks));
    CU(cudaEventRecord(ctx->ev1, ctx->stream));
    ctx->last = o; ctx->pending_n = n_photons; ctx->pending = true;   // have_run stays false until thor_wait
    return THOR_OK;
}

extern "C" thor_status thor_run(thor_ctx* ctx, unsigned long long n_photons, unsigned long long seed,
                                const thor_opts* opts) {
    const thor_status st = thor_run_async(ctx, n_photons, seed, opts);
    return st != THOR_OK ? st : run_finish(ctx);
}

// grid part of the kernel parameter block, shared by the ray operators
static thor::WalkParams grid_params(const thor_ctx* ctx) {
    const thor::LyaConstants K = thor::lya_constants();
    thor::WalkParams p{};
    p.g = ctx->g;
    p.nHI = ctx->f[0]; p.T = ctx->f[1]; p.vx = ctx->f[2]; p.vy = ctx->f[3]; p.vz = ctx->f[4]; p.kdust = ctx->f[5];
    p.packed = ctx->d_packed; p.has_dust = ctx->has_dust ? 1 : 0;
    p.sig_cell = (float)(K.c_sig * ctx->cell_cm);
    p.c_a = (float)K.c_a; p.c_vth = (float)K.c_vth; p.inv_c_vth = (float)(1.0 / K.c_vth);
    p.cell_cm = (float)ctx->cell_cm;
    p.gl_geom = -1;
    return p;
}

// ---- thor_run_noalloc: the walk for callers that cannot allocate at run time (include/thor.h) -------------------------------
// The kernels' scratch in one file-scope device array: [0, 256) six 64-bit words (photon counter, t_start, t_dry, max_nscat,
// pool_count, pool_next), then the pool ordering (one uint32 per slot), then the parked packets (48 words per slot).
// Every GPU that loads the library holds these 4.0 MB until exit; every call shares them.
static constexpr long long NOALLOC_SLOTS = (long long)THOR_NOALLOC_MAX_SM * 128;       // walk_pool_slots(THOR_NOALLOC_MAX_SM)
static constexpr int NOALLOC_PK_WORDS = 48;
static constexpr size_t NOALLOC_ORDER_OFF = 256, NOALLOC_POOL_OFF = NOALLOC_ORDER_OFF + (size_t)NOALLOC_SLOTS * 4,
                        NOALLOC_BYTES = NOALLOC_POOL_OFF + (size_t)NOALLOC_SLOTS * NOALLOC_PK_WORDS * 4;
static_assert(NOALLOC_BYTES == THOR_NOALLOC_SCRATCH_BYTES, "thor.h states the size of the scratch array");
static_assert(NOALLOC_POOL_OFF % 256 == 0, "the pool starts on a 256-byte boundary");
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];

// In host code `g_noalloc_scratch` is only a handle: its device address is looked up once per device, with that device
// current (the caller holds a DevGuard), and cached.
static cudaError_t noalloc_scratch_address(int device, unsigned char** out) {
    static std::mutex mu;
    static unsigned char* addr[64] = {};
    if (device < 0 || device >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[device]) {
        void* sym = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&sym, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        addr[device] = static_cast<unsigned char*>(sym);
    }
    *out = addr[device];
    return cudaSuccess;
}

extern "C" thor_status thor_run_noalloc(thor_ctx* ctx, unsigned long long n_photons, unsigned long long seed, const thor_opts* opts,
                                        unsigned long long* spectrum_out, unsigned long long* counters_out,
                                        unsigned long long* nscat_hist_out) {
    if (!ctx) return fail(nullptr, THOR_ERR_ARG, "thor_run_noalloc: ctx is NULL");
    { const thor_status st = run_finish(ctx); if (st != THOR_OK) return st; }
    if (ctx->gridless) return fail(ctx, THOR_ERR_UNSUPPORTED, "thor_run_noalloc: gridless datasets are not supported (use thor_run)");
    if (ctx->n_src <= 0) return fail(ctx, THOR_ERR_STATE, "thor_run_noalloc: call thor_sources_set first");
    thor_opts o;
    thor_opts_default(&o);
    if (opts) {
        if (opts->struct_size == 0 || opts->struct_size > sizeof o) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: opts->struct_size is not set (use thor_opts_default)");
        std::memcpy(&o, opts, opts->struct_size);
        o.struct_size = (uint32_t)sizeof o;
    }
    if (o.peel_on || o.raw_output || o.accumulate)
        return fail(ctx, THOR_ERR_UNSUPPORTED, "thor_run_noalloc: peel-off, raw_output and accumulate need memory this entry point may not allocate (use thor_run)");
    if (!counters_out || !nscat_hist_out || (o.spec_bins > 0 && !spectrum_out)) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: an output buffer is NULL");
    if (!phase_ok(o.phase_core) || !phase_ok(o.phase_wing)) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: unknown phase function");
    if (o.core_skip_mode < 0 || o.core_skip_mode > 2 || !(o.x_crit >= 0)) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: bad core-skip options");
    if (o.spec_bins < 0 || o.spec_bins > 4096) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: spec_bins must be in [0, 4096]");
    if (o.spec_bins > 0 && !(o.spec_hi > o.spec_lo)) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: spec_hi must exceed spec_lo");
    if (o.spec_mode != 0 && o.spec_mode != 1) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: spec_mode must be 0 or 1");
    if (o.spec_mode == 0 && !(o.spec_T_ref > 0)) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: spec_T_ref must be > 0");
    if (((o.walk_variant & ~16) != 0 && (o.walk_variant & ~16) != 3 && (o.walk_variant & ~16) != 4) || (o.drain_mode != 0 && o.drain_mode != 1)) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: bad walk_variant / drain_mode");
    if (!(o.dust_albedo >= 0 && o.dust_albedo <= 1) || !(o.dust_g >= -1 && o.dust_g <= 1)) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: dust_albedo must be in [0, 1] and dust_g in [-1, 1]");
    if (o.doublet_on && (!std::isfinite(o.doublet_dv_kms) || !(o.doublet_sigma_ratio >= 0) || !(o.doublet_a_ratio > 0) || !std::isfinite(o.doublet_sigma_ratio) || !std::isfinite(o.doublet_a_ratio)))
        return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: bad doublet options");
    if (!(o.hubble_eps > 0) || !(o.v_max_kms >= 0) || !std::isfinite(o.hubble_kms_per_cell)) return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: bad Hubble / v_max options");
    if (ctx->g.periodic == 7u && ctx->g.frozen != 7u && o.max_crossings == 0)
        return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: the grid is periodic on all three axes (no packet can leave it): set opts.max_crossings");
    // the one size this entry point cannot grow with: the pool holds walk_pool_slots(n_sm) parked packets
    const long long slots = thor::walk_pool_slots(ctx->n_sm);
    if (ctx->n_sm > THOR_NOALLOC_MAX_SM || slots > NOALLOC_SLOTS || thor::walk_pool_words() > NOALLOC_PK_WORDS)
        return fail(ctx, THOR_ERR_ARG, "thor_run_noalloc: this GPU has " + std::to_string(ctx->n_sm) + " multiprocessors and needs " + std::to_string(slots) +
                                       " pool slots; the static scratch holds " + std::to_string(NOALLOC_SLOTS) + " (THOR_NOALLOC_MAX_SM = " +
                                       std::to_string(THOR_NOALLOC_MAX_SM) + "): use thor_run");
    const thor::LyaConstants K = thor::lya_constants();
    thor::WalkParams p = grid_params(ctx);
    p.max_crossings = (o.max_crossings && o.max_crossings < 0xffffffffull) ? (unsigned)o.max_crossings : 0xffffffffu;
    p.n_src = ctx->n_src; p.src_pos = ctx->d_src_pos; p.src_sigma = ctx->d_src_sigma; p.src_cdf = ctx->d_src_cdf;
    p.phase_core = o.phase_core; p.phase_wing = o.phase_wing; p.phase_frame = o.phase_frame;
    p.phase_split_x = (float)o.phase_split_x;
    p.core_skip_mode = o.core_skip_mode; p.x_crit = (float)o.x_crit;
    p.spec_mode = o.spec_mode; p.spec_bins = o.spec_bins;
    p.spec_inv_vth_ref = (float)(1.0 / (K.c_vth * std::sqrt(o.spec_T_ref)));
    p.spec_lo = (float)o.spec_lo;
    p.spec_inv_width = o.spec_bins > 0 ? (float)(o.spec_bins / (o.spec_hi - o.spec_lo)) : 0.f;
    p.hubble = (float)o.hubble_kms_per_cell; p.hubble_eps = (float)o.hubble_eps; p.v_max = (float)o.v_max_kms;
    p.v_max_or_inf = p.v_max > 0.f ? p.v_max : INFINITY;
    p.peel_on = 0;
    p.id_offset = o.photon_id_offset; p.n_photons = n_photons; p.seed = seed; p.max_scatter = o.max_scatter;
    p.max_scatter_or_max = (o.max_scatter == 0 || o.max_scatter > 0xffffffffull) ? 0xffffffffu : (unsigned)o.max_scatter;
    p.walk_variant = o.walk_variant;
    p.dust_albedo = (float)o.dust_albedo; p.dust_g = (float)o.dust_g;
    p.doublet_on = o.doublet_on ? 1 : 0;
    p.db_dv = (float)o.doublet_dv_kms; p.db_rs = (float)o.doublet_sigma_ratio; p.db_ra = (float)o.doublet_a_ratio;
    DevGuard dev_guard(ctx->device);
    unsigned char* scratch = nullptr;
    CU(noalloc_scratch_address(ctx->device, &scratch));
    unsigned long long* small = reinterpret_cast<unsigned long long*>(scratch);
    // what must start at zero: the photon counter, max_nscat, the pool counters (words 0, 3, 4, 5); the timers start at ~0.
    // The pool and its ordering need no clearing: the kernels read only the slots this launch has written.
    CU(cudaMemsetAsync(small, 0, 6 * sizeof(unsigned long long), ctx->stream));
    CU(cudaMemsetAsync(small + 1, 0xFF, 2 * sizeof(unsigned long long), ctx->stream));
    CU(cudaMemsetAsync(counters_out, 0, thor::N_COUNTERS * sizeof(unsigned long long), ctx->stream));
    CU(cudaMemsetAsync(nscat_hist_out, 0, 64 * sizeof(unsigned long long), ctx->stream));
    if (o.spec_bins > 0) CU(cudaMemsetAsync(spectrum_out, 0, (size_t)(o.spec_bins + 2) * sizeof(unsigned long long), ctx->stream));
    p.next_photon = small + 0; p.t_start = small + 1; p.t_dry = small + 2; p.max_nscat = small + 3;
    p.pool_count = small + 4; p.pool_next = small + 5;
    p.pool_order = reinterpret_cast<unsigned int*>(scratch + NOALLOC_ORDER_OFF);
    p.pool = o.drain_mode == 0 ? reinterpret_cast<uint32_t*>(scratch + NOALLOC_POOL_OFF) : nullptr;
    p.pool_mid = nullptr; p.pool_mid_count = nullptr;       // single-pass tail: the static scratch holds one pool
    p.counters = counters_out; p.nscat_hist = nscat_hist_out; p.spectrum = spectrum_out;
    p.cube = nullptr; p.raw = nullptr;
    int blocks = 0;
    if (n_photons > 0) CU(thor::launch_walk(p, ctx->n_sm, ctx->stream, &blocks));
    return THOR_OK;
}

// HOST <-> DEVICE staging of the ray operators' buffers (THOR_RAYS_HOST): device twins owned for the length of one call.
struct Staged {
    std::vector<void*> dev;
    ~Staged() { for (void* d : dev) if (d) cudaFree(d); }
    cudaError_t in(const void* host, size_t bytes, cudaStream_t st, const float** out) {
        void* d = nullptr;
        cudaError_t e = cudaMalloc(&d, bytes);
        if (e != cudaSuccess) return e;
        dev.push_back(d);
        *out = static_cast<const float*>(d);
        return cudaMemcpyAsync(d, host, bytes, cudaMemcpyHostToDevice, st);
    }
    cudaError_t out(size_t bytes, float** out_dev) {
        void* d = nullptr;
        cudaError_t e = cudaMalloc(&d, bytes);
        if (e != cudaSuccess) return e;
        dev.push_back(d);
        *out_dev = static_cast<float*>(d);
        return cudaSuccess;
    }
};

extern "C" thor_status thor_raytrace_ex(thor_ctx* ctx, long long n_rays, const float* org_xyz, const float* dir_xyz,
                                        const thor_ray_opts* o, float* out_column, float* out_tmean, float* out_tau) {
    if (!ctx) return fail(nullptr, THOR_ERR_ARG, "thor_raytrace: ctx is NULL");
    if (ctx->gridless) return fail(ctx, THOR_ERR_UNSUPPORTED, "thor_raytrace: needs a grid dataset");
    if (!o || o->struct_size != sizeof(thor_ray_opts)) return fail(ctx, THOR_ERR_ARG, "thor_raytrace_ex: opts->struct_size is not set");
    if (n_rays <= 0 || !org_xyz || !dir_xyz) return fail(ctx, THOR_ERR_ARG, "thor_raytrace: no rays");
    if (!out_column && !out_tmean && !out_tau) return fail(ctx, THOR_ERR_ARG, "thor_raytrace: no output requested");
    if (out_tau && (o->n_v <= 0 || !(o->v_hi > o->v_lo))) return fail(ctx, THOR_ERR_ARG, "thor_raytrace: bad velocity axis");
    if (!std::isfinite(o->hubble_kms_per_cell) || !(o->hubble_eps >= 0) || !(o->max_length_cells >= 0) || !std::isfinite(o->max_length_cells))
        return fail(ctx, THOR_ERR_ARG, "thor_raytrace: bad Hubble term / sub-sampling / length");
    const thor::WalkParams p = grid_params(ctx);
    DevGuard dev_guard(ctx->device);
    const bool host = (o->flags & THOR_RAYS_HOST) != 0;
    const int n_v = out_tau ? o->n_v : 0;
    Staged st;
    const float *d_org = org_xyz, *d_dir = dir_xyz;
    float *d_col = out_column, *d_tm = out_tmean, *d_tau = out_tau;
    if (host) {
        CU(st.in(org_xyz, (size_t)n_rays * 12, ctx->stream, &d_org));
        CU(st.in(dir_xyz, (size_t)n_rays * 12, ctx->stream, &d_dir));
        if (out_column) CU(st.out((size_t)n_rays * 4, &d_col));
        if (out_tmean) CU(st.out((size_t)n_rays * 4, &d_tm));
        if (out_tau) CU(st.out((size_t)n_rays * n_v * 4, &d_tau));
    }
    CU(thor::launch_raytrace(p, n_rays, d_org, d_dir, (float)o->hubble_kms_per_cell, (float)o->hubble_eps,
                             (float)o->max_length_cells, n_v, (float)o->v_lo, n_v ? (float)((o->v_hi - o->v_lo) / n_v) : 0.f,
                             d_col, d_tm, d_tau, ctx->stream));
    if (host) {
        if (out_column) CU(cudaMemcpyAsync(out_column, d_col, (size_t)n_rays * 4, cudaMemcpyDeviceToHost, ctx->stream));
        if (out_tmean) CU(cudaMemcpyAsync(out_tmean, d_tm, (size_t)n_rays * 4, cudaMemcpyDeviceToHost, ctx->stream));
        if (out_tau) CU(cudaMemcpyAsync(out_tau, d_tau, (size_t)n_rays * n_v * 4, cudaMemcpyDeviceToHost, ctx->stream));
    }
    CU(cudaStreamSynchronize(ctx->stream));
    return THOR_OK;
}

extern "C" thor_status thor_raytrace(thor_ctx* ctx, long long n_rays, const float* org_xyz, const float* dir_xyz,
                                     double hubble_kms_per_cell, int n_v, double v_lo, double v_hi, float* out_column,
                                     float* out_tmean, float* out_tau) {
    thor_ray_opts o{};
    o.struct_size = (uint32_t)sizeof o;
    o.hubble_kms_per_cell = hubble_kms_per_cell;
    o.n_v = n_v; o.v_lo = v_lo; o.v_hi = v_hi;
    return thor_raytrace_ex(ctx, n_rays, org_xyz, dir_xyz, &o, out_column, out_tmean, out_tau);
}

extern "C" thor_status thor_volume_render_ex(thor_ctx* ctx, long long n_rays, const float* org_xyz, const float* dir_xyz,
                                             int n_peaks, const float* peaks, double n_ref, float* out_rgba, unsigned flags) {
    if (!ctx) return fail(nullptr, THOR_ERR_ARG, "thor_volume_render: ctx is NULL");
    if (ctx->gridless) return fail(ctx, THOR_ERR_UNSUPPORTED, "thor_volume_render: needs a grid dataset");
    if (n_rays <= 0 || !org_xyz || !dir_xyz || !out_rgba) return fail(ctx, THOR_ERR_ARG, "thor_volume_render: no rays or no output");
    if (!peaks || n_peaks < 1 || n_peaks > THOR_MAX_TF_PEAKS) return fail(ctx, THOR_ERR_ARG, "thor_volume_render: n_peaks out of range");
    if (!(n_ref >= 0.0) || !std::isfinite(n_ref)) return fail(ctx, THOR_ERR_ARG, "thor_volume_render: bad n_ref");
    static_assert(THOR_MAX_TF_PEAKS == thor::MAX_TF_PEAKS, "peak limit");
    thor::TransferFn tf{};
    tf.n_peaks = n_peaks;
    tf.weight_by_density = n_ref > 0.0 ? 1 : 0;
    const double l2_10 = 3.321928094887362;            // log2(10): log10 T = log2 T / log2 10
    for (int q = 0; q < n_peaks; ++q) {
        const float* k = peaks + 6 * q;
        for (int j = 0; j < 6; ++j)
            if (!std::isfinite(k[j])) return fail(ctx, THOR_ERR_ARG, "thor_volume_render: non-finite peak");
        if (!(k[1] > 0.f) || k[5] < 0.f) return fail(ctx, THOR_ERR_ARG, "thor_volume_render: width must be > 0 and A >= 0");
        const double s2 = (double)k[1] * l2_10;        // width in log2 T
        tf.centre[q] = (float)((double)k[0] * l2_10);
        tf.neg_inv_2s2[q] = (float)(-1.4426950408889634 / (2.0 * s2 * s2));
        tf.amp[q] = (float)(n_ref > 0.0 ? (double)k[5] / n_ref : (double)k[5]);
        tf.r[q] = k[2]; tf.g[q] = k[3]; tf.b[q] = k[4];
    }
    const thor::WalkParams p = grid_params(ctx);
    DevGuard dev_guard(ctx->device);
    const bool host = (flags & THOR_RAYS_HOST) != 0;
    Staged st;
    const float *d_org = org_xyz, *d_dir = dir_xyz;
    float* d_out = out_rgba;
    if (host) {
        CU(st.in(org_xyz, (size_t)n_rays * 12, ctx->stream, &d_org));
        CU(st.in(dir_xyz, (size_t)n_rays * 12, ctx->stream, &d_dir));
        CU(st.out((size_t)n_rays * 16, &d_out));
    }
    CU(thor::launch_volume_render(p, tf, n_rays, d_org, d_dir, d_out, ctx->stream));
    if (host) CU(cudaMemcpyAsync(out_rgba, d_out, (size_t)n_rays * 16, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return THOR_OK;
}

extern "C" thor_status thor_volume_render(thor_ctx* ctx, long long n_rays, const float* org_xyz, const float* dir_xyz,
                                          int n_peaks, const float* peaks, double n_ref, float* out_rgba) {
    return thor_volume_render_ex(ctx, n_rays, org_xyz, dir_xyz, n_peaks, peaks, n_ref, out_rgba, 0u);
}

extern "C" thor_status thor_slice(thor_ctx* ctx, long long n_points, const float* pos_xyz, int field, float* out, unsigned flags) {
    if (!ctx) return fail(nullptr, THOR_ERR_ARG, "thor_slice: ctx is NULL");
    if (ctx->gridless) return fail(ctx, THOR_ERR_UNSUPPORTED, "thor_slice: needs a grid dataset");
    if (n_points <= 0 || !pos_xyz || !out) return fail(ctx, THOR_ERR_ARG, "thor_slice: no points or no output");
    if (field < THOR_FIELD_NHI || field > THOR_FIELD_KDUST) return fail(ctx, THOR_ERR_ARG, "thor_slice: unknown field");
    if (field == THOR_FIELD_KDUST && !ctx->has_dust) return fail(ctx, THOR_ERR_ARG, "thor_slice: the grid has no dust field");
    const thor::WalkParams p = grid_params(ctx);
    DevGuard dev_guard(ctx->device);
    const bool host = (flags & THOR_RAYS_HOST) != 0;
    Staged st;
    const float* d_pos = pos_xyz;
    float* d_out = out;
    if (host) {
        CU(st.in(pos_xyz, (size_t)n_points * 12, ctx->stream, &d_pos));
        CU(st.out((size_t)n_points * 4, &d_out));
    }
    CU(thor::launch_slice(p, n_points, d_pos, field, d_out, ctx->stream));
    if (host) CU(cudaMemcpyAsync(out, d_out, (size_t)n_points * 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return THOR_OK;
}

extern "C" thor_status thor_last_run_ms(const thor_ctx* ctx, float* ms) {
    if (!ctx || !ms) return fail(nullptr, THOR_ERR_ARG, "thor_last_run_ms: NULL argument");
    if (ctx->pending) return fail(const_cast<thor_ctx*>(ctx), THOR_ERR_STATE, "thor_last_run_ms: a run is pending (thor_wait first)");
    if (!ctx->have_run) return fail(const_cast<thor_ctx*>(ctx), THOR_ERR_STATE, "thor_last_run_ms: no run yet");
    *ms = ctx->last_ms;
    return THOR_OK;
}

extern "C" thor_status thor_last_run_max_nscat(const thor_ctx* ctx, unsigned long long* n) {
    if (!ctx || !n) return fail(nullptr, THOR_ERR_ARG, "thor_last_run_max_nscat: NULL argument");
    if (ctx->pending) return fail(const_cast<thor_ctx*>(ctx), THOR_ERR_STATE, "thor_last_run_max_nscat: a run is pending (thor_wait first)");
    if (!ctx->have_run) return fail(const_cast<thor_ctx*>(ctx), THOR_ERR_STATE, "thor_last_run_max_nscat: no run yet");
    *n = ctx->last_max_nscat;
    return THOR_OK;
}

extern "C" thor_status thor_last_run_feed_ms(const thor_ctx* ctx, float* ms) {
    if (!ctx || !ms) return fail(nullptr, THOR_ERR_ARG, "thor_last_run_feed_ms: NULL argument");
    if (ctx->pending) return fail(const_cast<thor_ctx*>(ctx), THOR_ERR_STATE, "thor_last_run_feed_ms: a run is pending (thor_wait first)");
    if (!ctx->have_run) return fail(const_cast<thor_ctx*>(ctx), THOR_ERR_STATE, "thor_last_run_feed_ms: no run yet");
    *ms = ctx->last_feed_ms;
    return THOR_OK;
}

extern "C" thor_status thor_tally_get(thor_ctx* ctx, int kind, void* dst, size_t dst_bytes, size_t* needed) {
    if (!ctx) return fail(nullptr, THOR_ERR_ARG, "thor_tally_get: ctx is NULL");
    { const thor_status st = run_finish(ctx); if (st != THOR_OK) return st; }
    if (!ctx->have_run) return fail(ctx, THOR_ERR_STATE, "thor_tally_get: no completed run");
    const bool dev_dst = (kind & THOR_TALLY_DEVICE_DST) != 0;
    const int k = kind & ~THOR_TALLY_DEVICE_DST;
    const void* src = nullptr;
    size_t bytes = 0;
    switch (k) {
        case THOR_TALLY_SPECTRUM:
            src = ctx->d_small + SMALL_SPEC; bytes = ((size_t)ctx->last.spec_bins + 2) * 8; break;
        case THOR_TALLY_NSCAT_HIST: src = ctx->d_small + SMALL_HIST; bytes = 64 * 8; break;
        case THOR_TALLY_COUNTERS: src = ctx->d_small + SMALL_COUNTERS; bytes = (size_t)thor::N_COUNTERS * 8; break;
        case THOR_TALLY_CUBE:
            if (!ctx->last.peel_on || !ctx->d_cube) return fail(ctx, THOR_ERR_STATE, "thor_tally_get: the last run had no peel-off");
            src = ctx->d_cube; bytes = ctx->cube_elems * 8; break;
        case THOR_TALLY_RAW:
            if (!ctx->last.raw_output || !ctx->d_raw) return fail(ctx, THOR_ERR_STATE, "thor_tally_get: the last run kept no raw records");
            src = ctx->d_raw; bytes = (size_t)ctx->last_n * sizeof(thor::RawRecord); break;
        default: return fail(ctx, THOR_ERR_ARG, "thor_tally_get: unknown tally kind");
    }
    if (needed) *needed = bytes;
    if (!dst) return THOR_OK;
    if (dst_bytes < bytes) return fail(ctx, THOR_ERR_ARG, "thor_tally_get: dst_bytes too small");
    if (bytes == 0) return THOR_OK;
    DevGuard dev_guard(ctx->device);
    if (k == THOR_TALLY_CUBE && !dev_dst) {
        // fixed point -> double on the host
        std::vector<unsigned long long> tmp;
        try { tmp.resize(ctx->cube_elems); } catch (...) { return fail(ctx, THOR_ERR_OOM, "thor_tally_get: host allocation failed"); }
        CU(cudaMemcpyAsync(tmp.data(), src, bytes, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        double* d = static_cast<double*>(dst);
        for (size_t i = 0; i < ctx->cube_elems; ++i) d[i] = (double)tmp[i] / thor::CUBE_FIXED_SCALE;
        return THOR_OK;
    }
    CU(cudaMemcpyAsync(dst, src, bytes, dev_dst ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return THOR_OK;
}
