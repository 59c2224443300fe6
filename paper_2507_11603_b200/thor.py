"""Thin ctypes binding over the C-ABI of include/thor.h (libthor_b200.so).  Argument marshalling only: every step of
the path runs in the CUDA kernels.  torch supplies device memory and the stream.  There is no CPU fallback: loading
fails loudly if the library is missing, and every call raises ThorError on a non-zero status.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libthor_b200.so")

STATUS = {0: "THOR_OK", 1: "THOR_ERR_ARG", 2: "THOR_ERR_STATE", 3: "THOR_ERR_OOM", 4: "THOR_ERR_CUDA",
          5: "THOR_ERR_UNSUPPORTED"}
GRID_HOST, PERIODIC_X, PERIODIC_Y, PERIODIC_Z, GRID_NO_VALIDATE, GRID_PACK = 0x1, 0x10, 0x20, 0x40, 0x100, 0x200
GRID_L2_PERSIST, GRID_L2_FETCH32 = 0x400, 0x800
TALLY_SPECTRUM, TALLY_NSCAT_HIST, TALLY_COUNTERS, TALLY_CUBE, TALLY_RAW, TALLY_DEVICE_DST = 0, 1, 2, 3, 4, 0x100
COUNTER_NAMES = ["escaped", "absorbed", "terminated", "capped", "scatterings", "cell_crossings", "rejection_iters",
                 "peel_rays", "peel_cells", "dust_scatterings"]
RAW_DTYPE = np.dtype([("V", "<f4"), ("nscat", "<u4"), ("status", "<i4"), ("kx", "<f4"), ("ky", "<f4"), ("kz", "<f4")])

EXPORTS = ["thor_grid_create", "thor_dataset_create_gridless", "thor_grid_destroy", "thor_sources_set", "thor_opts_default", "thor_run", "thor_run_async", "thor_wait", "thor_run_noalloc",
           "thor_last_run_ms", "thor_last_run_feed_ms", "thor_last_run_max_nscat", "thor_raytrace", "thor_raytrace_ex", "thor_volume_render", "thor_volume_render_ex", "thor_slice", "thor_tally_get", "thor_last_error", "thor_unit_philox", "thor_unit_curand_philox", "thor_unit_dda_trace",
           "thor_unit_voigt", "thor_unit_scatter"]


class ThorError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class Opts(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32),
        ("phase_core", C.c_int32), ("phase_wing", C.c_int32), ("phase_frame", C.c_int32),
        ("phase_split_x", C.c_double),
        ("core_skip_mode", C.c_int32), ("x_crit", C.c_double),
        ("spec_mode", C.c_int32), ("spec_T_ref", C.c_double), ("spec_bins", C.c_int32),
        ("spec_lo", C.c_double), ("spec_hi", C.c_double),
        ("hubble_kms_per_cell", C.c_double), ("hubble_eps", C.c_double), ("v_max_kms", C.c_double),
        ("peel_on", C.c_int32), ("k_obs", C.c_double * 3),
        ("peel_nx", C.c_int32), ("peel_ny", C.c_int32), ("peel_nv", C.c_int32),
        ("peel_v_lo", C.c_double), ("peel_v_hi", C.c_double), ("peel_width_cells", C.c_double),
        ("tau_peel_max", C.c_double),
        ("photon_id_offset", C.c_uint64), ("max_scatter", C.c_uint64),
        ("raw_output", C.c_int32), ("accumulate", C.c_int32),
        ("max_crossings", C.c_uint64), ("walk_variant", C.c_int32), ("drain_mode", C.c_int32),
        ("dust_albedo", C.c_double), ("dust_g", C.c_double), ("doublet_on", C.c_int32),
        ("doublet_dv_kms", C.c_double), ("doublet_sigma_ratio", C.c_double), ("doublet_a_ratio", C.c_double),
    ]


class RayOpts(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("flags", C.c_uint32), ("hubble_kms_per_cell", C.c_double), ("hubble_eps", C.c_double),
                ("max_length_cells", C.c_double), ("n_v", C.c_int32), ("v_lo", C.c_double), ("v_hi", C.c_double)]


RAYS_HOST = 0x1
FIELDS = dict(nHI=0, T=1, vx=2, vy=3, vz=4, kdust=5)


class Gridless(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("geometry", C.c_int32), ("r_in", C.c_double), ("r_out", C.c_double),
                ("length_cm", C.c_double), ("n0", C.c_double), ("alpha_rho", C.c_double), ("T", C.c_double),
                ("v_max", C.c_double), ("alpha_v", C.c_double), ("kdust0", C.c_double), ("step_f", C.c_double)]


GRIDLESS_DEFAULTS = dict(geometry=0, r_in=0.0, r_out=1.0, length_cm=1.0, n0=0.0, alpha_rho=0.0, T=1e4, v_max=0.0, alpha_v=1.0,
                         kdust0=0.0, step_f=0.01)

_lib = None


def lib():
    """Loads libthor_b200.so (built by csrc/build.py / __graft_entry__.build()).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ThorError(5, f"{LIB_PATH} is missing: build it with `python -m paper_2507_11603_b200.csrc.build` "
                               "(CUDA, sm_100a); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        P, i32, i64, u32, u64, d, f = C.c_void_p, C.c_int, C.c_longlong, C.c_uint, C.c_uint64, C.c_double, C.c_float
        L.thor_grid_create.argtypes = [C.POINTER(P), i32, i32, i32, d, P, P, P, P, P, P, u32, P]
        L.thor_dataset_create_gridless.argtypes = [C.POINTER(P), C.POINTER(Gridless), P]
        L.thor_grid_destroy.argtypes = [P]
        L.thor_grid_destroy.restype = None
        L.thor_sources_set.argtypes = [P, i64, P, P, P]
        L.thor_opts_default.argtypes = [C.POINTER(Opts)]
        L.thor_opts_default.restype = None
        L.thor_run.argtypes = [P, C.c_ulonglong, C.c_ulonglong, C.POINTER(Opts)]
        L.thor_run_async.argtypes = [P, C.c_ulonglong, C.c_ulonglong, C.POINTER(Opts)]
        L.thor_wait.argtypes = [P]
        L.thor_run_noalloc.argtypes = [P, C.c_ulonglong, C.c_ulonglong, C.POINTER(Opts), P, P, P]
        L.thor_last_run_ms.argtypes = [P, C.POINTER(f)]
        L.thor_last_run_feed_ms.argtypes = [P, C.POINTER(f)]
        L.thor_last_run_max_nscat.argtypes = [P, C.POINTER(C.c_ulonglong)]
        L.thor_raytrace.argtypes = [P, i64, P, P, d, i32, d, d, P, P, P]
        L.thor_volume_render.argtypes = [P, i64, P, P, i32, P, d, P]
        L.thor_raytrace_ex.argtypes = [P, i64, P, P, C.POINTER(RayOpts), P, P, P]
        L.thor_volume_render_ex.argtypes = [P, i64, P, P, i32, P, d, P, u32]
        L.thor_slice.argtypes = [P, i64, P, i32, P, u32]
        L.thor_tally_get.argtypes = [P, i32, P, C.c_size_t, C.POINTER(C.c_size_t)]
        L.thor_last_error.argtypes = [P]
        L.thor_last_error.restype = C.c_char_p
        L.thor_unit_philox.argtypes = [u64, u64, i64, i32, P, P]
        L.thor_unit_curand_philox.argtypes = [u64, u64, i64, i32, P, P]
        L.thor_unit_dda_trace.argtypes = [i32, i32, i32, u32, i64, P, P, i64, P, P, P, P, P, P]
        L.thor_unit_voigt.argtypes = [i64, P, P, P, P]
        L.thor_unit_scatter.argtypes = [f, f, f, i32, u64, u64, i64, P, P, P, P, P]
        _lib = L
    return _lib


def _check(status, ctx=None):
    if status != 0:
        msg = lib().thor_last_error(ctx)
        raise ThorError(status, (msg or b"").decode())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def make_opts(**kw):
    o = Opts()
    lib().thor_opts_default(C.byref(o))
    for k, v in kw.items():
        if not hasattr(o, k):
            raise KeyError(f"unknown thor_opts field: {k}")
        if k == "k_obs":
            o.k_obs = (C.c_double * 3)(*v)
        else:
            setattr(o, k, v)
    return o


def _periodic_flags(periodic):
    return (PERIODIC_X if periodic[0] else 0) | (PERIODIC_Y if periodic[1] else 0) | (PERIODIC_Z if periodic[2] else 0)


class Context:
    """One grid + its sources + its tallies (thor_ctx).  Fields: torch CUDA float32 tensors [nz, ny, nx] (borrowed:
    kept referenced here) or numpy float32 arrays (host=True: copied to the device by the library)."""

    def __init__(self, nx, ny, nz, cell_cm, nHI, T, vx, vy, vz, kdust=None, periodic=(0, 0, 0), host=False,
                 validate=True, pack=False, extra_flags=0):
        self._ctx = C.c_void_p()
        fields = [nHI, T, vx, vy, vz, kdust]
        flags = _periodic_flags(periodic) | (0 if validate else GRID_NO_VALIDATE) | (GRID_PACK if pack else 0) | int(extra_flags)
        if host:
            self._keep = [None if a is None else np.ascontiguousarray(a, np.float32) for a in fields]
            ptrs = [None if a is None else a.ctypes.data_as(C.c_void_p) for a in self._keep]
            flags |= GRID_HOST
            stream = C.c_void_p(0)
            try:
                stream = _stream()
            except Exception:
                pass
        else:
            import torch
            for a in fields:
                if a is not None and not (a.is_cuda and a.dtype == torch.float32 and a.is_contiguous()):
                    raise ValueError("fields must be contiguous float32 CUDA tensors (or pass host=True)")
            self._keep = fields
            ptrs = [None if a is None else C.c_void_p(a.data_ptr()) for a in fields]
            stream = _stream()
        for a in self._keep:
            if a is not None and int(np.prod(a.shape)) != nx * ny * nz:
                raise ValueError("field size does not match nx*ny*nz")
        _check(lib().thor_grid_create(C.byref(self._ctx), nx, ny, nz, float(cell_cm), *ptrs, flags, stream))
        if pack:
            self._keep = None              # THOR_GRID_PACK: the library holds its own copy; release ours

    @classmethod
    def gridless(cls, **dataset):
        """A gridless shell / sphere / slab dataset (thor_dataset_create_gridless); keys of GRIDLESS_DEFAULTS."""
        unknown = set(dataset) - set(GRIDLESS_DEFAULTS)
        if unknown:
            raise KeyError(f"unknown gridless fields: {unknown}")
        d = Gridless(struct_size=C.sizeof(Gridless), **{**GRIDLESS_DEFAULTS, **dataset})
        self = cls.__new__(cls)
        self._ctx = C.c_void_p()
        self._keep = None
        _check(lib().thor_dataset_create_gridless(C.byref(self._ctx), C.byref(d), _stream()))
        return self

    @classmethod
    def from_workload(cls, grid, host=False, device="cuda", pack=False, extra_flags=0):
        """grid: the dict made by paper_2507_11603_b200.workloads (numpy float32 fields) or .workloads_device (CUDA
        tensors, borrowed as they are)."""
        keys = ("nHI", "T", "vx", "vy", "vz", "kdust")
        if host:
            arrs = [grid.get(k) for k in keys]
        else:
            import torch
            arrs = [None if grid.get(k) is None else
                    (grid[k] if isinstance(grid[k], torch.Tensor) else
                     torch.from_numpy(np.ascontiguousarray(grid[k], np.float32)).to(device)) for k in keys]
        return cls(grid["nx"], grid["ny"], grid["nz"], grid["cell_cm"], *arrs,
                   periodic=grid.get("periodic", (0, 0, 0)), host=host, pack=pack, extra_flags=extra_flags)

    def close(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            L = _lib                      # at interpreter shutdown the module globals may already be gone
            if L is not None:
                L.thor_grid_destroy(self._ctx)
            self._ctx = C.c_void_p()
        self._keep = None

    __del__ = close

    def sources_set(self, pos, lum, sigma):
        pos = np.ascontiguousarray(pos, np.float32).reshape(-1, 3)
        lum = np.ascontiguousarray(lum, np.float32)
        sigma = np.ascontiguousarray(sigma, np.float32)
        if not (pos.shape[0] == lum.shape[0] == sigma.shape[0]):
            raise ValueError("pos, lum, sigma lengths differ")
        _check(lib().thor_sources_set(self._ctx, pos.shape[0], pos.ctypes.data_as(C.c_void_p),
                                      lum.ctypes.data_as(C.c_void_p), sigma.ctypes.data_as(C.c_void_p)), self._ctx)

    def run(self, n_photons, seed, opts=None, **kw):
        if opts is None:
            opts = make_opts(**kw)
        elif isinstance(opts, dict):
            opts = make_opts(**{**opts, **kw})
        self._opts = opts
        self._n = int(n_photons)
        _check(lib().thor_run(self._ctx, int(n_photons), int(seed), C.byref(opts)), self._ctx)

    def run_async(self, n_photons, seed, opts=None, **kw):
        """thor_run_async: enqueue the run and return; wait() (or any tally getter) completes it."""
        if opts is None:
            opts = make_opts(**kw)
        elif isinstance(opts, dict):
            opts = make_opts(**{**opts, **kw})
        self._opts = opts
        self._n = int(n_photons)
        _check(lib().thor_run_async(self._ctx, int(n_photons), int(seed), C.byref(opts)), self._ctx)

    def wait(self):
        _check(lib().thor_wait(self._ctx), self._ctx)

    def run_noalloc(self, n_photons, seed, opts, spectrum_out, counters_out, nscat_hist_out):
        """thor_run_noalloc: the same walk without any device allocation; the tallies go into the caller's torch CUDA int64
        tensors (spectrum_out: spec_bins + 2, counters_out: len(COUNTER_NAMES), nscat_hist_out: 64).  Asynchronous on the
        context's stream; the context's own tallies are not touched."""
        if isinstance(opts, dict):
            opts = make_opts(**opts)
        ptr = lambda t: None if t is None else C.c_void_p(t.data_ptr())
        _check(lib().thor_run_noalloc(self._ctx, int(n_photons), int(seed), C.byref(opts), ptr(spectrum_out), ptr(counters_out),
                                      ptr(nscat_hist_out)), self._ctx)

    def last_run_ms(self):
        ms = C.c_float()
        _check(lib().thor_last_run_ms(self._ctx, C.byref(ms)), self._ctx)
        return ms.value

    def raytrace(self, origins, dirs, n_v=0, v_lo=0.0, v_hi=1.0, hubble_kms_per_cell=0.0, hubble_eps=0.0, max_length_cells=0.0):
        """Projection / absorption spectra along rays (thor_raytrace_ex with HOST buffers: the library does the copies).
        Returns dict(column, tmean[, tau])."""
        org = np.ascontiguousarray(origins, np.float32).reshape(-1, 3)
        dr = np.ascontiguousarray(dirs, np.float32).reshape(-1, 3)
        n = org.shape[0]
        col, tm = np.empty(n, np.float32), np.empty(n, np.float32)
        tau = np.empty((n, n_v), np.float32) if n_v > 0 else None
        o = RayOpts(struct_size=C.sizeof(RayOpts), flags=RAYS_HOST, hubble_kms_per_cell=float(hubble_kms_per_cell),
                    hubble_eps=float(hubble_eps), max_length_cells=float(max_length_cells), n_v=int(n_v), v_lo=float(v_lo), v_hi=float(v_hi))
        p = lambda a: None if a is None else a.ctypes.data_as(C.c_void_p)
        _check(lib().thor_raytrace_ex(self._ctx, n, p(org), p(dr), C.byref(o), p(col), p(tm), p(tau)), self._ctx)
        out = dict(column=col, tmean=tm)
        if tau is not None:
            out["tau"] = tau
        return out

    def volume_render(self, origins, dirs, peaks, n_ref=0.0):
        """Volume rendering along rays (thor_volume_render_ex, Eq. 12; HOST buffers).  Returns float32[n][4] = (C_R, C_G, C_B, opacity)."""
        org = np.ascontiguousarray(origins, np.float32).reshape(-1, 3)
        dr = np.ascontiguousarray(dirs, np.float32).reshape(-1, 3)
        pk = np.ascontiguousarray(peaks, np.float32).reshape(-1, 6)
        out = np.empty((org.shape[0], 4), np.float32)
        p = lambda a: a.ctypes.data_as(C.c_void_p)
        _check(lib().thor_volume_render_ex(self._ctx, org.shape[0], p(org), p(dr), pk.shape[0], p(pk), float(n_ref), p(out), RAYS_HOST), self._ctx)
        return out

    def slice(self, points, field):
        """Slice operator (thor_slice): the value of `field` ('nHI', 'T', 'vx', 'vy', 'vz', 'kdust') in the cell holding each point."""
        pts = np.ascontiguousarray(points, np.float32).reshape(-1, 3)
        out = np.empty(pts.shape[0], np.float32)
        _check(lib().thor_slice(self._ctx, pts.shape[0], pts.ctypes.data_as(C.c_void_p), FIELDS[field], out.ctypes.data_as(C.c_void_p), RAYS_HOST), self._ctx)
        return out

    def last_run_max_nscat(self):
        n = C.c_ulonglong()
        _check(lib().thor_last_run_max_nscat(self._ctx, C.byref(n)), self._ctx)
        return n.value

    def last_run_feed_ms(self):
        ms = C.c_float()
        _check(lib().thor_last_run_feed_ms(self._ctx, C.byref(ms)), self._ctx)
        return ms.value

    def _get(self, kind, dtype, shape):
        out = np.empty(shape, dtype)
        need = C.c_size_t()
        _check(lib().thor_tally_get(self._ctx, kind, out.ctypes.data_as(C.c_void_p), out.nbytes, C.byref(need)), self._ctx)
        assert need.value == out.nbytes, (need.value, out.nbytes)
        return out

    def tally_to_device(self, kind, tensor):
        """Copies tally `kind` into a CUDA tensor (THOR_TALLY_DEVICE_DST): no host round trip (multi-GPU reduce)."""
        nbytes = tensor.numel() * tensor.element_size()
        need = C.c_size_t()
        _check(lib().thor_tally_get(self._ctx, kind | TALLY_DEVICE_DST, C.c_void_p(tensor.data_ptr()), nbytes,
                                    C.byref(need)), self._ctx)
        assert need.value == nbytes, (need.value, nbytes)
        return tensor

    def spectrum(self):
        return self._get(TALLY_SPECTRUM, np.uint64, self._opts.spec_bins + 2)

    def nscat_hist(self):
        return self._get(TALLY_NSCAT_HIST, np.uint64, 64)

    def counters(self):
        c = self._get(TALLY_COUNTERS, np.uint64, len(COUNTER_NAMES))
        return dict(zip(COUNTER_NAMES, (int(v) for v in c)))

    def cube(self):
        o = self._opts
        return self._get(TALLY_CUBE, np.float64, (o.peel_ny, o.peel_nx, o.peel_nv))

    def raw(self):
        return self._get(TALLY_RAW, RAW_DTYPE, self._n)


def run_workload(w, n_photons=None, host=False, raw=True, pack=False, **opt_overrides):
    """Convenience: build a Context from a workloads.* dict (or dict(dataset=<gridless fields>, ...)), run it, return the
    tallies as a dict."""
    ctx = Context.gridless(**w["dataset"]) if "dataset" in w else Context.from_workload(w["grid"], host=host, pack=pack)
    try:
        ctx.sources_set(w["sources"]["pos"], w["sources"]["lum"], w["sources"]["sigma"])
        n = w["n_photons"] if n_photons is None else n_photons
        ctx.run(n, w["seed"], dict(w["opts"], raw_output=1 if raw else 0, **opt_overrides))
        out = dict(spectrum=ctx.spectrum(), nscat_hist=ctx.nscat_hist(), counters=ctx.counters(), ms=ctx.last_run_ms())
        out["cube"] = ctx.cube() if w["opts"].get("peel_on") else None
        out["raw"] = ctx.raw() if raw else None
        return out
    finally:
        ctx.close()


# ---- single steps (device tensors in, device tensors out) ----

def unit_philox(seed, id0, n_ids, n_draws):
    import torch
    out = torch.empty((n_ids, n_draws), dtype=torch.int32, device="cuda")
    _check(lib().thor_unit_philox(int(seed), int(id0), n_ids, n_draws, C.c_void_p(out.data_ptr()), _stream()))
    return out.cpu().numpy().view(np.uint32)


def unit_curand_philox(seed, id0, n_ids, n_draws):
    import torch
    out = torch.empty((n_ids, n_draws), dtype=torch.int32, device="cuda")
    _check(lib().thor_unit_curand_philox(int(seed), int(id0), n_ids, n_draws, C.c_void_p(out.data_ptr()), _stream()))
    return out.cpu().numpy().view(np.uint32)


def unit_dda_trace(dims, periodic, origins, dirs, max_steps=1 << 20, want_seq=False):
    import torch
    org = torch.from_numpy(np.ascontiguousarray(origins, np.float32)).cuda()
    dr = torch.from_numpy(np.ascontiguousarray(dirs, np.float32)).cuda()
    n = org.shape[0]
    hi = torch.empty(n, dtype=torch.int64, device="cuda")
    hl = torch.empty(n, dtype=torch.int64, device="cuda")
    cnt = torch.empty(n, dtype=torch.int32, device="cuda")
    si = sl = None
    if want_seq:
        si = torch.zeros(max_steps, dtype=torch.int64, device="cuda")
        sl = torch.zeros(max_steps, dtype=torch.float32, device="cuda")
    p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
    _check(lib().thor_unit_dda_trace(int(dims[0]), int(dims[1]), int(dims[2]), _periodic_flags(periodic), n, p(org), p(dr),
                                     int(max_steps), p(hi), p(hl), p(cnt), p(si), p(sl), _stream()))
    out = dict(hash_idx=hi.cpu().numpy().view(np.uint64), hash_len=hl.cpu().numpy().view(np.uint64),
               count=cnt.cpu().numpy().view(np.uint32))
    if want_seq:
        c = int(out["count"][0])
        out["seq_idx"] = si.cpu().numpy()[:c]
        out["seq_len"] = sl.cpu().numpy()[:c]
    return out


def unit_voigt(a, x):
    import torch
    a = torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda()
    x = torch.from_numpy(np.ascontiguousarray(x, np.float32)).cuda()
    out = torch.empty_like(x)
    _check(lib().thor_unit_voigt(x.numel(), C.c_void_p(a.data_ptr()), C.c_void_p(x.data_ptr()),
                                 C.c_void_p(out.data_ptr()), _stream()))
    return out.cpu().numpy()


def unit_scatter(a, x_in, n, x_crit=0.0, phase=0, seed=1, id0=0):
    import torch
    up = torch.empty(n, dtype=torch.float32, device="cuda")
    xo = torch.empty(n, dtype=torch.float32, device="cuda")
    ko = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    it = torch.empty(n, dtype=torch.int32, device="cuda")
    _check(lib().thor_unit_scatter(float(a), float(x_in), float(x_crit), int(phase), int(seed), int(id0), n,
                                   C.c_void_p(up.data_ptr()), C.c_void_p(xo.data_ptr()), C.c_void_p(ko.data_ptr()),
                                   C.c_void_p(it.data_ptr()), _stream()))
    return dict(u_par=up.cpu().numpy(), x_out=xo.cpu().numpy(), k_out=ko.cpu().numpy(), iters=it.cpu().numpy().view(np.uint32))
