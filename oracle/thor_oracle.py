"""ORACLE — TEST INFRASTRUCTURE ONLY.

ctypes loader for the fp64 CPU oracle (oracle/*.hpp, capi.cpp).  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the CUDA package.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboracle.so")
_SOURCES = ["capi.cpp", "walker.hpp", "gridless.hpp", "dda.hpp", "sampler.hpp", "voigt.hpp", "philox.hpp", "constants.hpp"]


def build(force=False):
    """Compile the oracle with g++ (no fast-math, no FMA contraction: PAPER.md:591; DDA spec needs it)."""
    srcs = [os.path.join(_HERE, s) for s in _SOURCES]
    if not force and os.path.exists(_LIB_PATH):
        if os.path.getmtime(_LIB_PATH) >= max(os.path.getmtime(s) for s in srcs):
            return _LIB_PATH
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           os.path.join(_HERE, "capi.cpp"), "-o", _LIB_PATH]
    subprocess.run(cmd, check=True)
    return _LIB_PATH


class _Opts(C.Structure):
    _fields_ = [
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
        ("photon_id_offset", C.c_uint64), ("max_scatter", C.c_uint64), ("max_crossings", C.c_uint64),
        ("dust_albedo", C.c_double), ("dust_g", C.c_double), ("doublet_on", C.c_int32),
        ("doublet_dv_kms", C.c_double), ("doublet_sigma_ratio", C.c_double), ("doublet_a_ratio", C.c_double),
    ]


OPT_DEFAULTS = dict(
    phase_core=0, phase_wing=0, phase_frame=0, phase_split_x=0.2, core_skip_mode=0, x_crit=0.0,
    spec_mode=0, spec_T_ref=1e4, spec_bins=0, spec_lo=0.0, spec_hi=1.0,
    hubble_kms_per_cell=0.0, hubble_eps=0.25, v_max_kms=0.0,
    peel_on=0, k_obs=(0.0, 0.0, 1.0), peel_nx=0, peel_ny=0, peel_nv=0, peel_v_lo=0.0, peel_v_hi=1.0,
    peel_width_cells=0.0, tau_peel_max=30.0, photon_id_offset=0, max_scatter=0, max_crossings=0,
    dust_albedo=0.0, dust_g=0.0, doublet_on=0, doublet_dv_kms=0.0, doublet_sigma_ratio=0.0, doublet_a_ratio=1.0,
)

RAW_DTYPE = np.dtype([("V", "<f4"), ("nscat", "<u4"), ("status", "<i4"), ("kx", "<f4"), ("ky", "<f4"), ("kz", "<f4")])
COUNTER_NAMES = ["escaped", "absorbed", "terminated", "capped", "scatterings", "cell_crossings", "rejection_iters",
                 "peel_rays", "peel_cells", "dust_scatterings"]

_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB_PATH)
        d, u64, i64, i32, u32 = C.c_double, C.c_uint64, C.c_int64, C.c_int32, C.c_uint32
        P = C.c_void_p
        for name in ("orc_vth_kms", "orc_voigt_a", "orc_sigma0_cm2", "orc_dawson", "orc_x_cw_exact", "orc_x_cw_b25"):
            getattr(L, name).restype = d
            getattr(L, name).argtypes = [d]
        L.orc_voigt_H.restype = d
        L.orc_voigt_H.argtypes = [d, d]
        L.orc_voigt_H_array.argtypes = [i64, P, P, P]
        L.orc_philox4x32_10.argtypes = [P, P, P]
        L.orc_draws_u32.argtypes = [u64, u64, i64, P]
        L.orc_u32_to_uniform.restype = d
        L.orc_u32_to_uniform.argtypes = [u32]
        L.orc_sample_upar.argtypes = [d, d, u64, u64, i64, i32, P, P]
        L.orc_upar_pdf.restype = d
        L.orc_upar_pdf.argtypes = [d, d, d]
        L.orc_upar_u0.restype = d
        L.orc_upar_u0.argtypes = [d, d]
        L.orc_sample_uperp.argtypes = [d, d, u64, u64, i64, P, P]
        L.orc_sample_mu.argtypes = [i32, u64, u64, i64, P]
        L.orc_dipole_mu.restype = d
        L.orc_dipole_mu.argtypes = [d]
        L.orc_hg_mu.restype = d
        L.orc_hg_mu.argtypes = [d, d]
        L.orc_hg_value.restype = d
        L.orc_hg_value.argtypes = [d, d]
        L.orc_scatter_once.argtypes = [d, d, d, i32, u64, u64, i64, P, P]
        L.orc_dda_trace.argtypes = [i32] * 6 + [i64, P, P, i64, i32, P, P, P, P, P]
        L.orc_raytrace.restype = None
        L.orc_raytrace.argtypes = [i32, i32, i32, d] + [P] * 6 + [i64, P, P, d, i32, d, d, P, P, P]
        L.orc_raytrace_ex.restype = None
        L.orc_raytrace_ex.argtypes = [i32] * 6 + [d] + [P] * 6 + [i64, P, P, d, d, d, i32, d, d, P, P, P]
        L.orc_volume_render.restype = None
        L.orc_volume_render.argtypes = [i32, i32, i32, P, P, i64, P, P, i32, P, d, P]
        L.orc_run_gridless.restype = d
        L.orc_run_gridless.argtypes = [i32] + [d] * 10 + [i64, P, P, P, P, u64, u64] + [P] * 4
        L.orc_run.restype = d
        L.orc_run.argtypes = [i32] * 6 + [d] + [P] * 6 + [i64, P, P, P, P, u64, u64] + [P] * 5
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def vth_kms(T): return lib().orc_vth_kms(float(T))
def voigt_a(T): return lib().orc_voigt_a(float(T))
def sigma0_cm2(T): return lib().orc_sigma0_cm2(float(T))
def dawson(x): return lib().orc_dawson(float(x))
def x_cw_exact(a): return lib().orc_x_cw_exact(float(a))
def x_cw_b25(a): return lib().orc_x_cw_b25(float(a))
def upar_pdf(a, x, u): return lib().orc_upar_pdf(float(a), float(x), float(u))
def upar_u0(a, x): return lib().orc_upar_u0(float(a), float(x))
def dipole_mu(r): return lib().orc_dipole_mu(float(r))
def hg_mu(g, r): return lib().orc_hg_mu(float(g), float(r))
def hg_value(g, mu): return lib().orc_hg_value(float(g), float(mu))
def u32_to_uniform(r): return lib().orc_u32_to_uniform(int(r))


def voigt_H(a, x):
    a = np.ascontiguousarray(np.broadcast_to(np.asarray(a, np.float64), np.broadcast(a, x).shape))
    x = np.ascontiguousarray(np.broadcast_to(np.asarray(x, np.float64), a.shape))
    out = np.empty(a.shape, np.float64)
    lib().orc_voigt_H_array(a.size, _ptr(a), _ptr(x), _ptr(out))
    return out


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, np.uint32).copy()
    k = np.asarray(key, np.uint32).copy()
    out = np.empty(4, np.uint32)
    lib().orc_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
    return out


def draws_u32(seed, photon_id, n):
    out = np.empty(n, np.uint32)
    lib().orc_draws_u32(int(seed), int(photon_id), n, _ptr(out))
    return out


def sample_upar(a, x, n, seed=1, photon_id=0, which=0):
    out = np.empty(n, np.float64)
    it = C.c_uint64(0)
    lib().orc_sample_upar(float(a), float(x), int(seed), int(photon_id), n, which, _ptr(out), C.addressof(it))
    return out, it.value


def sample_uperp(x_in, x_crit, n, seed=1, photon_id=0):
    o1 = np.empty(n, np.float64)
    o2 = np.empty(n, np.float64)
    lib().orc_sample_uperp(float(x_in), float(x_crit), int(seed), int(photon_id), n, _ptr(o1), _ptr(o2))
    return o1, o2


def sample_mu(phase, n, seed=1, photon_id=0):
    out = np.empty(n, np.float64)
    lib().orc_sample_mu(int(phase), int(seed), int(photon_id), n, _ptr(out))
    return out


def scatter_once(a, x_in, n, x_crit=0.0, phase=0, seed=1, photon_id=0):
    xo = np.empty(n, np.float64)
    ko = np.empty((n, 3), np.float64)
    lib().orc_scatter_once(float(a), float(x_in), float(x_crit), int(phase), int(seed), int(photon_id), n,
                           _ptr(xo), _ptr(ko))
    return xo, ko


def dda_trace(dims, periodic, origins, dirs, max_steps=1 << 20, real32=True, want_seq=False):
    """origins, dirs: float32 [n,3].  Returns dict(hash_idx, hash_len, count[, seq_idx, seq_len])."""
    org = np.ascontiguousarray(origins, np.float32)
    dr = np.ascontiguousarray(dirs, np.float32)
    n = org.shape[0]
    hi = np.empty(n, np.uint64)
    hl = np.empty(n, np.uint64)
    cnt = np.empty(n, np.uint32)
    seq_i = seq_l = None
    if want_seq:
        assert n == 1
        seq_i = np.zeros(max_steps, np.int64)
        seq_l = np.zeros(max_steps, np.float64)
    lib().orc_dda_trace(int(dims[0]), int(dims[1]), int(dims[2]), int(periodic[0]), int(periodic[1]),
                        int(periodic[2]), n, _ptr(org), _ptr(dr), int(max_steps), 1 if real32 else 0,
                        _ptr(hi), _ptr(hl), _ptr(cnt), _ptr(seq_i), _ptr(seq_l))
    out = dict(hash_idx=hi, hash_len=hl, count=cnt)
    if want_seq:
        out["seq_idx"] = seq_i[: cnt[0]]
        out["seq_len"] = seq_l[: cnt[0]]
    return out


def run(grid, sources, opts, n_photons, seed, want_raw=True):
    """grid: dict(nx, ny, nz, periodic=(px,py,pz), cell_cm, nHI, T, vx, vy, vz, kdust|None) with float32 arrays of
    shape [nz, ny, nx]; sources: dict(pos [n,3], lum [n], sigma [n]) float32; opts: dict over OPT_DEFAULTS."""
    f = lambda k: None if grid.get(k) is None else np.ascontiguousarray(grid[k], np.float32)
    nHI, T, vx, vy, vz, kd = (f(k) for k in ("nHI", "T", "vx", "vy", "vz", "kdust"))
    pos = np.ascontiguousarray(sources["pos"], np.float32).reshape(-1, 3)
    lum = np.ascontiguousarray(sources["lum"], np.float32)
    sig = np.ascontiguousarray(sources["sigma"], np.float32)
    o = dict(OPT_DEFAULTS)
    unknown = set(opts) - set(o)
    if unknown:
        raise KeyError(f"unknown opts: {unknown}")
    o.update(opts)
    oc = _Opts()
    for k, v in o.items():
        if k == "k_obs":
            oc.k_obs = (C.c_double * 3)(*v)
        else:
            setattr(oc, k, v)
    spectrum = np.zeros(o["spec_bins"] + 2, np.uint64)
    hist = np.zeros(64, np.uint64)
    counters = np.zeros(len(COUNTER_NAMES), np.uint64)
    cube = np.zeros((o["peel_ny"], o["peel_nx"], o["peel_nv"]), np.float64) if o["peel_on"] else None
    raw = np.zeros(n_photons, RAW_DTYPE) if want_raw else None
    per = grid.get("periodic", (0, 0, 0))
    secs = lib().orc_run(int(grid["nx"]), int(grid["ny"]), int(grid["nz"]), int(per[0]), int(per[1]), int(per[2]),
                         float(grid["cell_cm"]), _ptr(nHI), _ptr(T), _ptr(vx), _ptr(vy), _ptr(vz), _ptr(kd),
                         pos.shape[0], _ptr(pos), _ptr(lum), _ptr(sig), C.addressof(oc), int(n_photons), int(seed),
                         _ptr(spectrum), _ptr(hist), _ptr(counters), _ptr(cube), _ptr(raw))
    return dict(spectrum=spectrum, nscat_hist=hist, counters=dict(zip(COUNTER_NAMES, (int(c) for c in counters))),
                cube=cube, raw=raw, seconds=secs)


GRIDLESS_DEFAULTS = dict(geometry=0, r_in=0.0, r_out=1.0, length_cm=1.0, n0=0.0, alpha_rho=0.0, T=1e4, v_max=0.0, alpha_v=1.0,
                         kdust0=0.0, step_f=0.01)


def _opts_struct(opts):
    o = dict(OPT_DEFAULTS)
    unknown = set(opts) - set(o)
    if unknown:
        raise KeyError(f"unknown opts: {unknown}")
    o.update(opts)
    oc = _Opts()
    for k, v in o.items():
        if k == "k_obs":
            oc.k_obs = (C.c_double * 3)(*v)
        else:
            setattr(oc, k, v)
    return o, oc


def run_gridless(dataset, sources, opts, n_photons, seed, want_raw=True):
    """The walk through a gridless dataset (oracle/gridless.hpp).  dataset: dict over GRIDLESS_DEFAULTS (geometry 0 = shell /
    sphere, 1 = slab; lengths in the dataset's unit of length_cm centimetres); sources: pos in that unit, relative to the
    centre / midplane."""
    dd = dict(GRIDLESS_DEFAULTS)
    unknown = set(dataset) - set(dd)
    if unknown:
        raise KeyError(f"unknown gridless fields: {unknown}")
    dd.update(dataset)
    pos = np.ascontiguousarray(sources["pos"], np.float32).reshape(-1, 3)
    lum = np.ascontiguousarray(sources["lum"], np.float32)
    sig = np.ascontiguousarray(sources["sigma"], np.float32)
    o, oc = _opts_struct(opts)
    spectrum = np.zeros(o["spec_bins"] + 2, np.uint64)
    hist = np.zeros(64, np.uint64)
    counters = np.zeros(len(COUNTER_NAMES), np.uint64)
    raw = np.zeros(n_photons, RAW_DTYPE) if want_raw else None
    secs = lib().orc_run_gridless(int(dd["geometry"]), *(float(dd[k]) for k in ("r_in", "r_out", "length_cm", "n0", "alpha_rho", "T",
                                                                                  "v_max", "alpha_v", "kdust0", "step_f")),
                                  pos.shape[0], _ptr(pos), _ptr(lum), _ptr(sig), C.addressof(oc), int(n_photons), int(seed),
                                  _ptr(spectrum), _ptr(hist), _ptr(counters), _ptr(raw))
    return dict(spectrum=spectrum, nscat_hist=hist, counters=dict(zip(COUNTER_NAMES, (int(c) for c in counters))),
                raw=raw, seconds=secs)


def raytrace(grid, origins, dirs, n_v=0, v_lo=0.0, v_hi=1.0, hubble_kms_per_cell=0.0):
    """Projection and absorption spectra along rays (PAPER.md 3.5.1-3.5.2, Eq. 11).  Returns dict(column, tmean[, tau])."""
    f = lambda k: None if grid.get(k) is None else np.ascontiguousarray(grid[k], np.float32)
    nHI, T, vx, vy, vz, kd = (f(k) for k in ("nHI", "T", "vx", "vy", "vz", "kdust"))
    org = np.ascontiguousarray(origins, np.float32).reshape(-1, 3)
    dr = np.ascontiguousarray(dirs, np.float32).reshape(-1, 3)
    n = org.shape[0]
    col = np.zeros(n, np.float64)
    tm = np.zeros(n, np.float64)
    tau = np.zeros((n, n_v), np.float64) if n_v > 0 else None
    lib().orc_raytrace(int(grid["nx"]), int(grid["ny"]), int(grid["nz"]), float(grid["cell_cm"]), _ptr(nHI), _ptr(T),
                       _ptr(vx), _ptr(vy), _ptr(vz), _ptr(kd), n, _ptr(org), _ptr(dr), float(hubble_kms_per_cell),
                       int(n_v), float(v_lo), float(v_hi), _ptr(col), _ptr(tm), _ptr(tau))
    out = dict(column=col, tmean=tm)
    if tau is not None:
        out["tau"] = tau
    return out


def raytrace_ex(grid, origins, dirs, n_v=0, v_lo=0.0, v_hi=1.0, hubble_kms_per_cell=0.0, hubble_eps=0.25, max_length_cells=0.0):
    """Sight lines with periodic wrap-around up to max_length_cells and Hubble sub-sampling of Eq. 11."""
    f = lambda k: None if grid.get(k) is None else np.ascontiguousarray(grid[k], np.float32)
    nHI, T, vx, vy, vz, kd = (f(k) for k in ("nHI", "T", "vx", "vy", "vz", "kdust"))
    org = np.ascontiguousarray(origins, np.float32).reshape(-1, 3)
    dr = np.ascontiguousarray(dirs, np.float32).reshape(-1, 3)
    n = org.shape[0]
    col = np.zeros(n, np.float64)
    tm = np.zeros(n, np.float64)
    tau = np.zeros((n, n_v), np.float64) if n_v > 0 else None
    per = grid.get("periodic", (0, 0, 0))
    lib().orc_raytrace_ex(int(grid["nx"]), int(grid["ny"]), int(grid["nz"]), int(per[0]), int(per[1]), int(per[2]),
                          float(grid["cell_cm"]), _ptr(nHI), _ptr(T), _ptr(vx), _ptr(vy), _ptr(vz), _ptr(kd), n, _ptr(org), _ptr(dr),
                          float(hubble_kms_per_cell), float(hubble_eps), float(max_length_cells), int(n_v), float(v_lo), float(v_hi),
                          _ptr(col), _ptr(tm), _ptr(tau))
    out = dict(column=col, tmean=tm)
    if tau is not None:
        out["tau"] = tau
    return out


def slice_field(grid, points, field):
    """Slice operator: the value of `field` in the cell holding each point — by definition a plain lookup."""
    pts = np.asarray(points, np.float64).reshape(-1, 3)
    idx = [np.clip(np.floor(pts[:, a]).astype(np.int64), 0, grid[("nx", "ny", "nz")[a]] - 1) for a in range(3)]
    return np.asarray(grid[field])[idx[2], idx[1], idx[0]].astype(np.float64)


def volume_render(grid, origins, dirs, peaks, n_ref=0.0):
    """Volume rendering (PAPER.md 3.5.3, Eq. 12) with Gaussian-peak transfer function in log10 T.
    peaks: rows (log10 T centre, width in dex, R, G, B, A).  Returns float64[n][4] = (C_R, C_G, C_B, opacity)."""
    nHI = np.ascontiguousarray(grid["nHI"], np.float32)
    T = np.ascontiguousarray(grid["T"], np.float32)
    org = np.ascontiguousarray(origins, np.float32).reshape(-1, 3)
    dr = np.ascontiguousarray(dirs, np.float32).reshape(-1, 3)
    pk = np.ascontiguousarray(peaks, np.float64).reshape(-1, 6)
    out = np.zeros((org.shape[0], 4), np.float64)
    lib().orc_volume_render(int(grid["nx"]), int(grid["ny"]), int(grid["nz"]), _ptr(nHI), _ptr(T), org.shape[0],
                            _ptr(org), _ptr(dr), pk.shape[0], _ptr(pk), float(n_ref), _ptr(out))
    return out
