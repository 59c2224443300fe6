"""GPU parity of the ray-tracing operators (thor_raytrace: projection, PAPER.md 3.5.1, and absorption spectra, Eq. 11)
against the fp64 oracle on the same rays through the synthetic turbulent box and cosmic web, SoA and packed."""
import numpy as np
import pytest

from paper_2507_11603_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def thor():
    import torch
    assert torch.cuda.is_available()
    from paper_2507_11603_b200 import thor as t
    t.lib()
    return t


@pytest.mark.parametrize("pack", [False, True])
def test_projection_and_absorption_parity(thor, oracle, pack):
    w = W.cosmic_web(n=48, n_src=16, n_photons=1, mean_n=1e-9, map_pix=8)
    n = 48
    org, dirs = W.random_rays(4000, (n, n, n), seed=5)
    # add a pencil-beam image along +z through every (x, y) of a coarse raster, starting on the z = 0 face
    xs = (np.arange(12) + 0.5) * 4.0
    gx, gy = np.meshgrid(xs, xs)
    org = np.vstack([org, np.stack([gx.ravel(), gy.ravel(), np.zeros(gx.size)], 1)]).astype(np.float32)
    dirs = np.vstack([dirs, np.tile([0.0, 0.0, 1.0], (gx.size, 1))]).astype(np.float32)
    hc = w["opts"]["hubble_kms_per_cell"]
    ctx = thor.Context.from_workload(w["grid"], pack=pack)
    try:
        g = ctx.raytrace(org, dirs, n_v=48, v_lo=-150.0, v_hi=250.0, hubble_kms_per_cell=hc)
    finally:
        ctx.close()
    o = oracle.raytrace(w["grid"], org, dirs, n_v=48, v_lo=-150.0, v_hi=250.0, hubble_kms_per_cell=hc)
    # the GPU marches the fp32 DDA, the oracle its fp64 twin: a ray grazing a cell corner may visit one different
    # cell, so compare with a tolerance and allow a handful of outliers
    rel = np.abs(g["column"] - o["column"]) / np.maximum(o["column"], 1e-300)
    assert np.quantile(rel, 0.999) < 2e-5 and rel.max() < 1e-2
    relT = np.abs(g["tmean"] - o["tmean"]) / o["tmean"]
    assert np.quantile(relT, 0.999) < 2e-5
    scale = o["tau"].max(axis=1, keepdims=True) + 1e-30
    err = np.abs(g["tau"] - o["tau"]) / scale
    assert np.quantile(err, 0.999) < 5e-5 and err.max() < 1e-2
    assert o["tau"].max() > 0.1                      # the sight lines do absorb
    # pencil beams along +z: exact cell lists on both sides -> tight agreement
    k = gx.size
    assert np.allclose(g["column"][-k:], o["column"][-k:], rtol=5e-6)
    assert np.allclose(g["tau"][-k:], o["tau"][-k:], rtol=2e-4, atol=1e-7)


TF_PEAKS = np.array([[4.3, 0.15, 0.1, 0.3, 1.0, 0.8],     # (log10 T centre, width [dex], R, G, B, A): PAPER.md:510
                     [5.0, 0.20, 1.0, 0.6, 0.1, 0.5],
                     [5.5, 0.10, 1.0, 0.1, 0.1, 1.2]])


@pytest.mark.parametrize("pack", [False, True])
@pytest.mark.parametrize("n_ref", [0.0, 3e-9])
def test_volume_render_parity(thor, oracle, pack, n_ref):
    """Eq. 12 (PAPER.md 3.5.3) through the 48^3 cosmic web: random rays plus an image raster along +z."""
    w = W.cosmic_web(n=48, n_src=16, n_photons=1, mean_n=1e-9, map_pix=8)
    n = 48
    org, dirs = W.random_rays(4000, (n, n, n), seed=6)
    xs = (np.arange(12) + 0.5) * 4.0
    gx, gy = np.meshgrid(xs, xs)
    org = np.vstack([org, np.stack([gx.ravel(), gy.ravel(), np.zeros(gx.size)], 1)]).astype(np.float32)
    dirs = np.vstack([dirs, np.tile([0.0, 0.0, 1.0], (gx.size, 1))]).astype(np.float32)
    pk = TF_PEAKS.copy()
    pk[:, 0] -= 1.2                                   # the web's temperatures sit around 10^3-10^4.5 K
    pk[:, 5] *= 0.3 if n_ref == 0.0 else 0.15
    ctx = thor.Context.from_workload(w["grid"], pack=pack)
    try:
        g = ctx.volume_render(org, dirs, pk, n_ref=n_ref)
    finally:
        ctx.close()
    o = oracle.volume_render(w["grid"], org, dirs, pk.astype(np.float32), n_ref=n_ref)
    assert 0.05 < np.median(o[:, 3]) and o[:, 3].min() < 0.9       # neither transparent nor saturated everywhere
    # fp32 DDA against its fp64 twin: a ray grazing a corner may see one different cell (as in the projection test)
    err = np.abs(g - o) / np.maximum(np.abs(o).max(axis=1, keepdims=True), 1e-3)
    assert np.quantile(err, 0.999) < 1e-4 and err.max() < 1e-2
    k = gx.size
    assert np.allclose(g[-k:], o[-k:], rtol=1e-4, atol=1e-6)        # pencil beams: identical cell lists


def test_volume_render_argument_errors(thor):
    w = W.cosmic_web(n=16, n_src=4, n_photons=1, mean_n=1e-9, map_pix=8)
    org, dirs = W.random_rays(8, (16, 16, 16), seed=1)
    ctx = thor.Context.from_workload(w["grid"])
    try:
        bad = TF_PEAKS.copy()
        bad[1, 1] = 0.0                                # zero width
        with pytest.raises(thor.ThorError):
            ctx.volume_render(org, dirs, bad)
        with pytest.raises(thor.ThorError):
            ctx.volume_render(org, dirs, np.tile(TF_PEAKS, (3, 1)))     # 9 peaks > THOR_MAX_TF_PEAKS
        with pytest.raises(thor.ThorError):
            ctx.volume_render(org, dirs, TF_PEAKS, n_ref=-1.0)
        assert ctx.volume_render(org, dirs, TF_PEAKS).shape == (8, 4)   # context still usable
    finally:
        ctx.close()


def test_marcher_degenerate_rays(thor, oracle):
    """The constant-direction marcher on the cases its folded constants special-case: axis-aligned rays of either
    sign (two dead axes, +0 and -0 components), rays in a coordinate plane, origins on faces, edges and corners with
    inward and outward directions (zero-length first segments, reading A20)."""
    w = W.cosmic_web(n=24, n_src=4, n_photons=1, mean_n=1e-9, map_pix=8)
    n = 24.0
    s2, s3 = 1 / np.sqrt(2), 1 / np.sqrt(3)
    org, dirs = [], []
    for o in ([3.5, 7.25, 11.0], [0.0, 0.0, 0.0], [n, n, n], [12.0, 0.0, 5.0], [n, 6.0, 6.0], [8.0, 8.0, 8.0]):
        for k in ([1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1], [-1, -0.0, 0.0], [0.0, -0.0, 1],
                  [s2, s2, 0], [-s2, 0, s2], [0, -s2, -s2], [s3, s3, s3], [-s3, -s3, -s3], [s3, -s3, s3]):
            org.append(o)
            dirs.append(k)
    org, dirs = np.array(org, np.float32), np.array(dirs, np.float32)
    pk = TF_PEAKS.copy()
    pk[:, 0] -= 1.2
    pk[:, 5] *= 0.3
    for pack in (False, True):
        ctx = thor.Context.from_workload(w["grid"], pack=pack)
        try:
            g = ctx.raytrace(org, dirs, n_v=8, v_lo=-100.0, v_hi=100.0)
            gv = ctx.volume_render(org, dirs, pk)
        finally:
            ctx.close()
        o = oracle.raytrace(w["grid"], org, dirs, n_v=8, v_lo=-100.0, v_hi=100.0)
        ov = oracle.volume_render(w["grid"], org, dirs, pk.astype(np.float32))
        # these rays run along cell edges or through exact lattice points only where both sides take the same ties
        assert np.allclose(g["column"], o["column"], rtol=2e-5, atol=0)
        assert np.allclose(g["tmean"], o["tmean"], rtol=2e-5)
        assert np.allclose(g["tau"], o["tau"], rtol=5e-4, atol=1e-7 * o["tau"].max())
        assert np.allclose(gv, ov, rtol=2e-4, atol=1e-6)
        assert (o["column"] == 0).any() and (o["column"] > 0).any()      # outward rays from a corner see nothing


# ---------------------------------------------------------------- round 2: forest sight lines, slices, thin renders
@pytest.mark.parametrize("pack", [False, True])
def test_periodic_subsampled_sightlines_parity(thor, oracle, pack):
    """sight lines through the periodic box, wrapping at the faces up to a stated length, Eq. 11 sub-sampled so
    that a step shifts the line by <= 0.25 v_th — against the oracle's orc_raytrace_ex on the same rays."""
    n = 32
    w = W.cosmic_web(n=n, n_src=16, n_photons=1, mean_n=3e-9, map_pix=8)
    grid = dict(w["grid"], periodic=(1, 1, 1), T=(w["grid"]["T"] * 0.02).astype(np.float32))     # ~200 K: H_c ~ 1.3 v_th per cell
    org, dirs = W.random_rays(1500, (n, n, n), seed=8)
    hc = w["opts"]["hubble_kms_per_cell"]
    ctx = thor.Context.from_workload(grid, pack=pack)
    try:
        g = ctx.raytrace(org, dirs, n_v=40, v_lo=-100.0, v_hi=400.0, hubble_kms_per_cell=hc, hubble_eps=0.25, max_length_cells=2.5 * n)
        g1 = ctx.raytrace(org, dirs, n_v=40, v_lo=-100.0, v_hi=400.0, hubble_kms_per_cell=hc, hubble_eps=0.0, max_length_cells=2.5 * n)
    finally:
        ctx.close()
    o = oracle.raytrace_ex(grid, org, dirs, 40, -100.0, 400.0, hc, 0.25, 2.5 * n)
    rel = np.abs(g["column"] - o["column"]) / o["column"]
    assert np.quantile(rel, 0.999) < 3e-5 and rel.max() < 1e-2
    scale = o["tau"].max(axis=1, keepdims=True) + 1e-30
    err = np.abs(g["tau"] - o["tau"]) / scale
    assert np.quantile(err, 0.999) < 1e-4 and err.max() < 1e-2
    # every ray went the full 2.5 box lengths: columns well above any single crossing of the box
    single = oracle.raytrace(dict(grid, periodic=(0, 0, 0)), org, dirs)["column"]
    assert np.all(o["column"] > single * (1 - 1e-9)) and np.median(o["column"] / single) > 2.0
    # and the sub-sampling matters at this temperature: one midpoint per segment is off by far more than the parity bar
    assert (np.abs(g1["tau"] - o["tau"]) / scale).max() > 1e-2


def test_slice_and_host_buffers(thor, oracle):
    """Slice operator = plain lookup, exact; and the HOST-buffer flag of the ray operators gives the very
    bits the DEVICE-pointer entry points give."""
    import ctypes as C
    import torch
    w = W.turbulent_box(n=24, n_src=16, n_photons=1, peel_pix=4, peel_bins=4)
    grid = dict(w["grid"], kdust=(w["grid"]["nHI"] * 1e-20).astype(np.float32))
    rng = np.random.default_rng(2)
    pts = (rng.random((5000, 3)) * 24).astype(np.float32)
    org, dirs = W.random_rays(800, (24, 24, 24), seed=4)
    for pack in (False, True):
        ctx = thor.Context.from_workload(grid, pack=pack)
        try:
            for f in ("nHI", "T", "vx", "vy", "vz", "kdust"):
                assert np.array_equal(ctx.slice(pts, f).astype(np.float64), oracle.slice_field(grid, pts, f)), (f, pack)
            host = ctx.raytrace(org, dirs, n_v=8, v_lo=-50.0, v_hi=50.0)
            d = lambda a: torch.from_numpy(a).cuda()
            o_, d_ = d(org), d(dirs)
            col, tau = torch.empty(800, device="cuda"), torch.empty((800, 8), device="cuda")
            p = lambda t: C.c_void_p(t.data_ptr())
            assert thor.lib().thor_raytrace(ctx._ctx, 800, p(o_), p(d_), 0.0, 8, -50.0, 50.0, p(col), None, p(tau)) == 0
            assert np.array_equal(col.cpu().numpy(), host["column"]) and np.array_equal(tau.cpu().numpy(), host["tau"])
        finally:
            ctx.close()


def test_volume_render_thin_regime(thor, oracle):
    """Optically thin renders (total tau 1e-4 ... 1e-2, per-segment mu l down to 1e-6): 1 - e^{-y} must not be formed by
    subtracting an approximate exponential from one: colour and opacity agree with the fp64 oracle to 1e-4."""
    n = 48
    w = W.cosmic_web(n=n, n_src=16, n_photons=1, mean_n=1e-9, map_pix=8)
    org, dirs = W.random_rays(3000, (n, n, n), seed=6)
    peaks = TF_PEAKS.copy()
    peaks[:, 5] *= 2e-4                                   # amplitudes: tau per cell ~1e-6 ... 1e-4
    ctx = thor.Context.from_workload(w["grid"])
    try:
        g = ctx.volume_render(org, dirs, peaks).astype(np.float64)
    finally:
        ctx.close()
    o = oracle.volume_render(w["grid"], org, dirs, peaks)
    assert 1e-5 < np.median(o[:, 3]) < 1e-2
    sel = o[:, 3] > 1e-6
    rel = np.abs(g[sel] - o[sel]) / np.maximum(np.abs(o[sel]), 1e-12)
    assert np.quantile(rel[:, 3], 0.999) < 1e-4, np.quantile(rel[:, 3], 0.999)
    assert np.quantile(rel[:, :3], 0.999) < 1e-4
