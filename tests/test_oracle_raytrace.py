"""Pins for the oracle's ray-tracing operators (PAPER.md 3.5.1 projection, 3.5.2 / Eq. 11 absorption spectra): closed
forms that do not go through the oracle's DDA or its Voigt routine."""
import math

import numpy as np
import pytest
from scipy import integrate, special

from paper_2507_11603_b200 import workloads as W

N = 16
CELL = W.PC_CM


def _uniform_grid(n, T, v=(0.0, 0.0, 0.0), kd=None):
    shape = (N, N, N)
    full = lambda x: np.full(shape, x, np.float32)
    return dict(nx=N, ny=N, nz=N, periodic=(0, 0, 0), cell_cm=CELL, nHI=full(n), T=full(T), vx=full(v[0]), vy=full(v[1]),
                vz=full(v[2]), kdust=None if kd is None else full(kd))


def _chord(org, d):
    """Distance from org to the surface of the cube [0,N]^3 along d (slab method)."""
    t = np.inf
    for o, k in zip(org, d):
        if k > 0:
            t = min(t, (N - o) / k)
        elif k < 0:
            t = min(t, (0 - o) / k)
    return t


def test_column_density_is_density_times_chord(oracle):
    rng = np.random.default_rng(1)
    org = (rng.random((200, 3)) * N).astype(np.float32)
    d = rng.standard_normal((200, 3))
    d = (d / np.linalg.norm(d, axis=1)[:, None]).astype(np.float32)
    org = np.vstack([org, [[8, 8, 8], [0, 0, 0], [3.5, 8, 8]]]).astype(np.float32)
    d = np.vstack([d, [[1, 0, 0], [1 / math.sqrt(3)] * 3, [0, 0, -1]]]).astype(np.float32)
    n = float(np.float32(0.37))
    r = oracle.raytrace(_uniform_grid(n, 2e4), org, d)
    expect = np.array([n * _chord(o.astype(float), k.astype(float)) * CELL for o, k in zip(org, d)])
    assert np.allclose(r["column"], expect, rtol=1e-6)
    assert np.allclose(r["tmean"], 2e4, rtol=1e-12)
    assert r["column"][-3] == pytest.approx(n * 8 * CELL, rel=1e-12)      # centre to the +x face: 8 cells


def test_projection_weights_by_density(oracle):
    """Q / Q^ with q = T, w = n_HI: two slabs of different density and temperature along z."""
    g = _uniform_grid(1.0, 1e4)
    g["nHI"][8:, :, :] = 3.0
    g["T"][8:, :, :] = 5e4
    r = oracle.raytrace(g, np.array([[8.2, 7.7, 0.0]], np.float32), np.array([[0, 0, 1]], np.float32))
    assert r["column"][0] == pytest.approx((1.0 * 8 + 3.0 * 8) * CELL, rel=1e-12)
    assert r["tmean"][0] == pytest.approx((1.0 * 8 * 1e4 + 3.0 * 8 * 5e4) / (8 + 24), rel=1e-12)


def test_absorption_spectrum_static_uniform_gas(oracle):
    """Eq. 11 without motion: tau(V) = N_HI sigma_0 H(a, V / v_th), H from scipy's Faddeeva function; with a uniform
    bulk velocity the profile shifts by v.k; dust adds kappa L."""
    T, n = 1e4, 1e-6
    v = (30.0, -10.0, 20.0)
    kd = 0.2 / (N * CELL)
    org = np.array([[0.0, 5.3, 9.1]], np.float32)
    d = np.array([[1.0, 0.0, 0.0]], np.float32)
    nv, vlo, vhi = 64, -200.0, 200.0
    r = oracle.raytrace(_uniform_grid(n, T, v, kd), org, d, n_v=nv, v_lo=vlo, v_hi=vhi)
    V = vlo + (np.arange(nv) + 0.5) * (vhi - vlo) / nv
    a, vth, s0 = oracle.voigt_a(T), oracle.vth_kms(T), oracle.sigma0_cm2(T)
    H = special.wofz((V - v[0]) / vth + 1j * a).real
    expect = n * N * CELL * s0 * H + 0.2
    assert np.allclose(r["tau"][0], expect, rtol=1e-8)


def test_absorption_spectrum_hubble_flow(oracle):
    """Eq. 11 with the Hubble term: uniform static gas, tau(V) = n sigma_0 Int_0^L H(a, (V - Hc s)/v_th) ds.  The oracle
    uses the midpoint of each cell segment; with Hc = 1 km/s per cell << v_th = 12.8 km/s the midpoint rule agrees with
    adaptive quadrature to a few 1e-3."""
    T, n, Hc = 1e4, 1e-6, 1.0
    org = np.array([[0.0, 8.5, 8.5]], np.float32)
    d = np.array([[1.0, 0.0, 0.0]], np.float32)
    nv, vlo, vhi = 16, -20.0, 40.0
    r = oracle.raytrace(_uniform_grid(n, T), org, d, n_v=nv, v_lo=vlo, v_hi=vhi, hubble_kms_per_cell=Hc)
    a, vth, s0 = oracle.voigt_a(T), oracle.vth_kms(T), oracle.sigma0_cm2(T)
    V = vlo + (np.arange(nv) + 0.5) * (vhi - vlo) / nv
    expect = [n * s0 * CELL * integrate.quad(lambda s: special.wofz((v - Hc * s) / vth + 1j * a).real, 0, N, epsabs=0, epsrel=1e-10)[0]
              for v in V]
    assert np.allclose(r["tau"][0], expect, rtol=5e-3)
    # absorption is strongest where the line sweeps through the sight line: V between 0 and Hc * N
    assert 0.0 <= V[int(np.argmax(r["tau"][0]))] <= Hc * N


# ---- volume rendering (PAPER.md 3.5.3, Eq. 12) ----
PEAKS = np.array([[4.3, 0.15, 0.1, 0.3, 1.0, 0.8],      # cold: blue      (log10 T centre, width [dex], R, G, B, A)
                  [5.0, 0.20, 1.0, 0.6, 0.1, 0.5],      # warm: orange
                  [5.5, 0.10, 1.0, 0.1, 0.1, 1.2]])     # hot: red


def _tf(T, n, n_ref):
    """Transfer function written out independently: returns (mu, c_rgb)."""
    lt = math.log10(T)
    gp = PEAKS[:, 5] * np.exp(-0.5 * ((lt - PEAKS[:, 0]) / PEAKS[:, 1]) ** 2) * (n / n_ref if n_ref > 0 else 1.0)
    mu = gp.sum()
    return mu, (gp[:, None] * PEAKS[:, 2:5]).sum(0) / mu


def test_volume_render_uniform_medium_closed_form(oracle):
    """Constant c and mu: Eq. 12 integrates to C = c (1 - e^{-mu L}) with L the analytic chord."""
    rng = np.random.default_rng(3)
    org = (rng.random((100, 3)) * N).astype(np.float32)
    d = rng.standard_normal((100, 3))
    d = (d / np.linalg.norm(d, axis=1)[:, None]).astype(np.float32)
    T, n, n_ref = 10 ** 4.4, 0.02, 0.1
    g = _uniform_grid(n, T)
    out = oracle.volume_render(g, org, d, PEAKS, n_ref=n_ref)
    mu, c = _tf(float(np.float32(T)), float(np.float32(n)), n_ref)
    for o, k, rgba in zip(org, d, out):
        L = _chord(o.astype(float), k.astype(float))
        assert rgba[:3] == pytest.approx(c * (1 - math.exp(-mu * L)), rel=1e-6)
        assert rgba[3] == pytest.approx(1 - math.exp(-mu * L), rel=1e-6)
    # no density weighting: mu does not depend on n
    out1 = oracle.volume_render(g, org[:1], d[:1], PEAKS, n_ref=0.0)
    mu1, _ = _tf(float(np.float32(T)), 1.0, 0.0)
    assert out1[0, 3] == pytest.approx(1 - math.exp(-mu1 * _chord(org[0].astype(float), d[0].astype(float))), rel=1e-6)


def test_volume_render_front_slab_attenuates_back_slab(oracle):
    """Observer at s = 0: the near slab is seen unattenuated, the far slab through e^{-mu1 L1}; reversing the ray
    swaps the roles (catches a back-to-front / front-to-back mix-up)."""
    g = _uniform_grid(1.0, 10 ** 4.3)
    g["T"][8:, :, :] = 10 ** 5.5                       # z >= 8 hot (red), z < 8 cold (blue)
    mu1, c1 = _tf(float(g["T"][0, 0, 0]), 1.0, 0.0)
    mu2, c2 = _tf(float(g["T"][8, 0, 0]), 1.0, 0.0)
    fwd = oracle.volume_render(g, [[5.5, 6.5, 0.0]], [[0, 0, 1]], PEAKS)[0]
    bwd = oracle.volume_render(g, [[5.5, 6.5, 16.0]], [[0, 0, -1]], PEAKS)[0]
    a1, a2 = math.exp(-mu1 * 8), math.exp(-mu2 * 8)
    assert fwd[:3] == pytest.approx(c1 * (1 - a1) + a1 * c2 * (1 - a2), rel=1e-12)
    assert bwd[:3] == pytest.approx(c2 * (1 - a2) + a2 * c1 * (1 - a1), rel=1e-12)
    assert fwd[3] == pytest.approx(1 - a1 * a2, rel=1e-12) and bwd[3] == pytest.approx(fwd[3], rel=1e-12)
    assert not np.allclose(fwd[:3], bwd[:3], rtol=1e-3)


def test_volume_render_matches_quadrature_of_eq12(oracle):
    """Eq. 12 by nested adaptive quadrature on a random 6^3 grid, the fields looked up by floor(position) (no DDA)."""
    rng = np.random.default_rng(11)
    n6 = 6
    g = dict(nx=n6, ny=n6, nz=n6, periodic=(0, 0, 0), cell_cm=CELL,
             nHI=np.exp(rng.normal(0, 1, (n6, n6, n6))).astype(np.float32),
             T=(10 ** rng.uniform(4.0, 5.8, (n6, n6, n6))).astype(np.float32))
    n_ref = 2.0
    scale = 0.5                                        # keep the total optical depth O(1)
    pk = PEAKS.copy()
    pk[:, 5] *= scale
    for o, k in [((0.3, 2.2, 4.1), (0.61, 0.35, -0.71)), ((5.9, 5.2, 0.4), (-0.7, -0.5, 0.51))]:
        o = np.array(o, np.float32).astype(float)
        k = np.array(k) / np.linalg.norm(k)
        k = k.astype(np.float32).astype(float)
        t_end = min(((n6 - o[i]) / k[i] if k[i] > 0 else (0 - o[i]) / k[i]) for i in range(3))

        def mu_c(s):
            c = np.clip(np.floor(o + s * k).astype(int), 0, n6 - 1)
            T, n = float(g["T"][c[2], c[1], c[0]]), float(g["nHI"][c[2], c[1], c[0]])
            lt = math.log10(T)
            gp = pk[:, 5] * np.exp(-0.5 * ((lt - pk[:, 0]) / pk[:, 1]) ** 2) * n / n_ref
            return gp.sum(), (gp[:, None] * pk[:, 2:5]).sum(0)

        # breakpoints (face crossings) so that the adaptive rule sees the discontinuities
        br = sorted({(f - o[i]) / k[i] for i in range(3) for f in range(n6 + 1) if 0 < (f - o[i]) / k[i] < t_end})
        edges = [0.0] + br + [t_end]
        tau_at = [0.0]
        for a, b in zip(edges[:-1], edges[1:]):
            tau_at.append(tau_at[-1] + integrate.quad(lambda s: mu_c(s)[0], a, b)[0])
        C = np.zeros(3)
        for j, (a, b) in enumerate(zip(edges[:-1], edges[1:])):
            for ch in range(3):
                f = lambda s: mu_c(s)[1][ch] * math.exp(-(tau_at[j] + mu_c(0.5 * (a + b))[0] * (s - a)))
                C[ch] += integrate.quad(f, a, b)[0]
        out = oracle.volume_render(g, [o], [k], pk, n_ref=n_ref)[0]
        assert out[:3] == pytest.approx(C, rel=1e-7)
        assert out[3] == pytest.approx(1 - math.exp(-tau_at[-1]), rel=1e-7)
        assert 0.05 < out[3] < 0.999


# ---------------------------------------------------------------- round 2: periodic sight lines, Hubble sub-sampling
def test_forest_sightline_subsampled_against_quadrature(oracle):
    """cells are sub-sampled so that a ray step shifts the line by much less than its width.  Uniform static gas
    swept by H_c = 2.28 km/s per cell (BASELINE.json config 5's drift): tau(V) = n sigma_0 Delta Int_0^L H(a, (V - H_c s) / v_th) ds
    by scipy quad, to 1e-3 — at T = 1e3 K (0.56 v_th per cell; there even one midpoint per cell is accurate, the midpoint rule
    converging exponentially on a Gaussian) and at T = 60 K (2.3 v_th per cell), where one midpoint per cell fails by far."""
    from scipy import integrate, special
    for T, coarse_fails in ((1e3, False), (60.0, True)):
        _forest_case(oracle, T, coarse_fails)


def _forest_case(oracle, T, coarse_fails):
    from scipy import integrate, special
    Hc, L = 2.28, 40
    shape = (2, 2, L)
    tau_cell = 0.8
    n = tau_cell / (oracle.sigma0_cm2(T) * W.PC_CM)
    z = np.zeros(shape[::-1], np.float32)
    grid = dict(nx=2, ny=2, nz=L, periodic=(0, 0, 0), cell_cm=W.PC_CM, nHI=np.full(shape[::-1], n, np.float32),
                T=np.full(shape[::-1], T, np.float32), vx=z, vy=z, vz=z, kdust=None)
    org, dr = np.array([[1.0, 1.0, 0.0]], np.float32), np.array([[0.0, 0.0, 1.0]], np.float32)
    vth, a = oracle.vth_kms(T), oracle.voigt_a(T)
    n_v, v_lo, v_hi = 24, 20.0, 70.0
    fine = oracle.raytrace_ex(grid, org, dr, n_v, v_lo, v_hi, Hc, hubble_eps=0.25)["tau"][0]
    coarse = oracle.raytrace(grid, org, dr, n_v, v_lo, v_hi, Hc)["tau"][0]
    tau_real = float(np.float32(n)) * oracle.sigma0_cm2(T) * W.PC_CM
    worst_c = 0.0
    for j in range(n_v):
        V = v_lo + (j + 0.5) * (v_hi - v_lo) / n_v
        exact = tau_real * integrate.quad(lambda s: special.wofz((V - Hc * s) / vth + 1j * a).real, 0, L, points=[V / Hc],
                                          epsabs=1e-12, epsrel=1e-10, limit=400)[0]
        assert abs(fine[j] - exact) < 1e-3 * exact, (j, fine[j], exact)
        worst_c = max(worst_c, abs(coarse[j] - exact) / exact)
    assert (worst_c > 3e-2) == coarse_fails, worst_c


def test_periodic_sightline_wraps(oracle):
    """PAPER.md:520 "periodic boundary conditions": a ray of stated length wraps at periodic faces.  Pins: an axis-aligned ray
    of 2.5 box lengths collects 2.5 times the row's column; an oblique ray through the periodic box equals the same ray
    through the box tiled 3 x 3 x 3 without wrapping; a non-periodic axis still ends the ray."""
    rng = np.random.default_rng(3)
    N = 6
    f = lambda: rng.random((N, N, N)).astype(np.float32) + 0.1
    grid = dict(nx=N, ny=N, nz=N, periodic=(1, 1, 1), cell_cm=1.0, nHI=f(), T=f() * 1e4, vx=f() * 20, vy=f() * 20, vz=f() * 20, kdust=None)
    r = oracle.raytrace_ex(grid, np.array([[0.0, 2.5, 3.5]], np.float32), np.array([[1.0, 0.0, 0.0]], np.float32), max_length_cells=15.0)
    row = grid["nHI"][3, 2, :].astype(np.float64)
    assert abs(r["column"][0] - (2 * row.sum() + row[:3].sum())) < 1e-9
    org = np.array([[1.25, 4.5, 0.75]], np.float32)              # exact in fp32 also after adding N
    dr = np.array([[0.48, -0.6, 0.64]], np.float32)
    tiled = {k: (np.tile(grid[k], (3, 3, 3)) if isinstance(grid[k], np.ndarray) else grid[k]) for k in grid}
    tiled.update(nx=3 * N, ny=3 * N, nz=3 * N, periodic=(0, 0, 0))
    a = oracle.raytrace_ex(grid, org, dr, 8, -60.0, 60.0, 1.5, 0.25, max_length_cells=9.0)
    b = oracle.raytrace_ex(tiled, org + N, dr, 8, -60.0, 60.0, 1.5, 0.25, max_length_cells=9.0)
    assert abs(a["column"][0] - b["column"][0]) < 1e-9 * b["column"][0]
    assert np.allclose(a["tau"], b["tau"], rtol=1e-9)
    c = oracle.raytrace_ex(dict(grid, periodic=(0, 0, 0)), org, dr, max_length_cells=9.0)
    assert c["column"][0] < a["column"][0]                         # not periodic: ends at the first face


def test_slice_is_a_lookup(oracle):
    """PAPER.md:189 slices: the field value of the cell holding each point of the plane."""
    rng = np.random.default_rng(4)
    g = dict(nx=5, ny=4, nz=3, T=rng.random((3, 4, 5)).astype(np.float32))
    pts = np.array([[0.2, 0.9, 2.99], [4.99, 3.0, 0.0], [2.5, 1.5, 1.5]])
    assert np.array_equal(oracle.slice_field(g, pts, "T"), [g["T"][2, 0, 0], g["T"][0, 3, 4], g["T"][1, 1, 2]])
