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
