"""Pins for the oracle's gridless walker (oracle/gridless.hpp; PAPER.md 3.3, 197-198, 342-348, 380-382), CPU only.  With
analytic boundaries there is no voxelisation error, so the closed forms bind more tightly than on grids."""
import math

import numpy as np
import pytest
from scipy import integrate, special, stats

from paper_2507_11603_b200 import workloads as W

PC = W.PC_CM


def _central(sigma=0.0):
    return dict(pos=np.zeros((1, 3), np.float32), lum=np.ones(1, np.float32), sigma=np.full(1, sigma, np.float32))


def _sphere(oracle, tau0, T, **kw):
    return dict(dict(geometry=0, r_in=0.0, r_out=1.0, length_cm=PC, n0=tau0 / (oracle.sigma0_cm2(T) * PC), T=T), **kw)


def _slab(oracle, tau0, T, **kw):
    return dict(dict(geometry=1, r_out=1.0, length_cm=PC, n0=tau0 / (oracle.sigma0_cm2(T) * PC), T=T), **kw)


def test_unscattered_fractions_are_exact(oracle):
    """P7 without voxelisation: central line-centre source, P(N_scat = 0) = exp(-tau0 H(a,0)) in a sphere and
    E_2(tau0 H(a,0)) in a slab (scipy's expn and Faddeeva function)."""
    n, T = 40_000, 1e4
    H0 = special.wofz(1j * oracle.voigt_a(T)).real
    opts = dict(spec_bins=10, spec_lo=-20.0, spec_hi=20.0, spec_T_ref=T)
    for tau0 in (0.4, 2.0):
        r = oracle.run_gridless(_sphere(oracle, tau0, T), _central(), opts, n, seed=3)
        p = math.exp(-tau0 * H0)
        assert abs(r["nscat_hist"][0] / n - p) < 4.5 * math.sqrt(p * (1 - p) / n), ("sphere", tau0)
        assert r["counters"]["escaped"] == n
        r = oracle.run_gridless(_slab(oracle, tau0, T), _central(), opts, n, seed=4)
        p = special.expn(2, tau0 * H0)
        assert abs(r["nscat_hist"][0] / n - p) < 4.5 * math.sqrt(p * (1 - p) / n), ("slab", tau0)


def test_dust_only_sphere_escape_fraction(oracle):
    """P6's exact special case: no gas, absorbing dust of radial depth tau_d: f_esc = exp(-tau_d) — exact on the analytic
    sphere (the voxelised twin of this test needs a direction average over chords).  Also a shell with a dust-free cavity."""
    n = 100_000
    opts = dict(spec_bins=4, spec_lo=-1.0, spec_hi=1.0)
    for r_in, tau_d in ((0.0, 0.7), (0.6, 1.3)):
        d = dict(geometry=0, r_in=r_in, r_out=1.0, length_cm=PC, n0=0.0, T=1e4, kdust0=tau_d / ((1.0 - r_in) * PC))
        r = oracle.run_gridless(d, _central(), opts, n, seed=5)
        p = math.exp(-tau_d)
        assert r["counters"]["scatterings"] == 0 and r["counters"]["escaped"] + r["counters"]["absorbed"] == n
        assert abs(r["counters"]["escaped"] / n - p) < 4.5 * math.sqrt(p * (1 - p) / n), (r_in, tau_d)


def test_dijkstra_sphere_and_neufeld_slab_without_voxelisation(oracle):
    """P4 on the analytic geometries (the paper's own validation) at a tau0 >= 1e4, where the asymptotic
    solutions are good: escaped |x| against tanh(k|x|^3/2) (sphere) and (4/pi) atan(tanh(k|x|^3/2)) (slab), KS distance
    <= 0.02 — on the 32^3 / 256-cell grids the same pins are held at 0.05-0.08."""
    n = 12_000
    T = 10.0
    a = oracle.voigt_a(T)
    tau0 = 1e6                                                     # a tau0 = 1.49e4
    xc = 0.2 * (a * tau0) ** (1 / 3)
    opts = dict(spec_bins=10, spec_lo=-200.0, spec_hi=200.0, spec_T_ref=T, core_skip_mode=1, x_crit=xc)
    r = oracle.run_gridless(_sphere(oracle, tau0, T), _central(), opts, n, seed=1)
    ax = np.abs(r["raw"]["V"].astype(float)) / oracle.vth_kms(T)
    k = math.sqrt(2 * math.pi ** 3 / 27) / (a * tau0)
    ks = stats.kstest(ax, lambda x: np.tanh(k * x ** 3 / 2))
    assert ks.statistic < 0.02, ks
    assert abs(r["raw"]["kz"].mean()) < 4 / math.sqrt(3 * n)
    r = oracle.run_gridless(_slab(oracle, tau0, T), _central(), dict(opts, phase_core=1), n, seed=2)
    ax = np.abs(r["raw"]["V"].astype(float)) / oracle.vth_kms(T)
    k = math.sqrt(math.pi ** 3 / 54) / (a * tau0)
    ks = stats.kstest(ax, lambda x: 4 / math.pi * np.arctan(np.tanh(k * x ** 3 / 2)))
    assert ks.statistic < 0.02, ks
    assert np.all(np.abs(r["raw"]["kz"]) > 0)


def test_expanding_sphere_sweeps_the_line(oracle):
    """PAPER.md:197 (v = v_max r / r_o) with the step limiter of PAPER.md:382: a central line-centre source in a linearly
    expanding homogeneous sphere sees the gas recede, so along any radius the line is swept from x = 0 to -v_max / v_th:
    P(N_scat = 0) = exp(-tau0 Int_0^1 H(a, v_max s / v_th) ds), by quadrature of scipy's Faddeeva function."""
    n, T, v_max, tau0 = 40_000, 1e4, 60.0, 3.0
    vth, a = oracle.vth_kms(T), oracle.voigt_a(T)
    tau = tau0 * integrate.quad(lambda s: special.wofz(v_max * s / vth + 1j * a).real, 0, 1, epsabs=1e-12)[0]
    p = math.exp(-tau)
    assert 0.3 < p < 0.7
    opts = dict(spec_mode=1, spec_bins=10, spec_lo=-300.0, spec_hi=300.0)
    r = oracle.run_gridless(_sphere(oracle, tau0, T, v_max=v_max, alpha_v=1.0, step_f=0.01), _central(), opts, n, seed=6)
    assert abs(r["nscat_hist"][0] / n - p) < 4.5 * math.sqrt(p * (1 - p) / n), (r["nscat_hist"][0] / n, p)
    assert r["counters"]["cell_crossings"] > 50 * n                # the limiter really cuts the path into steps
    # the outflow reddens what escapes after scattering (dv = -V > 0)
    sc = r["raw"][r["raw"]["nscat"] > 0]
    assert (-sc["V"]).mean() > 4 * sc["V"].std() / math.sqrt(len(sc))


def test_step_limiter_converges_and_power_laws(oracle):
    """Reading A29/A30: with rho ∝ r^-2, v ∝ r^0.5 in a shell the spectrum at f = 0.01 equals the one at
    f = 0.003 (two-sample KS): the midpoint rule has converged; and the radial column is the analytic integral, seen
    through the unscattered fraction of far-wing photons, exp(-N sigma_0 H(a, x))."""
    n, T = 3000, 1e4
    r_in, n0 = 0.25, 2e18 / (0.25 * (1 / 0.25 - 1) * PC) / 16.0   # column N = n0 Int (r/r_o)^-2 dr = n0 r_o (1/r_in - 1)
    d = dict(geometry=0, r_in=r_in, r_out=1.0, length_cm=PC, n0=n0, alpha_rho=-2.0, T=T, v_max=150.0, alpha_v=0.5)
    opts = dict(spec_mode=1, spec_bins=10, spec_lo=-1500.0, spec_hi=1500.0)
    a1 = oracle.run_gridless(dict(d, step_f=0.01), _central(50.0), opts, n, seed=7)
    a2 = oracle.run_gridless(dict(d, step_f=0.003), _central(50.0), opts, n, seed=8)
    assert stats.ks_2samp(a1["raw"]["V"], a2["raw"]["V"]).pvalue > 0.01
    assert stats.ks_2samp(a1["raw"]["nscat"], a2["raw"]["nscat"]).pvalue > 0.01
    # static twin, photons emitted 40 v_th off resonance (sigma = 0 source in a moving frame is not available: use the
    # wing of a wide Gaussian): unscattered fraction against the analytic column
    N = n0 * PC * (1 / r_in - 1)
    ds = dict(d, v_max=0.0)
    b = oracle.run_gridless(ds, _central(2000.0), opts, 40_000, seed=9)
    V = b["raw"]["V"].astype(float)                                # unscattered packets keep their emission frequency
    # expectation of exp(-N sigma0 H(a, V/vth)) over the emitted Gaussian, by quadrature
    vth, a = oracle.vth_kms(T), oracle.voigt_a(T)
    f = lambda v: math.exp(-N * oracle.sigma0_cm2(T) * special.wofz(v / vth + 1j * a).real) * stats.norm.pdf(v, 0, 2000.0)
    p = integrate.quad(f, -2e4, 2e4, points=[-100, 0, 100], limit=400)[0]
    got = b["nscat_hist"][0] / 40_000
    assert abs(got - p) < 4.5 * math.sqrt(p * (1 - p) / 40_000), (got, p)


def test_gridless_agrees_with_the_voxelised_walker(oracle):
    """The two walkers of the oracle share samplers but no geometry code: a homogeneous static sphere walked gridless and
    on a 64^3 grid (voxelised surface: tau0 by direction differs by ~1 %) give the same escape spectrum and counts."""
    n, T, tau0 = 5000, 10.0, 1e3
    g = W.static_sphere(n=64, tau0=tau0, T=T, n_photons=n)
    a = oracle.run(g["grid"], g["sources"], g["opts"], n, seed=11)
    # the recipe's sigma0 literal sets the grid's density: use the same density gridless (radius = 32 cells of 1 pc)
    dens = float(g["grid"]["nHI"].max())
    d = dict(geometry=0, r_in=0.0, r_out=32.0, length_cm=PC, n0=dens, T=T)
    b = oracle.run_gridless(d, _central(), g["opts"], n, seed=12)
    assert stats.ks_2samp(a["raw"]["V"], b["raw"]["V"]).pvalue > 0.01
    ma, mb = a["raw"]["nscat"].astype(float), b["raw"]["nscat"].astype(float)
    assert abs(ma.mean() - mb.mean()) < 4 * math.sqrt(ma.var() / n + mb.var() / n) + 0.02 * mb.mean()
