"""GPU parity of the walk through the paper's GRIDLESS datasets (thor_dataset_create_gridless; PAPER.md 3.3, 197-198,
380-382) against the oracle's gridless walker (oracle/gridless.hpp, pinned in tests/test_oracle_gridless.py), at
BASELINE.json's bars, plus the closed forms that hold exactly on analytic geometry."""
import math

import numpy as np
import pytest
from scipy import special, stats

from paper_2507_11603_b200 import workloads as W
from conftest import scaled, statistical
from test_gpu_walk import _bins_within_4sigma, _conserved, _statistical_parity

pytestmark = pytest.mark.gpu
PC = W.PC_CM


@pytest.fixture(scope="module")
def thor():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2507_11603_b200 import thor as t
    t.lib()
    return t


def _central(sigma=0.0):
    return dict(pos=np.zeros((1, 3), np.float32), lum=np.ones(1, np.float32), sigma=np.full(1, sigma, np.float32))


def _both(thor, oracle, dataset, sources, opts, n, seed=1):
    g = thor.run_workload(dict(dataset=dataset, sources=sources, opts=opts, n_photons=n, seed=seed))
    o = oracle.run_gridless(dataset, sources, opts, n, seed)
    _conserved(g, n)
    return g, o


@statistical()
def test_static_sphere_and_slab(thor, oracle):
    """The Neufeld / Dijkstra problems on the analytic geometries the paper validates on: sphere without
    core-skipping at tau0 = 1e3, slab with x_crit core-skipping at tau0 = 1e6 (a tau0 = 1.5e4, T = 10 K)."""
    n, T = scaled(10_000), 10.0
    sig0 = oracle.sigma0_cm2(T)
    opts = dict(spec_bins=100, spec_lo=-30.0, spec_hi=30.0, spec_T_ref=T)
    g, o = _both(thor, oracle, dict(geometry=0, r_out=1.0, length_cm=PC, n0=1e3 / (sig0 * PC), T=T), _central(), opts, n)
    _statistical_parity(g, o, n, n)
    a = oracle.voigt_a(T)
    opts = dict(spec_bins=100, spec_lo=-120.0, spec_hi=120.0, spec_T_ref=T, core_skip_mode=1, x_crit=0.2 * (a * 1e6) ** (1 / 3),
                phase_core=1)
    g, o = _both(thor, oracle, dict(geometry=1, r_out=2.0, length_cm=PC, n0=1e6 / (sig0 * 2.0 * PC), T=T), _central(), opts, n)
    _statistical_parity(g, o, n, n)
    ax = np.abs(g["raw"]["V"].astype(float)) / oracle.vth_kms(T)
    k = math.sqrt(math.pi ** 3 / 54) / (a * 1e6)
    assert stats.kstest(ax, lambda x: 4 / math.pi * np.arctan(np.tanh(k * x ** 3 / 2))).statistic < 0.025    # P4, no voxelisation


def test_exact_unscattered_and_dust_fractions(thor, oracle):
    """Closed forms on the GPU path itself: P(N = 0) = exp(-tau0 H(a,0)) (sphere) and E_2 (slab); dust-only f_esc = e^-tau_d."""
    n, T = 200_000, 1e4
    H0 = special.wofz(1j * oracle.voigt_a(T)).real
    sig0 = oracle.sigma0_cm2(T)
    opts = dict(spec_bins=10, spec_lo=-20.0, spec_hi=20.0, spec_T_ref=T)
    for geom, tau0 in ((0, 0.4), (0, 2.0), (1, 0.4), (1, 2.0)):
        g = thor.run_workload(dict(dataset=dict(geometry=geom, r_out=1.0, length_cm=PC, n0=tau0 / (sig0 * PC), T=T),
                                   sources=_central(), opts=opts, n_photons=n, seed=3), raw=False)
        p = math.exp(-tau0 * H0) if geom == 0 else special.expn(2, tau0 * H0)
        assert abs(g["nscat_hist"][0] / n - p) < 4.5 * math.sqrt(p * (1 - p) / n), (geom, tau0)
    g = thor.run_workload(dict(dataset=dict(geometry=0, r_in=0.6, r_out=1.0, length_cm=PC, n0=0.0, T=T, kdust0=1.3 / (0.4 * PC)),
                               sources=_central(), opts=opts, n_photons=n, seed=5), raw=False)
    p = math.exp(-1.3)
    assert g["counters"]["scatterings"] == 0
    assert abs(g["counters"]["escaped"] / n - p) < 4.5 * math.sqrt(p * (1 - p) / n)


@statistical()
def test_expanding_shell_with_power_laws_and_dust(thor, oracle):
    """rho ∝ r^-2, v ∝ r^0.5 between r_in and r_out, with dust and the step limiter f = 0.01;
    and the linearly expanding sphere of PAPER.md:352."""
    n, T = scaled(6000), 1e4
    r_in = 0.25
    n0 = 2e18 / (0.25 * (1 / 0.25 - 1) * PC) / 16.0
    d = dict(geometry=0, r_in=r_in, r_out=1.0, length_cm=PC, n0=n0, alpha_rho=-2.0, T=T, v_max=150.0, alpha_v=0.5,
             kdust0=0.3 / (0.75 * PC) / 16.0, step_f=0.01)
    opts = dict(spec_mode=1, spec_bins=100, spec_lo=-1000.0, spec_hi=1000.0)
    g, o = _both(thor, oracle, d, _central(50.0), opts, n)
    _statistical_parity(g, o, n, n)
    assert 0.02 * n < g["counters"]["absorbed"] < 0.98 * n
    assert abs(g["counters"]["cell_crossings"] / o["counters"]["cell_crossings"] - 1) < 0.05       # steps of the limiter
    d = dict(geometry=0, r_out=1.0, length_cm=PC, n0=2e19 / PC, T=2e4, v_max=200.0, alpha_v=1.0, step_f=0.01)
    g, o = _both(thor, oracle, d, _central(), dict(opts, max_scatter=50_000), n)
    _statistical_parity(g, o, n, n)
    assert (-g["raw"]["V"]).mean() > 50.0                        # outflow: red peak


def test_gridless_edge_cases_and_drain_identity(thor):
    T = 1e4
    d = dict(geometry=0, r_out=1.0, length_cm=PC, n0=3e3 / (5.9e-14 * PC), T=T)
    w = dict(dataset=d, sources=_central(), opts=dict(spec_bins=50, spec_lo=-40.0, spec_hi=40.0, spec_T_ref=T), n_photons=3000, seed=2)
    a = thor.run_workload(w, drain_mode=0)
    b = thor.run_workload(w, drain_mode=1)
    assert a["raw"].tobytes() == b["raw"].tobytes() and a["counters"] == b["counters"]
    ctx = thor.Context.gridless(**d)
    try:
        with pytest.raises(thor.ThorError) as e:
            ctx.sources_set(np.array([[0.9, 0.9, 0.0]], np.float32), np.ones(1, np.float32), np.zeros(1, np.float32))
        assert e.value.status == 1                               # outside r_out
        ctx.sources_set(np.array([[0.3, -0.2, 0.1]], np.float32), np.ones(1, np.float32), np.zeros(1, np.float32))
        for bad in (dict(peel_on=1, peel_nx=4, peel_ny=4, peel_nv=4, peel_width_cells=2.0), dict(hubble_kms_per_cell=1.0),
                    dict(core_skip_mode=2)):
            with pytest.raises(thor.ThorError) as e:
                ctx.run(10, 1, dict(w["opts"], **bad))
            assert e.value.status == 5                           # THOR_ERR_UNSUPPORTED
        ctx.run(1000, 1, dict(w["opts"], raw_output=1))
        assert ctx.counters()["escaped"] == 1000
        with pytest.raises(thor.ThorError):
            ctx.raytrace(np.zeros((1, 3), np.float32), np.array([[0, 0, 1.0]], np.float32))
    finally:
        ctx.close()
    for bad in (dict(r_out=0.0), dict(r_in=1.0, r_out=1.0), dict(T=0.0), dict(n0=-1.0), dict(geometry=7), dict(alpha_rho=-2.0)):
        with pytest.raises(thor.ThorError) as e:
            thor.Context.gridless(**dict(d, **bad))
        assert e.value.status == 1
