"""Pins for the oracle's dust scattering (PAPER.md 2.3.2, Eq. 8-9) and doublet interactor, CPU only."""
import math

import numpy as np
from scipy import integrate, special, stats

from paper_2507_11603_b200 import workloads as W

PC = W.PC_CM


def _central(sigma=0.0):
    return dict(pos=np.zeros((1, 3), np.float32), lum=np.ones(1, np.float32), sigma=np.full(1, sigma, np.float32))


def test_henyey_greenstein_sampler(oracle):
    """Eq. 9: closed-form inversion against the closed-form CDF, F(mu) = (1 - g^2)/(2g) [1/sqrt(1 + g^2 - 2 g mu) - 1/(1 + g)],
    <mu> = g; hg_value is 2 P_HG (isotropic -> 1) and integrates to 2 over mu."""
    r = (np.arange(200_000) + 0.5) / 200_000
    for g in (0.73, -0.4, 0.05):
        mu = np.array([oracle.hg_mu(g, x) for x in r[::20]])
        cdf = lambda m: (1 - g * g) / (2 * g) * (1 / np.sqrt(1 + g * g - 2 * g * m) - 1 / (1 + g))
        assert np.abs(cdf(mu) - r[::20]).max() < 1e-12
        assert abs(np.mean([oracle.hg_mu(g, x) for x in r[::20]]) - g) < 2e-4
        assert abs(integrate.quad(lambda m: oracle.hg_value(g, m), -1, 1)[0] - 2.0) < 1e-9
    assert oracle.hg_mu(0.0, 0.25) == -0.5 and oracle.hg_value(0.0, 0.3) == 1.0


def test_dust_scattering_closed_forms(oracle):
    """(i) Deep inside thick dust nothing escapes and every interaction scatters with probability A: the number of dust
    scatterings before destruction is geometric, mean A / (1 - A).  (ii) Forward scattering (g -> 1) never turns a packet:
    along a path of extinction depth tau it survives iff every interaction scatters: f_esc = exp(-tau (1 - A)).
    (iii) A = 1 destroys nothing."""
    n, A = 40_000, 0.32
    opts = dict(spec_bins=4, spec_lo=-1.0, spec_hi=1.0)
    d = dict(geometry=0, r_out=1.0, length_cm=PC, n0=0.0, T=1e4, kdust0=60.0 / PC)
    r = oracle.run_gridless(d, _central(), dict(opts, dust_albedo=A, dust_g=0.0), n, seed=1)
    assert r["counters"]["absorbed"] == n
    mean = r["counters"]["dust_scatterings"] / n
    assert abs(mean - A / (1 - A)) < 4.5 * math.sqrt(A / (1 - A) ** 2 / n)
    tau = 2.5
    d = dict(d, kdust0=tau / PC)
    r = oracle.run_gridless(d, _central(), dict(opts, dust_albedo=A, dust_g=1.0 - 1e-9), n, seed=2)
    p = math.exp(-tau * (1 - A))
    assert abs(r["counters"]["escaped"] / n - p) < 4.5 * math.sqrt(p * (1 - p) / n)
    r = oracle.run_gridless(d, _central(), dict(opts, dust_albedo=1.0, dust_g=0.73), 5000, seed=3)
    assert r["counters"]["escaped"] == 5000 and r["counters"]["dust_scatterings"] > 5000
    # the voxelised walker: same geometric law in a thick dusty cube, and forward scattering along the chord
    N = 8
    z = np.zeros((N, N, N), np.float32)
    grid = dict(nx=N, ny=N, nz=N, periodic=(0, 0, 0), cell_cm=PC, nHI=z, T=np.full((N, N, N), 1e4, np.float32), vx=z, vy=z, vz=z,
                kdust=np.full((N, N, N), 15.0 / PC, np.float32))
    src = dict(pos=np.array([[4.0, 4.0, 4.0]], np.float32), lum=np.ones(1, np.float32), sigma=np.zeros(1, np.float32))
    r = oracle.run(grid, src, dict(opts, dust_albedo=A, dust_g=0.73), n, seed=4)
    assert r["counters"]["absorbed"] == n
    assert abs(r["counters"]["dust_scatterings"] / n - A / (1 - A)) < 4.5 * math.sqrt(A / (1 - A) ** 2 / n)


def test_dust_scattering_keeps_the_bulk_frame_frequency(oracle):
    """Reading A33: grains move with the gas and are heavy, so a dust scattering leaves the frequency unchanged in the
    cell's bulk frame: V' = V - v.k + v.k'.  Pure scattering dust (A = 1) moving at v = (0, 0, 100) km/s: every packet leaves
    with V = v k_z' whatever happened in between (emitted at the bulk-frame line centre)."""
    N, n = 6, 4000
    z = np.zeros((N, N, N), np.float32)
    grid = dict(nx=N, ny=N, nz=N, periodic=(0, 0, 0), cell_cm=PC, nHI=z, T=np.full((N, N, N), 1e4, np.float32), vx=z, vy=z,
                vz=np.full((N, N, N), 100.0, np.float32), kdust=np.full((N, N, N), 1.0 / PC, np.float32))
    src = dict(pos=np.array([[3.0, 3.0, 3.0]], np.float32), lum=np.ones(1, np.float32), sigma=np.zeros(1, np.float32))
    r = oracle.run(grid, src, dict(spec_mode=1, spec_bins=4, spec_lo=-200.0, spec_hi=200.0, dust_albedo=1.0, dust_g=0.73), n, seed=5)
    assert r["counters"]["escaped"] == n and r["counters"]["dust_scatterings"] > n
    assert np.allclose(r["raw"]["V"], 100.0 * r["raw"]["kz"], atol=2e-4)


def test_doublet_cross_sections_add(oracle):
    """the overall cross-section is the sum over the transitions.  A broad source behind a static slab of a
    species with a second line 300 km/s away (sigma_0 ratio 0.5): packets that never scatter keep their emission
    frequency, so their spectrum is the source Gaussian times E_2-like transmission through tau(V) = N sigma_0 [H(a, V/v_th)
    + 0.5 H(a r_a, (V - 300)/v_th)]: both troughs, at the right place and depth (chi^2 over bins, scipy's Faddeeva function)."""
    n, T = 200_000, 1e4
    vth, a, sig0 = oracle.vth_kms(T), oracle.voigt_a(T), oracle.sigma0_cm2(T)
    tau0 = 3.0
    w = W.static_slab(nz=4, tau0=tau0, T=T, core_skip=False, n_photons=n)
    w["sources"]["sigma"][:] = 250.0
    opts = dict(w["opts"], spec_mode=1, spec_bins=40, spec_lo=-400.0, spec_hi=700.0, doublet_on=1, doublet_dv_kms=300.0,
                doublet_sigma_ratio=0.5, doublet_a_ratio=2.0)
    r = oracle.run(w["grid"], w["sources"], opts, n, seed=6)
    un = r["raw"][r["raw"]["nscat"] == 0]
    tau_real = tau0 * sig0 / W.RECIPE_SIGMA0_T4
    edges = np.linspace(-400.0, 700.0, 45)
    got, _ = np.histogram(un["V"], edges)
    def dens(V):
        t = tau_real * (special.wofz(V / vth + 1j * a).real + 0.5 * special.wofz((V - 300.0) / vth + 2j * a).real)
        return stats.norm.pdf(V, 0, 250.0) * special.expn(2, t)        # slab, isotropic emission from the midplane: E_2
    exp = np.array([integrate.quad(dens, lo, hi, points=[p for p in (0.0, 300.0) if lo < p < hi] or None, limit=200)[0]
                    for lo, hi in zip(edges[:-1], edges[1:])]) * n
    chi2 = ((got - exp) ** 2 / np.maximum(exp, 1.0)).sum()
    assert stats.chi2.sf(chi2, len(exp)) > 1e-3, chi2
    i0, i1 = np.searchsorted(edges, 0.0) - 1, np.searchsorted(edges, 300.0) - 1
    assert got[i0] < 0.5 * got[i0 - 3] and got[i1] < 0.8 * got[i1 + 3]                 # two troughs
    # interaction i with probability tau_i / tau: photons emitted exactly at the second line's centre and
    # scattered once or more end up redistributed about 300 km/s, not about 0
    w["sources"]["sigma"][:] = 0.0
    grid2 = dict(w["grid"], vz=np.zeros_like(w["grid"]["vz"]))
    sc = oracle.run(grid2, w["sources"], dict(opts, doublet_dv_kms=0.0, doublet_sigma_ratio=3.0, doublet_a_ratio=1.0), 20_000, seed=7)
    one = oracle.run(grid2, w["sources"], dict(w["opts"], spec_mode=1, spec_bins=40, spec_lo=-400.0, spec_hi=700.0), 20_000, seed=7)
    # dv = 0 with ratio 3 is one line of 4 x the cross-section: unscattered fraction E_2(4 tau H0) against E_2(tau H0)
    H0 = special.wofz(1j * a).real
    for res, f in ((sc, 4.0), (one, 1.0)):
        p = special.expn(2, f * tau_real * H0)
        assert abs(res["nscat_hist"][0] / 20_000 - p) < 4.5 * math.sqrt(p * (1 - p) / 20_000)
