"""Pins for the oracle's building blocks (CPU only).  Each test checks oracle/ against something other than itself:
a value the paper prints, a closed form, a library routine, an invariant, or brute force.  Pin numbers: DESIGN.md."""
import math
import os

import numpy as np
import pytest
from scipy import integrate, special, stats

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden_rows(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


# ---------------------------------------------------------------- P13 Philox
def test_philox_known_answers(oracle):
    for row in _golden_rows("philox4x32_10_kat.txt"):
        v = [int(h, 16) for h in row]
        out = oracle.philox4x32_10(v[0:4], v[4:6])
        assert [int(o) for o in out] == v[6:10]


def test_draw_stream_layout(oracle):
    """Draw d of packet id = word d&3 of block d>>2 with counter (block_lo, block_hi, id_lo, id_hi), key = seed."""
    seed, pid = 0x123456789ABCDEF0, 0x0FEDCBA987654321
    d = oracle.draws_u32(seed, pid, 11)
    for blk in range(3):
        ref = oracle.philox4x32_10([blk, 0, pid & 0xFFFFFFFF, pid >> 32], [seed & 0xFFFFFFFF, seed >> 32])
        for w in range(4):
            if 4 * blk + w < 11:
                assert d[4 * blk + w] == ref[w]


def test_uniform_mapping_open_interval(oracle):
    assert oracle.u32_to_uniform(0) == 0.5 / 2 ** 23
    assert oracle.u32_to_uniform(0xFFFFFFFF) == 1.0 - 0.5 / 2 ** 23
    assert oracle.u32_to_uniform(0x80000000) == (2 ** 22 + 0.5) / 2 ** 23
    # every value is representable in fp32 (so the CUDA path can form exactly the same uniforms)
    for r in (0, 0x1FF, 0x200, 0x7FFFFFFF, 0x80000000, 0xFFFFFE00, 0xFFFFFFFF):
        u = oracle.u32_to_uniform(r)
        assert float(np.float32(u)) == u and 0.0 < u < 1.0
    u = np.array([oracle.u32_to_uniform(int(r)) for r in oracle.draws_u32(1, 0, 4000)])
    assert stats.kstest(u, stats.uniform(0, 1).cdf).pvalue > 1e-3


# ---------------------------------------------------------------- constants
def test_lya_constants(oracle):
    got = dict(vth_kms_1e4K=oracle.vth_kms(1e4), a_1e4K=oracle.voigt_a(1e4), sigma0_1e4K=oracle.sigma0_cm2(1e4),
               a_10K=oracle.voigt_a(10.0))
    for name, val, tol in _golden_rows("lya_constants.txt"):
        assert abs(got[name] / float(val) - 1.0) < float(tol), name
    # scalings with temperature
    assert abs(oracle.vth_kms(4e4) / oracle.vth_kms(1e4) - 2.0) < 1e-12
    assert abs(oracle.voigt_a(4e4) / oracle.voigt_a(1e4) - 0.5) < 1e-12
    assert abs(oracle.sigma0_cm2(4e4) / oracle.sigma0_cm2(1e4) - 0.5) < 1e-12
    # BASELINE.json config 1: a tau0 ≈ 1.5e3
    assert abs(oracle.voigt_a(10.0) * 1e5 - 1.5e3) < 20


# ---------------------------------------------------------------- P1 Voigt
def test_voigt_vs_faddeeva_lattice(oracle):
    a = np.geomspace(1e-6, 5e-2, 80)[:, None]
    x = np.concatenate([np.linspace(0, 12, 2401), np.geomspace(12, 1e4, 600)])[None, :]
    H = oracle.voigt_H(a, x)
    ref = special.wofz(x + 1j * a).real
    assert np.max(np.abs(H - ref) / ref) < 1e-10
    # symmetric in x
    assert np.array_equal(oracle.voigt_H(a, -x), H)


def test_voigt_line_centre_closed_form(oracle):
    for a in (1e-5, 4.7e-4, 1.49e-2, 4.7e-2):
        assert abs(oracle.voigt_H(a, 0.0) / (math.exp(a * a) * math.erfc(a)) - 1.0) < 1e-13


def test_voigt_normalisation(oracle):
    """Int H dx = sqrt(pi).  Integrate |x| < X numerically and add the wing a/(sqrt(pi) x^2)(1 + 3/(2x^2)) tail."""
    for a in (4.7e-4, 1.49e-2):
        X = 200.0
        xs = np.concatenate([np.linspace(0, 10, 200001), np.linspace(10, X, 400001)[1:]])
        core = 2.0 * integrate.simpson(oracle.voigt_H(a, xs), x=xs)
        tail = 2.0 * a / math.sqrt(math.pi) * (1.0 / X + 0.5 / X ** 3)
        assert abs((core + tail) / math.sqrt(math.pi) - 1.0) < 1e-8


def test_voigt_wing_limit(oracle):
    for a in (5e-5, 4.7e-4, 1.49e-2):
        for x in (30.0, 100.0, 1000.0):
            lim = a / (math.sqrt(math.pi) * x * x) * (1 + 1.5 / x ** 2 + 3.75 / x ** 4)
            assert abs(oracle.voigt_H(a, x) / lim - 1.0) < 2e-5


def test_voigt_defining_integral(oracle):
    """Direct quadrature of (a/pi) Int exp(-y^2)/((x-y)^2+a^2) dy with y = x + a sinh(s)."""
    def H_quad(a, x):
        f = lambda s: math.exp(-(x + a * math.sinh(s)) ** 2) / math.cosh(s)
        smax = math.asinh((abs(x) + 7.0) / a)
        s0 = -math.asinh(x / a)                                  # image of the Gaussian core y = 0
        pts = sorted({-smax, s0 - 3.0 / max(1.0, abs(x)), s0, s0 + 3.0 / max(1.0, abs(x)), 0.0, smax})
        tot = 0.0
        for lo, hi in zip(pts[:-1], pts[1:]):
            tot += integrate.quad(f, lo, hi, epsabs=0, epsrel=1e-12, limit=400)[0]
        return tot / math.pi
    for a, x in [(1.49e-2, 0.0), (1.49e-2, 1.0), (4.7e-4, 2.5), (4.7e-4, 3.3), (1.49e-2, 5.0), (4.7e-4, 9.0)]:
        assert abs(oracle.voigt_H(a, x) / H_quad(a, x) - 1.0) < 1e-8, (a, x)


def test_dawson_vs_scipy(oracle):
    xs = np.concatenate([np.linspace(-12, 12, 4801), [1e-8, 0.19999, 0.2, 0.924]])
    d = np.array([oracle.dawson(x) for x in xs])
    ref = special.dawsn(xs)
    assert np.max(np.abs(d - ref)) < 2e-15


# ---------------------------------------------------------------- P2 x_cw
def test_x_cw_root_and_b25(oracle):
    coeffs = {r[0]: float(r[1]) for r in _golden_rows("x_cw_b25_coeffs.txt")}
    for T in np.geomspace(1.0, 1e7, 29):
        a = oracle.voigt_a(T)
        xcw = oracle.x_cw_exact(a)
        assert abs(math.exp(-xcw * xcw) - a / (math.sqrt(math.pi) * xcw * xcw)) < 1e-12
        L = math.log(a)
        poly = sum(coeffs[f"c{i}"] * L ** i for i in range(5))
        assert abs(oracle.x_cw_b25(a) - poly) < 1e-12             # the oracle carries the printed coefficients
        assert abs(poly / xcw - 1.0) < coeffs["max_rel_dev"]       # <= 0.5 % (0.53 % at 1e7 K)
    assert abs(oracle.x_cw_exact(oracle.voigt_a(1e4)) - 3.2544) < 2e-3


# ---------------------------------------------------------------- P3 u_par
def _upar_cdf(oracle, a, x):
    """CDF of Eq. 6 by trapezoid on a grid that resolves both the Gaussian bulk and the Lorentzian peak."""
    g = np.union1d(np.linspace(-7.0, 7.0 + abs(x), 40001), x + a * np.sinh(np.linspace(-14, 14, 8001)))
    g = g[(g > -7.5) & (g < abs(x) + 7.5)]
    H = oracle.voigt_H(a, x).item()
    pdf = (a / math.pi) * np.exp(-g * g) / ((x - g) ** 2 + a * a) / H
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (pdf[1:] + pdf[:-1]) * np.diff(g))])
    assert abs(cdf[-1] - 1.0) < 2e-5, (a, x, cdf[-1])             # Eq. 6 integrates to one (fixes H's normalisation)
    return lambda u: np.interp(u, g, cdf / cdf[-1])


@pytest.mark.parametrize("a", [1.49e-2, 4.72e-4, 5e-5])
@pytest.mark.parametrize("x", [0.0, 0.5, 1.0, 2.0, 3.0, "xcw", 4.0, 6.0, 7.9, 8.0, 10.0, 30.0, -2.0, -12.0])
def test_upar_distribution(oracle, a, x):
    if x == "xcw":
        x = oracle.x_cw_exact(a)
    n = 200_000
    u, iters = oracle.sample_upar(a, x, n, seed=5, photon_id=int(1000 * abs(x)) + 7)
    ks = stats.kstest(u, _upar_cdf(oracle, a, x))
    assert ks.pvalue > 1e-3, (a, x, ks)
    assert iters >= n


@pytest.mark.parametrize("which", [1, 2])
def test_upar_both_schemes_everywhere(oracle, which):
    """Each of the two rejection schemes is exact for any x (only their efficiency differs)."""
    a = 4.72e-4
    for x in (1.0, 5.0, 9.0):
        if which == 2 and x < 4:
            continue                                            # far scheme's acceptance collapses in the core
        u, _ = oracle.sample_upar(a, x, 40_000, seed=9, photon_id=which, which=which)
        assert stats.kstest(u, _upar_cdf(oracle, a, x)).pvalue > 1e-3, (which, x)


def test_upar_symmetry_and_iterations(oracle):
    a = 4.72e-4
    up, _ = oracle.sample_upar(a, 2.5, 50_000, seed=2, photon_id=4)
    um, _ = oracle.sample_upar(a, -2.5, 50_000, seed=2, photon_id=4)
    assert np.array_equal(up, -um)                                # f(u; -x) = f(-u; x), same stream
    # efficiency in kind with PAPER.md:1050-1052 (expected iterations a few, tens at worst near x ~ 3-4)
    for x, lim in [(0.0, 2.0), (1.0, 2.0), (2.0, 2.5), (3.5, 40.0), (5.0, 20.0), (12.0, 6.0), (40.0, 3.0)]:
        _, it = oracle.sample_upar(a, x, 20_000, seed=3, photon_id=1)
        assert it / 20_000 < lim, (x, it / 20_000)


# ---------------------------------------------------------------- u_perp, phase functions (P10), Eq. 7 (P9)
def test_uperp_moments_and_core_skip(oracle):
    u1, u2 = oracle.sample_uperp(0.0, 0.0, 400_000)
    for u in (u1, u2):                                             # Eq. 5: pdf ∝ exp(-u^2): variance 1/2
        assert abs(u.mean()) < 4 * math.sqrt(0.5 / u.size)
        assert abs(u.var() - 0.5) < 0.005
        assert stats.kstest(u, stats.norm(0, math.sqrt(0.5)).cdf).pvalue > 1e-3
    assert abs(np.mean(u1 * u2)) < 0.005
    xc = 3.0
    s1, s2 = oracle.sample_uperp(1.0, xc, 200_000)                 # |x_in| < x_crit: magnitude left-truncated at x_crit
    m2 = s1 * s1 + s2 * s2
    assert m2.min() >= xc * xc
    assert stats.kstest(m2 - xc * xc, stats.expon.cdf).pvalue > 1e-3       # m^2 - x_crit^2 ~ Exp(1)
    t1, t2 = oracle.sample_uperp(3.5, xc, 100_000)                 # |x_in| >= x_crit: untouched
    assert abs((t1 * t1 + t2 * t2).mean() - 1.0) < 0.02


def test_phase_functions(oracle):
    n = 400_000
    iso = oracle.sample_mu(0, n)
    dip = oracle.sample_mu(1, n)
    mix = oracle.sample_mu(2, n)
    se = 1.0 / math.sqrt(n)
    assert abs(iso.mean()) < 4 * se and abs((iso ** 2).mean() - 1 / 3) < 4 * se
    assert abs(dip.mean()) < 4 * se and abs((dip ** 2).mean() - 2 / 5) < 4 * se
    assert abs((mix ** 2).mean() - (1 / 3 * 1 / 3 + 2 / 3 * 2 / 5)) < 4 * se
    dip_cdf = lambda m: (3 * m + m ** 3 + 4) / 8
    assert stats.kstest(dip, dip_cdf).pvalue > 1e-3
    assert stats.kstest(iso, stats.uniform(-1, 2).cdf).pvalue > 1e-3
    for r in (0.0, 0.1, 0.5, 0.77, 1.0):
        m = oracle.dipole_mu(r)
        assert abs(dip_cdf(m) - r) < 1e-12


def _upar_moments(oracle, a, x):
    f = lambda u, p: u ** p * (a / math.pi) * math.exp(-u * u) / ((x - u) ** 2 + a * a)
    H = oracle.voigt_H(a, x).item()
    out = []
    for p in (1, 2):
        pts = [x - 50 * a, x, x + 50 * a, 0.0]
        v = integrate.quad(f, -9, 9 + abs(x), args=(p,), points=sorted(pts), epsabs=0, epsrel=1e-10, limit=2000)[0]
        out.append(v / H)
    return out


@pytest.mark.parametrize("x_in", [0.0, 1.5, 5.0, 10.0, 20.0])
def test_single_scatter_redistribution(oracle, x_in):
    """Eq. 7 with isotropic scattering: <dx> = -<u_par>, <dx^2> = 4/3 <u_par^2> + 1/3 (moments of Eq. 6 by
    quadrature); wing limit <dx> -> -1/x_in, rms -> 1."""
    a, n = 4.72e-4, 400_000
    xo, ko = oracle.scatter_once(a, x_in, n, phase=0, seed=11, photon_id=3)
    dx = xo - x_in
    m1, m2 = _upar_moments(oracle, a, x_in)
    var = 4 / 3 * m2 + 1 / 3 - m1 * m1
    assert abs(dx.mean() + m1) < 4.5 * math.sqrt(var / n)
    assert abs((dx ** 2).mean() - (4 / 3 * m2 + 1 / 3)) < 0.02
    if x_in >= 5:
        assert abs(dx.mean() + 1 / x_in + 1.5 / x_in ** 3) < 0.01
        assert abs(dx.std() - 1.0) < 0.03
    assert np.max(np.abs(np.sum(ko * ko, 1) - 1.0)) < 1e-12        # k' is a unit vector
    phi = np.arctan2(ko[:, 1], ko[:, 0])
    assert stats.kstest(phi, stats.uniform(-math.pi, 2 * math.pi).cdf).pvalue > 1e-3
    assert stats.kstest(ko[:, 2], stats.uniform(-1, 2).cdf).pvalue > 1e-3     # mu about k_in = +z


def test_single_scatter_dipole_correlation(oracle):
    """With a dipole phase function <mu^2> = 2/5: <dx^2> = <u_par^2>(1 + 2/5) + (1 - 2/5)/2."""
    a, n, x_in = 4.72e-4, 300_000, 6.0
    xo, ko = oracle.scatter_once(a, x_in, n, phase=1, seed=12, photon_id=1)
    m1, m2 = _upar_moments(oracle, a, x_in)
    assert abs(((xo - x_in) ** 2).mean() - (1.4 * m2 + 0.3)) < 0.02
    assert abs((ko[:, 2] ** 2).mean() - 0.4) < 0.005


# ---------------------------------------------------------------- P11 DDA
def _brute_force_cells(dims, org, d):
    """All cells whose box the ray pierces with positive length, ordered by entry parameter (fp64)."""
    hits = []
    for iz in range(dims[2]):
        for iy in range(dims[1]):
            for ix in range(dims[0]):
                lo = np.array([ix, iy, iz], float)
                t0, t1 = 0.0, np.inf
                ok = True
                for ax in range(3):
                    if d[ax] == 0:
                        if not (lo[ax] <= org[ax] <= lo[ax] + 1):
                            ok = False
                        continue
                    ta, tb = (lo[ax] - org[ax]) / d[ax], (lo[ax] + 1 - org[ax]) / d[ax]
                    t0, t1 = max(t0, min(ta, tb)), min(t1, max(ta, tb))
                if ok and t1 - t0 > 1e-9:
                    hits.append((t0, (iz * dims[1] + iy) * dims[0] + ix, t1 - t0))
    hits.sort()
    return [h[1] for h in hits], [h[2] for h in hits]


@pytest.mark.parametrize("real32", [True, False])
def test_dda_brute_force_small_grid(oracle, real32):
    from paper_2507_11603_b200 import workloads
    dims = (5, 4, 6)
    org, dirs = workloads.random_rays(150, dims, seed=21)
    for i in range(org.shape[0]):
        t = oracle.dda_trace(dims, (0, 0, 0), org[i:i + 1], dirs[i:i + 1], max_steps=64, real32=real32, want_seq=True)
        cells, lens = _brute_force_cells(dims, org[i].astype(float), dirs[i].astype(float))
        seq = [int(c) for c, l in zip(t["seq_idx"], t["seq_len"]) if l > 1e-6]      # drop grazing zero-length cells
        cells = [c for c, l in zip(cells, lens) if l > 1e-6]
        assert seq == cells, i
        # total length = chord through the grid
        assert abs(t["seq_len"].sum() - sum(lens)) < (2e-5 if real32 else 1e-10)
        # consecutive cells differ by one step on exactly one axis
        idx = t["seq_idx"]
        c3 = np.stack([idx % dims[0], (idx // dims[0]) % dims[1], idx // (dims[0] * dims[1])], 1)
        assert np.all(np.abs(np.diff(c3, axis=0)).sum(1) == 1)


def test_dda_special_cases(oracle):
    dims = (8, 8, 8)
    # source on a cell corner (reading A20): cell = floor(pos), f = 0; negative components take a zero-length step
    t = oracle.dda_trace(dims, (0, 0, 0), np.array([[4, 4, 4]], np.float32), np.array([[-0.6, 0.0, 0.8]], np.float32),
                         max_steps=64, want_seq=True)
    assert t["seq_idx"][0] == (4 * 8 + 4) * 8 + 4 and t["seq_len"][0] == 0.0
    assert t["seq_idx"][1] == (4 * 8 + 4) * 8 + 3
    # axis-aligned ray, zero components (t = +inf on those axes)
    t = oracle.dda_trace(dims, (0, 0, 0), np.array([[2.5, 3.5, 0.25]], np.float32), np.array([[0, 0, 1]], np.float32),
                         max_steps=64, want_seq=True)
    assert list(t["seq_idx"]) == [(z * 8 + 3) * 8 + 2 for z in range(8)]
    assert abs(t["seq_len"].sum() - 7.75) < 1e-6
    # tie: exact diagonal leaves through x first, then y, then z
    t = oracle.dda_trace(dims, (0, 0, 0), np.array([[0, 0, 0]], np.float32), np.array([[1, 1, 1]], np.float32),
                         max_steps=8, want_seq=True)
    assert list(t["seq_idx"][:4]) == [0, 1, 1 + 8, 1 + 8 + 64]
    # periodic wrap
    t = oracle.dda_trace(dims, (1, 0, 0), np.array([[7.5, 0.5, 0.5]], np.float32), np.array([[1, 0, 0]], np.float32),
                         max_steps=20, want_seq=True)
    assert list(t["seq_idx"][:3]) == [7, 0, 1] and t["count"][0] == 20
    # an axis that is periodic with extent 1 is infinite: never crossed
    t = oracle.dda_trace((1, 1, 16), (1, 1, 0), np.array([[0.5, 0.5, 8.0]], np.float32),
                         np.array([[0.7, 0.1, 0.7071]], np.float32), max_steps=64, want_seq=True)
    assert list(t["seq_idx"]) == list(range(8, 16))
    assert abs(t["seq_len"].sum() - 8 / 0.7071) < 1e-4


def test_dda_reflection_symmetry_and_fp64_twin(oracle):
    from paper_2507_11603_b200 import workloads
    dims = (16, 16, 16)
    org, dirs = workloads.random_rays(2000, dims, seed=5)
    a = oracle.dda_trace(dims, (0, 0, 0), org, dirs, real32=True)
    b = oracle.dda_trace(dims, (0, 0, 0), org, dirs, real32=False)
    assert np.array_equal(a["count"], b["count"]) or np.mean(a["count"] != b["count"]) < 0.01
    assert np.mean(a["hash_idx"] == b["hash_idx"]) > 0.98          # fp32 and fp64 agree except at near-ties
    # mirror in x: same number of cells
    org_m = org.copy()
    org_m[:, 0] = np.float32(16) - org[:, 0]
    dirs_m = dirs.copy()
    dirs_m[:, 0] = -dirs[:, 0]
    m = oracle.dda_trace(dims, (0, 0, 0), org_m, dirs_m, real32=False)
    assert np.mean(m["count"] == b["count"]) > 0.99
