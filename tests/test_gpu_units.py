"""GPU parity, single steps of the path (a1, a4, a6, a8-a11 of DESIGN.md) through the C-ABI (thor_unit_*), against the
fp64 oracle on the same seeded inputs.  Bars (BASELINE.json north_star): Philox and DDA cell-index sequences
bit-exact; Voigt within 1e-5 relative; sampled variates statistically (KS against Eq. 6 itself and against the
oracle's draws)."""
import math

import numpy as np
import pytest
from scipy import stats

from paper_2507_11603_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def thor():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2507_11603_b200 import thor as t
    t.lib()                                   # raises if libthor_b200.so is missing: no fallback
    return t


# ---------------------------------------------------------------- a1 Philox (bit-exact)
def test_philox_bit_exact(thor, oracle):
    seed = 0x1234_5678_9ABC_DEF0
    for id0, n_ids, n_draws in [(0, 257, 37), ((1 << 32) - 5, 64, 9), ((1 << 63) + 11, 33, 130)]:
        g = thor.unit_philox(seed, id0, n_ids, n_draws)
        for i in (0, 1, n_ids // 2, n_ids - 1):
            o = oracle.draws_u32(seed, (id0 + i) % (1 << 64), n_draws)
            assert np.array_equal(g[i], o), (id0, i)


def test_philox_known_answer_on_device(thor):
    """Philox4x32-10 known answer (tests/golden/philox4x32_10_kat.txt): ctr = key = 0 -> 6627e8d5 e169c58d bc57ac4c
    9b00dbd8.  Stream layout: photon id 0, seed 0, draws 0..3 are the four words of counter block 0."""
    g = thor.unit_philox(0, 0, 1, 4)
    assert [hex(v) for v in g[0]] == ["0x6627e8d5", "0xe169c58d", "0xbc57ac4c", "0x9b00dbd8"]


# ---------------------------------------------------------------- a4 DDA (bit-exact on 1e6 random rays)
def _compare_dda(thor, oracle, dims, periodic, org, dirs, max_steps):
    g = thor.unit_dda_trace(dims, periodic, org, dirs, max_steps=max_steps)
    o = oracle.dda_trace(dims, periodic, org, dirs, max_steps=max_steps, real32=True)
    bad = np.flatnonzero((g["hash_idx"] != o["hash_idx"]) | (g["count"] != o["count"]) |
                         (g["hash_len"] != o["hash_len"]))
    if bad.size:                               # replay the first mismatching ray index by index
        i = int(bad[0])
        gs = thor.unit_dda_trace(dims, periodic, org[i:i + 1], dirs[i:i + 1], max_steps=max_steps, want_seq=True)
        os_ = oracle.dda_trace(dims, periodic, org[i:i + 1], dirs[i:i + 1], max_steps=max_steps, want_seq=True)
        m = min(len(gs["seq_idx"]), len(os_["seq_idx"]))
        first = np.flatnonzero(gs["seq_idx"][:m] != os_["seq_idx"][:m])
        pytest.fail(f"{bad.size} of {len(org)} rays differ; ray {i} org {org[i]} dir {dirs[i]} counts "
                    f"{gs['count'][0]} vs {os_['count'][0]}, first differing step {first[:1]}")
    return g


def test_dda_bit_exact_1e6_rays(thor, oracle):
    dims = (128, 128, 128)
    org, dirs = W.random_rays(1_000_000, dims, seed=3)
    g = _compare_dda(thor, oracle, dims, (0, 0, 0), org, dirs, max_steps=4096)
    assert g["count"].min() >= 1 and g["count"].max() <= 3 * 128
    assert 60 < g["count"].mean() < 140          # mean chord of a cube ~ (2/3) n per axis-crossing family


def test_dda_bit_exact_ragged_and_periodic(thor, oracle):
    for dims, per, steps in [((37, 5, 61), (0, 0, 0), 4096), ((16, 16, 16), (1, 1, 0), 300), ((1, 1, 256), (1, 1, 0), 4096),
                             ((8, 1, 8), (0, 1, 1), 500)]:
        org, dirs = W.random_rays(50_000, dims, seed=11)
        _compare_dda(thor, oracle, dims, per, org, dirs, max_steps=steps)


def test_dda_special_rays(thor, oracle):
    """Reading A20 / A9: origins exactly on cell corners and faces, directions with zero components, axis-aligned
    and diagonal rays (ties between axes), rays starting on the upper boundary."""
    dims = (32, 32, 32)
    s = 1 / math.sqrt(2.0)
    t = 1 / math.sqrt(3.0)
    dirs = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, 0, -1], [s, s, 0], [-s, 0, s], [t, t, t], [-t, -t, -t],
                     [t, -t, t], [0.6, 0.8, 0], [0, -0.6, 0.8], [1e-8, 1, 0], [-1e-20, 0, 1]], np.float32)
    orgs = np.array([[16, 16, 16], [0, 0, 0], [32, 32, 32], [16, 16.5, 3.25], [31.999998, 0, 16], [16, 16, 0]], np.float32)
    org = np.repeat(orgs, len(dirs), axis=0)
    dr = np.tile(dirs, (len(orgs), 1))
    g = _compare_dda(thor, oracle, dims, (0, 0, 0), org, dr, max_steps=4096)
    # a ray along +x from the centre corner visits exactly 16 cells
    assert g["count"][0] == 16


# ---------------------------------------------------------------- a6 Voigt (<= 1e-5 relative)
def test_voigt_lattice(thor, oracle):
    a = np.array([5e-5, 1e-4, 4.72e-4, 1.5e-3, 4.7e-3, 1.0e-2, 1.492e-2, 2.0e-2])
    x = np.concatenate([np.linspace(0, 12, 3841), np.geomspace(12, 1e3, 400), [0.924, 7.9999, 8.0, 8.0001]])
    x = np.concatenate([x, -x[1::7]])
    A, X = np.meshgrid(a, x, indexing="ij")
    g = thor.unit_voigt(A.ravel(), X.ravel()).astype(np.float64)
    o = oracle.voigt_H(A.ravel().astype(np.float32).astype(np.float64), X.ravel().astype(np.float32).astype(np.float64))
    rel = np.abs(g - o) / o
    i = int(rel.argmax())
    assert rel.max() <= 1e-5, (rel.max(), A.ravel()[i], X.ravel()[i])


def test_voigt_random_points(thor, oracle):
    rng = np.random.default_rng(5)
    n = 400_000
    a = np.exp(rng.uniform(math.log(5e-5), math.log(2e-2), n)).astype(np.float32)
    x = (rng.standard_normal(n) * 6).astype(np.float32)
    g = thor.unit_voigt(a, x).astype(np.float64)
    o = oracle.voigt_H(a.astype(np.float64), x.astype(np.float64))
    assert (np.abs(g - o) / o).max() <= 1e-5


# ---------------------------------------------------------------- a8-a11 scattering variates
def _upar_cdf(oracle, a, x):
    """CDF of Eq. 6 by trapezoid; H from the oracle's Voigt routine."""
    g = np.union1d(np.linspace(-7.0, 7.0 + abs(x), 40001), x + a * np.sinh(np.linspace(-14, 14, 8001)))
    g = g[(g > -7.5) & (g < abs(x) + 7.5)]
    pdf = np.exp(-g * g) / ((x - g) ** 2 + a * a)
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (pdf[1:] + pdf[:-1]) * np.diff(g))])
    return lambda u: np.interp(u, g, cdf / cdf[-1])


@pytest.mark.parametrize("a", [1.49e-2, 4.72e-4, 5e-5])
@pytest.mark.parametrize("x", [0.0, 0.03, 0.5, 1.0, 1.49, 1.5, 2.0, 3.0, "xcw", 4.0, 6.0, 8.0, 10.0, 30.0, 200.0, -2.0, -12.0])
def test_upar_against_eq6(thor, oracle, a, x):
    if x == "xcw":
        x = oracle.x_cw_exact(a)
    n = 400_000
    s = thor.unit_scatter(a, x, n, seed=9, id0=1 << 20)
    u = s["u_par"].astype(np.float64)
    assert np.all(np.isfinite(u))
    ks = stats.kstest(u, _upar_cdf(oracle, a, float(np.float32(x))))
    assert ks.pvalue > 1e-3, (a, x, ks)
    assert s["iters"].min() >= 1
    assert s["iters"].mean() < 8.0, s["iters"].mean()       # the envelope's worst case is ~5 near x_cw


@pytest.mark.parametrize("a,x_in,x_crit,phase", [(1.49e-2, 0.0, 0.0, 0), (4.72e-4, 1.0, 0.0, 1), (4.72e-4, 3.3, 0.0, 0),
                                                  (4.72e-4, 1.0, 3.354, 0), (4.72e-4, 6.0, 0.0, 2), (5e-5, 20.0, 0.0, 1),
                                                  (1.49e-2, -4.0, 2.3, 2)])
def test_single_scatter_against_oracle(thor, oracle, a, x_in, x_crit, phase):
    n = 300_000
    g = thor.unit_scatter(a, x_in, n, x_crit=x_crit, phase=phase, seed=3, id0=77)
    xo, ko = oracle.scatter_once(a, x_in, n, x_crit=x_crit, phase=phase, seed=4, photon_id=5)
    assert stats.ks_2samp(g["x_out"], xo).pvalue > 1e-3
    uo, _ = oracle.sample_upar(a, x_in, n, seed=6, photon_id=1)
    assert stats.ks_2samp(g["u_par"], uo).pvalue > 1e-3
    k = g["k_out"].astype(np.float64)
    assert np.abs(np.linalg.norm(k, axis=1) - 1).max() < 5e-6
    assert stats.ks_2samp(k[:, 2], ko[:, 2]).pvalue > 1e-3            # mu = k_out . k_in (k_in = +z)
    phi = np.arctan2(k[:, 1], k[:, 0])
    assert stats.kstest(phi, stats.uniform(-math.pi, 2 * math.pi).cdf).pvalue > 1e-3
    m2 = {0: 1 / 3, 1: 2 / 5, 2: (1 / 3) * (1 / 3) + (2 / 3) * (2 / 5)}[phase]   # pin P10
    assert abs((k[:, 2] ** 2).mean() - m2) < 5 * 0.3 / math.sqrt(n)


def test_dda_linear_index_beyond_2_31(thor, oracle):
    """a4 with 64-bit cell indices (BASELINE.json config 5 has 3.6e9 cells): random rays through VIRTUAL grids of 2.15e9
    and 4.3e9 cells (the trace reads no field; the second is beyond 2^32 as well) — hashes of the 64-bit linear indices
    and of the fp32 segment lengths equal the oracle's."""
    for dims, n_rays in (((2049, 1024, 1024), 60_000), ((1024, 1024, 4100), 40_000)):
        org, dirs = W.random_rays(n_rays, dims, seed=17)
        g = thor.unit_dda_trace(dims, (0, 0, 0), org, dirs, max_steps=1 << 14)
        o = oracle.dda_trace(dims, (0, 0, 0), org, dirs, max_steps=1 << 14)
        assert np.array_equal(g["count"], o["count"])
        assert np.array_equal(g["hash_idx"], o["hash_idx"]) and np.array_equal(g["hash_len"], o["hash_len"])
    # the grid really is beyond 2^32: a ray in the top slabs visits indices above it
    far = thor.unit_dda_trace((1024, 1024, 4100), (0, 0, 0), np.array([[1000.5, 1000.5, 4097.5]], np.float32),
                              np.array([[0.6, 0.0, 0.8]], np.float32), max_steps=64, want_seq=True)
    assert far["seq_idx"].min() > 2 ** 32


def test_gathers_beyond_2_31_on_a_borrowed_grid(thor):
    """A borrowed 1024 x 1024 x 2304 grid (2.4e9 cells) whose five field pointers alias ONE 9.7 GB device buffer holding an
    index-dependent pattern; everything below happens in the slabs z >= 2048, whose linear indices exceed 2^31:
    (i) thor_raytrace's column density equals sum(buffer[idx] * len) over the index / length sequence of the DDA unit
    trace (itself pinned to the oracle above); (ii) the walk emits from source cells up there with
    V = v_cell . k = buffer[idx] (kx + ky + kz) and crosses exactly the cells the DDA counts."""
    import torch
    nx, ny, nz = 1024, 1024, 2304
    N = nx * ny * nz
    buf = torch.empty(N, dtype=torch.float32, device="cuda")
    step = 1 << 27
    for i0 in range(0, N, step):                              # pattern: 50 + (i mod 977), exact in fp32
        i1 = min(N, i0 + step)
        buf[i0:i1] = (torch.arange(i0, i1, device="cuda", dtype=torch.int64) % 977 + 50).float()
    f = buf.view(nz, ny, nx)
    ctx = thor.Context(nx, ny, nz, 1.0, f, f, f, f, f, None, validate=False)     # cell_cm = 1 cm: transparent
    try:
        org = np.array([[1000.5, 1020.5, 2100.25], [500.25, 900.5, 2200.75], [1023.5, 1023.5, 2303.5]], np.float32)
        dirs = np.array([[0.6, 0.0, 0.8], [0.48, 0.6, 0.64], [-0.8, -0.6, 0.0]], np.float32)
        col = ctx.raytrace(org, dirs)["column"]
        for j in range(3):
            t = thor.unit_dda_trace((nx, ny, nz), (0, 0, 0), org[j:j + 1], dirs[j:j + 1], max_steps=4096, want_seq=True)
            idx = torch.from_numpy(t["seq_idx"]).cuda()
            assert int(idx.min()) > 2 ** 31
            vals = buf[idx].double().cpu().numpy()
            expect = float((vals * t["seq_len"].astype(np.float64)).sum())
            assert abs(col[j] - expect) <= 2e-5 * expect, (j, col[j], expect)
        n = 2000
        src = np.array([[1000.5, 1020.5, 2100.25], [1020.5, 700.5, 2290.5]], np.float32)
        ctx.sources_set(src, np.ones(2, np.float32), np.zeros(2, np.float32))
        ctx.run(n, 5, dict(spec_mode=1, spec_bins=10, spec_lo=-1e4, spec_hi=1e4, raw_output=1))
        raw, c = ctx.raw(), ctx.counters()
        assert c["escaped"] == n and c["scatterings"] == 0
        k = np.stack([raw["kx"], raw["ky"], raw["kz"]], 1)
        lin = (np.floor(src[:, 2]).astype(np.int64) * ny + np.floor(src[:, 1]).astype(np.int64)) * nx + np.floor(src[:, 0]).astype(np.int64)
        assert lin.min() > 2 ** 31
        vcell = (lin % 977 + 50).astype(np.float64)
        ksum = k.astype(np.float64).sum(1)
        which = np.argmin(np.abs(raw["V"][:, None].astype(np.float64) - vcell[None, :] * ksum[:, None]), axis=1)
        assert np.allclose(raw["V"], vcell[which] * ksum, rtol=2e-6, atol=1e-3)
        assert 0.4 < which.mean() < 0.6                          # both sources emit
        cnt = thor.unit_dda_trace((nx, ny, nz), (0, 0, 0), src[which], k, max_steps=1 << 13)["count"]
        assert int(cnt.astype(np.int64).sum()) == c["cell_crossings"]
    finally:
        ctx.close()
        del buf, f
        torch.cuda.empty_cache()


def test_philox_layout_is_curands(thor):
    """S§8(c) P13 / reading A16: the walk's Philox stream for (seed, photon id) is, word for word, what cuRAND's own device
    API gives for curand_init(seed, subsequence = id, offset = 0) + curand4() — across 32-bit boundaries of seed and id."""
    for seed, id0 in ((1, 0), (0xDEADBEEFCAFEF00D, (1 << 32) - 3), ((1 << 64) - 1, (1 << 40) + 17)):
        a = thor.unit_philox(seed, id0, 50, 23)
        b = thor.unit_curand_philox(seed, id0, 50, 23)
        assert np.array_equal(a, b), (seed, id0)
