"""The device-side input generators (paper_2507_11603_b200/workloads_device.py), run here on the CPU at small sizes: they
must realise the recipe of DESIGN.md 3 — unit-variance Gaussian fields with the stated spectral slope, lognormal density with
the stated mean, sources inside the grid and concentrated where the weight is."""
import numpy as np
import torch

from paper_2507_11603_b200 import workloads_device as WD


def _slope(field):
    n = field.shape[0]
    p = np.abs(np.fft.fftn(field)) ** 2
    k = np.sqrt(sum(np.meshgrid(*(np.fft.fftfreq(n) ** 2,) * 3, indexing="ij")))
    sel = (k > 2.0 / n) & (k < 0.25)
    return np.polyfit(np.log(k[sel]), np.log(p[sel]), 1)[0]


def test_gaussian_field_variance_and_slope():
    gen = torch.Generator(device="cpu")
    gen.manual_seed(5)
    for slope in (-3.0, -4.0):
        g = WD.gaussian_field(48, slope, gen, "cpu").numpy()
        assert g.shape == (48, 48, 48) and abs(g.std() - 1.0) < 1e-4 and abs(g.mean()) < 1e-4
        assert abs(_slope(g.astype(np.float64)) - slope) < 0.25          # Rayleigh scatter of |F|^2 biases the log fit a little
    # chunked passes == one 3-D inverse transform of the same coefficients: a tiny chunk size changes nothing
    gen.manual_seed(9)
    a = WD.gaussian_field(16, -3.0, gen, "cpu")
    old = WD._CHUNK_BYTES
    try:
        WD._CHUNK_BYTES = 16 * 9 * 8 * 16                                 # 16 planes per chunk: the same draws
        gen.manual_seed(9)
        b = WD.gaussian_field(16, -3.0, gen, "cpu")
    finally:
        WD._CHUNK_BYTES = old
    assert torch.allclose(a, b, atol=1e-5)


def test_cosmic_web_and_turbulent_box_recipes():
    w = WD.cosmic_web(n=32, n_src=4000, n_photons=10, map_pix=16, device="cpu")
    g = w["grid"]
    opd = g["nHI"].double().numpy() / 1e-6
    assert abs(np.log(opd).std() - 1.5) < 0.02 and abs(np.log(opd).mean() + 1.125) < 0.02     # lognormal, mean 1 in expectation
    assert np.allclose(g["T"].numpy(), 1e4 * opd ** 0.6, rtol=1e-4)
    v2 = sum(float((g[k].double() ** 2).mean()) for k in ("vx", "vy", "vz"))
    assert abs(v2 - 100.0 ** 2) < 1.0                                     # 3-D dispersion 100 km/s
    pos = w["sources"]["pos"]
    assert pos.shape == (4000, 3) and pos.min() >= 0 and pos.max() <= 32
    # sources ∝ (1+delta)^2: the mean weight of source cells is the weight-weighted mean, far above the plain mean
    c = np.minimum(pos.astype(int), 31)
    wsrc = opd[c[:, 2], c[:, 1], c[:, 0]] ** 2
    expect = (opd ** 4).sum() / (opd ** 2).sum()
    assert abs(wsrc.mean() / expect - 1.0) < 0.25 and wsrc.mean() > 5 * (opd ** 2).mean()
    assert abs(w["opts"]["hubble_kms_per_cell"] - 203.6 * 11.2e-3) < 1e-5
    t = WD.turbulent_box(n=32, n_src=500, n_photons=10, peel_pix=8, peel_bins=10, device="cpu")
    ln = np.log(t["grid"]["nHI"].double().numpy())
    assert abs(ln.std() - 2.0) < 0.02 and abs(np.log(t["grid"]["T"].double().numpy()).std() - 0.5) < 0.01
    h = WD.to_host(t)
    assert isinstance(h["grid"]["nHI"], np.ndarray) and t["opts"]["core_skip_mode"] == 2
