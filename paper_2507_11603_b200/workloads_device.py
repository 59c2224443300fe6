"""Seeded synthetic inputs generated ON THE DEVICE (torch), for the grids the numpy generators of workloads.py cannot
reach: BASELINE.json config 5 at its stated 1536^3 (72.5 GB of SoA fp32 fields) and config 4 at 512^3.  Same recipes as
workloads.cosmic_web / workloads.turbulent_box, different random stream (torch's Philox generator instead
of numpy's PCG64), so a grid made here is not cell-for-cell the numpy one of the same seed — both are realisations of the
same recipe.  Harness side only: no method arithmetic, imports neither the binding nor oracle/.

Memory plan at n = 1536 (one field = 14.5 GB): a Gaussian random field is drawn directly in Fourier space (complex white
noise times k^(slope/2), half spectrum: 14.5 GB) and brought back by three passes of 1-D inverse transforms in chunks
(torch.fft on slices of <= ~1 GB), so the peak is two field-sized buffers beside the fields already made — 5 fields +
2 buffers = 102 GB of the B200's 180 GB.  (A single 3-D cuFFT plan of 3.6e9 points would need a workspace of unknown size.)
"""
import math

import numpy as np
import torch

from .workloads import PC_CM

_CHUNK_BYTES = 1 << 30


def gaussian_field(n, slope, gen, device):
    """Unit-variance real Gaussian random field on an n^3 periodic grid with P(k) ∝ k^slope, float32 [n, n, n]."""
    m = n // 2 + 1
    fk = torch.empty((n, n, m), dtype=torch.complex64, device=device)
    kz = torch.fft.rfftfreq(n, device=device)[None, None, :] ** 2
    ky = torch.fft.fftfreq(n, device=device)[None, :, None] ** 2
    kx = torch.fft.fftfreq(n, device=device)
    c0 = max(1, _CHUNK_BYTES // (n * m * 8))
    for i0 in range(0, n, c0):
        i1 = min(n, i0 + c0)
        k2 = kx[i0:i1, None, None] ** 2 + ky + kz
        if i0 == 0:
            k2[0, 0, 0] = 1.0
        amp = k2 ** (slope / 4.0)
        if i0 == 0:
            amp[0, 0, 0] = 0.0
        re = torch.randn((i1 - i0, n, m), dtype=torch.float32, device=device, generator=gen)
        im = torch.randn((i1 - i0, n, m), dtype=torch.float32, device=device, generator=gen)
        fk[i0:i1] = torch.complex(re * amp, im * amp)
        del re, im, amp, k2
    # inverse transform, one axis at a time, in chunks (scaling is irrelevant: the field is normalised below)
    c1 = max(1, _CHUNK_BYTES // (n * m * 8))
    for j0 in range(0, n, c1):                                   # axis 0, chunked over axis 1
        j1 = min(n, j0 + c1)
        fk[:, j0:j1] = torch.fft.ifft(fk[:, j0:j1], dim=0)
    for i0 in range(0, n, c1):                                   # axis 1, chunked over axis 0
        i1 = min(n, i0 + c1)
        fk[i0:i1] = torch.fft.ifft(fk[i0:i1], dim=1)
    out = torch.empty((n, n, n), dtype=torch.float32, device=device)
    for i0 in range(0, n, c1):                                   # axis 2: half spectrum -> real
        i1 = min(n, i0 + c1)
        out[i0:i1] = torch.fft.irfft(fk[i0:i1], n=n, dim=2)
    del fk
    if device != "cpu":
        torch.cuda.empty_cache()
    # unit variance, in chunks and in fp64 (the mean is zero by construction: the k = 0 mode is removed)
    ss = 0.0
    for i0 in range(0, n, c1):
        ss += float((out[i0:min(n, i0 + c1)].double() ** 2).sum())
    out.mul_(1.0 / math.sqrt(ss / n ** 3))
    return out


def _draw_sources(weight_of_slab, n, n_src, gen, device):
    """n_src positions drawn ∝ a per-cell weight without a field-sized CDF: pick the z-slab ∝ its summed weight, then the
    cell inside the slab by that slab's own cumulative sum; uniform inside the cell.  weight_of_slab(z) -> float64 [n, n]."""
    sums = torch.stack([weight_of_slab(z).sum() for z in range(n)])
    cdf = torch.cumsum(sums, 0)
    u = torch.rand(n_src, dtype=torch.float64, device=device, generator=gen) * cdf[-1]
    slab = torch.clamp(torch.searchsorted(cdf, u), max=n - 1)
    order = torch.argsort(slab)
    slab_sorted = slab[order]
    counts = torch.bincount(slab_sorted, minlength=n).cpu().numpy()
    cell = torch.empty(n_src, dtype=torch.int64, device=device)
    start = 0
    for z in np.nonzero(counts)[0]:
        c = int(counts[z])
        wc = torch.cumsum(weight_of_slab(int(z)).reshape(-1), 0)
        uu = torch.rand(c, dtype=torch.float64, device=device, generator=gen) * wc[-1]
        cell[start:start + c] = torch.clamp(torch.searchsorted(wc, uu), max=n * n - 1)
        start += c
    iz = slab_sorted
    iy, ix = cell // n, cell % n
    pos = torch.stack([ix, iy, iz], 1).double() + torch.rand((n_src, 3), dtype=torch.float64, device=device, generator=gen)
    return pos.float().cpu().numpy()


def cosmic_web(n=1536, n_src=1 << 22, n_photons=100_000_000, seed=11, mean_n=1e-6, sigma_ln=1.5, sigma_v3d=100.0,
               cell_kpc=11.2, hubble_kms_per_mpc=203.6, map_pix=2048, bins=1000, v_max=1233.0, device="cuda"):
    """BASELINE.json config 5 (recipe of workloads.cosmic_web): lognormal overdensity (sigma_ln 1.5) on mean n_HI 1e-6,
    T = 1e4 (1+delta)^0.6, Gaussian peculiar velocities (3-D dispersion 100 km/s, k^-4), Hubble drift, sources
    ∝ (1+delta)^2, stop at |V| > 5 Å, surface-brightness map by peel-off along +z.  Fields are torch tensors on `device`."""
    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    g = gaussian_field(n, -3.0, gen, device)
    nHI = g.mul_(sigma_ln).add_(-0.5 * sigma_ln ** 2).exp_()          # 1 + delta, mean 1 (in place: g is gone)
    T = nHI.pow(0.6).mul_(1e4)
    pos = _draw_sources(lambda z: nHI[z].double() ** 2, n, n_src, gen, device)
    nHI.mul_(mean_n)
    s1 = sigma_v3d / math.sqrt(3.0)
    vx, vy, vz = (gaussian_field(n, -4.0, gen, device).mul_(s1) for _ in range(3))
    cell_cm = cell_kpc * 1e3 * PC_CM
    hc = hubble_kms_per_mpc * cell_kpc * 1e-3
    grid = dict(nx=n, ny=n, nz=n, periodic=(0, 0, 0), cell_cm=cell_cm, nHI=nHI, T=T, vx=vx, vy=vy, vz=vz, kdust=None)
    src = dict(pos=pos, lum=np.ones(n_src, np.float32), sigma=np.zeros(n_src, np.float32))
    opts = dict(phase_core=0, phase_wing=0, core_skip_mode=2, spec_mode=1, spec_bins=bins, spec_lo=-v_max, spec_hi=v_max,
                hubble_kms_per_cell=float(np.float32(hc)), hubble_eps=0.25, v_max_kms=v_max,
                peel_on=1, k_obs=(0.0, 0.0, 1.0), peel_nx=map_pix, peel_ny=map_pix, peel_nv=1,
                peel_v_lo=-1e30, peel_v_hi=1e30, peel_width_cells=float(n), tau_peel_max=30.0)
    return dict(name=f"cosmic_web_n{n}", grid=grid, sources=src, opts=opts, n_photons=n_photons, seed=1)


def turbulent_box(n=512, n_src=1 << 20, n_photons=10_000_000, seed=7, mean_n=1e-2, sigma_ln_n=2.0, sigma_ln_T=0.5,
                  sigma_v3d=50.0, cell_pc=10.0, peel_pix=256, peel_bins=400, v_range=1500.0, device="cuda"):
    """BASELINE.json config 4 (recipe of workloads.turbulent_box) at its stated 512^3: lognormal n_HI (mean 1e-2,
    sigma_ln 2) and T (about 1e4 K, sigma_ln 0.5) on k^-3 fields, Gaussian k^-4 velocities with 3-D dispersion 50 km/s,
    sources ∝ n_HI^2, local core-skipping, peel-off along +z into a 256 x 256 x 400 cube."""
    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    nHI = gaussian_field(n, -3.0, gen, device).mul_(sigma_ln_n).add_(math.log(mean_n) - 0.5 * sigma_ln_n ** 2).exp_()
    T = gaussian_field(n, -3.0, gen, device).mul_(sigma_ln_T).add_(math.log(1e4)).exp_()
    s1 = sigma_v3d / math.sqrt(3.0)
    vx, vy, vz = (gaussian_field(n, -4.0, gen, device).mul_(s1) for _ in range(3))
    pos = _draw_sources(lambda z: nHI[z].double() ** 2, n, n_src, gen, device)
    grid = dict(nx=n, ny=n, nz=n, periodic=(0, 0, 0), cell_cm=cell_pc * PC_CM, nHI=nHI, T=T, vx=vx, vy=vy, vz=vz, kdust=None)
    src = dict(pos=pos, lum=np.ones(n_src, np.float32), sigma=np.zeros(n_src, np.float32))
    opts = dict(phase_core=0, phase_wing=0, core_skip_mode=2, spec_mode=1, spec_bins=400, spec_lo=-v_range,
                spec_hi=v_range, peel_on=1, k_obs=(0.0, 0.0, 1.0), peel_nx=peel_pix, peel_ny=peel_pix,
                peel_nv=peel_bins, peel_v_lo=-v_range, peel_v_hi=v_range, peel_width_cells=float(n),
                tau_peel_max=30.0)
    return dict(name=f"turbulent_box_n{n}", grid=grid, sources=src, opts=opts, n_photons=n_photons, seed=1)


def to_host(w):
    """The same workload with numpy fields (for the oracle); only for grids that fit host memory."""
    g = dict(w["grid"])
    for k in ("nHI", "T", "vx", "vy", "vz", "kdust"):
        if g.get(k) is not None:
            g[k] = g[k].cpu().numpy()
    return dict(w, grid=g)
