"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 1-5; recipe in DESIGN.md §Inputs).

This module serves BOTH the CUDA path and the oracle and therefore holds none of the method's arithmetic: it only
fills float32 arrays (grid fields, source lists) and option dictionaries from recipe numbers.  It imports neither
the binding nor oracle/.  The two recipe constants below are plain numbers of the recipe (they decide how dense the
synthetic gas is), not something either implementation reads.

Grid dict:    nx, ny, nz, periodic (px,py,pz), cell_cm, nHI, T, vx, vy, vz, kdust|None  — float32 [nz, ny, nx]
Sources dict: pos float32 [n,3] (cell units), lum float32 [n], sigma float32 [n] (km/s)
Opts dict:    keys of thor_opts (include/thor.h)
"""
import math

import numpy as np

PC_CM = 3.0857e18
# Recipe constant: Lyα line-centre cross-section at 1e4 K used to turn a requested tau_0 into a density.
RECIPE_SIGMA0_T4 = 5.8981e-14      # cm^2, scales as T4^-1/2
RECIPE_VTH_T4 = 12.845             # km/s, scales as T4^+1/2
RECIPE_A_T4 = 4.7184e-4            # Voigt parameter at 1e4 K, scales as T4^-1/2


def _recipe_sigma0(T):
    return RECIPE_SIGMA0_T4 / math.sqrt(T / 1e4)


def _cell_centres(n):
    z, y, x = np.meshgrid(np.arange(n[2]) + 0.5, np.arange(n[1]) + 0.5, np.arange(n[0]) + 0.5, indexing="ij")
    return x, y, z


def static_sphere(n=32, tau0=1e5, T=10.0, n_photons=1000, bins=200, x_range=60.0):
    """Config 1 (Dijkstra test): n^3 grid, sphere of radius n/2 cells of uniform n_HI with line-centre optical depth
    tau0 centre-to-edge, temperature T, no motion, no dust, central source at line centre, isotropic scattering."""
    R = n / 2.0
    x, y, z = _cell_centres((n, n, n))
    r = np.sqrt((x - R) ** 2 + (y - R) ** 2 + (z - R) ** 2)
    inside = r < R
    cell_cm = PC_CM
    dens = tau0 / (_recipe_sigma0(T) * R * cell_cm)
    grid = dict(nx=n, ny=n, nz=n, periodic=(0, 0, 0), cell_cm=cell_cm,
                nHI=np.where(inside, dens, 0.0).astype(np.float32),
                T=np.full((n, n, n), T, np.float32),
                vx=np.zeros((n, n, n), np.float32), vy=np.zeros((n, n, n), np.float32),
                vz=np.zeros((n, n, n), np.float32), kdust=None)
    src = dict(pos=np.array([[R, R, R]], np.float32), lum=np.ones(1, np.float32), sigma=np.zeros(1, np.float32))
    opts = dict(phase_core=0, phase_wing=0, spec_mode=0, spec_T_ref=T, spec_bins=bins, spec_lo=-x_range,
                spec_hi=x_range)
    return dict(name=f"static_sphere_n{n}_tau{tau0:g}_T{T:g}", grid=grid, sources=src, opts=opts,
                n_photons=n_photons, seed=1)


def expanding_shell(n=128, N_HI=1e20, T=1e4, v_exp=200.0, tau_d=1.0, sigma_src=50.0, n_photons=1_000_000,
                    bins=400, v_range=1500.0, inner=0.8):
    """Config 2: n^3 grid, shell between inner*R and R (R = n/2 cells) with radial column N_HI, temperature T,
    radial outflow v_exp, dust ABSORPTION depth tau_d radially through the shell; empty elsewhere; central source
    with Gaussian line of width sigma_src."""
    R = n / 2.0
    x, y, z = _cell_centres((n, n, n))
    dx, dy, dz = x - R, y - R, z - R
    r = np.sqrt(dx * dx + dy * dy + dz * dz)
    shell = (r > inner * R) & (r <= R)
    cell_cm = PC_CM
    thick_cm = (1.0 - inner) * R * cell_cm
    dens = N_HI / thick_cm
    kd = tau_d / thick_cm
    rs = np.maximum(r, 1e-30)
    f32 = lambda a: np.ascontiguousarray(a, np.float32)
    grid = dict(nx=n, ny=n, nz=n, periodic=(0, 0, 0), cell_cm=cell_cm,
                nHI=f32(np.where(shell, dens, 0.0)), T=f32(np.full_like(r, T)),
                vx=f32(np.where(shell, v_exp * dx / rs, 0.0)), vy=f32(np.where(shell, v_exp * dy / rs, 0.0)),
                vz=f32(np.where(shell, v_exp * dz / rs, 0.0)), kdust=f32(np.where(shell, kd, 0.0)))
    src = dict(pos=np.array([[R, R, R]], np.float32), lum=np.ones(1, np.float32),
               sigma=np.full(1, sigma_src, np.float32))
    opts = dict(phase_core=0, phase_wing=0, spec_mode=1, spec_bins=bins, spec_lo=-v_range, spec_hi=v_range)
    return dict(name=f"expanding_shell_n{n}", grid=grid, sources=src, opts=opts, n_photons=n_photons, seed=1)


def static_slab(nz=256, tau0=1e7, T=1e4, core_skip=True, n_photons=1_000_000, bins=400, x_range=80.0,
                tau_d=0.0, phase_core=1, phase_wing=0):
    """Config 3 (Neufeld test): 1 x 1 x nz cells, periodic in x and y, line-centre optical depth tau0 from the
    midplane to either face, source at line centre in the midplane; dipole phase function in the core and isotropic
    in the wings (as BASELINE.json states it); x_crit = 0.2 (a tau0)^(1/3) core-skipping when a tau0 >= 1."""
    half = nz / 2.0
    cell_cm = PC_CM
    dens = tau0 / (_recipe_sigma0(T) * half * cell_cm)
    shape = (nz, 1, 1)
    kd = None
    if tau_d > 0:
        kd = np.full(shape, tau_d / (half * cell_cm), np.float32)
    grid = dict(nx=1, ny=1, nz=nz, periodic=(1, 1, 0), cell_cm=cell_cm,
                nHI=np.full(shape, dens, np.float32), T=np.full(shape, T, np.float32),
                vx=np.zeros(shape, np.float32), vy=np.zeros(shape, np.float32), vz=np.zeros(shape, np.float32),
                kdust=kd)
    src = dict(pos=np.array([[0.5, 0.5, half]], np.float32), lum=np.ones(1, np.float32),
               sigma=np.zeros(1, np.float32))
    a_tau0 = RECIPE_A_T4 / math.sqrt(T / 1e4) * tau0
    x_crit = 0.2 * a_tau0 ** (1.0 / 3.0) if (core_skip and a_tau0 >= 1.0) else 0.0
    opts = dict(phase_core=phase_core, phase_wing=phase_wing, core_skip_mode=1 if x_crit > 0 else 0,
                x_crit=float(np.float32(x_crit)), spec_mode=0, spec_T_ref=T, spec_bins=bins, spec_lo=-x_range,
                spec_hi=x_range)
    return dict(name=f"static_slab_nz{nz}_tau{tau0:g}", grid=grid, sources=src, opts=opts, n_photons=n_photons,
                seed=1)


def _gaussian_field(rng, n, slope):
    """Unit-variance Gaussian random field with power spectrum P(k) ∝ k^slope on an n^3 periodic grid (numpy FFT)."""
    white = rng.standard_normal((n, n, n)).astype(np.float32)
    fk = np.fft.rfftn(white)
    kx = np.fft.fftfreq(n)[:, None, None]
    ky = np.fft.fftfreq(n)[None, :, None]
    kz = np.fft.rfftfreq(n)[None, None, :]
    k2 = kx * kx + ky * ky + kz * kz
    k2[0, 0, 0] = 1.0
    amp = k2 ** (slope / 4.0)
    amp[0, 0, 0] = 0.0
    out = np.fft.irfftn(fk * amp, s=(n, n, n)).astype(np.float32)
    out /= out.std()
    return out


def turbulent_box(n=64, n_src=4096, n_photons=10_000, seed=7, mean_n=1e-2, sigma_ln_n=2.0, sigma_ln_T=0.5,
                  sigma_v3d=50.0, cell_pc=10.0, peel_pix=64, peel_bins=100, v_range=1500.0):
    """Config 4 at size n (512 in BASELINE.json): lognormal n_HI (mean mean_n, sigma_ln 2), lognormal T about 1e4 K
    (sigma_ln 0.5), Gaussian velocity field with 3-D dispersion 50 km/s and k^-4 spectrum, sources drawn ∝ n_HI^2
    placed uniformly inside their cells, local core-skipping, peel-off along +z to a cube."""
    rng = np.random.default_rng(seed)
    g1 = _gaussian_field(rng, n, -3.0)
    g2 = _gaussian_field(rng, n, -3.0)
    nHI = np.exp(np.log(mean_n) - 0.5 * sigma_ln_n ** 2 + sigma_ln_n * g1).astype(np.float32)
    T = np.exp(np.log(1e4) + sigma_ln_T * g2).astype(np.float32)
    s1 = sigma_v3d / math.sqrt(3.0)
    vx, vy, vz = (np.ascontiguousarray(s1 * _gaussian_field(rng, n, -4.0), np.float32) for _ in range(3))
    w = nHI.astype(np.float64).ravel() ** 2
    cdf = np.cumsum(w)
    pick = np.searchsorted(cdf, rng.random(n_src) * cdf[-1])
    pick = np.minimum(pick, w.size - 1)
    iz, iy, ix = np.unravel_index(pick, nHI.shape)
    pos = np.stack([ix, iy, iz], 1).astype(np.float64) + rng.random((n_src, 3))
    grid = dict(nx=n, ny=n, nz=n, periodic=(0, 0, 0), cell_cm=cell_pc * PC_CM, nHI=nHI, T=T, vx=vx, vy=vy, vz=vz,
                kdust=None)
    src = dict(pos=pos.astype(np.float32), lum=np.ones(n_src, np.float32), sigma=np.zeros(n_src, np.float32))
    opts = dict(phase_core=0, phase_wing=0, core_skip_mode=2, spec_mode=1, spec_bins=400, spec_lo=-v_range,
                spec_hi=v_range, peel_on=1, k_obs=(0.0, 0.0, 1.0), peel_nx=peel_pix, peel_ny=peel_pix,
                peel_nv=peel_bins, peel_v_lo=-v_range, peel_v_hi=v_range, peel_width_cells=float(n),
                tau_peel_max=30.0)
    return dict(name=f"turbulent_box_n{n}", grid=grid, sources=src, opts=opts, n_photons=n_photons, seed=1)


def cosmic_web(n=64, n_src=4096, n_photons=10_000, seed=11, mean_n=1e-6, sigma_ln=1.5, sigma_v3d=100.0,
               cell_kpc=11.2, hubble_kms_per_mpc=203.6, map_pix=128, bins=1000, v_max=1233.0):
    """Config 5 at size n (1536 in BASELINE.json): lognormal overdensity (sigma_ln 1.5) on mean n_HI = 1e-6,
    T = 1e4 (1+delta)^0.6, Hubble flow as a frequency drift plus Gaussian peculiar velocities (3-D dispersion
    100 km/s, k^-4), sources ∝ (1+delta)^2, stop at |V| > v_max (5 Å), surface-brightness map by peel-off along +z,
    local core-skipping as in the paper's simulation runs (reading A28)."""
    rng = np.random.default_rng(seed)
    g = _gaussian_field(rng, n, -3.0)
    opd = np.exp(-0.5 * sigma_ln ** 2 + sigma_ln * g)              # 1 + delta, mean 1
    nHI = (mean_n * opd).astype(np.float32)
    T = (1e4 * opd ** 0.6).astype(np.float32)
    s1 = sigma_v3d / math.sqrt(3.0)
    vx, vy, vz = (np.ascontiguousarray(s1 * _gaussian_field(rng, n, -4.0), np.float32) for _ in range(3))
    w = opd.astype(np.float64).ravel() ** 2
    cdf = np.cumsum(w)
    pick = np.minimum(np.searchsorted(cdf, rng.random(n_src) * cdf[-1]), w.size - 1)
    iz, iy, ix = np.unravel_index(pick, nHI.shape)
    pos = np.stack([ix, iy, iz], 1).astype(np.float64) + rng.random((n_src, 3))
    cell_cm = cell_kpc * 1e3 * PC_CM
    hc = hubble_kms_per_mpc * cell_kpc * 1e-3
    grid = dict(nx=n, ny=n, nz=n, periodic=(0, 0, 0), cell_cm=cell_cm, nHI=nHI, T=T, vx=vx, vy=vy, vz=vz, kdust=None)
    src = dict(pos=pos.astype(np.float32), lum=np.ones(n_src, np.float32), sigma=np.zeros(n_src, np.float32))
    opts = dict(phase_core=0, phase_wing=0, core_skip_mode=2, spec_mode=1, spec_bins=bins, spec_lo=-v_max, spec_hi=v_max,
                hubble_kms_per_cell=float(np.float32(hc)), hubble_eps=0.25, v_max_kms=v_max,
                peel_on=1, k_obs=(0.0, 0.0, 1.0), peel_nx=map_pix, peel_ny=map_pix, peel_nv=1,
                peel_v_lo=-1e30, peel_v_hi=1e30, peel_width_cells=float(n), tau_peel_max=30.0)
    return dict(name=f"cosmic_web_n{n}", grid=grid, sources=src, opts=opts, n_photons=n_photons, seed=1)


def random_rays(n_rays, dims, seed=3):
    """Ray origins uniform in the grid and isotropic unit directions, float32, for the DDA parity test
    (BASELINE.json: 'bit-exact on 1e6 random rays')."""
    rng = np.random.default_rng(seed)
    org = (rng.random((n_rays, 3)) * np.asarray(dims, np.float64)).astype(np.float32)
    org = np.minimum(org, np.nextafter(np.asarray(dims, np.float32), np.float32(0)))
    mu = 2.0 * rng.random(n_rays) - 1.0
    phi = 2.0 * math.pi * rng.random(n_rays)
    st = np.sqrt(1.0 - mu * mu)
    dirs = np.stack([st * np.cos(phi), st * np.sin(phi), mu], 1).astype(np.float32)
    return org, dirs
