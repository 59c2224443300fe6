"""bench.py — throughput of the Lyα random walk (the whole hot path, DESIGN.md §1 rows a1-a14) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload web1536|web512|turb512|shell|sphere|slab|gather|project|render]
                    [--impl reference] [--no-subs]

A "step" is one thor_run over one batch of packets.  The headline workload is BASELINE.json's largest single-GPU
configuration, configs[4]: the 1536^3 cosmic web (72.5 GB of SoA fp32 fields generated on the device, borrowed by the
library), with Hubble drift, termination at 5 Å and a 2048^2 surface-brightness map by peel-off; each step walks a STATED
subsample of the config's 1e8 packets (config.n_photons_per_step_per_gpu of config.n_photons_subsample_of).  value =
scatterings/s over the timed steps (whole job, all ranks), with packets/s and cell crossings/s beside it; inputs are
resident in HBM when the timed region starts.  Steps are independent batches: up to --in-flight of them (default 3) run at
once, each in a context, stream and host thread of its own on the shared resident grid, so that the tail of one step (a few
long packets) overlaps the feed phase of the next; ms_per_step = timed region / steps, serial_ms_per_step = the
warm-up steps, which run one at a time.  `e2e` is the same metric through the C-ABI with HOST buffers for what a
step takes in and gives back (the source list in, the tallies out; the 72.5 GB grid is the resident dataset).  `roofline` is the
issue-slot ("alu") roofline of the walk kernel, `roofline_hbm` the cell-gather bandwidth beside it;
`workloads` holds the other configurations measured in the same run (configs[1], [2], [3] at 512^3, the scaled configs[0],
the gather regime), a few steps each; `cpu_baseline` is the fp64 oracle timed on this box's host cores.

N > 1 (torchrun): the path shards by photon id: every rank walks its own id range of the same size on its
own replica of the grid (weak scaling), and the tallies are summed with one NCCL all-reduce.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

from paper_2507_11603_b200 import workloads as W

# Issue-slot roofline constants: algorithmic thread-instructions per unit of work, SURVEY.md §8(d)'s a-priori budgets
# (~600 per scattering, ~60 per cell crossing) — fixed numbers that do not come from this kernel, so a slower or fatter
# kernel cannot raise its own fraction.  What the kernel actually executes per unit is in profiles/r02_*.md.
INST_PER_SCATTERING = 600.0
INST_PER_CROSSING = 60.0
SCHEDULERS_PER_SM, LANES = 4, 32
BYTES_PER_CROSSING = 20.0                              # n_HI, T, v_x, v_y, v_z (24 with dust)
# dram__bytes_read.sum + dram__bytes_write.sum of walk_kernel per launch at the default packet counts, from the ncu
# captures summarised under profiles/ (bench.py cannot measure this itself); None = no capture of that workload
TRAFFIC = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))) if os.path.exists(os.path.join(ROOT, "profiles", "traffic.json")) else {}

HEADLINE = "web1536"
SUBS = ["shell", "sphere", "slab", "slab_paper", "gather", "turb512"]


def make_workload(name, n_photons=None, device="cuda"):
    """name -> (workload dict, pack flag, note).  Device-generated grids hold CUDA tensors, the others numpy arrays."""
    pack, note = False, None
    if name == "web1536":    # BASELINE.json configs[4] as stated; a stated subsample of its 1e8 packets per step
        from paper_2507_11603_b200 import workloads_device as WD
        w = WD.cosmic_web(n=1536, n_src=1 << 22, n_photons=400_000, map_pix=2048, device=device)
        note = dict(n_photons_subsample_of=100_000_000)
    elif name == "web512":   # configs[4]'s recipe at 512^3
        from paper_2507_11603_b200 import workloads_device as WD
        w = WD.cosmic_web(n=512, n_src=1 << 18, n_photons=400_000, map_pix=2048, device=device)
        note = dict(n_photons_subsample_of=100_000_000, reduced_grid_of=1536)
    elif name == "turb512":  # configs[3] as stated (512^3, 256 x 256 x 400 cube); a stated subsample of its 1e7 packets,
        # each capped at 1e5 scatterings (the densest source cells have tau_0 > 1e7 per cell: DESIGN.md 5)
        from paper_2507_11603_b200 import workloads_device as WD
        w = WD.turbulent_box(n=512, n_src=1 << 20, n_photons=100_000, device=device)
        w["opts"]["max_scatter"] = 100_000
        note = dict(n_photons_subsample_of=10_000_000, max_scatter=100_000)
    elif name == "shell":    # configs[1] as stated
        w = W.expanding_shell(n=128, n_photons=1_000_000)
    elif name == "sphere":   # configs[0] scaled to fill the GPU (same physics, more packets), tau0 = 1e4
        w = W.static_sphere(n=32, tau0=1e4, T=10.0, n_photons=1_000_000)
        note = dict(scaled_from="configs[0]: tau0 1e5 -> 1e4, 1e3 -> 1e6 packets")
    elif name == "slab":     # configs[2] as stated
        w = W.static_slab(n_photons=1_000_000)
    elif name == "neufeld":  # the paper's own benchmark problem (Table 2): homogeneous static sphere, tau0 = 1e6,
        # T = 2e4 K, 2e5 packets injected at line centre, no core-skipping — on the gridless dataset the paper uses
        T, tau0 = 2e4, 1e6
        w = dict(name="neufeld_sphere_gridless_tau1e6", n_photons=200_000, seed=1,
                 dataset=dict(geometry=0, r_in=0.0, r_out=1.0, length_cm=W.PC_CM, T=T,
                              n0=tau0 / (W.RECIPE_SIGMA0_T4 / (T / 1e4) ** 0.5 * W.PC_CM)),
                 sources=dict(pos=np.zeros((1, 3), np.float32), lum=np.ones(1, np.float32), sigma=np.zeros(1, np.float32)),
                 opts=dict(phase_core=0, phase_wing=0, spec_mode=0, spec_T_ref=T, spec_bins=400, spec_lo=-60.0, spec_hi=60.0))
    elif name == "slab_paper":  # configs[2] with the PAPER's phase functions (1/3-2/3 mix in the core, dipole in the wings)
        w = W.static_slab(n_photons=1_000_000, phase_core=2, phase_wing=1)
        w["name"] += "_paper_phases"
        note = dict(phase_assignment="PAPER.md:132 (mix core / dipole wing) instead of BASELINE.json's dipole core / isotropic wing")
    elif name == "gather":   # the cell-gather regime: configs[4]'s recipe at 512^3 made optically thin (mean n_HI 1e-11), so
        # packets stream through ~340 cells each and the walk is bound by the HBM gathers, not by scatterings
        w = W.cosmic_web(n=512, n_src=1 << 16, n_photons=4_000_000, map_pix=2048, mean_n=1e-11)
        w["opts"].update(peel_on=0, v_max_kms=0.0)
        w["name"] = "cosmic_web_n512_thin_gather"
        pack = True
    else:
        raise SystemExit(f"unknown workload {name}")
    if n_photons:
        w["n_photons"] = int(n_photons)
    return w, pack, note


def oracle_workload(name):
    """What the oracle walks for `name`: the same workload, except where its grid cannot exist on the host — there the
    same recipe at 128^3 (numpy generator), which the `sample` text says."""
    if name in ("web1536", "web512"):
        w = W.cosmic_web(n=128, n_src=1 << 14, n_photons=1 << 20, map_pix=2048)
        return w, "the same recipe at 128^3 (the 1536^3 grid cannot be held in host arrays for the oracle)"
    if name == "turb512":
        w = W.turbulent_box(n=128, n_src=1 << 14, n_photons=1 << 20, peel_pix=256, peel_bins=400)
        w["opts"]["max_scatter"] = 100_000
        return w, "the same recipe at 128^3"
    w, _, _ = make_workload(name)
    return w, "the same workload and seed"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML every 100 ms while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz, self._stop_evt = index, [], set(), None, threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap", nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            self._stop_evt.wait(0.1)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return dict(sm_mhz=med, sm_max_mhz=self.max_mhz, reasons=sorted(self.reasons), samples=len(self.samples))


def _oracle_worker(args):
    """One host process of the timed oracle: walks photon ids [first, first + k chunk) of the workload, chunk by chunk,
    until budget_s seconds of walking are spent.  Returns (scatterings, packets, crossings, seconds walked)."""
    name, first, stride, budget_s, chunk = args
    from oracle import thor_oracle
    w, _ = oracle_workload(name)
    scat = pk = cross = 0
    secs = 0.0
    off = first
    while secs < budget_s:
        o = dict(w["opts"], photon_id_offset=off)
        if "dataset" in w:
            r = thor_oracle.run_gridless(w["dataset"], w["sources"], o, chunk, w["seed"], want_raw=False)
        else:
            r = thor_oracle.run(w["grid"], w["sources"], o, chunk, w["seed"], want_raw=False)
        secs += r["seconds"]
        scat += r["counters"]["scatterings"]
        cross += r["counters"]["cell_crossings"]
        pk += chunk
        off += stride
    return scat, pk, cross, secs


def oracle_timed(name, budget_s, chunk, procs):
    """The oracle, as it stands, on `procs` host processes over disjoint photon-id ranges (valid because the RNG is keyed
    on photon id): process p walks ids [p chunk, (p+1) chunk), [(p + procs) chunk, ...), ...  Aggregate rate =
    total scatterings / the longest process's walking time."""
    from oracle import thor_oracle
    thor_oracle.build()
    jobs = [(name, p * chunk, procs * chunk, budget_s, chunk) for p in range(procs)]
    if procs == 1:
        res = [_oracle_worker(jobs[0])]
    else:
        import multiprocessing as mp
        with mp.get_context("spawn").Pool(procs) as pool:
            res = pool.map(_oracle_worker, jobs)
    scat = sum(r[0] for r in res)
    pk = sum(r[1] for r in res)
    secs = max(r[3] for r in res)
    return scat, pk, secs


def host_cores():
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


def cpu_baseline(name, budget_s, chunk):
    """cpu_baseline object: the oracle single-threaded (its definition) and on all P host cores, on a bounded sample."""
    _, what = oracle_workload(name)
    P = host_cores()
    s1, p1, t1 = oracle_timed(name, budget_s, chunk, 1)
    out = {"value": s1 / t1, "unit": "scatterings/s", "cores": 1, "kind": "oracle", "packets_per_sec": p1 / t1,
           "sample": f"photon ids [0, {p1}) of {what}, single thread, fp64, {t1:.1f} s"}
    if P > 1:
        sP, pP, tP = oracle_timed(name, budget_s, chunk, P)
        out["all_cores"] = {"value": sP / tP, "unit": "scatterings/s", "cores": P, "packets_per_sec": pP / tP,
                            "sample": f"{pP} packets of {what} in {P} processes over disjoint id ranges, fp64, {tP:.1f} s each"}
    return out


def run_reference(args):
    """--impl reference: the oracle, as it stands, on all of the box's host cores, same config / metric / unit; each step
    a bounded sample of the workload (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    name = args.workload
    w, what = oracle_workload(name)
    P = host_cores()
    chunk = max(1, args.ref_chunk)
    for _ in range(min(args.warmup, 1)):
        oracle_timed(name, 0.0, max(1, chunk // 10), 1)
    scat = pk = 0
    secs = 0.0
    for _ in range(args.steps):
        s, p, t = oracle_timed(name, args.ref_budget, chunk, P)
        scat += s
        pk += p
        secs += t
    v = scat / secs
    sample = f"{pk // args.steps} packets of {what} per step x {args.steps} steps, {P} processes over disjoint id ranges, fp64"
    print(json.dumps({
        "impl": "reference", "metric": "lya_scatterings_per_sec", "value": v, "unit": "scatterings/s",
        "packets_per_sec": pk / secs, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(name), "oracle_grid": w["name"], "n_photons_per_step": pk // args.steps},
        "cpu_baseline": {"value": v, "unit": "scatterings/s", "cores": P, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "scatterings/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def workload_label(name):
    return {"web1536": "cosmic_web_n1536", "web512": "cosmic_web_n512", "turb512": "turbulent_box_n512",
            "shell": "expanding_shell_n128", "sphere": "static_sphere_n32_tau10000_T10", "slab": "static_slab_nz256_tau1e+07", "neufeld": "neufeld_sphere_gridless_tau1e6", "slab_paper": "static_slab_nz256_tau1e+07_paper_phases",
            "gather": "cosmic_web_n512_thin_gather"}.get(name, name)

def run_operators(args):
    """--workload project|render: one step = one 2048^2 image through the 512^3 cosmic-web fields (config 5's recipe at
    512^3) with thor_raytrace (column density, PAPER.md 3.5.1) or thor_volume_render (Eq. 12), oblique parallel rays
    from the z = 0 face.  The NEXT-row operators at the same measurement bar as the walk."""
    import ctypes as C
    import torch
    import torch.distributed as dist
    from paper_2507_11603_b200.csrc import build as cuda_build
    rank, local, world = (int(os.environ.get(k, "0")) for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"))
    world = max(world, 1)
    if rank == 0:
        cuda_build.build()
    from paper_2507_11603_b200 import thor
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()
    L = thor.lib()
    n, pix = 512, 2048
    w = W.cosmic_web(n=n, n_src=16, n_photons=1, mean_n=1e-9, map_pix=8)
    pack = bool(args.pack) if args.pack >= 0 else True
    ctx = thor.Context.from_workload(w["grid"], pack=pack)
    xs = (np.arange(pix) + 0.5) * (n / pix)
    gx, gy = np.meshgrid(xs, xs)
    org = np.stack([gx.ravel(), gy.ravel(), np.zeros(gx.size)], 1).astype(np.float32)
    k = np.array([0.35, 0.25, 0.9]) / np.linalg.norm([0.35, 0.25, 0.9])
    dirs = np.tile(k.astype(np.float32), (gx.size, 1))
    # cells per ray from the slab exit point: 1 + face crossings on each axis (host arithmetic, not the kernel's)
    o64, k64 = org.astype(np.float64), dirs[0].astype(np.float64)
    t_exit = np.min(np.where(k64 > 0, (n - o64) / k64, np.inf), axis=1)
    crossings = int((1 + np.abs(np.floor(np.minimum(o64 + t_exit[:, None] * k64, n - 1e-9)) - np.floor(o64)).sum(1)).sum())
    peaks = np.array([[3.1, 0.15, 0.1, 0.3, 1.0, 0.016], [3.8, 0.2, 1.0, 0.6, 0.1, 0.01], [4.3, 0.1, 1.0, 0.1, 0.1, 0.024]],
                     np.float32)                      # three Gaussian peaks in log10 T
    render = args.workload == "render"
    n_rays = org.shape[0]
    h_org, h_dir = torch.from_numpy(org).pin_memory(), torch.from_numpy(dirs).pin_memory()
    d_org, d_dir = h_org.cuda(), h_dir.cuda()
    out = torch.empty((n_rays, 4 if render else 1), dtype=torch.float32, device="cuda")
    h_out = torch.empty(out.shape, dtype=torch.float32).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def launch(o, d):
        if render:
            st = L.thor_volume_render(ctx._ctx, n_rays, C.c_void_p(o.data_ptr()), C.c_void_p(d.data_ptr()), len(peaks),
                                      peaks.ctypes.data_as(C.c_void_p), 0.0, C.c_void_p(out.data_ptr()))
        else:
            st = L.thor_raytrace(ctx._ctx, n_rays, C.c_void_p(o.data_ptr()), C.c_void_p(d.data_ptr()), 0.0, 0, 0.0, 1.0,
                                 C.c_void_p(out.data_ptr()), None, None)
        assert st == 0, thor.lib().thor_last_error(ctx._ctx)

    def timed(fn, steps):
        ms = []
        for _ in range(steps):
            flush.zero_()
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        return ms

    def e2e_step():
        # the C-ABI call with HOST buffers: the library copies rays in and the image out inside the call
        ho, hd, hout = (C.c_void_p(t.data_ptr()) for t in (h_org, h_dir, h_out))
        if render:
            st = L.thor_volume_render_ex(ctx._ctx, n_rays, ho, hd, len(peaks), peaks.ctypes.data_as(C.c_void_p), 0.0, hout, thor.RAYS_HOST)
        else:
            ro = thor.RayOpts(struct_size=C.sizeof(thor.RayOpts), flags=thor.RAYS_HOST)
            st = L.thor_raytrace_ex(ctx._ctx, n_rays, ho, hd, C.byref(ro), hout, None, None)
        assert st == 0, thor.lib().thor_last_error(ctx._ctx)

    timed(lambda: launch(d_org, d_dir), max(args.warmup, 3))
    sampler = ClockSampler(local)
    sampler.start()
    ms = timed(lambda: launch(d_org, d_dir), args.steps)
    clocks = sampler.stop()
    ms_e2e = timed(e2e_step, args.steps)
    tot = torch.tensor([sum(ms), sum(ms_e2e)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(tot, op=dist.ReduceOp.MAX)
    t, t_e2e = (float(x) * 1e-3 for x in tot)
    if rank != 0:
        return
    I_C = 80.0                                         # thread-instructions per cell crossing: DDA 45, gather 10, accumulate ~25
    peak = 148 * 4 * 32 * (clocks["sm_max_mhz"] or 1965) * 1e-3
    val = crossings * args.steps * world / t
    line = {"metric": "ray_cell_crossings_per_sec", "value": val, "unit": "cell crossings/s", "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": t * 1e3 / args.steps,
            "images_per_sec": args.steps * world / t, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{args.workload}_web512_2048sq", "grid": [n, n, n], "rays": n_rays,
                       "crossings_per_image": crossings, "direction": [float(x) for x in k],
                       "layout": "packed 32 B/cell" if pack else "SoA fp32", "parallelism": f"one image per rank x{world}",
                       "l2": "flushed between timed iterations (256 MB memset)"},
            "clocks": clocks, "gpu_launches": args.steps,
            "e2e": {"value": crossings * args.steps * world / t_e2e, "unit": "cell crossings/s",
                    "h2d_bytes_per_step": int(h_org.numel() * 4 + h_dir.numel() * 4), "d2h_bytes_per_step": int(h_out.numel() * 4)},
            "roofline": {"bound": "alu", "achieved": I_C * val * 1e-9, "peak": peak, "unit": "G thread-inst/s",
                         "frac": I_C * val * 1e-9 / peak,
                         "traffic": {"render": 3.53e9, "project": 3.16e9}[args.workload] if pack else None,
                         "traffic_source": "ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, profiles/r01_ray_operators_ncu.md",
                         "kernel": "volume_render_kernel" if render else "raytrace_kernel",
                         "kernel_ms_per_launch": t * 1e3 / args.steps,
                         "peak_source": "148 SMs x 4 schedulers x 32 lanes x clocks.max.sm, derived in DESIGN.md 5",
                         "hbm_GBs_algorithmic": (8 if render else 4) * n ** 3 / (t / args.steps) * 1e-9},
            "cpu_baseline": None}
    if not args.no_cpu_baseline:
        from oracle import thor_oracle as orc          # the timed CPU baseline: the oracle on a bounded sample of the rays
        orc.build()
        sel = np.random.default_rng(0).choice(n_rays, 2000, replace=False)
        t0 = time.perf_counter()
        if render:
            orc.volume_render(w["grid"], org[sel], dirs[sel], peaks)
        else:
            orc.raytrace(w["grid"], org[sel], dirs[sel])
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": crossings * (len(sel) / n_rays) / dt, "unit": "cell crossings/s", "cores": 1,
                                "kind": "oracle", "sample": f"2000 of the {n_rays} rays, single thread, fp64, {dt:.1f} s"}
    print(json.dumps(line))



def measure_walk(args, name, steps, warmup, rank, local, world, n_photons=0, sample_clocks=False, want_e2e=False):
    """Builds workload `name`, runs warmup + steps thor_run calls (L2 flushed between timed iterations), returns the result
    object of that workload (value, ms_per_step, counters, phases, rooflines, optional e2e).  Collective under torchrun."""
    import torch
    import torch.distributed as dist
    from paper_2507_11603_b200 import shard, thor
    w, pack, note = make_workload(name, n_photons)
    if args.pack >= 0:
        pack = bool(args.pack)
    n = w["n_photons"]
    opts = dict(w["opts"], raw_output=0)
    if args.max_scatter >= 0:
        opts["max_scatter"] = args.max_scatter
    id0 = args.photon_id_offset
    gridless = "dataset" in w
    # Steps in flight: consecutive steps are independent batches, so up to C of them run at once, each in a context of its own
    # on a stream of its own (one host thread each; thor_run is synchronous), all borrowing the same resident grid.  A step is
    # tail-bound (its last seconds walk a few long packets): with several in flight the tail of one step overlaps
    # the feed phase of the next, as in a production run of many batches.  --in-flight 1 runs them one after the other.
    C = max(1, min(args.in_flight, steps))
    if not gridless:                                               # small host-made grids: uploaded once, shared by every context
        gsh = dict(w["grid"])
        for key in ("nHI", "T", "vx", "vy", "vz", "kdust"):
            if gsh.get(key) is not None and not isinstance(gsh[key], torch.Tensor):
                gsh[key] = torch.from_numpy(np.ascontiguousarray(gsh[key], np.float32)).cuda()
    streams = [torch.cuda.current_stream()] + [torch.cuda.Stream() for _ in range(C - 1)]
    ctxs = []
    for j in range(C):
        with torch.cuda.stream(streams[j]):                        # the context keeps the stream it is created on
            cx = thor.Context.gridless(**w["dataset"]) if gridless else thor.Context.from_workload(gsh, pack=pack, extra_flags=args.grid_flags)
            cx.sources_set(w["sources"]["pos"], w["sources"]["lum"], w["sources"]["sigma"])   # resident before the timed region
        ctxs.append(cx)
    ctx = ctxs[0]
    flush = [torch.empty(256 << 20, dtype=torch.uint8, device="cuda") for _ in range(C)]   # > 126 MB L2
    n_spec, n_cnt = opts["spec_bins"] + 2, len(thor.COUNTER_NAMES)
    spec_dev = [torch.zeros(n_spec, dtype=torch.int64, device="cuda") for _ in range(C)]
    cnt_dev = [torch.zeros(n_cnt, dtype=torch.int64, device="cuda") for _ in range(C)]
    spec_sum = [torch.zeros(n_spec, dtype=torch.int64, device="cuda") for _ in range(C)]
    cnt_sum = [torch.zeros(n_cnt, dtype=torch.int64, device="cuda") for _ in range(C)]

    def step(j, i):
        # rank r walks photon ids [r n, (r+1) n) of step i's seed
        cx = ctxs[j]
        cx.run(n, w["seed"] + (i if not id0 else 0), dict(opts, photon_id_offset=id0 + rank * n))
        cx.tally_to_device(thor.TALLY_SPECTRUM, spec_dev[j])
        cx.tally_to_device(thor.TALLY_COUNTERS, cnt_dev[j])
        return cx.last_run_ms(), cx.last_run_feed_ms(), cx.last_run_max_nscat()

    serial_ms = []
    for i in range(warmup):                                        # warm-up: one step at a time, on every context in turn
        j = i % C
        with torch.cuda.stream(streams[j]):
            t0 = time.perf_counter()
            step(j, -1 - i)
            streams[j].synchronize()
            serial_ms.append(1e3 * (time.perf_counter() - t0))
    for j in range(min(warmup, C), C):                             # contexts the warm-up did not reach: a short run each
        with torch.cuda.stream(streams[j]):
            ctxs[j].run(min(n, 1024), w["seed"], dict(opts, photon_id_offset=id0 + rank * n))
    sampler = ClockSampler(local) if sample_clocks else None
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    kern_ms, feed_ms, max_nscat = [0.0] * steps, [0.0] * steps, [0] * steps
    nxt, lock, errors = [0], threading.Lock(), []
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def worker(j):
        try:
            torch.cuda.set_device(local)
            with torch.cuda.stream(streams[j]):
                while True:
                    with lock:
                        i = nxt[0]
                        nxt[0] += 1
                    if i >= steps:
                        return
                    flush[j].zero_()                               # L2 flush before every timed step (on this step's stream)
                    kern_ms[i], feed_ms[i], max_nscat[i] = step(j, i)
                    spec_sum[j] += spec_dev[j]
                    cnt_sum[j] += cnt_dev[j]
        except Exception as e:                                     # surfaced after the join
            errors.append(e)

    ev0.record()
    if C == 1:
        worker(0)
    else:
        th = [threading.Thread(target=worker, args=(j,)) for j in range(C)]
        [t.start() for t in th]
        [t.join() for t in th]
    for st in streams:
        st.synchronize()
    ev1.record()
    torch.cuda.synchronize()
    if errors:
        raise errors[0]
    spec_tot, cnt_tot = sum(spec_sum[1:], spec_sum[0]), sum(cnt_sum[1:], cnt_sum[0])
    shard.allreduce_tallies([spec_tot, cnt_tot])                   # the one exchange step; no-op at N = 1
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if sampler else None
    totals = cnt_tot.cpu().numpy()
    step_ms = ev0.elapsed_time(ev1)                                # the whole timed region, device clock
    t = torch.tensor([step_ms, sum(kern_ms)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    step_ms, kernel_ms = float(t[0]), float(t[1])
    if C > 1:
        kernel_ms = step_ms                                        # launches overlap: the region is their span
    c = dict(zip(thor.COUNTER_NAMES, (int(v) for v in totals)))
    packets = c["escaped"] + c["absorbed"] + c["terminated"] + c["capped"]
    assert packets == n * world * steps, (packets, n, world, steps)
    secs = step_ms * 1e-3
    crossings = c["cell_crossings"] + c["peel_cells"]
    g = w.get("grid") or dict(nx=0, ny=0, nz=0)
    out = {
        "metric": "lya_scatterings_per_sec", "value": c["scatterings"] / secs, "unit": "scatterings/s",
        "packets_per_sec": packets / secs, "cell_crossings_per_sec": crossings / secs,
        "steps": steps, "warmup": warmup, "ms_per_step": step_ms / steps,
        "serial_ms_per_step": float(np.mean(serial_ms)) if serial_ms else None,
        "config": {"workload": workload_label(name), "grid": [g["nx"], g["ny"], g["nz"]], "n_photons_per_step_per_gpu": n,
                   "layout": "gridless (analytic sphere, fp64 geometry)" if gridless else "packed 32 B/cell (THOR_GRID_PACK)" if pack else "SoA fp32, borrowed",
                   "parallelism": f"photon-id shards x{world}, grid replicated",
                   "steps_in_flight": C,
                   "steps_in_flight_note": (f"{C} independent steps at a time, each in its own context / stream / host thread on the shared resident grid; "
                                            "ms_per_step = timed region / steps; serial_ms_per_step = the warm-up steps, run one at a time") if C > 1 else "steps run one after the other",
                   "l2": "flushed before every timed step (256 MB memset on the step's stream)",
                   "scatterings_per_packet": c["scatterings"] / packets,
                   "crossings_per_packet": crossings / packets,
                   "rejection_iters_per_scattering": c["rejection_iters"] / max(1, c["scatterings"]),
                   "phase_functions": f"core {opts.get('phase_core', 0)} / wing {opts.get('phase_wing', 0)} (0 isotropic, 1 dipole, 2 mix)"},
        # how the kernel time splits: until the photon counter runs dry the walk is fed (throughput phase); after that
        # the launch only drains the packets in flight, and lasts as long as its longest single packet
        "phases": {"feed_ms_per_step": float(np.mean(feed_ms)),
                   "drain_ms_per_step": float(np.mean(kern_ms)) - float(np.mean(feed_ms)),
                   "launch_ms_per_step": float(np.mean(kern_ms)),
                   "longest_packet_scatterings": [int(v) for v in max_nscat],
                   "drain_ns_per_scattering_of_longest_packet": float(np.mean([1e6 * (k - f) / max(1, m) for k, f, m in
                                                                               zip(kern_ms, feed_ms, max_nscat)])),
                   "source": "device %globaltimer at kernel entry and when the photon counter is first found exhausted (thor_last_run_feed_ms)",
                   "note": ("launches of different steps overlap: a launch's span (launch_ms_per_step, and the drain figures derived from it) includes the time its kernels "
                            "wait for SMs held by the other steps; serial_ms_per_step is the span of a step alone") if C > 1 else "one step at a time"},
        "counters": c,
    }
    if note:
        out["config"].update(note)
    if clocks:
        out["clocks"] = clocks
    # ---- rooflines of the dominant (only) kernel
    sm_hz = 1e6 * float((clocks or {}).get("sm_max_mhz") or 1965.0)
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    peak = n_sm * SCHEDULERS_PER_SM * LANES * sm_hz * world
    inst = INST_PER_SCATTERING * c["scatterings"] + INST_PER_CROSSING * crossings
    achieved = inst / (kernel_ms * 1e-3)
    tr = TRAFFIC.get(name)
    traffic = tr["bytes_per_launch"] * n / tr["n_photons"] if tr else None      # measured at tr[n_photons] packets, scaled to n
    alu = {"bound": "alu", "achieved": achieved / 1e9, "peak": peak / 1e9, "unit": "G thread-inst/s", "frac": achieved / peak,
           "traffic": traffic, "traffic_source": (tr["source"] + f"; measured at {tr['n_photons']} packets, scaled linearly to {n}") if tr else None,
           "peak_source": f"{n_sm} SMs x 4 schedulers x 32 lanes x {sm_hz / 1e6:.0f} MHz (clocks.max.sm), derived in DESIGN.md 5",
           "kernel": "walk_kernel + drain_kernel (one thor_run)", "kernel_ms_per_launch": kernel_ms / steps,
           "kernel_ms_note": "CUDA events around the timed region / steps (launches of different steps overlap)" if C > 1 else "thor_last_run_ms: CUDA events around the launch on the context's stream",
           "inst_per_scattering": INST_PER_SCATTERING, "inst_per_crossing": INST_PER_CROSSING,
           "constants_source": "SURVEY.md 8(d) a-priori budgets"}
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0)) * world
    gbs = BYTES_PER_CROSSING * crossings / (kernel_ms * 1e-3) / 1e9
    hbm = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak, "traffic": traffic,
           "algorithmic_bytes_per_launch": BYTES_PER_CROSSING * crossings / steps, "bytes_per_crossing": BYTES_PER_CROSSING,
           "dram_bytes_per_crossing": (traffic / (crossings / steps / world)) if traffic else None,
           "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if peaks else "6650 GB/s (of fallback)"}
    if name == "gather":                                            # the HBM roofline is the binding one there
        out["roofline"], out["roofline_alu"] = hbm, alu
    else:
        out["roofline"], out["roofline_hbm"] = alu, hbm

    # ---- e2e: the same step through the C-ABI with HOST buffers for what a step takes in and gives back: the source list
    # goes host -> device (thor_sources_set), the tallies come back device -> host (thor_tally_get), all inside the timed
    # region.  Small grids are re-created from host arrays each step as well; the 72.5 GB grid stays resident (dataset).
    if want_e2e:
        regrid = not gridless and not isinstance(g["nHI"], torch.Tensor)
        src = w["sources"]
        h2d = sum(np.asarray(src[k]).nbytes for k in ("pos", "lum", "sigma"))
        if regrid:
            h2d += sum(g[k].nbytes for k in ("nHI", "T", "vx", "vy", "vz", "kdust") if g.get(k) is not None)
        cube_bytes = opts.get("peel_nx", 0) * opts.get("peel_ny", 0) * opts.get("peel_nv", 0) * 8 if opts.get("peel_on") else 0
        d2h = (opts["spec_bins"] + 2 + 64 + len(thor.COUNTER_NAMES)) * 8 + cube_bytes
        e_steps = steps
        e_scat = [0.0] * e_steps

        def e2e_step(j, i):
            with torch.cuda.stream(streams[j]):
                flush[j].zero_()
                cx = thor.Context.from_workload(g, host=True, pack=pack) if regrid else ctxs[j]
                cx.sources_set(src["pos"], src["lum"], src["sigma"])
                cx.run(n, w["seed"] + (max(i, 0) if not id0 else 0), dict(opts, photon_id_offset=id0 + rank * n))
                cx.spectrum(); cx.nscat_hist()
                if cube_bytes:
                    cx.cube()
                cc = cx.counters()
                if regrid:
                    cx.close()
                return float(cc["scatterings"])

        if regrid:
            e2e_step(0, -1)                                         # small grids: one untimed pass warms the re-creation path
        nxt[0] = 0
        del errors[:]

        def e2e_worker(j):
            try:
                torch.cuda.set_device(local)
                while True:
                    with lock:
                        i = nxt[0]
                        nxt[0] += 1
                    if i >= e_steps:
                        return
                    e_scat[i] = e2e_step(j, i)
            except Exception as e:
                errors.append(e)

        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        if C == 1:
            e2e_worker(0)
        else:
            th = [threading.Thread(target=e2e_worker, args=(j,)) for j in range(C)]
            [t.start() for t in th]
            [t.join() for t in th]
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if errors:
            raise errors[0]
        tt = torch.tensor([dt, float(sum(e_scat))], dtype=torch.float64, device="cuda")
        if world > 1:
            mx = tt.clone(); dist.all_reduce(mx, op=dist.ReduceOp.MAX)
            dist.all_reduce(tt)
            tt[0] = mx[0]
        e_secs, e_tot = float(tt[0]), float(tt[1])
        out["e2e"] = {"value": e_tot / e_secs, "unit": "scatterings/s", "h2d_bytes_per_step": int(h2d),
                      "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * e_secs / e_steps, "steps": e_steps, "steps_in_flight": C,
                      "timing": ("host wall clock around " + str(e_steps) + " steps of " + ("create(host arrays)+" if regrid else "") +
                                 "sources_set(host arrays)+run+tally_get(host: spectrum, histogram, counters" +
                                 (", cube" if cube_bytes else "") + ")" + ("+destroy" if regrid else "") +
                                 f", {C} in flight, device synchronised on both sides, max over ranks" +
                                 ("" if regrid else "; the grid is the resident dataset and is not re-copied"))}
    for cx in ctxs:
        cx.close()
    del ctxs, ctx, flush, w, g
    if not gridless:
        del gsh
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default=HEADLINE)
    ap.add_argument("--n-photons", type=int, default=0)
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of oracle work for each cpu_baseline leg")
    ap.add_argument("--ref-budget", type=float, default=10.0, help="seconds of oracle work per reference step")
    ap.add_argument("--ref-chunk", type=int, default=20, help="packets per oracle call")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-subs", action="store_true", help="skip the `workloads` sub-dict")
    ap.add_argument("--sub-steps", type=int, default=3)
    ap.add_argument("--photon-id-offset", type=int, default=0, help="first photon id of rank 0 (with --n-photons 1: one chosen packet alone on the GPU, the lone-lane regime of DESIGN.md 4.6)")
    ap.add_argument("--max-scatter", type=int, default=-1, help="override the workload's scattering cap")
    ap.add_argument("--grid-flags", type=lambda v: int(v, 0), default=0, help="extra thor_grid_create flags (0x400 L2 persistence window, 0x800 32-byte L2 fetch granularity)")
    ap.add_argument("--in-flight", type=int, default=3, help="independent steps run at once, each in its own context and stream (1 = one after the other)")
    ap.add_argument("--pack", type=int, default=-1, help="THOR_GRID_PACK (1/0); default: on for the gather workload")
    args = ap.parse_args()
    if args.workload in ("project", "render"):
        if args.impl == "reference":
            raise SystemExit("--impl reference times the walk workloads only")
        return run_operators(args)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2507_11603_b200.csrc import build as cuda_build
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank == 0:
        cuda_build.build()
    from paper_2507_11603_b200 import thor
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()
    thor.lib()
    t0 = time.perf_counter()
    head = measure_walk(args, args.workload, args.steps, args.warmup, rank, local, world, n_photons=args.n_photons,
                        sample_clocks=True, want_e2e=not args.no_e2e)
    out = {"metric": head["metric"], "value": head["value"], "unit": head["unit"], "packets_per_sec": head["packets_per_sec"],
           "cell_crossings_per_sec": head["cell_crossings_per_sec"], "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "serial_ms_per_step": head["serial_ms_per_step"], "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": head["config"], "clocks": head.get("clocks"),
           "gpu_launches": 5 * args.steps, "phases": head["phases"], "counters": head["counters"],
           "roofline": head["roofline"]}
    for k in ("roofline_hbm", "roofline_alu", "e2e"):
        if k in head:
            out[k] = head[k]
    out["headline_wall_s"] = time.perf_counter() - t0
    # ---- the other configurations, measured in the same run (a few steps each): steady-state and straggler regimes
    if not args.no_subs and args.workload == HEADLINE and not args.n_photons:
        out["workloads"] = {}
        for name in SUBS:
            r = measure_walk(args, name, args.sub_steps, 3, rank, local, world)
            out["workloads"][name] = {k: r[k] for k in ("value", "unit", "packets_per_sec", "cell_crossings_per_sec", "steps",
                                                         "warmup", "ms_per_step", "serial_ms_per_step", "config", "phases", "roofline")}
            out["workloads"][name]["roofline_other"] = r.get("roofline_hbm") or r.get("roofline_alu")
            out["gpu_launches"] += 5 * args.sub_steps
    # ---- cpu_baseline: the oracle on a bounded sample, rank 0 at N = 1 only
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.workload, args.cpu_budget, max(1, args.ref_chunk))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(out))


if __name__ == "__main__":
    main()
