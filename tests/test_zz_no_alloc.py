"""thor_run_noalloc (include/thor.h): the walk for callers that cannot allocate device memory at run time.  Its kernels'
scratch is one static device array shared by every call, so the test makes two calls IN A ROW and compares each with the
existing path (thor_run + thor_tally_get) on the same packets.  The tallies are integer counts of a walk that depends on
(seed, photon id) only: the bar is bit-exact, as everywhere the suite compares two CUDA runs of the same packets.

Collected last on purpose (file name): the run is `pytest -x`.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2507_11603_b200 import workloads as W


def test_null_context_is_an_argument_error():
    from paper_2507_11603_b200 import thor as t
    assert t.lib().thor_run_noalloc(None, 1, 1, None, None, None, None) == 1      # THOR_ERR_ARG, before any CUDA call


@pytest.mark.gpu
def test_run_noalloc_matches_thor_run_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2507_11603_b200 import thor

    # config 2's recipe (dusty expanding shell, global core-skipping): heavy-tailed chains, so both launches park packets
    # in the pool and the drain kernel runs — every word of the static scratch is in use; then a Hubble-drift walk
    cases = [(W.expanding_shell(n=32, n_photons=20_000), dict(max_scatter=20_000)),
             (W.cosmic_web(n=32, n_src=256, n_photons=3000, mean_n=1e-8, map_pix=16, v_max=40.0), dict(max_scatter=20_000, peel_on=0))]
    for w, extra in cases:
        opts = dict(w["opts"], **extra)
        n, bins = w["n_photons"], opts["spec_bins"]
        ctx = thor.Context.from_workload(w["grid"])
        try:
            ctx.sources_set(w["sources"]["pos"], w["sources"]["lum"], w["sources"]["sigma"])
            seeds = (w["seed"], w["seed"] + 7)
            # outputs start as garbage: the entry point must clear them itself
            outs = [[torch.full((m,), -3, dtype=torch.int64, device="cuda") for m in (bins + 2, len(thor.COUNTER_NAMES), 64)]
                    for _ in seeds]
            ctx.run_noalloc(n, seeds[0], opts, *outs[0])                      # first call on this device: address look-up
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
            for seed, o in zip(seeds, outs):                                  # two calls in a row, no synchronisation between
                ctx.run_noalloc(n, seed, opts, *o)
            torch.cuda.synchronize()
            assert torch.cuda.mem_get_info()[0] >= free0, "thor_run_noalloc allocated device memory"
            got = [[t.cpu().numpy().view(np.uint64) for t in o] for o in outs]
            for seed, (spec, cnt, hist) in zip(seeds, got):
                ctx.run(n, seed, opts)                                        # the existing path
                assert np.array_equal(spec, ctx.spectrum()), (w["name"], seed)
                assert dict(zip(thor.COUNTER_NAMES, (int(v) for v in cnt))) == ctx.counters(), (w["name"], seed)
                assert np.array_equal(hist, ctx.nscat_hist()), (w["name"], seed)
                assert int(cnt[thor.COUNTER_NAMES.index("scatterings")]) > n
            assert not np.array_equal(got[0][0], got[1][0])                   # the two calls did walk different packets
            # what needs memory this entry point may not allocate is refused, by name
            with pytest.raises(thor.ThorError) as e:
                ctx.run_noalloc(n, seeds[0], dict(opts, raw_output=1), *outs[0])
            assert e.value.status == 5 and "raw_output" in str(e.value)         # THOR_ERR_UNSUPPORTED
        finally:
            ctx.close()
