"""CPU-only checks of the boundary: libthor_b200.so builds for sm_100a, loads, and exports every symbol include/thor.h
declares; argument errors are reported as status codes; without a GPU the product path fails loudly (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def thor():
    from paper_2507_11603_b200.csrc import build
    build.build()
    from paper_2507_11603_b200 import thor as t
    return t


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "thor.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(thor_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_all_exported(thor):
    names = _declared_symbols()
    assert set(thor.EXPORTS) <= set(names)
    assert len(names) >= 12
    L = C.CDLL(thor.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/thor.h but not exported"


def test_opts_struct_matches_header(thor):
    o = thor.make_opts()
    assert o.struct_size == C.sizeof(thor.Opts)
    assert (o.phase_split_x, o.hubble_eps, o.tau_peel_max, o.spec_T_ref) == (0.2, 0.25, 30.0, 1e4)
    assert tuple(o.k_obs) == (0.0, 0.0, 1.0)
    with pytest.raises(KeyError):
        thor.make_opts(no_such_field=1)


def test_argument_errors_are_status_codes(thor):
    L = thor.lib()
    ctx = C.c_void_p()
    a = np.ones(8, np.float32)
    p = a.ctypes.data_as(C.c_void_p)
    assert L.thor_grid_create(None, 2, 2, 2, 1.0, p, p, p, p, p, None, thor.GRID_HOST, None) == 1
    assert L.thor_grid_create(C.byref(ctx), 0, 2, 2, 1.0, p, p, p, p, p, None, thor.GRID_HOST, None) == 1
    assert L.thor_grid_create(C.byref(ctx), 2, 2, 2, -1.0, p, p, p, p, p, None, thor.GRID_HOST, None) == 1
    assert L.thor_grid_create(C.byref(ctx), 2, 2, 2, 1.0, None, p, p, p, p, None, thor.GRID_HOST, None) == 1
    assert b"NULL" in L.thor_last_error(None)
    assert L.thor_sources_set(None, 1, p, p, p) == 1
    assert L.thor_run(None, 1, 1, None) == 1
    assert L.thor_tally_get(None, 0, None, 0, None) == 1
    assert L.thor_unit_voigt(0, p, p, p, None) == 1
    assert L.thor_raytrace(None, 1, p, p, 0.0, 0, 0.0, 1.0, p, None, None) == 1
    assert L.thor_last_run_feed_ms(None, None) == 1
    L.thor_grid_destroy(None)   # no-op


def test_no_cpu_fallback_without_gpu(thor):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    a = np.ones((2, 2, 2), np.float32)
    with pytest.raises(thor.ThorError) as e:
        thor.Context(2, 2, 2, 1.0, a, a, a, a, a, host=True)
    assert e.value.status == 5 and "no CPU fallback" in str(e.value)


def test_product_does_not_import_oracle():
    """The product path shares nothing with oracle/: no import, include, dlopen or path reference."""
    pkg = os.path.join(ROOT, "paper_2507_11603_b200")
    pat = re.compile(r"(import\s+oracle|from\s+oracle|#include\s*[\"<][^\n]*oracle|liboracle|oracle/[a-z_]+\.(py|hpp|cpp|so))")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inc")):
                s = open(os.path.join(d, f)).read()
                assert not pat.search(s), f
    for f in ("include/thor.h",):
        assert not pat.search(open(os.path.join(ROOT, f)).read())
