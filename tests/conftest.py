import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle():
    """The fp64 CPU oracle (test infrastructure; built on first use with g++)."""
    from oracle import thor_oracle
    thor_oracle.build()
    return thor_oracle


RETRIES = []          # (test id, first-attempt failure) of every statistical test that needed its second sample
_ATTEMPT = 0


def scaled(n):
    """Packet count of a statistical test: n on the first attempt, 2n on the retry (a larger independent sample, so a
    small real bias that slipped past once is less likely to slip past twice)."""
    return int(n) * (2 if _ATTEMPT else 1)


def statistical(retries=1):
    """Decorator for tests whose verdict is a statistical comparison at BASELINE.json's bar (KS p > 0.01, bins within
    4 sigma).  Each such test holds 3-6 comparisons at alpha = 0.01 and the suite ~40, so under a true null one of them
    fails every few runs; a failure must therefore REPRODUCE on an independent, twice as large sample to count
    (per comparison this makes alpha = 1e-4, per test ~5e-4).  The re-run shifts the workload seeds (both
    sides draw new packets), doubles the packet counts taken through scaled(), is held to the same bar — and is never
    silent: it raises a warning naming the test and the first failure and the session ends with a 'statistical retries'
    summary line."""
    import functools
    import warnings

    def deco(fn):
        @functools.wraps(fn)
        def wrapper(*args, **kwargs):
            global _ATTEMPT
            from paper_2507_11603_b200 import workloads as W
            names = ["static_sphere", "expanding_shell", "static_slab", "turbulent_box", "cosmic_web"]
            last = None
            for attempt in range(retries + 1):
                saved = {n: getattr(W, n) for n in names}

                def shifted(f, k):
                    def g(*a, **kw):
                        w = f(*a, **kw)
                        w["seed"] = w["seed"] + 1000 * k
                        return w
                    return g
                try:
                    _ATTEMPT = attempt
                    for n in names:
                        setattr(W, n, shifted(saved[n], attempt))
                    return fn(*args, **kwargs)
                except AssertionError as e:
                    last = e
                    if attempt < retries:
                        first = " ".join(str(e).split())[:300]
                        RETRIES.append((fn.__name__, first))
                        warnings.warn(f"statistical retry: {fn.__name__} failed its first sample ({first}); "
                                      "re-running on an independent sample of twice the size")
                finally:
                    _ATTEMPT = 0
                    for n in names:
                        setattr(W, n, saved[n])
            raise last
        return wrapper
    return deco


def pytest_terminal_summary(terminalreporter):
    terminalreporter.write_line(f"statistical retries: {len(RETRIES)}" +
                                "".join(f"\n  retried: {name}: {why}" for name, why in RETRIES))
