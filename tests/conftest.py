import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


_CFG_CACHE = {}


@pytest.fixture(scope="session")
def config_oracle(oracle_mod):
    """config index -> (ViewBatch, params, OracleResult with seed dump), computed once per session."""
    from emu_synth import default_params, make_config

    def get(c, seed_dump=True):
        if c not in _CFG_CACHE:
            b = make_config(c)
            p = default_params(c)
            r = oracle_mod.track_views(p, b.grains, b.view_off, "cells", 1, seed_dump=seed_dump)
            _CFG_CACHE[c] = (b, p, r)
        return _CFG_CACHE[c]
    return get
