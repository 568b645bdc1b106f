import os
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
for p in (str(ROOT), str(ROOT / "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_collection_modifyitems(config, items):
    """GPU tests never silently pass without a device: they are skipped only when deselected by -m."""
    return


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session")
def gen_mod():
    from paper_1712_09416_b200 import gen
    return gen


def make_geometry(oracle, gen, ev):
    return oracle.Geometry(ev.n_sectors, gen.row_x().astype(np.float32), gen.TAN_HALF_ANGLE, ev.sigma, ev.sigma,
                           ev.bz)


@pytest.fixture(scope="session")
def geometry_of(oracle_mod, gen_mod):
    return lambda ev: make_geometry(oracle_mod, gen_mod, ev)


_cache = {}


@pytest.fixture(scope="session")
def event_and_oracle(oracle_mod, gen_mod):
    """(recipe name, precision) -> (event, oracle result), cached for the session."""
    def get(name, precision="float", event=0):
        key = (name, precision, event)
        if key not in _cache:
            ev = gen_mod.generate(name, event)
            res = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z,
                                         ev.row, precision=precision)
            _cache[key] = (ev, res)
        return _cache[key]
    return get
