"""Shared fixtures. ``-m "not gpu"`` tests run on the CPU box; ``-m gpu`` tests need a B200."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (parity tests through the C-ABI)")


@pytest.fixture(scope="session")
def geom():
    from paper_2207_08207_b200 import synth
    return synth.make_geometry()


@pytest.fixture(scope="session")
def mmap(geom):
    """The module map used as INPUT by the oracle and GPU tests: the test-side generator (tests/mapgen.py)."""
    import mapgen
    return mapgen.make_module_map(geom)


@pytest.fixture(scope="session")
def o32():
    from oracle import oracle
    return oracle.load("f32")


@pytest.fixture(scope="session")
def o64():
    from oracle import oracle
    return oracle.load("f64")


@pytest.fixture(scope="session")
def run_oracle(geom, mmap):
    """run_oracle(lib, event, **kw) -> OracleResult on the standard geometry and map."""
    def _run(lib, ev, **kw):
        return lib.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side, **kw)
    return _run
