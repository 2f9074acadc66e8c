import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _ensure_built():
    """The package refuses to import without libhr_b200.so (no CPU fallback), so a stale or
    missing library is (re)built here by loading its build script by path."""
    import importlib.util
    spec = importlib.util.spec_from_file_location(
        "_hr_cuda_build", os.path.join(ROOT, "paper_2501_14030_b200", "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.build()
    from oracle import build as oracle_build
    oracle_build.build()


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    _ensure_built()


@pytest.fixture(scope="session")
def oracle_mod():
    from oracle import hr_oracle
    hr_oracle.lib()
    return hr_oracle
