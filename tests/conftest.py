import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FULL_MODULE = "test_zfull_registration"
_full_refs = None


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_collection_finish(session):
    """The full-size registration tests need minutes of oracle time: start their references in background
    processes now (tests/full_refs.py), so they are computed while the other GPU tests run."""
    global _full_refs
    wanted = any(FULL_MODULE in item.nodeid for item in session.items)
    if not wanted or _full_refs is not None:
        return
    import torch
    if not torch.cuda.is_available():
        return
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    import full_refs
    _full_refs = full_refs.FullRefs()


def pytest_sessionfinish(session, exitstatus):
    global _full_refs
    if _full_refs is not None:
        _full_refs.close()
        _full_refs = None


@pytest.fixture(scope="session")
def full_refs():
    if _full_refs is None:
        pytest.skip("no CUDA device: the full-size references were not started")
    return _full_refs


@pytest.fixture(scope="session")
def oracle():
    from oracle import oracle as O
    O.build()
    return O
