import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")


@pytest.fixture(scope="session", autouse=True)
def built_library():
    """Build libwolff_b200.so in-tree when it is missing or older than its sources (the .so is not in the history).
    Needs nvcc, not a GPU; without nvcc the tests that load the library fail loudly -- there is no fallback."""
    from paper_1110_0899_b200 import build
    try:
        build.build()
    except RuntimeError as e:          # nvcc absent or the compile failed: let the ABI / GPU tests report it
        sys.stderr.write("libwolff_b200.so not built: %s\n" % e)


def pytest_collection_finish(session):
    """Protocol-length parity tests: start their oracle chains (minutes of sequential CPU work at 2D L=4096) in
    background threads as soon as such a test is known to run, so that they overlap with the other GPU tests."""
    names = set()
    for item in session.items:
        if item.module.__name__.endswith("test_gpu_protocol") or item.module.__name__.endswith("test_gpu_measure"):
            callspec = getattr(item, "callspec", None)
            if callspec is not None and "name" in callspec.params:
                names.add(callspec.params["name"])
    if names:
        import protocol_farm
        # longest first: the pool runs them all at once, but start order decides who gets a core first on a small box
        order = ["C3", "C3-stretch", "C5a", "C2", "C4", "C5b", "C5b-literal", "C2-literal", "C3-literal", "C4-literal", "C5a-literal"]
        protocol_farm.start([n for n in order if n in names])
