import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_sessionstart(session):
    """A fresh checkout has no libbcf.so (built artefacts are git-ignored): build it in-tree before any test
    imports the binding, exactly as __graft_entry__.build() does.  A no-op when the library is up to date; a
    build failure is left for the ABI tests to report."""
    try:
        from paper_1306_5076_b200 import build as cuda_build
        cuda_build.build()
    except Exception as e:      # noqa: BLE001
        print("conftest: could not build libbcf.so: %r" % (e,), file=sys.stderr)


@pytest.fixture(scope="session")
def repo_root():
    return ROOT
