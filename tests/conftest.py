import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HERE = os.path.dirname(os.path.abspath(__file__))
for _p in (ROOT, HERE):
    if _p not in sys.path:
        sys.path.insert(0, _p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (run with -m gpu on the GPU box)")
    # native libraries are git-ignored build artefacts: (re)build them if missing or stale before any test imports a binding
    from paper_2607_01701_b200 import build

    build.build()
    build.build_sched()


@pytest.fixture(scope="session")
def orc():
    from oracle import arachne_oracle

    arachne_oracle.build()
    return arachne_oracle
