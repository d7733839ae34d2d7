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


@pytest.fixture
def record(request):
    """Record what a parity test MEASURED (max deviation, dev / sigma, counts ...): printed (pytest -s or a
    failure shows it) and appended as one JSON line to gpurun_out/parity_stats.jsonl when that directory
    exists (the GPU box's scratch folder).  DESIGN.md §5 tabulates one such run."""
    import json

    def _rec(stats):
        row = dict(test=request.node.name, **stats)
        print("PARITY-STATS " + json.dumps(row))
        out = os.path.join(ROOT, "gpurun_out")
        if os.path.isdir(out):
            with open(os.path.join(out, "parity_stats.jsonl"), "a") as fh:
                fh.write(json.dumps(row) + "\n")

    return _rec
