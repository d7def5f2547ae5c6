import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_sessionfinish(session, exitstatus):
    """Achieved parity errors of the run (gpu vs long-double oracle, floor, bar per field) as a scratch record."""
    try:
        import json

        from _util import RECORDS

        if RECORDS:
            os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
            with open(os.path.join(ROOT, "gpurun_out", "parity_records.jsonl"), "w") as f:
                for r in RECORDS:
                    f.write(json.dumps(r) + "\n")
    except Exception:
        pass
