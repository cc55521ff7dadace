import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


# Measured parity figures (rel-L2, max-abs, flipped bins ...) of the -m gpu tests: record(name, key=value, ...) from a
# test; written to gpurun_out/parity_measured.json when the session ends (quoted under profiles/).
_MEASURED = {}


def record(name, **values):
    _MEASURED.setdefault(name, {}).update({k: (float(v) if isinstance(v, float) else v) for k, v in values.items()})


def pytest_sessionfinish(session, exitstatus):
    if not _MEASURED:
        return
    import json
    out = os.path.join(ROOT, "gpurun_out")
    try:
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_measured.json"), "w") as f:
            json.dump(_MEASURED, f, indent=1, sort_keys=True, default=lambda o: o.item() if hasattr(o, "item") else str(o))
    except OSError:
        pass


def golden(name):
    """Rows of a whitespace-separated golden text file under tests/golden/ ('#' starts a comment)."""
    rows = []
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows
