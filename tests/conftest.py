import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")


class ParityReport:
    """Measured parity errors of the -m gpu tests (reading L asks for two figures): max|g-o| / max|o| over the
    array and the element-wise max |g-o| / |o| over the elements with |o| > 1e-30 max|o|.  One JSON object per line in
    gpurun_out/parity_report.jsonl (scratch; the summary committed under profiles/ is written from it)."""

    def __init__(self):
        self.path = os.path.join(ROOT, "gpurun_out", "parity_report.jsonl")
        os.makedirs(os.path.dirname(self.path), exist_ok=True)
        open(self.path, "w").close()

    def add(self, test, config, what, got, want, bar, precision="f64"):
        import json
        import numpy as np
        g = np.asarray(got, dtype=np.float64)
        w = np.asarray(want, dtype=np.float64)
        scale = float(np.abs(w).max())
        diff = np.abs(g - w)
        rel_inf = float(diff.max() / scale) if scale > 0 else float(diff.max())
        mask = np.abs(w) > 1e-30 * scale
        elem = float((diff[mask] / np.abs(w[mask])).max()) if mask.any() else 0.0
        with open(self.path, "a") as fh:
            fh.write(json.dumps({"test": test, "config": config, "precision": precision, "what": what,
                                 "max_rel_inf": rel_inf, "max_elementwise_rel": elem, "bar": bar, "n": int(g.size)}) + "\n")
        return rel_inf


_REPORT = None


@pytest.fixture(scope="session")
def parity_report():
    global _REPORT
    if _REPORT is None:
        _REPORT = ParityReport()
    return _REPORT
