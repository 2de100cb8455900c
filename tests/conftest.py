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
    gpurun_out/parity_report.jsonl (scratch).  At the end of the session `summary()` condenses it to
    gpurun_out/parity_summary.md -- worst figure per test, config group and precision -- and the file committed under
    profiles/ (rN_parity.md) is a copy of that summary."""

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


    def summary(self):
        import json
        rows = {}
        with open(self.path) as fh:
            for line in fh:
                r = json.loads(line)
                key = (r["test"], r["config"], r["precision"], r["what"])
                w = rows.setdefault(key, {"n": 0, "rel": 0.0, "elem": 0.0, "bar": r["bar"]})
                w["n"] += 1
                w["rel"] = max(w["rel"], r["max_rel_inf"])
                w["elem"] = max(w["elem"], r["max_elementwise_rel"])
        if not rows:
            return None
        out = os.path.join(os.path.dirname(self.path), "parity_summary.md")
        with open(out, "w") as fh:
            fh.write("# Measured parity errors, CUDA path against the oracle\n\n"
                     "Written by tests/conftest.py at the end of `python -m pytest tests -q -m gpu` from every comparison the\n"
                     "tests recorded.  rel = max|g-o| / max|o| (gated by `bar`); elem = element-wise max|g-o|/|o| (recorded only).\n\n"
                     "| test | config | precision | what | comparisons | worst rel | bar | worst rel / bar | worst elem |\n|---|---|---|---|---|---|---|---|---|\n")
            for (test, cfg, prec, what), w in sorted(rows.items()):
                fh.write(f"| {test} | {cfg} | {prec} | {what} | {w['n']} | {w['rel']:.2e} | {w['bar']:.0e} | {w['rel'] / w['bar']:.3f} | {w['elem']:.2e} |\n")
        return out


_REPORT = None


@pytest.fixture(scope="session")
def parity_report():
    global _REPORT
    if _REPORT is None:
        _REPORT = ParityReport()
    return _REPORT


def pytest_sessionfinish(session, exitstatus):
    if _REPORT is not None:
        _REPORT.summary()
