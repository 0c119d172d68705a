import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

GOLDEN = Path(__file__).resolve().parent / "golden"


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def read_kv(name):
    """Parse a `key = value  # comment` golden file."""
    out = {}
    for line in (GOLDEN / name).read_text().splitlines():
        line = line.split("#", 1)[0].strip()
        if not line or "=" not in line:
            continue
        k, v = line.split("=", 1)
        out[k.strip()] = float(v)
    return out


def read_table(name):
    rows = []
    for line in (GOLDEN / name).read_text().splitlines():
        line = line.split("#", 1)[0].strip()
        if line:
            rows.append([float(t) for t in line.split()])
    return rows


@pytest.fixture(scope="session")
def oracle():
    from oracle import Oracle
    return Oracle()


# ---- achieved error against the tolerance, per config and variant ("print the achieved max |dF| / tolerance") ----
MARGINS = []


def record_margin(config, variant, what, err, tol):
    """Called by the GPU parity tests; the table is written to gpurun_out/ at the end of the session."""
    MARGINS.append((str(config), str(variant), str(what), float(err), float(tol)))


def pytest_sessionfinish(session, exitstatus):
    if not MARGINS:
        return
    out = ROOT / "gpurun_out"
    out.mkdir(exist_ok=True)
    worst = {}
    for cfg, var, what, err, tol in MARGINS:
        k = (cfg, var, what)
        if k not in worst or err / tol > worst[k][0] / worst[k][1]:
            worst[k] = (err, tol)
    lines = ["# Achieved error over tolerance in the GPU parity tests (worst case per config, variant and quantity)", "",
             "Command: `python -m pytest tests -m gpu -q` (written by tests/conftest.py at the end of the session).",
             "Tolerances (BASELINE.json north_star): forces and torques 1e-4 max|F_oracle| + 1e-6 per component, energies 1e-5 relative.", "",
             "| config | variant | quantity | max abs error | tolerance | error / tolerance |", "|---|---|---|---|---|---|"]
    for (cfg, var, what), (err, tol) in sorted(worst.items()):
        lines.append(f"| {cfg} | {var} | {what} | {err:.3e} | {tol:.3e} | {err / tol:.4f} |")
    (out / "parity_margins.md").write_text("\n".join(lines) + "\n")
