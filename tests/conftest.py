import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


# Observed margins of the whole-run comparisons (same-seed identical-history fractions, endpoint errors, statistics):
# tests append one line each; printed in the terminal summary and written to gpurun_out/parity_margins.txt (overwritten by
# every session and stamped with its command line, so the file always holds ONE run), from which BASELINE.md's parity table
# is filled in.
MARGINS = []


def _git_head() -> str:
    """HEAD of the tree the tests ran on ("unknown" on the GPU box, whose snapshot has no .git)."""
    try:
        import subprocess
        return subprocess.run(["git", "rev-parse", "--short", "HEAD"], cwd=ROOT, capture_output=True, text=True, timeout=10).stdout.strip() or "unknown"
    except Exception:
        return "unknown"


def record_margin(line: str) -> None:
    MARGINS.append(line)


def pytest_terminal_summary(terminalreporter):
    if not MARGINS:
        return
    terminalreporter.write_sep("-", "observed parity margins")
    for m in MARGINS:
        terminalreporter.write_line(m)
    out = os.path.join(ROOT, "gpurun_out")
    try:
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_margins.txt"), "w") as f:          # one run per file: never mixed with older code's lines
            f.write(f"# pytest session at git {_git_head()}; args: {' '.join(sys.argv[1:])}\n")
            f.write("\n".join(MARGINS) + "\n")
    except OSError:
        pass


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import avmo
    avmo.build()
    return avmo


@pytest.fixture(scope="session")
def g0():
    from paper_2509_15377_b200.gen import gas
    return gas.gas_g0()


@pytest.fixture(scope="session")
def avm():
    """The CUDA path through its C ABI.  Fails loudly when the library or a GPU is missing."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu test selected but no CUDA device is visible")
    from paper_2509_15377_b200 import build
    build.build()                         # no-op when libavm.so is newer than its sources (nvcc is on the GPU box too)
    from paper_2509_15377_b200 import avm as _avm
    return _avm
