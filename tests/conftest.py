import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def repo_root():
    return ROOT


def _verdict_rows():
    try:
        import parity_utils
    except Exception:
        return []
    return list(parity_utils.VERDICTS)


def pytest_terminal_summary(terminalreporter):
    """End-to-end v+ verdicts of the GPU session (parity_utils.check_step_parity): the tally goes to the terminal and
    the full table to gpurun_out/parity_verdicts.md (copied to profiles/ by hand after a GPU run)."""
    rows = _verdict_rows()
    if not rows:
        return
    tally = {}
    for _, kind, *_ in rows:
        tally[kind] = tally.get(kind, 0) + 1
    terminalreporter.write_line("end-to-end v+ verdicts: " + ", ".join(f"{n} {k}" for k, n in sorted(tally.items())))
    out_dir = os.path.join(ROOT, "gpurun_out")
    try:
        os.makedirs(out_dir, exist_ok=True)
        fmt = lambda x: "-" if x is None else f"{x:.2e}"
        with open(os.path.join(out_dir, "parity_verdicts.md"), "w") as f:
            f.write("# End-to-end v+ verdicts (tests/parity_utils.py: check_step_parity)\n\n"
                    "Command: `python -m pytest tests -q -m gpu` on a B200.  `match` = |v+ - oracle v+| < 1e-4 outright; otherwise the\n"
                    "test asserted the isolated-update reproduction and the weight-sensitivity bound (see the docstring).\n\n"
                    f"Tally: {', '.join(f'{n} {k}' for k, n in sorted(tally.items()))}.\n\n"
                    "| case | verdict | max abs err of v+ | max abs dS~ (live samples) | gap of the two smallest S~ | bound |\n|---|---|---|---|---|---|\n")
            for name, kind, err, D, gap, bound in rows:
                f.write(f"| {name} | {kind} | {err:.2e} | {fmt(D)} | {fmt(gap)} | {fmt(bound)} |\n")
    except OSError:
        pass
