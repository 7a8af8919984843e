import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


# Exemption accounting of the relaxation parity tests (tests/test_gpu_parity.py appends one record per comparison):
# how many (pixel, z-step) samples missed the 2e-3 Å tolerance, how many of those carry north_star's end-point flag
# (smallest Hessian eigenvalue < 1e-3 eV/Å^2 at the relaxed point of this or the previous z-step, or not converged),
# and how many are exempt ONLY through the trajectory flag of reading S17.  Printed at the end of the session.
PARITY_LOG = []


def pytest_terminal_summary(terminalreporter, exitstatus, config):
    if not PARITY_LOG:
        return
    tr = terminalreporter
    tr.write_sep("-", "relaxation parity: samples outside 2e-3 Å and how they are exempt (reading S17)")
    tr.write_line(f"{'case':58s} {'samples':>9s} {'fail':>6s} {'end-point flag':>15s} {'trajectory flag only':>21s} "
                  f"{'inherited':>10s} {'valid minima':>13s} {'saddles':>8s} {'max |dr| ok (Å)':>16s}")
    for r in PARITY_LOG:
        tr.write_line(f"{r['what'][:58]:58s} {r['samples']:9d} {r['fail']:6d} {r['fail_endpoint_flag']:15d} "
                      f"{r['fail_traj_only']:21d} {r.get('fail_inherited', 0):10d} {r.get('exempt_validated', 0):13d} {r.get('exempt_saddle', 0):8d} "
                      f"{r['max_ok_dist']:16.2e}")
    out = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out) and not os.environ.get("PPFM_CHECKS_OUT"):      # not from the checked build's child session
        import json
        with open(os.path.join(out, "parity_exemptions.jsonl"), "w") as fh:
            for r in PARITY_LOG:
                fh.write(json.dumps(r) + "\n")


def pytest_sessionfinish(session, exitstatus):
    """Under the checked build (PPFM_LIBRARY=.../libppfm_chk.so, tests/test_checked_build.py) write the kernels' own
    bounds / ring check counts of this session to the file named by PPFM_CHECKS_OUT."""
    path = os.environ.get("PPFM_CHECKS_OUT")
    if not path:
        return
    import json

    from paper_2401_14564_b200 import ppfm_bench
    with open(path, "w") as fh:
        json.dump({"exitstatus": int(exitstatus), "counts": ppfm_bench.checks_read()}, fh)


def pytest_collection_modifyitems(config, items):
    # GPU tests must never pass silently on a box without a device: they are deselected by `-m "not gpu"`;
    # when explicitly selected without a GPU they fail loudly inside the binding (no CPU fallback exists).
    pass
