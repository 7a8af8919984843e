"""The checked build (libppfm_chk.so, -DPPFM_CHECKS; include/ppfm_bench.h) stands in for compute-sanitizer, which is
closed on the GPU pool: a second pytest process runs the force-field tests with multi-chunk atom rings and ragged
tiles, every relaxation kernel instance, the periodic / clamped / tri-cubic scans, the df kernels and config 0 end to end
against libppfm_chk.so.  Parity must still hold there, and the kernels' own counters must show checks executed and
not one ring or bounds violation."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SELECT = ("test_ff_ragged_tiles_and_tails or test_ff_charged_neutral_partition or test_ff_nonorthogonal_grid_and_cell or "
          "test_ff_batch_cfg3_matches_oracle_and_single_calls or test_relax_every_kernel_instance or "
          "test_relax_periodic_wrap_and_clamp or test_relax_zero_field_and_ragged_scan or "
          "test_relax_tricubic_periodic_skewed_batch_and_edges or test_df_column_and_gather_kernels_all_window_lengths or "
          "test_relax_scan_stiffness_closed_forms or test_stiffness_zero_field_periodic_nonorthogonal_and_batch or "
          "test_scan_host_equals_device_path or "
          "(test_relax_and_df_full_scan and 0)")


@pytest.mark.gpu
def test_parity_under_the_checked_build_and_no_violation(tmp_path):
    from paper_2401_14564_b200 import build as B
    assert os.path.exists(B.CHK_LIB), "libppfm_chk.so not built (python -m paper_2401_14564_b200.build)"
    out = tmp_path / "checks.json"
    env = dict(os.environ, PPFM_LIBRARY=B.CHK_LIB, PPFM_CHECKS_OUT=str(out))
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_gpu_parity.py"), "-m", "gpu", "-q",
                        "-x", "-k", SELECT, "-p", "no:cacheprovider"], env=env, capture_output=True, text=True,
                       cwd=ROOT, timeout=1500)
    assert r.returncode == 0, r.stdout[-4000:] + r.stderr[-2000:]
    rec = json.loads(out.read_text())
    counts = rec["counts"]
    assert counts is not None, "the child process did not load the checked build"
    print("checked build:", counts)
    gp = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(gp):
        with open(os.path.join(gp, "checked_build_counts.json"), "w") as fh:
            json.dump({"selected": SELECT, "pytest_tail": r.stdout.strip().splitlines()[-1], "counts": counts}, fh)
    assert counts["visits"] > 1_000_000
    bad = {k: v for k, v in counts.items() if k != "visits" and v}
    assert not bad, f"violations under the checked build: {bad}"


def test_product_build_has_no_checks():
    """libppfm.so answers PPFM_EINVAL to ppfm_checks_read: none of the instrumentation is compiled into the product."""
    from paper_2401_14564_b200 import ppfm, ppfm_bench
    if os.environ.get("PPFM_LIBRARY"):
        pytest.skip("running under another build")
    ppfm.lib()
    assert ppfm_bench.checks_read() is None
