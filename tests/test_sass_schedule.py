"""Build-time check of the relaxation kernels' instruction schedule (no GPU needed: reads the SASS of the built library).

DESIGN.md §6.2 / §7: for a lone warp the FIRE iteration is a dependent chain, and whether ptxas issues the spring
chain's MUFU.SQRT well ahead of the stale-cell vote or directly in front of its MUFU.RCP changes the relaxation time of
small scans by 15-40 %.  The placement follows from the register budget (`RX_MIN_CTAS` in relax.cu), not from anything the
source orders, so it is asserted here for every tri-linear instantiation the dispatcher can pick: in the FIRE loop at
least 12 instructions lie between each MUFU.SQRT / MUFU.RCP pair that brackets a stale-cell vote.  Also: the hot kernels
carry the sm_100a instructions the design relies on (FFMA2 / UBLKCP in ff_kernel) and no local-memory traffic in the
relaxation kernels."""
import os
import re
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
LIB = os.path.join(ROOT, "paper_2401_14564_b200", "libppfm.so")
CUOBJDUMP = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"


@pytest.fixture(scope="module")
def sass():
    if not os.path.exists(CUOBJDUMP):
        pytest.skip("cuobjdump not available")
    from paper_2401_14564_b200 import build
    build.build()
    out = subprocess.run([CUOBJDUMP, "-sass", LIB], capture_output=True, text=True, check=True).stdout
    funcs, name = {}, None
    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            name = m.group(1)
            funcs[name] = []
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(.*?);", line)
        if m and name:
            t = m.group(1).split()
            funcs[name].append(t[1] if t[0].startswith("@") else t[0])
    return funcs


def test_relax_kernels_issue_sqrt_well_ahead_of_its_reciprocal(sass):
    names = [n for n in sass if re.search(r"relax_(batch_)?kernelILb[01]ELb[01]ELb[01]ELb0ELb[01]E", n)]
    assert len(names) == 32, len(names)           # 8 tri-linear variants x {plain, stiffness} x {single, batch}
    for n in names:
        ops = sass[n]
        votes = [i for i, o in enumerate(ops) if o == "VOTE.ANY"]
        assert len(votes) >= 2, n
        checked = 0
        for v in votes[:2]:                        # the two unrolled FIRE iterations of the loop body
            near = [i for i in range(max(v - 60, 0), min(v + 30, len(ops))) if ops[i] == "MUFU.SQRT"]
            assert near, n
            sq = min(near, key=lambda i: abs(i - v))                        # the spring chain's square root
            rc = next(i for i in range(sq + 1, len(ops)) if ops[i] == "MUFU.RCP")
            assert rc - sq >= 12, f"{n}: MUFU.SQRT and MUFU.RCP only {rc - sq} instructions apart around the vote"
            checked += 1
        assert checked == 2
        assert not any(o.startswith("LDL") or o.startswith("STL") for o in ops), f"{n}: local-memory traffic"


def test_hot_kernels_carry_the_sm100a_instructions_the_design_relies_on(sass):
    ff = [n for n in sass if re.search(r"ff_(batch_)?kernelILi\d+ELb[01]ELb[01]E", n)]
    assert ff
    for n in ff:
        ops = sass[n]
        assert ops.count("FFMA2") > 100 and "UBLKCP" in " ".join(ops), n       # packed FP32x2 math, TMA bulk copies
        assert any(o.startswith("SYNCS") for o in ops), n                      # mbarrier ring
        assert any(o.startswith("STG.E.128") for o in ops), n                  # float4 stores
    df = [n for n in sass if "df_column_kernel" in n]
    assert len(df) == 64                                                        # n + 1 = 2 .. 33, float4 and plain stacks
