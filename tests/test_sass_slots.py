"""The roofline's "operations per pair" (bench.py SLOTS / SLOTS_V_ONLY, reading 20) are
the builder's own counts; this test checks them against the machine code.  For every headline
kernel the built library is disassembled (cuobjdump -sass: no GPU needed), the innermost loop that
holds the reciprocal-square-root seeds (MUFU.RSQ / MUFU.RSQ64H: exactly one per pair) is found, and
the arithmetic-pipe lane operations in it are counted per seed: packed FFMA2 / FMUL2 / FADD2 count
two (two points per instruction), scalar FP32 and every DP instruction one.  The count must equal
the table's figure, plus at most the summation-tree adds of the FP32 kernels (a quarter operation
per pair; half of one in the kernels whose last tree level is compensated); a kernel that silently did more -- or less -- work per pair than the roofline assumes
would fail here.
"""
import os
import re
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PACKED = ("FFMA2", "FMUL2", "FADD2")
SCALAR = ("FFMA", "FMUL", "FADD")
DP = ("DFMA", "DMUL", "DADD")

# (mangled kernel, layout, precision, potential only, dz table, compensated row sums)
KERNELS = [
    # <2, 8, false, true, true, 0, VONLY, ACCV>: the batched kernels of config 3 -- V + E with accurate V (default),
    # V + E fast (qmmm_field_set_accurate_v(h, 0)), potential only
    ("_ZN4qmmm17grid_kernel_f32x2ILi2ELi8ELb0ELb1ELb1ELi0ELb0ELb1EEEvNS_10PairParamsE", "grid", "fp32", False, True, True),
    ("_ZN4qmmm17grid_kernel_f32x2ILi2ELi8ELb0ELb1ELb1ELi0ELb0ELb0EEEvNS_10PairParamsE", "grid", "fp32", False, True, False),
    ("_ZN4qmmm17grid_kernel_f32x2ILi2ELi8ELb0ELb1ELb1ELi0ELb1ELb0EEEvNS_10PairParamsE", "grid", "fp32", True, True, True),
    ("_ZN4qmmm17grid_kernel_f32x2ILi2ELi8ELb0ELb1ELb0ELi0ELb0ELb0EEEvNS_10PairParamsE", "grid", "fp32", False, False, False),
    ("_ZN4qmmm17pair_kernel_f32x2ILi4ELi8EEEvNS_10PairParamsE", "list", "fp32", False, False, False),
    ("_ZN4qmmm15grid_kernel_f64ILi4ELb1ELi8ELb0ELb1EEEvNS_10PairParamsE", "grid", "fp64", False, True, False),
    ("_ZN4qmmm15grid_kernel_f64ILi4ELb0ELi8ELb0ELb1EEEvNS_10PairParamsE", "grid", "fp64", True, True, False),
    ("_ZN4qmmm15grid_kernel_f64ILi4ELb1ELi8ELb0ELb0EEEvNS_10PairParamsE", "grid", "fp64", False, False, False),
    ("_ZN4qmmm11pair_kernelIdLi4ELb1EEEvNS_10PairParamsE", "list", "fp64", False, False, False),
    ("_ZN4qmmm11pair_kernelIdLi4ELb0EEEvNS_10PairParamsE", "list", "fp64", True, False, False),
]


def hot_loop(lib, sym, seed):
    """Instructions of the smallest backward-branch loop that holds at least 8 seeds."""
    txt = subprocess.run(["cuobjdump", "-sass", "-fun", sym, lib], capture_output=True, text=True, check=True).stdout
    ins = []
    for ln in txt.splitlines():
        m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", ln)
        if m:
            ins.append((int(m.group(1), 16), re.sub(r"^@!?U?P\d+\s+", "", m.group(2).strip())))
    assert ins, f"{sym}: not found in {lib}"
    best = None
    for addr, text in ins:
        m = re.match(r"BRA(?:\.\w+)*\s+(?:!?U?P\d+,\s*)?(0x[0-9a-f]+)", text)
        if not m or int(m.group(1), 16) >= addr:
            continue
        body = [t for (a, t) in ins if int(m.group(1), 16) <= a <= addr]
        seeds = sum(1 for t in body if t.split()[0] == seed)
        if seeds >= 8 and (best is None or len(body) < len(best)):
            best = body
    assert best is not None, f"{sym}: no loop with {seed} found"
    return best


@pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump (CUDA toolkit) not on PATH")
@pytest.mark.parametrize("sym,layout,prec,v_only,dzt,comp", KERNELS)
def test_lane_operations_per_pair_match_the_roofline_table(sym, layout, prec, v_only, dzt, comp):
    from paper_1011_4687_b200 import build
    import bench
    lib = build.build()
    info = {"last_dz_table": 1 if dzt else 0}
    if prec == "fp32" and v_only:
        claimed = bench.SLOTS_V_ONLY_F32_GRID
    else:
        claimed = bench.slots_for(layout, prec, info, v_only=v_only)
    seed = "MUFU.RSQ" if prec == "fp32" else "MUFU.RSQ64H"
    body = hot_loop(lib, sym, seed)
    ops = [t.split()[0] for t in body]
    seeds = ops.count(seed)
    if prec == "fp32":
        lane_ops = 2 * sum(ops.count(k) for k in PACKED) + sum(ops.count(k) for k in SCALAR)
        assert sum(ops.count(k) for k in DP) == 0, "FP64 arithmetic inside the FP32 hot loop"
        per_pair = lane_ops / seeds
        # one seed per pair; the V0 / T summation trees add at most a quarter operation per pair,
        # the compensated last tree level of the potential-only and the accurate V + E kernel (fast
        # two-sum, once per 16 nodes) another quarter
        extra = 0.5 if comp else 0.25
        assert claimed <= per_pair <= claimed + extra + 1e-9, (sym, per_pair, claimed)
    else:
        per_pair = sum(ops.count(k) for k in DP) / seeds
        assert per_pair == pytest.approx(claimed, abs=1e-9), (sym, per_pair, claimed)
