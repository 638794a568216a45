"""Writes tests/golden/config0_oracle.txt: V, Ex, Ey, Ez of config 0 (BASELINE.json
configs[0]; 8 points x 4,096 sources + 16 nuclei, seed 0) from the CPU ORACLE ONLY.

Run:  python tests/golden/make_config0_golden.py
The values are the oracle's (oracle/qmmm_oracle.c, following PAPER.md:59-60 Eq. 4);
tests/test_oracle_pins.py::test_mpmath_config0_and_golden re-derives two of the rows
with 50-digit mpmath arithmetic.  Nothing here touches the CUDA path.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1011_4687_b200.workloads import make_workload  # noqa: E402

w = make_workload(0)
res = oracle.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, w.elec_xyz)
out = np.column_stack([res.V, res.E])
path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config0_oracle.txt")
np.savetxt(path, out, fmt="%.17e",
           header="config 0 (seed 0): V Ex Ey Ez per evaluation point, hartree/e and hartree/(e bohr);\n"
                  "written by tests/golden/make_config0_golden.py from oracle/qmmm_oracle.c "
                  "(PAPER.md:59-60 Eq. 4; V = -U_ES)")
print("wrote", path)
