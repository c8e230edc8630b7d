"""Writes tests/golden/dphi_anchors.txt: values of the von Karman structure function D_phi (Eq.53,
reading G2) and of the Hudgin / Fried slope variances (Eq.50, Eq.56) computed by the ORACLE only (oracle/vonkarman.py,
oracle/covariance.py).  The library's host builder is checked against this file in tests/test_host_builder.py.

    python tests/golden/make_anchors.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import covariance as cov  # noqa: E402
from oracle import vonkarman as vk  # noqa: E402

r0, L0 = 0.15, 25.0
lines = ["# name | value | r0 | L0 -- written by tests/golden/make_anchors.py from oracle/ only"]
for r in (0.05, 0.2567, 0.5, 1.0, 5.0, 25.0, 74.0):
    lines.append(f"dphi_r{r} | {float(vk.structure_function(np.array(r), r0, L0)):.12e} | {r0} | {L0}")
lines.append(f"dphi_inf | {vk.structure_function_inf(r0, L0):.12e} | {r0} | {L0}")
z = np.zeros((1, 2))
for model in ("hudgin", "fried"):
    v = cov.cov_slope_slope(z, 0, 0, 0.5, 2.0, r0, L0, model)[0]
    lines.append(f"slope_var_{model}_d0.5 | {float(v):.12e} | {r0} | {L0}")
open(os.path.join(ROOT, "tests", "golden", "dphi_anchors.txt"), "w").write("\n".join(lines) + "\n")
print("\n".join(lines))
