"""Offline reconstructor matrix by the fast 2RBT products ("the proposed method can also be used to compute
the tomographic reconstructor off-line, solving Sigma_ss R = Sigma_phi-s one column at a time with the 2RBT MVM").

R = M_phi W_phi Sigma_phi-s W_s^T M_s^T (M_s (W_s Sigma_ss W_s^T + Sigma_eta) M_s^T)^+ M_s        (Eq.5, Eq.12-13)
Column j of R is the whole hot path (tomo_solve_batch: A1-A8) applied to the unit slope vector e_j, so the columns are
independent right-hand sides and go through the batch path max_batch at a time.  Argument marshalling only: every
arithmetic step runs in the library's kernels.
"""
from __future__ import annotations

from typing import Optional, Sequence


def reconstructor_columns(plan, n_iter: int, columns: Optional[Sequence[int]] = None, minres: bool = False):
    """Returns a CUDA tensor [len(columns)][n_targets * n_vphi] (row c = column columns[c] of R); default: all columns."""
    import torch
    cols = list(range(plan.slopes_len)) if columns is None else list(columns)
    B = plan.max_batch
    out = torch.empty((len(cols), plan.wavefront_len), dtype=torch.float32, device="cuda")
    rhs = torch.zeros((B, plan.slopes_len), dtype=torch.float32, device="cuda")
    wf = torch.empty((B, plan.wavefront_len), dtype=torch.float32, device="cuda")
    for c0 in range(0, len(cols), B):
        chunk = cols[c0:c0 + B]
        rhs.zero_()
        rhs[torch.arange(len(chunk), device="cuda"), torch.tensor(chunk, device="cuda")] = 1.0
        if minres:
            plan.solve_minres(rhs, wf, len(chunk), n_iter)
        else:
            plan.solve_batch(rhs, wf, len(chunk), n_iter)
        out[c0:c0 + len(chunk)] = wf[:len(chunk)]
    return out
