"""Shared helpers for the GPU parity tests: run the CUDA path and the oracle on the same tensors."""
import numpy as np
import torch

import oracle
from paper_2607_07740_b200 import workloads as W

# BASELINE.json north_star tolerances
TOL = {torch.bfloat16: dict(out_abs=2e-2, out_rel=5e-3, lse=1e-3),
       torch.float32: dict(out_abs=1e-4, out_rel=1e-4, lse=1e-5)}


def oracle_rows(Q, K, V, rows, heads, *, w_local, w_pretrained, rope_theta, mode="bifocal", q_pos_rows=None):
    """Oracle on the same bits: tensors are widened to fp32 (exact) and handed to the fp64 C oracle."""
    Kf = K.float().cpu().numpy()
    Vf = V.float().cpu().numpy()
    ri = torch.as_tensor(rows, dtype=torch.long)
    hi = torch.as_tensor(heads, dtype=torch.long)
    Qr = Q[ri.to(Q.device) if q_pos_rows is None else torch.as_tensor(q_pos_rows).to(Q.device), hi.to(Q.device)]
    Qr = Qr.float().cpu().numpy()
    return oracle.attend_rows((Qr, Q.shape[1]), Kf, Vf, rows, heads, w_local=w_local, w_pretrained=w_pretrained,
                              rope_theta=rope_theta, mode=mode, q_is_compact=True)


def check(out_gpu, lse_gpu, out_ref, lse_ref, dtype, what=""):
    """out_gpu [n,d] tensor, lse_gpu [n]; refs are float64 numpy.  Asserts the north_star tolerances."""
    tol = TOL[dtype]
    og = out_gpu.double().cpu().numpy()
    lg = lse_gpu.double().cpu().numpy()
    assert np.isfinite(og).all() and np.isfinite(lg).all(), what + ": non-finite output"
    err_abs = np.abs(og - out_ref).max()
    rel = np.linalg.norm(og - out_ref) / max(np.linalg.norm(out_ref), 1e-30)
    err_lse = np.abs(lg - lse_ref).max()
    msg = "%s: out max-abs %.3e (tol %.0e), rel-L2 %.3e (tol %.0e), lse %.3e (tol %.0e)" % (
        what, err_abs, tol["out_abs"], rel, tol["out_rel"], err_lse, tol["lse"])
    assert err_abs <= tol["out_abs"] and rel <= tol["out_rel"] and err_lse <= tol["lse"], msg
    return dict(out_abs=float(err_abs), out_rel=float(rel), lse=float(err_lse))


def gather(out, lse, rows, heads):
    ri = torch.as_tensor(rows, dtype=torch.long, device=out.device)
    hi = torch.as_tensor(heads, dtype=torch.long, device=out.device)
    return out[ri, hi], lse[hi, ri]


def all_pairs(L, H_q):
    rows = np.repeat(np.arange(L, dtype=np.int64), H_q)
    heads = np.tile(np.arange(H_q, dtype=np.int32), L)
    return rows, heads
