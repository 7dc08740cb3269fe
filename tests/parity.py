"""Parity metric of DESIGN.md reading R14 (SURVEY.md 8(c) "tolerance metric"), used by the -m gpu tests.

pass  <=>  for all l: |gpu_l - or_l| <= tol * max(|or_l|, S_l)
S_l = max |or| over the element containing l  (ax_e, ax, G, x, r, p)
    = max |addend| over the copies of l's node (gs)
"""
import numpy as np


def elem_scale(ref: np.ndarray, P: int) -> np.ndarray:
    s = np.abs(ref.reshape(-1, P)).max(axis=1)
    return np.repeat(s, P)


def scaled_err(got: np.ndarray, ref: np.ndarray, scale: np.ndarray) -> float:
    """max_l |got-ref| / max(|ref|, scale); 0/0 counts as 0 (both exactly zero)."""
    den = np.maximum(np.abs(ref), scale)
    num = np.abs(got - ref)
    with np.errstate(invalid="ignore", divide="ignore"):
        q = np.where(den > 0, num / den, np.where(num > 0, np.inf, 0.0))
    return float(q.max()) if q.size else 0.0


def elem_err(got, ref, P) -> float:
    return scaled_err(np.asarray(got), np.asarray(ref), elem_scale(np.asarray(ref), P))


def gs_scale(v_in: np.ndarray, glo_num: np.ndarray) -> np.ndarray:
    """max |addend| over the copies of each local point's node."""
    _, inv = np.unique(glo_num, return_inverse=True)
    m = np.zeros(inv.max() + 1)
    np.maximum.at(m, inv, np.abs(v_in))
    return m[inv]


def maxnorm_rel(got, ref) -> float:
    d = np.abs(np.asarray(got) - np.asarray(ref)).max()
    s = np.abs(np.asarray(ref)).max()
    return float(d / s) if s > 0 else float(d)
