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


def oracle_variants(mesh, f, niter):
    """Histories (and solutions) of the oracle's OTHER correct evaluations of the same iteration: the build with
    FMA contraction on, and plain double pairwise-free dot products instead of long double ones.  Their distance
    from the reference run is the oracle's own rounding band (R15)."""
    from oracle.nko import Oracle
    out = []
    ofm = Oracle.from_mesh(mesh, fma=True)
    out.append(ofm.cg(f, niter))
    ofm.close()
    od = Oracle.from_mesh(mesh)
    od.set_dot_mode(1)
    out.append(od.cg(f, niter))
    od.close()
    return out


def history_parity(h_gpu, h_or, h_or_band, tol=1e-10, band_ok=1e-11, converged=1e-9):
    """R15 protocol for a residual history (SURVEY.md 8(c) "CG sensitivity", parts 3-4).

    h_or is the oracle's history, h_or_band one or several histories of other correct evaluations by the
    oracle itself (oracle_variants: contraction on, double instead of long double dot products); the running
    maximum of their relative distance from h_or is the oracle's own rounding band.  Once rounding noise
    grows (x1000 per three iterations on a 63-unknown mesh) a single pair is one sample of it, so the band is
    the maximum over the variants.  Returns (passed, worst, kstar):
      * k with band <= band_ok:   |gpu - or| <= tol * or                      (the flat 1e-10)
      * beyond:                   |gpu - or| <= max(tol, 10 band) * or, or both sides have converged
                                  (<= converged * h[0]: the recursive residual is rounding noise there)
    worst = max relative difference over the flat part, kstar = last index of the flat part."""
    h_gpu, h_or = np.asarray(h_gpu, dtype=np.float64), np.asarray(h_or, dtype=np.float64)
    alts = np.atleast_2d(np.asarray(h_or_band, dtype=np.float64))
    den = np.where(h_or > 0, h_or, 1.0)
    band = np.maximum.accumulate((np.abs(alts - h_or[None, :]) / den[None, :]).max(axis=0))
    diff = np.abs(h_gpu - h_or) / den
    flat = band <= band_ok
    done = (h_gpu <= converged * h_or[0]) & (h_or <= converged * h_or[0])
    ok = np.where(flat, diff <= tol, (diff <= np.maximum(tol, 10.0 * band)) | done)
    kstar = int(np.nonzero(flat)[0].max()) if flat.any() else -1
    worst = float(diff[flat].max()) if flat.any() else float("nan")
    return bool(ok.all()), worst, kstar
