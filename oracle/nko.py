"""ctypes binding of the oracle library (libnko.so).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this module.  It never imports `paper_2606_12650_b200`.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_c_double_p = C.POINTER(C.c_double)
_c_int64_p = C.POINTER(C.c_int64)


class NkoError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"nko error {code}: {msg}")
        self.code = code


NKO_ERR_ARG, NKO_ERR_ALLOC, NKO_ERR_ID, NKO_ERR_MASK, NKO_ERR_GEOM = -1, -2, -3, -4, -5

_libs = {}


def _load(fma: bool = False):
    key = bool(fma)
    if key in _libs:
        return _libs[key]
    _build.build()
    path = _build.LIB_FMA if fma else _build.LIB
    lib = C.CDLL(path)
    vp = C.c_void_p
    sig = {
        "nko_basis": [C.c_int, vp, vp, vp],
        "nko_setup": [C.POINTER(vp), C.c_int64, C.c_int, vp, vp, vp],
        "nko_ax_e": [vp, vp, vp],
        "nko_gs": [vp, vp],
        "nko_mask": [vp, vp],
        "nko_ax": [vp, vp, vp],
        "nko_dot": [vp, vp, vp, vp],
        "nko_cg": [vp, vp, vp, C.c_int, vp],
        "nko_pcg": [vp, vp, vp, C.c_int, vp],
        "nko_diag": [vp, vp],
        "nko_cg_step": [vp, vp, vp, vp, vp, vp],
        "nko_cg_init": [vp, vp, vp, vp, vp, vp],
        "nko_set_dot_mode": [vp, C.c_int],
        "nko_get_sizes": [vp, vp, vp, vp, vp],
        "nko_get_mult": [vp, vp],
        "nko_get_geom": [vp, vp, vp],
        "nko_get_D": [vp, vp, vp, vp],
    }
    for name, args in sig.items():
        fn = getattr(lib, name)
        fn.argtypes = args
        fn.restype = C.c_int
    lib.nko_free.argtypes = [vp]
    lib.nko_free.restype = None
    lib.nko_num_threads.argtypes = []
    lib.nko_num_threads.restype = C.c_int
    lib.nko_set_num_threads.argtypes = [C.c_int]
    lib.nko_set_num_threads.restype = None
    lib.nko_strerror.argtypes = [C.c_int]
    lib.nko_strerror.restype = C.c_char_p
    _libs[key] = lib
    return lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None and a.shape != shape:
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _check(lib, rc: int):
    if rc != 0:
        raise NkoError(rc, lib.nko_strerror(rc).decode())


def num_threads() -> int:
    return int(_load().nko_num_threads())


def set_num_threads(n: int) -> None:
    """OpenMP threads of later calls (bench.py's 1-thread figure); values do not depend on it."""
    _load().nko_set_num_threads(int(n))


def basis(N: int, fma: bool = False):
    """(xi, w, D) for order N -- O1."""
    lib = _load(fma)
    n = N + 1
    xi, w, D = np.empty(n), np.empty(n), np.empty((n, n))
    _check(lib, lib.nko_basis(N, _p(xi), _p(w), _p(D)))
    return xi, w, D


class Oracle:
    """One mesh.  Vectors are float64 numpy arrays of length L in element-local layout."""

    def __init__(self, E: int, N: int, coords, glo_num, mask, fma: bool = False):
        self._lib = _load(fma)
        self._ctx = C.c_void_p()
        n = N + 1
        self.E, self.N, self.n = int(E), int(N), n
        self.L = self.E * n ** 3
        coords = _f64(coords).reshape(-1)
        glo_num = np.ascontiguousarray(glo_num, dtype=np.int64)
        mask = _f64(mask)
        if coords.size != 3 * self.L or glo_num.size != self.L or mask.size != self.L:
            raise ValueError("coords/glo_num/mask size does not match E*(N+1)^3")
        rc = self._lib.nko_setup(C.byref(self._ctx), self.E, self.N, _p(coords), _p(glo_num), _p(mask))
        _check(self._lib, rc)

    @classmethod
    def from_mesh(cls, mesh, fma: bool = False):
        return cls(mesh.E, mesh.N, mesh.coords, mesh.glo_num, mesh.mask, fma=fma)

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx:
            self._lib.nko_free(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- operators -----------------------------------------------------------------------
    def ax_e(self, u):
        u = _f64(u, (self.L,))
        w = np.empty(self.L)
        _check(self._lib, self._lib.nko_ax_e(self._ctx, _p(u), _p(w)))
        return w

    def gs(self, v):
        v = np.array(v, dtype=np.float64, copy=True)
        _check(self._lib, self._lib.nko_gs(self._ctx, _p(v)))
        return v

    def mask(self, v):
        v = np.array(v, dtype=np.float64, copy=True)
        _check(self._lib, self._lib.nko_mask(self._ctx, _p(v)))
        return v

    def ax(self, u):
        u = _f64(u, (self.L,))
        w = np.empty(self.L)
        _check(self._lib, self._lib.nko_ax(self._ctx, _p(u), _p(w)))
        return w

    def dot(self, a, b) -> float:
        a, b = _f64(a, (self.L,)), _f64(b, (self.L,))
        out = np.empty(1)
        _check(self._lib, self._lib.nko_dot(self._ctx, _p(a), _p(b), _p(out)))
        return float(out[0])

    def cg(self, f, niter: int):
        f = _f64(f, (self.L,))
        x = np.empty(self.L)
        hist = np.empty(niter + 1)
        _check(self._lib, self._lib.nko_cg(self._ctx, _p(f), _p(x), int(niter), _p(hist)))
        return x, hist

    def pcg(self, f, niter: int):
        """Jacobi-preconditioned CG."""
        f = _f64(f, (self.L,))
        x = np.empty(self.L)
        hist = np.empty(niter + 1)
        _check(self._lib, self._lib.nko_pcg(self._ctx, _p(f), _p(x), int(niter), _p(hist)))
        return x, hist

    def diag(self):
        """Q Q^T diag(A_L) in local layout."""
        d = np.empty(self.L)
        _check(self._lib, self._lib.nko_diag(self._ctx, _p(d)))
        return d

    def cg_init(self, f):
        f = _f64(f, (self.L,))
        x, r, p = np.empty(self.L), np.empty(self.L), np.empty(self.L)
        rho = np.empty(1)
        _check(self._lib, self._lib.nko_cg_init(self._ctx, _p(f), _p(x), _p(r), _p(p), _p(rho)))
        return x, r, p, float(rho[0])

    def cg_step(self, x, r, p, rho: float):
        """One iteration; x, r, p (numpy arrays) are updated IN PLACE.  Returns (w, dict)."""
        for a in (x, r, p):
            if a.dtype != np.float64 or not a.flags.c_contiguous or a.shape != (self.L,):
                raise ValueError("x, r, p must be contiguous float64 arrays of length L")
        w = np.empty(self.L)
        scal = np.zeros(5)
        scal[0] = rho
        _check(self._lib, self._lib.nko_cg_step(self._ctx, _p(x), _p(r), _p(p), _p(w), _p(scal)))
        return w, dict(rho=scal[0], pap=scal[1], alpha=scal[2], rho_new=scal[3], beta=scal[4])

    def set_dot_mode(self, mode: int):
        _check(self._lib, self._lib.nko_set_dot_mode(self._ctx, int(mode)))

    # -- introspection -------------------------------------------------------------------
    def sizes(self):
        v = [C.c_int64() for _ in range(4)]
        _check(self._lib, self._lib.nko_get_sizes(self._ctx, *[C.byref(a) for a in v]))
        return dict(n_local=v[0].value, n_unique=v[1].value,
                    n_shared_unique=v[2].value, n_masked_unique=v[3].value)

    def mult(self):
        m = np.empty(self.L)
        _check(self._lib, self._lib.nko_get_mult(self._ctx, _p(m)))
        return m

    def geom(self):
        G = np.empty((6, self.L))
        J = np.empty(self.L)
        _check(self._lib, self._lib.nko_get_geom(self._ctx, _p(G), _p(J)))
        return G, J

    def basis(self):
        n = self.n
        D, xi, w = np.empty((n, n)), np.empty(n), np.empty(n)
        _check(self._lib, self._lib.nko_get_D(self._ctx, _p(D), _p(xi), _p(w)))
        return xi, w, D
