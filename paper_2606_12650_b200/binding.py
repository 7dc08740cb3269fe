"""Thin ctypes binding of libnk.so (include/nk.h): argument marshalling only.

Every numerical step runs in the CUDA kernels behind the C-ABI; PyTorch supplies device memory
(`torch.Tensor.data_ptr()`) and the current stream.  There is no CPU fallback: if libnk.so is
missing, `load()` raises; on a box without a CUDA device every compute call returns NK_ERR_CUDA.
This module never imports `oracle`.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libnk.so")

NK_OK, NK_ERR_ARG, NK_ERR_WORKSPACE, NK_ERR_ID, NK_ERR_MASK = 0, -1, -2, -3, -4
NK_ERR_GEOM, NK_ERR_CUDA, NK_ERR_ALLOC, NK_ERR_MULT = -5, -6, -7, -8

# every symbol include/nk.h declares: name -> (restype, argtypes)
_vp, _i, _i64, _sz, _d = C.c_void_p, C.c_int, C.c_int64, C.c_size_t, C.c_double
EXCHANGE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int, C.c_void_p)        # nk_exchange_fn
SIGNATURES = {
    "nk_workspace_bytes": (_i, [_i64, _i, C.POINTER(_sz)]),
    "nk_setup": (_i, [C.POINTER(_vp), _i64, _i, _vp, _vp, _vp, _vp, _sz, _vp]),
    "nk_free": (None, [_vp]),
    "nk_set_host_threads": (_i, [_i]),
    "nk_static_setup": (_i, []),
    "nk_dot_static_max_n": (_i64, []),
    "nk_dot_static": (_i, [_vp, _vp, _vp, _i64, _vp, _vp]),
    "nk_set_plan_builder": (_i, [_i]),
    "nk_ax_e": (_i, [_vp, _vp, _vp, _vp]),
    "nk_gs": (_i, [_vp, _vp, _vp]),
    "nk_ax": (_i, [_vp, _vp, _vp, _vp]),
    "nk_dot": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "nk_cg": (_i, [_vp, _vp, _vp, _i, _vp, _vp]),
    "nk_pcg": (_i, [_vp, _vp, _vp, _i, _vp, _vp]),
    "nk_get_diag": (_i, [_vp, _vp, _vp]),
    "nk_cg_host": (_i, [_vp, _vp, _vp, _i, _vp, _vp]),
    "nk_cg_host_batch": (_i, [_vp, _i, _vp, _vp, _i, _vp, _vp]),
    "nk_cg_init": (_i, [_vp, _vp, _vp, _vp]),
    "nk_cg_load_state": (_i, [_vp, _vp, _vp, _d, _vp]),
    "nk_cg_step": (_i, [_vp, _vp, _vp]),
    "nk_cg_get_state": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "nk_get_scalars": (_i, [_vp, _vp, _vp]),
    "nk_set_option": (_i, [_vp, C.c_char_p, _i]),
    "nk_get_option": (_i, [_vp, C.c_char_p, C.POINTER(_i)]),
    "nk_get_sizes": (_i, [_vp, C.POINTER(_i64), C.POINTER(_i64), C.POINTER(_i64), C.POINTER(_i64)]),
    "nk_get_setup_info": (_i, [_vp, C.POINTER(_i), C.POINTER(_d), C.POINTER(_d)]),
    "nk_get_plan_array": (_i, [_vp, _i, C.POINTER(_vp), C.POINTER(_sz)]),
    "nk_get_gs_sizes": (_i, [_vp, C.POINTER(_i64), C.POINTER(_i64), C.POINTER(_i64)]),
    "nk_get_mult": (_i, [_vp, _vp, _vp]),
    "nk_get_geom": (_i, [_vp, _vp, _vp]),
    "nk_get_D": (_i, [_vp, _vp, _vp, _vp]),
    "nk_get_kernel_times": (_i, [_vp, _vp, _vp, _vp]),
    "nk_dist_candidates": (_i, [_i64, _i, _vp, _vp, C.POINTER(_i64)]),
    "nk_dist_setup": (_i, [_vp, _i, _i, _vp, _vp, _vp, _vp]),
    "nk_dist_info": (_i, [_vp, C.POINTER(_i), C.POINTER(_i64), C.POINTER(_i64), C.POINTER(_i64)]),
    "nk_dist_neighbors": (_i, [_vp, _vp, _vp, _vp]),
    "nk_dist_set_buffers": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "nk_dist_set_mult": (_i, [_vp, _vp, _vp]),
    "nk_dist_gs": (_i, [_vp, _vp, _i, _vp, _vp, _vp]),
    "nk_dist_dot": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "nk_dist_cg": (_i, [_vp, _vp, _vp, _i, _vp, _vp, _vp, _vp]),
    "nk_get_launch_count": (_i, [_vp, C.POINTER(_i64)]),
    "nk_get_cg_path": (_i, [_vp, C.POINTER(_i), C.POINTER(_i)]),
    "nk_fp64_peak": (_i, [C.POINTER(_d), C.POINTER(_d), _vp]),
    "nk_ax_batch_elements": (_i, [_i]),
    "nk_get_ax_launch": (_i, [_vp, C.POINTER(_i), C.POINTER(_i), C.POINTER(_i64)]),
    "nk_strerror": (C.c_char_p, [_i]),
    "nk_last_cuda_error": (_i, []),
    "nk_version": (C.c_char_p, []),
}

_lib = None


class NkError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"nk error {code}: {msg}")
        self.code = code


def load():
    """dlopen libnk.so (built in-tree by `python -m paper_2606_12650_b200.build`).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: run `python -m paper_2606_12650_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _check(rc: int):
    if rc != NK_OK:
        raise NkError(rc, load().nk_strerror(rc).decode())


def workspace_bytes(E: int, N: int) -> int:
    out = _sz()
    _check(load().nk_workspace_bytes(int(E), int(N), C.byref(out)))
    return int(out.value)


def ax_batch_elements(N: int) -> int:
    """Elements per batch of the persistent ax_e kernel of order N (a compile-time constant)."""
    rc = load().nk_ax_batch_elements(int(N))
    if rc <= 0:
        _check(rc if rc < 0 else NK_ERR_ARG)
    return int(rc)


def fp64_peak() -> dict:
    """DFMA-only microbenchmark on the current device: measured fp64 TFLOP/s (2 flops per DFMA)."""
    t, r = _d(), _d()
    _check(load().nk_fp64_peak(C.byref(t), C.byref(r), _stream()))
    return dict(tflops=float(t.value), dfma_per_clk_per_sm_at_max_clock=float(r.value))


def set_host_threads(n: int) -> None:
    """Host threads of later set-ups (0 = all cores); the plan they build does not depend on it."""
    _check(load().nk_set_host_threads(int(n)))


def dot_static_max_n() -> int:
    return int(load().nk_dot_static_max_n())


def dot_static(a, b, c=None, out=None, n=None):
    """out[0] = sum c_i a_i b_i (c None: plain dot) over CUDA float64 tensors, through nk_dot_static: no context, no
    workspace, no allocation inside the call (scratch is a fixed __device__ array in the library; n <= 2^27)."""
    import torch
    n = a.numel() if n is None else int(n)
    for t in (a, b) + (() if c is None else (c,)):
        if t.dtype != torch.float64 or not t.is_cuda or not t.is_contiguous() or t.numel() < n:
            raise ValueError("contiguous CUDA float64 tensors of at least n entries")
    out = torch.empty(1, dtype=torch.float64, device=a.device) if out is None else out
    _check(load().nk_dot_static(_vp(a.data_ptr()), _vp(b.data_ptr()), _vp(c.data_ptr()) if c is not None else None,
                                n, _vp(out.data_ptr()), _stream()))
    return out


def set_plan_builder(which: str) -> None:
    """Builder of the gather-scatter plan in later set-ups: "device" (default) or "host"; same arrays bit for bit."""
    _check(load().nk_set_plan_builder({"device": 0, "host": 1}[which]))


def _np_ptr(a: np.ndarray):
    return a.ctypes.data_as(_vp)


def _stream():
    import torch
    return _vp(torch.cuda.current_stream().cuda_stream)


class Nekbone:
    """One mesh on the current CUDA device.  Vectors are float64 CUDA tensors of length L."""

    def __init__(self, E: int, N: int, coords, glo_num, mask, device="cuda"):
        import torch
        self._lib = load()
        self._ctx = _vp()
        self.E, self.N, self.n = int(E), int(N), int(N) + 1
        self.L = self.E * self.n ** 3
        self.device = torch.device(device)
        coords = np.ascontiguousarray(coords, dtype=np.float64).reshape(-1)
        glo_num = np.ascontiguousarray(glo_num, dtype=np.int64).reshape(-1)
        mask = np.ascontiguousarray(mask, dtype=np.float64).reshape(-1)
        if coords.size != 3 * self.L or glo_num.size != self.L or mask.size != self.L:
            raise ValueError("coords/glo_num/mask size does not match E*(N+1)^3")
        nbytes = workspace_bytes(self.E, self.N)
        # caller-owned workspace: one torch allocation (256-B aligned by the caching allocator)
        self._ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        with torch.cuda.device(self.device):
            rc = self._lib.nk_setup(C.byref(self._ctx), self.E, self.N, _np_ptr(coords), _np_ptr(glo_num),
                                    _np_ptr(mask), _vp(self._ws.data_ptr()), nbytes, _stream())
        _check(rc)

    @classmethod
    def from_mesh(cls, mesh, device="cuda"):
        return cls(mesh.E, mesh.N, mesh.coords, mesh.glo_num, mesh.mask, device=device)

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx:
            self._lib.nk_free(self._ctx)
            self._ctx = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers -------------------------------------------------------------------------
    def _vec(self, t, name="vector"):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64
                and t.is_contiguous() and t.numel() == self.L):
            raise ValueError(f"{name}: need a contiguous float64 CUDA tensor of length {self.L}")
        return _vp(t.data_ptr())

    def empty(self):
        import torch
        return torch.empty(self.L, dtype=torch.float64, device=self.device)

    # -- operators -----------------------------------------------------------------------
    def ax_e(self, u, w=None):
        w = self.empty() if w is None else w
        _check(self._lib.nk_ax_e(self._ctx, self._vec(u, "u"), self._vec(w, "w"), _stream()))
        return w

    def gs(self, v):
        """In place."""
        _check(self._lib.nk_gs(self._ctx, self._vec(v, "v"), _stream()))
        return v

    def ax(self, u, w=None):
        w = self.empty() if w is None else w
        _check(self._lib.nk_ax(self._ctx, self._vec(u, "u"), self._vec(w, "w"), _stream()))
        return w

    def dot(self, a, b, out=None):
        import torch
        out = torch.empty(1, dtype=torch.float64, device=self.device) if out is None else out
        _check(self._lib.nk_dot(self._ctx, self._vec(a, "a"), self._vec(b, "b"), _vp(out.data_ptr()), _stream()))
        return out

    def cg(self, f, niter: int, x=None, res_hist=None):
        """Device-resident CG: returns (x, res_hist) CUDA tensors; does not synchronise.
        On meshes where nk_cg replays a recorded CUDA graph (it keeps the last two, keyed by f, x, res_hist, niter and
        the options) pass the same x and res_hist tensors on every call: fresh ones mean a new capture each time."""
        import torch
        x = self.empty() if x is None else x
        if res_hist is None:
            res_hist = torch.empty(int(niter) + 1, dtype=torch.float64, device=self.device)
        _check(self._lib.nk_cg(self._ctx, self._vec(f, "f"), self._vec(x, "x"), int(niter),
                               _vp(res_hist.data_ptr()), _stream()))
        return x, res_hist

    def pcg(self, f, niter: int, x=None, res_hist=None):
        """Jacobi-preconditioned CG: returns (x, res_hist) CUDA tensors."""
        import torch
        x = self.empty() if x is None else x
        if res_hist is None:
            res_hist = torch.empty(int(niter) + 1, dtype=torch.float64, device=self.device)
        _check(self._lib.nk_pcg(self._ctx, self._vec(f, "f"), self._vec(x, "x"), int(niter),
                                _vp(res_hist.data_ptr()), _stream()))
        return x, res_hist

    def diag(self):
        d = self.empty()
        _check(self._lib.nk_get_diag(self._ctx, self._vec(d), _stream()))
        return d

    def cg_host(self, f_host: np.ndarray, niter: int, x_host=None, hist_host=None):
        """End-to-end call with HOST buffers (numpy, ideally pinned): H2D f, CG, D2H x + history."""
        if f_host.dtype != np.float64 or f_host.size != self.L or not f_host.flags.c_contiguous:
            raise ValueError("f_host: contiguous float64 array of length L")
        x_host = np.empty(self.L) if x_host is None else x_host
        hist_host = np.empty(int(niter) + 1) if hist_host is None else hist_host
        _check(self._lib.nk_cg_host(self._ctx, _np_ptr(f_host), _np_ptr(x_host), int(niter),
                                    _np_ptr(hist_host), _stream()))
        return x_host, hist_host

    def cg_host_batch(self, f_hosts, niter: int, x_hosts, hist_hosts):
        """Several solves with HOST buffers (lists of numpy arrays, ideally pinned), copies overlapped with the solves."""
        n = len(f_hosts)
        if len(x_hosts) != n or len(hist_hosts) != n:
            raise ValueError("f_hosts, x_hosts, hist_hosts: lists of equal length")
        for f, x, h in zip(f_hosts, x_hosts, hist_hosts):
            for a, size in ((f, self.L), (x, self.L), (h, int(niter) + 1)):
                if a.dtype != np.float64 or a.size != size or not a.flags.c_contiguous:
                    raise ValueError("contiguous float64 arrays of length L, L, niter + 1")
        arr = lambda xs: (C.c_void_p * max(n, 1))(*[a.ctypes.data for a in xs])
        fa, xa, ha = arr(f_hosts), arr(x_hosts), arr(hist_hosts)
        _check(self._lib.nk_cg_host_batch(self._ctx, n, fa, xa, int(niter), ha, _stream()))
        return x_hosts, hist_hosts

    # -- lock-step test entry points -----------------------------------------------------
    def cg_init(self, f, x):
        _check(self._lib.nk_cg_init(self._ctx, self._vec(f, "f"), self._vec(x, "x"), _stream()))

    def cg_load_state(self, r, p, rho: float):
        _check(self._lib.nk_cg_load_state(self._ctx, self._vec(r, "r"), self._vec(p, "p"), float(rho), _stream()))

    def cg_step(self, x):
        _check(self._lib.nk_cg_step(self._ctx, self._vec(x, "x"), _stream()))

    def cg_get_state(self):
        r, p, w = self.empty(), self.empty(), self.empty()
        _check(self._lib.nk_cg_get_state(self._ctx, self._vec(r), self._vec(p), self._vec(w), _stream()))
        return r, p, w

    def scalars(self) -> dict:
        out = np.empty(5)
        _check(self._lib.nk_get_scalars(self._ctx, _np_ptr(out), _stream()))
        return dict(rho=out[0], pap=out[1], alpha=out[2], rho_new=out[3], beta=out[4])

    # -- options / introspection ---------------------------------------------------------
    def set_option(self, name: str, value: int):
        _check(self._lib.nk_set_option(self._ctx, name.encode(), int(value)))

    def get_option(self, name: str) -> int:
        v = _i()
        _check(self._lib.nk_get_option(self._ctx, name.encode(), C.byref(v)))
        return int(v.value)

    def sizes(self) -> dict:
        v = [_i64() for _ in range(4)]
        _check(self._lib.nk_get_sizes(self._ctx, *[C.byref(a) for a in v]))
        return dict(n_local=v[0].value, n_unique=v[1].value, n_shared_unique=v[2].value,
                    n_masked_unique=v[3].value)

    def gs_sizes(self) -> dict:
        v = [_i64() for _ in range(3)]
        _check(self._lib.nk_get_gs_sizes(self._ctx, *[C.byref(a) for a in v]))
        return dict(n_rows=v[0].value, n_listed=v[1].value, n_sum_rows=v[2].value)

    def setup_info(self) -> dict:
        b, tp, tt = _i(), _d(), _d()
        _check(self._lib.nk_get_setup_info(self._ctx, C.byref(b), C.byref(tp), C.byref(tt)))
        return dict(plan_builder=("device", "host")[b.value], plan_s=tp.value, total_s=tt.value)

    PLAN_ARRAYS = ("code", "row_off", "row_idx", "pk", "gs_desc", "nbr", "gx", "gx_rows", "gx_blk", "ctab", "mtab")

    def plan_arrays(self) -> dict:
        """The arrays of the gather-scatter plan as byte views of the workspace (name -> uint8 tensor)."""
        out = {}
        for which, name in enumerate(self.PLAN_ARRAYS):
            ptr, n = _vp(), _sz()
            _check(self._lib.nk_get_plan_array(self._ctx, which, C.byref(ptr), C.byref(n)))
            start = (ptr.value or 0) - self._ws.data_ptr()
            assert 0 <= start and start + n.value <= self._ws.numel()
            out[name] = self._ws[start:start + n.value]
        return out

    def mult(self):
        m = self.empty()
        _check(self._lib.nk_get_mult(self._ctx, self._vec(m), _stream()))
        return m

    def geom(self):
        import torch
        G = torch.empty(6 * self.L, dtype=torch.float64, device=self.device)
        _check(self._lib.nk_get_geom(self._ctx, _vp(G.data_ptr()), _stream()))
        return G.view(6, self.L)

    def basis(self):
        n = self.n
        D, xi, w = np.empty((n, n)), np.empty(n), np.empty(n)
        _check(self._lib.nk_get_D(self._ctx, _np_ptr(D), _np_ptr(xi), _np_ptr(w)))
        return xi, w, D

    KERNEL_CLASSES = ("ax_e", "gs", "dot", "update_xr", "update_p", "cg_init")

    def kernel_times(self) -> dict:
        """{class: (total device ms, launches)} recorded since the last call (option "profile" = 1)."""
        ms, cnt = np.zeros(6), np.zeros(6, dtype=np.int64)
        _check(self._lib.nk_get_kernel_times(self._ctx, _np_ptr(ms), _np_ptr(cnt), _stream()))
        return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(self.KERNEL_CLASSES)}

    def ax_launch(self) -> dict:
        """How ax_e is scheduled here: elements per batch, persistent CTAs, batches of the busiest CTA."""
        e, g, b = _i(), _i(), _i64()
        _check(self._lib.nk_get_ax_launch(self._ctx, C.byref(e), C.byref(g), C.byref(b)))
        return dict(batch_elements=int(e.value), ctas=int(g.value), max_batches_per_cta=int(b.value))

    CG_PATHS = ("launches", "graph", "cooperative")

    def solve_path(self) -> str:
        """How nk_cg runs with the current options: "launches" (one by one), "graph" (CUDA graph replay) or
        "cooperative" (one persistent cooperative launch for the whole solve)."""
        v = _i()
        _check(self._lib.nk_get_cg_path(self._ctx, C.byref(v), None))
        return self.CG_PATHS[int(v.value)]

    def pdl_effective(self) -> int:
        """The "pdl" option resolved for this mesh: 0 plain launches, 1 ax_e and the vector kernels are
        programmatic dependents, 2 the kernels with gathers too."""
        v, m = _i(), _i()
        _check(self._lib.nk_get_cg_path(self._ctx, C.byref(v), C.byref(m)))
        return int(m.value)

    def launch_count(self) -> int:
        v = _i64()
        _check(self._lib.nk_get_launch_count(self._ctx, C.byref(v)))
        return int(v.value)
