"""CG over an element partition, one rank per GPU (include/nk.h "Distributed").

Each rank sets the library up on its own elements with GLOBAL node ids.  The plan (which nodes other ranks hold,
who the neighbours are, the exchange layout), every kernel and the per-iteration sequence live in the library
(`nk_dist_*`); this file is the caller's side of that interface:

* which elements a rank owns (`element_range`, `brick_partition`) and in what ORDER -- the elements that touch
  another rank's first, so that the library can overlap the halo exchange with ax_e on the rest;
* the transfers, as the callback the library invokes (`nk_exchange_fn`): one grouped send/recv with the
  neighbours and all-gathers of one double, through a communicator object.  `TorchComm` wraps torch.distributed
  (NCCL for CUDA tensors, gloo for the CPU tests); the GPU tests drive several ranks inside one process through
  the same class with an in-process communicator (tests/dist_common.py).

A communicator has `rank`, `world`, `all_gather_object(obj) -> list` (set-up only), `all_gather(send, out)` and
`exchange(send, recv, neighbours)` with neighbours = [(rank, offset, count), ...] on tensors.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .binding import EXCHANGE_FN, Nekbone, _check, _i, _i64, _stream, _vp, load


def element_range(E: int, world: int, rank: int):
    """Contiguous, balanced: the first E % world ranks get one element more."""
    if not (0 <= rank < world) or world < 1:
        raise ValueError("need 0 <= rank < world")
    base, extra = divmod(int(E), int(world))
    e0 = rank * base + min(rank, extra)
    return e0, e0 + base + (1 if rank < extra else 0)


def brick_partition(nx: int, ny: int, nz: int, px: int, py: int, pz: int, rank: int) -> np.ndarray:
    """Element indices (e = ex + nx (ey + ny ez), ascending) of sub-brick `rank` = rx + px (ry + py rz) of a
    px x py x pz partition of an nx x ny x nz brick of elements (balanced per axis)."""
    if not 0 <= rank < px * py * pz:
        raise ValueError("need 0 <= rank < px py pz")
    rx, ry, rz = rank % px, (rank // px) % py, rank // (px * py)
    ax = [np.arange(*element_range(n, p, r)) for n, p, r in ((nx, px, rx), (ny, py, ry), (nz, pz, rz))]
    ez, ey, ex = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return np.sort((ex + nx * (ey + ny * ez)).reshape(-1))


def local_part(E: int, N: int, coords, glo_num, mask, elements):
    """The rank's element-local arrays, elements in the given order: coords (3, L) -> (3, L_r); ids stay GLOBAL.
    `elements` may be an index array or an (e0, e1) range."""
    P = (N + 1) ** 3
    if isinstance(elements, tuple):
        elements = np.arange(elements[0], elements[1])
    elements = np.asarray(elements, dtype=np.int64)
    coords = np.asarray(coords, dtype=np.float64).reshape(3, E, P)
    return (np.ascontiguousarray(coords[:, elements, :].reshape(3, -1)),
            np.ascontiguousarray(np.asarray(glo_num).reshape(E, P)[elements].reshape(-1)),
            np.ascontiguousarray(np.asarray(mask).reshape(E, P)[elements].reshape(-1)))


def candidates(E: int, N: int, glo_num: np.ndarray) -> np.ndarray:
    """nk_dist_candidates: the distinct ids on element boundaries, ascending (HOST; needs no device)."""
    n = N + 1
    glo_num = np.ascontiguousarray(glo_num, dtype=np.int64).reshape(-1)
    out = np.empty(max(1, E * (n ** 3 - max(n - 2, 0) ** 3)), dtype=np.int64)
    cnt = _i64()
    _check(load().nk_dist_candidates(int(E), int(N), glo_num.ctypes.data_as(_vp), out.ctypes.data_as(_vp), C.byref(cnt)))
    return out[:cnt.value].copy()


class TorchComm:
    """torch.distributed (NCCL for CUDA tensors, gloo for CPU tensors) as the communicator."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self._dist, self._group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def all_gather_object(self, obj):
        out = [None] * self.world
        self._dist.all_gather_object(out, obj, group=self._group)
        return out

    def all_gather(self, send, out):
        if send.is_cuda:
            self._dist.all_gather_into_tensor(out, send, group=self._group)
        else:                                     # gloo (CPU tests): the list form
            self._dist.all_gather(list(out.view(self.world, -1).unbind(0)), send, group=self._group)

    def exchange(self, send, recv, neighbours):
        """One grouped send/recv: segment [off, off + cnt) of `send` to, and of `recv` from, every neighbour."""
        d = self._dist
        ops = []
        for r, off, cnt in neighbours:
            ops.append(d.P2POp(d.isend, send[off:off + cnt], r, group=self._group))
            ops.append(d.P2POp(d.irecv, recv[off:off + cnt], r, group=self._group))
        for w in d.batch_isend_irecv(ops) if ops else []:
            w.wait()


class DistNekbone:
    """One rank's share of a mesh.  Vectors are float64 CUDA tensors over the rank's OWN local points, its elements
    in the order `self.elements` (global element indices; interface elements first)."""

    def __init__(self, E: int, N: int, coords, glo_num, mask, comm, elements=None, device="cuda"):
        import torch
        self.comm = comm
        self.rank, self.world = comm.rank, comm.world
        self.E_global, self.N = int(E), int(N)
        P = (self.N + 1) ** 3
        if elements is None:
            elements = np.arange(*element_range(E, self.world, self.rank))
        elements = np.asarray(elements, dtype=np.int64)
        if elements.size == 0:
            raise ValueError("a rank without elements: use at most E ranks")
        glo_all = np.asarray(glo_num, dtype=np.int64).reshape(self.E_global, P)
        # every rank's candidate ids (nodes on element boundaries): which of mine do others hold?
        mine = candidates(elements.size, self.N, glo_all[elements].reshape(-1))
        lists = comm.all_gather_object(mine)
        if self.world > 1:
            ids, counts = np.unique(np.concatenate(lists), return_counts=True)
            touches = np.isin(glo_all[elements], ids[counts > 1]).any(axis=1)
            elements = np.concatenate([elements[touches], elements[~touches]])       # interface elements first
        self.elements = elements
        c, g, m = local_part(E, N, coords, glo_num, mask, elements)
        self.glo_num = g
        self.nk = Nekbone(elements.size, N, c, g, m, device=device)
        self.L = self.nk.L
        self.device = self.nk.device
        lib, ctx = self.nk._lib, self.nk._ctx
        cand = np.ascontiguousarray(np.concatenate(lists), dtype=np.int64)
        cnts = np.array([len(x) for x in lists], dtype=np.int64)
        _check(lib.nk_dist_setup(ctx, self.rank, self.world, g.ctypes.data_as(_vp), cand.ctypes.data_as(_vp),
                                 cnts.ctypes.data_as(_vp), _stream()))
        nn, nx, ni, ne = _i(), _i64(), _i64(), _i64()
        _check(lib.nk_dist_info(ctx, C.byref(nn), C.byref(nx), C.byref(ni), C.byref(ne)))
        self.n_neighbors, self.n_exchange = int(nn.value), int(nx.value)
        self.n_interface_nodes, self.n_interface_elements = int(ni.value), int(ne.value)
        ranks = np.zeros(max(1, self.n_neighbors), dtype=np.int32)
        offs, cnt = np.zeros_like(ranks, dtype=np.int64), np.zeros_like(ranks, dtype=np.int64)
        _check(lib.nk_dist_neighbors(ctx, ranks.ctypes.data_as(_vp), offs.ctypes.data_as(_vp), cnt.ctypes.data_as(_vp)))
        self.neighbours = [(int(ranks[k]), int(offs[k]), int(cnt[k])) for k in range(self.n_neighbors)]
        dev = self.device
        self._send = torch.zeros(max(1, self.n_exchange), dtype=torch.float64, device=dev)
        self._recv = torch.zeros(max(1, self.n_exchange), dtype=torch.float64, device=dev)
        self._ssend = torch.zeros(1, dtype=torch.float64, device=dev)
        self._sgath = torch.zeros(self.world, dtype=torch.float64, device=dev)
        _check(lib.nk_dist_set_buffers(ctx, _vp(self._send.data_ptr()), _vp(self._recv.data_ptr()),
                                       _vp(self._ssend.data_ptr()), _vp(self._sgath.data_ptr())))
        self._cb_error = None
        self._cb = EXCHANGE_FN(self._exchange)               # keep the callback object alive
        self._cb_ptr = C.cast(self._cb, _vp)
        # global multiplicity = gs of ones without the mask (S 8(a) a1), then the weights c = 1/mult
        ones = torch.ones(self.L, dtype=torch.float64, device=dev)
        self.gs(ones, with_mask=False)
        _check(lib.nk_dist_set_mult(ctx, _vp(ones.data_ptr()), _stream()))

    @classmethod
    def from_mesh(cls, mesh, comm, elements=None, device="cuda"):
        return cls(mesh.E, mesh.N, mesh.coords, mesh.glo_num, mesh.mask, comm, elements=elements, device=device)

    def close(self):
        self.nk.close()

    def empty(self):
        return self.nk.empty()

    def local(self, v_global):
        """The rank's part of an element-local vector over the whole mesh (elements in the rank's order)."""
        P = (self.N + 1) ** 3
        return np.ascontiguousarray(np.asarray(v_global).reshape(self.E_global, P)[self.elements].reshape(-1))

    def scatter_into(self, v_global, v_local):
        """Inverse of `local`: writes the rank's entries into a whole-mesh vector (numpy)."""
        P = (self.N + 1) ** 3
        v_global.reshape(self.E_global, P)[self.elements] = np.asarray(v_local).reshape(-1, P)

    # -- the transfers (nk_exchange_fn) -----------------------------------------------------
    def _exchange(self, user, kind, stream):
        import torch
        try:
            s = torch.cuda.ExternalStream(stream) if stream else torch.cuda.default_stream(self.device)
            with torch.cuda.stream(s):
                if kind & 1:
                    self.comm.exchange(self._send, self._recv, self.neighbours)
                if kind & 2:
                    self.comm.all_gather(self._ssend, self._sgath)
            return 0
        except BaseException as e:                           # noqa: BLE001 - re-raised by _call
            self._cb_error = e
            return 1

    def _call(self, rc):
        if self._cb_error is not None:
            e, self._cb_error = self._cb_error, None
            raise e
        _check(rc)

    # -- operators ------------------------------------------------------------------------
    def gs(self, v, with_mask=False):
        """v <- Q Q^T v over ALL ranks (and the Dirichlet mask if asked), in place."""
        self._call(self.nk._lib.nk_dist_gs(self.nk._ctx, self.nk._vec(v, "v"), int(bool(with_mask)), self._cb_ptr, None,
                                           _stream()))
        return v

    def ax(self, u, w=None):
        """w = M Q Q^T A_L u with the sum over all ranks."""
        w = self.nk.ax_e(u, w)
        return self.gs(w, with_mask=True)

    def dot(self, a, b):
        """<a, b>_c over all ranks (c = 1 / global multiplicity): a 1-element CUDA tensor."""
        import torch
        out = torch.empty(1, dtype=torch.float64, device=self.device)
        self._call(self.nk._lib.nk_dist_dot(self.nk._ctx, self.nk._vec(a, "a"), self.nk._vec(b, "b"), _vp(out.data_ptr()),
                                            self._cb_ptr, None, _stream()))
        return out

    def mult(self):
        return self.nk.mult()

    # -- the solver -----------------------------------------------------------------------
    def cg(self, f, niter: int, x=None, res_hist=None):
        """`niter` CG iterations from x = 0 (fixed count, no preconditioner).  Returns (x, history);
        history[k] = sqrt(<r_k, r_k>_c), the same on every rank.  One library call: the sequence of kernels and
        transfers of every iteration is nk_dist_cg's."""
        import torch
        x = self.empty() if x is None else x
        hist = torch.empty(niter + 1, dtype=torch.float64, device=self.device) if res_hist is None else res_hist
        if hist.numel() < niter + 1:
            raise ValueError("res_hist too short")
        self._call(self.nk._lib.nk_dist_cg(self.nk._ctx, self.nk._vec(f, "f"), self.nk._vec(x, "x"), int(niter),
                                           _vp(hist.data_ptr()), self._cb_ptr, None, _stream()))
        return x, hist
