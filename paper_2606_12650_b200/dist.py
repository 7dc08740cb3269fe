"""CG over an element partition, one rank per GPU (include/nk.h "Distributed").

Each rank sets the library up on a contiguous range of elements with GLOBAL node ids.  The one exchange
of gather-scatter and the two scalar sums per iteration are all-gathers (torch.distributed, NCCL) issued
between the library's `nk_dist_*` calls on the same stream; all arithmetic is in the library's kernels.

Host side (this file): the element ranges, the interface plan (which global ids more than one rank holds,
one exchange slot each), buffer ownership, and the sequence of calls.  `comm` is anything with
`rank`, `world`, `all_gather_object(obj) -> list` (set-up only) and `all_gather(send, out)` on CUDA
tensors: `TorchComm` wraps torch.distributed; the tests drive several ranks inside one process through
the same class with an in-process communicator.
"""
from __future__ import annotations

import numpy as np

from .binding import Nekbone, _check, _stream, _vp


def element_range(E: int, world: int, rank: int):
    """Contiguous, balanced: the first E % world ranks get one element more."""
    if not (0 <= rank < world) or world < 1:
        raise ValueError("need 0 <= rank < world")
    base, extra = divmod(int(E), int(world))
    e0 = rank * base + min(rank, extra)
    return e0, e0 + base + (1 if rank < extra else 0)


def local_part(E: int, N: int, coords, glo_num, mask, e0: int, e1: int):
    """The rank's slice of element-local arrays: coords (3, L) -> (3, L_r); ids stay GLOBAL."""
    P = (N + 1) ** 3
    coords = np.asarray(coords, dtype=np.float64).reshape(3, E * P)
    sl = slice(e0 * P, e1 * P)
    return (np.ascontiguousarray(coords[:, sl]), np.ascontiguousarray(np.asarray(glo_num).reshape(-1)[sl]),
            np.ascontiguousarray(np.asarray(mask).reshape(-1)[sl]))


def interface_plan(glo_local: np.ndarray, unique_ids_per_rank):
    """Interface nodes = global ids that more than one rank holds; slots in ascending id order (the same list on
    every rank).  Returns (n_slots, pack[n_slots] int32, unpack_loc int32, unpack_slot int32) for this rank:
    pack[s] = first local index carrying slot s's id, -1 if the rank does not hold it; unpack lists every local copy."""
    allids = np.concatenate([np.asarray(u, dtype=np.int64) for u in unique_ids_per_rank])
    ids, counts = np.unique(allids, return_counts=True)
    iface = ids[counts > 1]                                   # ascending
    glo_local = np.asarray(glo_local, dtype=np.int64).reshape(-1)
    pack = np.full(iface.size, -1, dtype=np.int32)
    if iface.size == 0:
        return 0, pack, np.zeros(0, dtype=np.int32), np.zeros(0, dtype=np.int32)
    pos = np.minimum(np.searchsorted(iface, glo_local), iface.size - 1)
    on = iface[pos] == glo_local
    uloc = np.nonzero(on)[0].astype(np.int32)                 # ascending local index
    uslot = pos[on].astype(np.int32)
    held, first = np.unique(uslot, return_index=True)         # first occurrence = smallest local index
    pack[held] = uloc[first]
    return int(iface.size), pack, uloc, uslot


class TorchComm:
    """torch.distributed (NCCL for CUDA tensors) as the communicator."""

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


class DistNekbone:
    """One rank's share of a mesh.  Vectors are float64 CUDA tensors over the rank's OWN local points."""

    def __init__(self, E: int, N: int, coords, glo_num, mask, comm, device="cuda"):
        import torch
        self.comm = comm
        self.rank, self.world = comm.rank, comm.world
        self.E_global, self.N = int(E), int(N)
        self.e0, self.e1 = element_range(E, self.world, self.rank)
        if self.e1 == self.e0:
            raise ValueError("a rank without elements: use at most E ranks")
        c, g, m = local_part(E, N, coords, glo_num, mask, self.e0, self.e1)
        self.glo_num = g
        self.nk = Nekbone(self.e1 - self.e0, N, c, g, m, device=device)
        self.L = self.nk.L
        self.device = self.nk.device
        uniq = comm.all_gather_object(np.unique(g))
        self.n_slots, pack, uloc, uslot = interface_plan(g, uniq)
        dev = self.device
        self._pack = torch.from_numpy(pack).to(dev)
        self._uloc = torch.from_numpy(uloc).to(dev)
        self._uslot = torch.from_numpy(uslot).to(dev)
        S = self.n_slots + 1
        self._send = torch.zeros(S, dtype=torch.float64, device=dev)
        self._gath = torch.zeros(self.world * S, dtype=torch.float64, device=dev)
        self._ssend = torch.zeros(1, dtype=torch.float64, device=dev)
        self._sgath = torch.zeros(self.world, dtype=torch.float64, device=dev)
        lib, ctx = self.nk._lib, self.nk._ctx
        _check(lib.nk_dist_attach(ctx, self.rank, self.world, self.n_slots, _vp(self._pack.data_ptr()), int(uloc.size),
                                  _vp(self._uloc.data_ptr()), _vp(self._uslot.data_ptr()), _vp(self._send.data_ptr()),
                                  _vp(self._gath.data_ptr()), _vp(self._ssend.data_ptr()), _vp(self._sgath.data_ptr())))
        # global multiplicity = gs of ones without the mask (S 8(a) a1), then the weights c = 1/mult
        ones = torch.ones(self.L, dtype=torch.float64, device=dev)
        self.gs(ones, with_mask=False)
        _check(lib.nk_dist_set_mult(ctx, _vp(ones.data_ptr()), _stream()))

    @classmethod
    def from_mesh(cls, mesh, comm, device="cuda"):
        return cls(mesh.E, mesh.N, mesh.coords, mesh.glo_num, mesh.mask, comm, device=device)

    def close(self):
        self.nk.close()

    def empty(self):
        return self.nk.empty()

    def local(self, v_global):
        """The rank's slice of an element-local vector over the whole mesh."""
        P = (self.N + 1) ** 3
        return np.ascontiguousarray(np.asarray(v_global).reshape(-1)[self.e0 * P:self.e1 * P])

    # -- operators ------------------------------------------------------------------------
    def gs(self, v, with_mask=False):
        """v <- Q Q^T v over ALL ranks (and the Dirichlet mask if asked), in place."""
        lib, ctx = self.nk._lib, self.nk._ctx
        _check(lib.nk_dist_gs_begin(ctx, self.nk._vec(v, "v"), int(bool(with_mask)), _stream()))
        self.comm.all_gather(self._send, self._gath)
        _check(lib.nk_dist_gs_end(ctx, self.nk._vec(v, "v"), _stream()))
        return v

    def ax(self, u, w=None):
        """w = M Q Q^T A_L u with the sum over all ranks."""
        w = self.nk.ax_e(u, w)
        return self.gs(w, with_mask=True)

    def dot(self, a, b):
        """<a, b>_c over all ranks (c = 1 / global multiplicity): a 1-element CUDA tensor."""
        import torch
        lib, ctx = self.nk._lib, self.nk._ctx
        out = torch.empty(1, dtype=torch.float64, device=self.device)
        _check(lib.nk_dist_dot_begin(ctx, self.nk._vec(a, "a"), self.nk._vec(b, "b"), _stream()))
        self.comm.all_gather(self._ssend, self._sgath)
        _check(lib.nk_dist_dot_end(ctx, _vp(out.data_ptr()), _stream()))
        return out

    def mult(self):
        return self.nk.mult()

    # -- the solver -----------------------------------------------------------------------
    def cg(self, f, niter: int, x=None, res_hist=None):
        """`niter` CG iterations from x = 0 (fixed count, no preconditioner).  Returns (x, history);
        history[k] = sqrt(<r_k, r_k>_c), the same on every rank."""
        import torch
        lib, ctx = self.nk._lib, self.nk._ctx
        x = self.empty() if x is None else x
        hist = torch.empty(niter + 1, dtype=torch.float64, device=self.device) if res_hist is None else res_hist
        if hist.numel() < niter + 1:
            raise ValueError("res_hist too short")
        h0 = hist.data_ptr()
        xp = self.nk._vec(x, "x")
        _check(lib.nk_dist_cg_begin(ctx, self.nk._vec(f, "f"), xp, _stream()))
        self.comm.all_gather(self._ssend, self._sgath)
        _check(lib.nk_dist_cg_begin_end(ctx, _vp(h0), _stream()))
        for k in range(1, niter + 1):
            _check(lib.nk_dist_iter_a(ctx, _stream()))
            self.comm.all_gather(self._send, self._gath)
            _check(lib.nk_dist_iter_b(ctx, _stream()))
            self.comm.all_gather(self._ssend, self._sgath)
            _check(lib.nk_dist_iter_c(ctx, xp, _vp(h0 + 8 * k), _stream()))
        return x, hist
