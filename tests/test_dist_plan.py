"""Host side of the distributed path (paper_2606_12650_b200/dist.py, nk_dist_candidates) on
CPU: element ranges and sub-brick partitions, the candidate ids against brute force, and the exchange protocol
(partial sums of interface nodes, neighbour-wise send/recv, totals in rank order) replayed in numpy over gloo with
two and three ranks through the same TorchComm the GPU path uses."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2606_12650_b200.dist import brick_partition, candidates, element_range, local_part   # noqa: E402
from workloads import brick_mesh                                                                 # noqa: E402


@pytest.mark.parametrize("E,world", [(8, 1), (8, 2), (8, 3), (10, 4), (7, 7), (512, 8)])
def test_element_range_partitions(E, world):
    r = [element_range(E, world, k) for k in range(world)]
    assert r[0][0] == 0 and r[-1][1] == E
    assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
    sizes = [b - a for a, b in r]
    assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        element_range(E, world, world)


@pytest.mark.parametrize("brick,part", [((4, 4, 4), (2, 2, 2)), ((6, 4, 3), (3, 2, 1)), ((5, 3, 2), (2, 3, 2)), ((8, 8, 8), (2, 2, 2))])
def test_brick_partition_is_a_partition_into_bricks(brick, part):
    nx, ny, nz = brick
    world = part[0] * part[1] * part[2]
    parts = [brick_partition(nx, ny, nz, *part, r) for r in range(world)]
    allel = np.concatenate(parts)
    assert np.array_equal(np.sort(allel), np.arange(nx * ny * nz))
    for p in parts:
        ex, ey, ez = p % nx, (p // nx) % ny, p // (nx * ny)
        spans = [np.unique(a) for a in (ex, ey, ez)]
        assert p.size == spans[0].size * spans[1].size * spans[2].size            # a full box of elements
        assert all(np.array_equal(s, np.arange(s[0], s[-1] + 1)) for s in spans)
    with pytest.raises(ValueError):
        brick_partition(nx, ny, nz, *part, world)


@pytest.mark.parametrize("N", [1, 2, 3, 5])
def test_candidates_are_the_ids_on_element_boundaries(N):
    """nk_dist_candidates (host code of libnk.so, no device): every id on an element face, nothing else."""
    mesh = brick_mesh(3, 2, 2, N, 0.05)
    n = N + 1
    got = candidates(mesh.E, N, mesh.glo_num)
    idx = np.arange(n)
    on = (idx == 0) | (idx == n - 1)
    face = on[None, None, :] | on[None, :, None] | on[:, None, None]                # (k, j, i)
    want = np.unique(mesh.glo_num.reshape(mesh.E, n, n, n)[:, face])
    assert np.array_equal(got, want)
    # any id two elements share is among them (so is any id two RANKS share)
    ids, cnt = np.unique(mesh.glo_num, return_counts=True)
    assert np.isin(ids[cnt > 1], got).all()


def _local_gs(v, glo):
    _, inv = np.unique(glo, return_inverse=True)
    return np.bincount(inv, weights=v)[inv]


def _plan(rank, lists):
    """What nk_dist_setup derives: neighbours (ascending rank) with the ids shared with each (ascending)."""
    out = []
    for r, other in enumerate(lists):
        if r != rank:
            sh = np.intersect1d(lists[rank], other)
            if sh.size:
                out.append((r, sh))
    return out


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    from paper_2606_12650_b200.dist import TorchComm
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    comm = TorchComm()
    mesh = brick_mesh(2, 2, 3, 3, 0.05)
    P = mesh.n ** 3
    els = np.arange(*element_range(mesh.E, world, rank))
    _, glo, _ = local_part(mesh.E, mesh.N, mesh.coords, mesh.glo_num, mesh.mask, els)
    lists = comm.all_gather_object(candidates(els.size, mesh.N, glo))
    plan = _plan(rank, lists)
    v = np.random.Generator(np.random.PCG64(4)).integers(-8, 9, mesh.L).astype(np.float64)   # exact sums
    vl = v.reshape(mesh.E, P)[els].reshape(-1)
    w = _local_gs(vl, glo)                                         # this rank's own sums
    first = {int(g): int(np.nonzero(glo == g)[0][0]) for _, sh in plan for g in sh}
    send = torch.tensor([w[first[int(g)]] for _, sh in plan for g in sh], dtype=torch.float64)
    recv = torch.zeros_like(send)
    nbrs, off = [], 0
    for r, sh in plan:
        nbrs.append((r, off, sh.size))
        off += sh.size
    comm.exchange(send, recv, nbrs)
    # totals in ascending rank order over the holders
    got = w.copy()
    iface = np.unique(np.concatenate([sh for _, sh in plan])) if plan else np.zeros(0, dtype=np.int64)
    for g in iface:
        terms = [(rank, w[first[int(g)]])]
        for (r, o, c), (_, sh) in zip(nbrs, plan):
            k = np.searchsorted(sh, g)
            if k < sh.size and sh[k] == g:
                terms.append((r, float(recv[o + k])))
        got[glo == g] = sum(t for _, t in sorted(terms))
    want = _local_gs(v, mesh.glo_num).reshape(mesh.E, P)[els].reshape(-1)
    # the scalar path: an all-gather of one double per rank, summed in rank order
    s = torch.tensor([float(rank + 1)], dtype=torch.float64)
    out = torch.zeros(world, dtype=torch.float64)
    comm.all_gather(s, out)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, bool(np.array_equal(got, want)), len(plan), out.tolist()))


@pytest.mark.parametrize("world", [2, 3])
def test_gloo_ranks_neighbour_exchange(world):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000 + world
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=240) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(r[1] for r in res)
    assert all(r[2] >= 1 for r in res)
    assert all(r[3] == [float(k + 1) for k in range(world)] for r in res)
