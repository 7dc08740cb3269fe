"""Host side of the distributed path (paper_2606_12650_b200/dist.py) on CPU: element
ranges, the interface plan against brute force, and the exchange protocol (local sums, pack, all-gather,
rank-ordered total, unpack) replayed in numpy -- in-process and over gloo with two ranks."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2606_12650_b200.dist import element_range, interface_plan, local_part   # noqa: E402
from workloads import brick_mesh                                                    # noqa: E402


@pytest.mark.parametrize("E,world", [(8, 1), (8, 2), (8, 3), (10, 4), (7, 7), (512, 8)])
def test_element_range_partitions(E, world):
    r = [element_range(E, world, k) for k in range(world)]
    assert r[0][0] == 0 and r[-1][1] == E
    assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
    sizes = [b - a for a, b in r]
    assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        element_range(E, world, world)


def _parts(mesh, world):
    out = []
    for r in range(world):
        e0, e1 = element_range(mesh.E, world, r)
        out.append(local_part(mesh.E, mesh.N, mesh.coords, mesh.glo_num, mesh.mask, e0, e1) + (e0, e1))
    return out


@pytest.mark.parametrize("world", [2, 3, 5])
def test_interface_plan_against_brute_force(world):
    mesh = brick_mesh(3, 2, 2, 3, 0.05)
    parts = _parts(mesh, world)
    uniq = [np.unique(p[1]) for p in parts]
    holders = {}
    for r, u in enumerate(uniq):
        for g in u.tolist():
            holders.setdefault(g, []).append(r)
    iface = sorted(g for g, h in holders.items() if len(h) > 1)
    for r, p in enumerate(parts):
        glo = p[1]
        n_slots, pack, uloc, uslot = interface_plan(glo, uniq)
        assert n_slots == len(iface)
        for s, g in enumerate(iface):
            if r in holders[g]:
                assert glo[pack[s]] == g and pack[s] == np.nonzero(glo == g)[0][0]
            else:
                assert pack[s] == -1
        want = [(l, iface.index(g)) for l, g in enumerate(glo.tolist()) if len(holders[g]) > 1]
        assert list(zip(uloc.tolist(), uslot.tolist())) == want


def _local_gs(v, glo):
    _, inv = np.unique(glo, return_inverse=True)
    return np.bincount(inv, weights=v)[inv]


def _exchange(v_local, glo, plan, gather):
    """The protocol of include/nk.h: local sums, one value per held slot, all-gather, rank-ordered total, unpack."""
    n_slots, pack, uloc, uslot = plan
    w = _local_gs(v_local, glo)
    send = np.where(pack >= 0, w[np.maximum(pack, 0)], 0.0)
    rows = gather(send)
    tot = np.zeros(n_slots)
    for row in rows:
        tot = tot + row
    w[uloc] = tot[uslot]
    return w


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_protocol_equals_global_gather_scatter(world):
    mesh = brick_mesh(2, 3, 2, 4, 0.05)
    v = np.random.Generator(np.random.PCG64(3)).integers(-8, 9, mesh.L).astype(np.float64)   # exact sums
    want = _local_gs(v, mesh.glo_num)
    parts = _parts(mesh, world)
    uniq = [np.unique(p[1]) for p in parts]
    plans = [interface_plan(p[1], uniq) for p in parts]
    P = mesh.n ** 3
    sends = []
    for p, plan in zip(parts, plans):
        w = _local_gs(v[p[3] * P:p[4] * P], p[1])
        sends.append(np.where(plan[1] >= 0, w[np.maximum(plan[1], 0)], 0.0))
    for p, plan in zip(parts, plans):
        got = _exchange(v[p[3] * P:p[4] * P], p[1], plan, lambda send: sends)
        assert np.array_equal(got, want[p[3] * P:p[4] * P])
    # global multiplicity the same way (what DistNekbone feeds nk_dist_set_mult)
    ones_sends = []
    for p, plan in zip(parts, plans):
        w = _local_gs(np.ones(p[1].size), p[1])
        ones_sends.append(np.where(plan[1] >= 0, w[np.maximum(plan[1], 0)], 0.0))
    gm = _local_gs(np.ones(mesh.L), mesh.glo_num)
    for p, plan in zip(parts, plans):
        got = _exchange(np.ones(p[1].size), p[1], plan, lambda send: ones_sends)
        assert np.array_equal(got, gm[p[3] * P:p[4] * P])


def _gloo_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    from paper_2606_12650_b200.dist import TorchComm
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    comm = TorchComm()
    mesh = brick_mesh(2, 2, 3, 3, 0.05)
    P = mesh.n ** 3
    e0, e1 = element_range(mesh.E, world, rank)
    _, glo, _ = local_part(mesh.E, mesh.N, mesh.coords, mesh.glo_num, mesh.mask, e0, e1)
    plan = interface_plan(glo, comm.all_gather_object(np.unique(glo)))
    v = np.random.Generator(np.random.PCG64(4)).integers(-8, 9, mesh.L).astype(np.float64)

    def gather(send):
        out = torch.empty(world * send.size, dtype=torch.float64)
        comm.all_gather(torch.from_numpy(send), out)
        return out.view(world, -1).numpy()

    got = _exchange(v[e0 * P:e1 * P], glo, plan, gather)
    want = _local_gs(v, mesh.glo_num)[e0 * P:e1 * P]
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, bool(np.array_equal(got, want)), plan[0]))


def test_gloo_two_ranks_exchange():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] and res[1][1]
    assert res[0][2] == res[1][2] > 0
