"""-m gpu parity of the distributed path (include/nk.h "Distributed") on ONE GPU: the ranks
are host threads of this process (tests/dist_common.py), each with its own context on its own elements; the
oracle is set up once on the WHOLE mesh and knows nothing about partitions.  Slab partitions (contiguous element
ranges), sub-brick partitions up to 2 x 2 x 2 (a rank then has up to seven neighbours and nodes held by eight
ranks), ragged ones.  Plus one real NCCL run with a process group of size 1 (all this box has)."""
import os

import numpy as np
import pytest

from parity import elem_err, gs_scale, scaled_err
from gpu_common import to_dev, to_np, TOL_OP, TOL_CG
from dist_common import run_ranks
from workloads import CONFIGS, brick_mesh, config_mesh, config_rhs, rhs_unique

pytestmark = pytest.mark.gpu

# name -> (mesh factory, partition or None for contiguous ranges)
MESHES = {
    "config1": (lambda: config_mesh("config1"), None),
    "config2": (lambda: config_mesh("config2"), None),
    "ragged": (lambda: brick_mesh(3, 2, 2, 5, 0.05), None),
    "bricks222": (lambda: brick_mesh(4, 4, 4, 3, 0.05), (2, 2, 2)),
    "bricks321": (lambda: brick_mesh(6, 4, 3, 4, 0.05), (3, 2, 1)),
    "config2_222": (lambda: config_mesh("config2"), (2, 2, 2)),
}


def _make(name, world, comm):
    from paper_2606_12650_b200.dist import DistNekbone, brick_partition
    mesh = MESHES[name][0]()
    part = MESHES[name][1]
    elements = None
    if part is not None:
        assert part[0] * part[1] * part[2] == world
        elements = brick_partition(mesh.nx, mesh.ny, mesh.nz, *part, comm.rank)
    return mesh, DistNekbone.from_mesh(mesh, comm, elements=elements)


def _assemble(mesh, res, key):
    out = np.full(mesh.L, np.nan)
    P = mesh.n ** 3
    for r in res:
        out.reshape(mesh.E, P)[r["elements"]] = r[key].reshape(-1, P)
    assert not np.isnan(out).any()
    return out


@pytest.mark.parametrize("name,world", [("config1", 2), ("config1", 3), ("ragged", 5), ("config2", 2), ("config2", 3),
                                        ("bricks222", 8), ("bricks321", 6)])
def test_dist_operators_against_whole_mesh_oracle(name, world):
    from oracle.nko import Oracle
    mesh = MESHES[name][0]()
    P = mesh.n ** 3
    rng = np.random.Generator(np.random.PCG64(21))
    u = rng.uniform(-1, 1, mesh.L)                    # copies differ: gs really sums
    a = rng.uniform(-1, 1, mesh.L)

    def rank(comm):
        _, d = _make(name, world, comm)
        v = to_dev(d.local(u))
        out = dict(elements=d.elements, mult=to_np(d.mult()), gs=to_np(d.gs(v.clone())), ax=to_np(d.ax(v)),
                   dot=float(d.dot(v, to_dev(d.local(a)))[0]), nbrs=d.neighbours, n_if=d.n_interface_nodes,
                   e_if=d.n_interface_elements, E=d.nk.E)
        d.close()
        return out

    res = run_ranks(world, rank)
    orc = Oracle.from_mesh(mesh)
    assert np.array_equal(_assemble(mesh, res, "mult"), orc.mult())
    assert scaled_err(_assemble(mesh, res, "gs"), orc.gs(u), gs_scale(u, mesh.glo_num)) <= TOL_OP
    assert elem_err(_assemble(mesh, res, "ax"), orc.ax(u), P) <= TOL_OP
    want = orc.dot(u, a)
    scale = float(np.abs(u * a / orc.mult()).sum())
    assert all(abs(r["dot"] - want) <= TOL_OP * scale for r in res)
    assert len({r["dot"] for r in res}) == 1           # rank-ordered totals: the same bits on every rank
    # the exchange is symmetric: r lists s with the count s lists r with; every rank has a neighbour
    table = [{n[0]: n[2] for n in r["nbrs"]} for r in res]
    for r in range(world):
        assert table[r] and all(table[s][r] == cnt for s, cnt in table[r].items())
    assert all(r["n_if"] > 0 and 0 < r["e_if"] <= r["E"] for r in res)
    if name == "bricks222":                             # every sub-brick touches the seven others
        assert all(len(t) == 7 for t in table)
    orc.close()


@pytest.mark.parametrize("name,world", [("config1", 2), ("config1", 3), ("ragged", 4), ("config2", 2), ("config2", 4),
                                        ("bricks222", 8), ("config2_222", 8)])
def test_dist_cg_against_whole_mesh_oracle(name, world):
    from oracle.nko import Oracle
    mesh = MESHES[name][0]()
    P = mesh.n ** 3
    base = name.split("_")[0]
    niter = CONFIGS[base]["niter"] if base in CONFIGS else 30
    f = config_rhs(base, mesh) if base in CONFIGS else rhs_unique(mesh, 1234)

    def rank(comm):
        _, d = _make(name, world, comm)
        x, h = d.cg(to_dev(d.local(f)), niter)
        x2, h2 = d.cg(to_dev(d.local(f)), niter)      # reruns are bitwise equal
        out = dict(elements=d.elements, x=to_np(x), h=to_np(h), same=bool((x == x2).all() and (h == h2).all()),
                   interior=d.nk.E - d.n_interface_elements)
        d.close()
        return out

    res = run_ranks(world, rank)
    orc = Oracle.from_mesh(mesh)
    xo, ho = orc.cg(f, niter)
    orc.close()
    for r in res:
        assert np.array_equal(r["h"], res[0]["h"])     # one history, bit for bit, on every rank
        assert r["same"]
    assert np.all(np.abs(res[0]["h"] - ho) <= TOL_CG * ho), float(np.abs(res[0]["h"] / ho - 1).max())
    xg = _assemble(mesh, res, "x")
    assert elem_err(xg, xo, P) <= TOL_CG
    assert np.all(xg[mesh.mask == 0.0] == 0.0)
    if name in ("config2", "config2_222"):              # these partitions leave interior elements: the overlapped path ran
        assert any(r["interior"] > 0 for r in res)


def test_dist_world_one_over_nccl_equals_single_gpu_solver():
    """A real NCCL communicator (size 1): DistNekbone through torch.distributed is nk_cg, bit for bit."""
    import torch
    import torch.distributed as dist
    from paper_2606_12650_b200 import Nekbone
    from paper_2606_12650_b200.dist import DistNekbone, TorchComm
    mesh = config_mesh("config2")
    f = to_dev(config_rhs("config2", mesh))
    port = 33500 + os.getpid() % 2000
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1,
                            device_id=torch.device("cuda:0"))
    try:
        d = DistNekbone.from_mesh(mesh, TorchComm())
        assert d.n_neighbors == 0 and d.n_exchange == 0
        xd, hd = d.cg(f, 50)
        one = Nekbone.from_mesh(mesh)
        xs, hs = one.cg(f, 50)
        torch.cuda.synchronize()
        assert bool((hd == hs).all()) and bool((xd == xs).all())
        v = to_dev(np.random.Generator(np.random.PCG64(5)).uniform(-1, 1, mesh.L))
        assert bool((d.gs(v.clone()) == one.gs(v.clone())).all())
        assert float(d.dot(v, f)[0]) == float(one.dot(v, f)[0])
        d.close()
        one.close()
    finally:
        dist.destroy_process_group()


def test_dist_calls_need_setup():
    from paper_2606_12650_b200 import Nekbone
    from paper_2606_12650_b200.binding import NkError, _check, _stream, _vp
    mesh = config_mesh("config1")
    nk = Nekbone.from_mesh(mesh)
    v = nk.empty()
    with pytest.raises(NkError):
        _check(nk._lib.nk_dist_gs(nk._ctx, _vp(v.data_ptr()), 0, None, None, _stream()))
    nk.close()
