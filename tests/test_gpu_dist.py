"""-m gpu parity of the distributed path (include/nk.h "Distributed") on ONE GPU: the ranks
are host threads of this process (tests/dist_common.py), each with its own context on its own elements; the
oracle is set up once on the WHOLE mesh and knows nothing about partitions.  Plus one real NCCL run with a
process group of size 1 (all this box has)."""
import os

import numpy as np
import pytest

from parity import elem_err, gs_scale, scaled_err
from gpu_common import to_dev, to_np, TOL_OP, TOL_CG
from dist_common import run_ranks
from workloads import CONFIGS, brick_mesh, config_mesh, config_rhs

pytestmark = pytest.mark.gpu


def _assemble(parts):
    return np.concatenate(parts)


def _mesh(name):
    return brick_mesh(3, 2, 2, 5, 0.05) if name == "ragged" else config_mesh(name)


@pytest.mark.parametrize("name,world", [("config1", 2), ("config1", 3), ("ragged", 5), ("config2", 2), ("config2", 3)])
def test_dist_operators_against_whole_mesh_oracle(name, world):
    from oracle.nko import Oracle
    from paper_2606_12650_b200.dist import DistNekbone
    mesh = _mesh(name)
    P = mesh.n ** 3
    rng = np.random.Generator(np.random.PCG64(21))
    u = rng.uniform(-1, 1, mesh.L)                    # copies differ: gs really sums
    a = rng.uniform(-1, 1, mesh.L)

    def rank(comm):
        d = DistNekbone.from_mesh(mesh, comm)
        v = to_dev(d.local(u))
        out = dict(mult=to_np(d.mult()), gs=to_np(d.gs(v.clone())), ax=to_np(d.ax(v)),
                   dot=float(d.dot(v, to_dev(d.local(a)))[0]), slots=d.n_slots)
        d.close()
        return out

    res = run_ranks(world, rank)
    orc = Oracle.from_mesh(mesh)
    assert np.array_equal(_assemble([r["mult"] for r in res]), orc.mult())
    assert scaled_err(_assemble([r["gs"] for r in res]), orc.gs(u), gs_scale(u, mesh.glo_num)) <= TOL_OP
    assert elem_err(_assemble([r["ax"] for r in res]), orc.ax(u), P) <= TOL_OP
    want = orc.dot(u, a)
    scale = float(np.abs(u * a / orc.mult()).sum())
    assert all(abs(r["dot"] - want) <= TOL_OP * scale for r in res)
    assert len({r["dot"] for r in res}) == 1           # rank-ordered totals: the same bits on every rank
    assert len({r["slots"] for r in res}) == 1 and res[0]["slots"] > 0
    orc.close()


@pytest.mark.parametrize("name,world", [("config1", 2), ("config1", 3), ("ragged", 4), ("config2", 2), ("config2", 4)])
def test_dist_cg_against_whole_mesh_oracle(name, world):
    from oracle.nko import Oracle
    from paper_2606_12650_b200.dist import DistNekbone
    mesh = _mesh(name)
    P = mesh.n ** 3
    niter = CONFIGS[name]["niter"] if name in CONFIGS else 30
    from workloads import rhs_unique
    f = config_rhs(name, mesh) if name in CONFIGS else rhs_unique(mesh, 1234)

    def rank(comm):
        d = DistNekbone.from_mesh(mesh, comm)
        x, h = d.cg(to_dev(d.local(f)), niter)
        x2, h2 = d.cg(to_dev(d.local(f)), niter)      # reruns are bitwise equal
        out = (to_np(x), to_np(h), bool((x == x2).all() and (h == h2).all()))
        d.close()
        return out

    res = run_ranks(world, rank)
    orc = Oracle.from_mesh(mesh)
    xo, ho = orc.cg(f, niter)
    orc.close()
    for r in res:
        assert np.array_equal(r[1], res[0][1])         # one history, bit for bit, on every rank
        assert r[2]
    assert np.all(np.abs(res[0][1] - ho) <= TOL_CG * ho), float(np.abs(res[0][1] / ho - 1).max())
    xg = _assemble([r[0] for r in res])
    assert elem_err(xg, xo, P) <= TOL_CG
    assert np.all(xg[mesh.mask == 0.0] == 0.0)


def test_dist_world_one_over_nccl_equals_single_gpu_solver():
    """A real NCCL communicator (size 1): DistNekbone through torch.distributed against nk_cg on the same mesh."""
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
        assert d.n_slots == 0
        xd, hd = d.cg(f, 50)
        one = Nekbone.from_mesh(mesh)
        xs, hs = one.cg(f, 50)
        torch.cuda.synchronize()
        assert np.all(np.abs(to_np(hd) - to_np(hs)) <= 1e-12 * to_np(hs))
        assert elem_err(to_np(xd), to_np(xs), mesh.n ** 3) <= 1e-12
        d.close()
        one.close()
    finally:
        dist.destroy_process_group()


def test_dist_calls_need_attach():
    from paper_2606_12650_b200 import Nekbone
    from paper_2606_12650_b200.binding import NkError
    mesh = config_mesh("config1")
    nk = Nekbone.from_mesh(mesh)
    v = nk.empty()
    with pytest.raises(NkError):
        from paper_2606_12650_b200.binding import _check, _stream, _vp
        _check(nk._lib.nk_dist_gs_begin(nk._ctx, _vp(v.data_ptr()), 0, _stream()))
    nk.close()
