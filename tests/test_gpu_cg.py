"""-m gpu parity of the CG iteration (SURVEY.md 8(c) protocol parts 2-4; R15):
lock-step single iterations from oracle-provided state at 1e-12, free-running CG at 1e-10 where
the oracle's own rounding band allows, every fusion option against the others, degenerate inputs."""
import numpy as np
import pytest

from parity import elem_err, maxnorm_rel
from gpu_common import pair_for_brick, pair_for_config, to_dev, to_np, TOL_OP, TOL_CG
from workloads import CONFIGS, brick_mesh, config_rhs, rhs_unique

pytestmark = pytest.mark.gpu

# launch-by-launch paths ("coop" = 0) with every fusion option, the graph replay, and the cooperative whole-solve launch
OPTION_SETS = [dict(coop=0, fuse_pap=1, fuse_p=1, fuse_gs=1, graph=0), dict(coop=0, fuse_pap=0, fuse_p=0, fuse_gs=1, graph=0),
               dict(coop=0, fuse_pap=1, fuse_p=0, fuse_gs=1, graph=0), dict(coop=0, fuse_pap=0, fuse_p=1, fuse_gs=1, graph=0),
               dict(coop=0, fuse_pap=1, fuse_p=1, fuse_gs=0, graph=0), dict(coop=0, fuse_pap=1, fuse_p=0, fuse_gs=0, graph=0),
               dict(coop=0, fuse_pap=1, fuse_p=1, fuse_gs=1, graph=1), dict(coop=1)]
DEFAULTS = dict(coop=2, fuse_pap=1, fuse_p=2, fuse_gs=2, graph=2)


def _set(gpu, opts):
    for k, v in opts.items():
        gpu.set_option(k, v)
        assert gpu.get_option(k) == v


def _rel(a, b):
    return abs(a - b) / abs(b) if b != 0 else abs(a)


@pytest.mark.parametrize("name", ["config1", "config2"])
@pytest.mark.parametrize("opts", OPTION_SETS[:6])
def test_lockstep_iterations(name, opts):
    """Load the ORACLE's state at iteration k into the GPU, run one GPU iteration, compare
    (w, pap, alpha, x, r, rho', beta, p) -- every iteration-level formula, zero amplification."""
    pr = pair_for_config(name)
    _set(pr.gpu, opts)
    niter = CONFIGS[name]["niter"]
    f = config_rhs(name, pr.mesh)
    x, r, p, rho = pr.orc.cg_init(f)
    checks = {k for k in (1, 2, 5, 10, 25, 50, 75, 100) if k <= niter}
    for k in range(1, niter + 1):
        if k in checks:
            xd = to_dev(x)
            pr.gpu.cg_load_state(to_dev(r), to_dev(p), rho)
            pr.gpu.cg_step(xd)
            rg, pg, wg = (to_np(t) for t in pr.gpu.cg_get_state())
            sg = pr.gpu.scalars()
        w, so = pr.orc.cg_step(x, r, p, rho)          # advances x, r, p in place
        if k in checks:
            assert elem_err(wg, w, pr.P) <= TOL_OP, k
            for key in ("pap", "alpha", "rho_new", "beta"):
                assert _rel(sg[key], so[key]) <= TOL_OP, (k, key, sg[key], so[key])
            assert elem_err(to_np(xd), x, pr.P) <= TOL_OP, k
            assert elem_err(rg, r, pr.P) <= TOL_OP, k
            assert elem_err(pg, p, pr.P) <= TOL_OP, k
        rho = so["rho_new"]
    _set(pr.gpu, DEFAULTS)


@pytest.mark.parametrize("name", ["config1", "config2"])
@pytest.mark.parametrize("opts", OPTION_SETS)
def test_free_running_cg(name, opts):
    pr = pair_for_config(name)
    _set(pr.gpu, opts)
    niter = CONFIGS[name]["niter"]
    f = config_rhs(name, pr.mesh)
    xo, ho = pr.orc.cg(f, niter)
    xg, hg = pr.gpu.cg(to_dev(f), niter)
    xg, hg = to_np(xg), to_np(hg)
    assert hg.shape == (niter + 1,)
    assert np.all(np.abs(hg - ho) <= TOL_CG * ho), np.abs(hg / ho - 1).max()
    assert elem_err(xg, xo, pr.P) <= TOL_CG
    assert np.all(xg[pr.mesh.mask == 0.0] == 0.0)
    _set(pr.gpu, DEFAULTS)


def test_golden_history_config1():
    """tests/golden/config1_cg.txt was written by tests/golden/make_golden.py from the oracle only."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "config1_cg.txt")
    gold = np.array([float(l.split()[-1]) for l in open(path) if l.strip() and not l.startswith("#")])
    pr = pair_for_config("config1")
    xg, hg = pr.gpu.cg(to_dev(config_rhs("config1", pr.mesh)), 20)
    hg = to_np(hg)
    assert gold.size == 22 and np.all(np.abs(hg - gold[:21]) <= TOL_CG * gold[:21])
    assert abs(float(xg.abs().max()) - gold[21]) <= TOL_CG * gold[21]


def test_cg_host_entry_equals_device_entry():
    pr = pair_for_config("config2")
    f = config_rhs("config2", pr.mesh)
    xd, hd = pr.gpu.cg(to_dev(f), 30)
    xh, hh = pr.gpu.cg_host(f, 30)
    assert np.array_equal(to_np(xd), xh) and np.array_equal(to_np(hd), hh)


@pytest.mark.parametrize("path", ["cooperative", "graph", "launches"])
def test_cg_host_batch_equals_one_call_per_rhs(path):
    """nk_cg_host_batch pipelines the copies of right-hand side j+1 and of solution j-1 with solve j (two copy streams,
    two sets of staging buffers); every solve must equal, bit for bit, nk_cg_host on the same right-hand side -- five
    different ones, pinned buffers, so that a copy racing a solve would show."""
    import torch
    pr = pair_for_config("config2")
    gpu = pr.gpu
    saved = {k: gpu.get_option(k) for k in ("coop", "graph")}
    try:
        gpu.set_option("coop", 1 if path == "cooperative" else 0)
        gpu.set_option("graph", 0 if path == "launches" else 1)
        assert gpu.solve_path() == path
        rng = np.random.Generator(np.random.PCG64(41))
        _, inv = np.unique(pr.mesh.glo_num, return_inverse=True)
        fs = [torch.from_numpy(rng.uniform(-1, 1, inv.max() + 1)[inv] * (j + 1)).pin_memory() for j in range(5)]
        xs = [torch.empty(pr.L, dtype=torch.float64).pin_memory() for _ in range(5)]
        hs = [torch.empty(26, dtype=torch.float64).pin_memory() for _ in range(5)]
        gpu.cg_host_batch([f.numpy() for f in fs], 25, [x.numpy() for x in xs], [h.numpy() for h in hs])
        for f, x, h in zip(fs, xs, hs):
            x1, h1 = gpu.cg_host(f.numpy(), 25)
            assert np.array_equal(x.numpy(), x1) and np.array_equal(h.numpy(), h1)
        assert gpu.cg_host_batch([], 25, [], []) == ([], [])
    finally:
        for k, v in saved.items():
            gpu.set_option(k, v)


@pytest.mark.parametrize("niter", [1, 2, 3, 7, 12])
@pytest.mark.parametrize("fuse_p,fuse_gs", [(0, 0), (0, 1), (1, 1)])
def test_deferred_x_update_is_bitwise_the_plain_one(niter, fuse_p, fuse_gs):
    """"defer_x": two iterations share one pass over x (x = fma(alpha', p', fma(alpha, p, x)), the direction kept in two
    vectors).  Same operations in the same order: x, the history and the state the context is left in (r, p, w) are
    bit for bit those of the plain update -- odd and even iteration counts, launch by launch and graphed, with the
    caller's x only 16-byte aligned (the 256-bit accesses fall back to 128-bit ones on x).  With "fuse_p" the second
    ax_e of a pair forms its direction out of place and the fused gs update applies both steps to x; the direction
    ends in either of the two vectors depending on the count, the context always shows it in p."""
    import torch
    pr = pair_for_brick(7, 6, 5, 6, 0.05)                    # 72030 points: two past the last quad
    gpu = pr.gpu
    saved = {k: gpu.get_option(k) for k in ("coop", "fuse_p", "fuse_gs", "graph", "defer_x")}
    try:
        gpu.set_option("coop", 0)
        gpu.set_option("fuse_p", fuse_p)
        gpu.set_option("fuse_gs", fuse_gs)
        f = to_dev(rhs_unique(pr.mesh, 77))
        xbuf = torch.empty(pr.L + 2, dtype=torch.float64, device="cuda")
        out = {}
        for defer in (0, 1):
            for graph in (0, 1):
                gpu.set_option("defer_x", defer)
                gpu.set_option("graph", graph)
                x = xbuf[2:] if defer else gpu.empty()        # 16-byte aligned only
                x, h = gpu.cg(f, niter, x=x)
                out[defer, graph] = (to_np(x),) + tuple(to_np(t) for t in gpu.cg_get_state()) + (to_np(h),)
        for key in ((0, 1), (1, 0), (1, 1)):
            for a, b in zip(out[0, 0], out[key]):
                assert np.array_equal(a, b), key
    finally:
        for k, v in saved.items():
            gpu.set_option(k, v)


def test_cached_graphs_are_keyed_by_every_option():
    """nk_cg keeps two recorded graphs (nk_cg_host_batch alternates between two sets of buffers).  Each option has a
    bit field of its own in the cache key: with fuse_gs = 2 and pdl = 3 sharing a bit, the graph recorded for
    fuse_gs = 0 was replayed for fuse_gs = 2.  1 M points, so fuse_gs = 2 means fused; fused and separate gs differ in
    the rounding of rho', which tells the replayed graphs apart."""
    mesh = brick_mesh(16, 16, 8, 7, 0.05)
    from paper_2606_12650_b200 import Nekbone
    gpu = Nekbone.from_mesh(mesh)
    try:
        rng = np.random.Generator(np.random.PCG64(5))
        _, inv = np.unique(mesh.glo_num, return_inverse=True)
        f = to_dev(rng.uniform(-1, 1, inv.max() + 1)[inv])
        gpu.set_option("coop", 0)
        gpu.set_option("graph", 1)
        x, h = gpu.empty(), gpu.empty()[:32]
        hist = {}
        for fuse_gs in (0, 1, 2, 0, 2, 1):                    # same buffers every time: only the key tells them apart
            gpu.set_option("fuse_gs", fuse_gs)
            assert gpu.solve_path() == "graph"
            gpu.cg(f, 30, x=x, res_hist=h)
            hn = to_np(h)[:31].copy()
            if fuse_gs in hist:
                assert np.array_equal(hist[fuse_gs], hn), fuse_gs
            hist[fuse_gs] = hn
        assert np.array_equal(hist[2], hist[1])               # 2 = fused at this size
        assert not np.array_equal(hist[0], hist[1])           # ... and the two are distinguishable here
        assert np.all(np.abs(hist[0] - hist[1]) <= 1e-10 * hist[0])
    finally:
        gpu.close()


def test_cg_reproducible_and_ignores_incoming_x():
    pr = pair_for_config("config2")
    f = to_dev(config_rhs("config2", pr.mesh))
    x1, h1 = pr.gpu.cg(f, 40)
    x2 = to_dev(np.full(pr.L, 123.0))
    x2, h2 = pr.gpu.cg(f, 40, x=x2)
    assert bool((x1 == x2).all()) and bool((h1 == h2).all())


def test_degenerate_inputs():
    import torch
    pr = pair_for_config("config1")
    f = config_rhs("config1", pr.mesh)
    # niter = 0: hist[0] only, x = 0
    xg, hg = pr.gpu.cg(to_dev(f), 0)
    xo, ho = pr.orc.cg(f, 0)
    assert hg.numel() == 1 and abs(float(hg[0]) - ho[0]) <= TOL_OP * ho[0] and not bool(xg.any())
    # f = 0: x = 0, history identically 0, no NaN
    xg, hg = pr.gpu.cg(torch.zeros(pr.L, dtype=torch.float64, device="cuda"), 5)
    assert not bool(xg.any()) and not bool(hg.any())
    # far past convergence rho underflows to 0: guards keep everything finite
    xg, hg = pr.gpu.cg(to_dev(f), 400)
    assert bool(torch.isfinite(xg).all()) and bool(torch.isfinite(hg).all())
    xo, _ = pr.orc.cg(f, 400)
    assert elem_err(to_np(xg), xo, pr.P) <= TOL_CG


def test_mask_all_zero_and_single_element():
    from oracle.nko import Oracle
    from paper_2606_12650_b200 import Nekbone
    from workloads import brick_mesh
    m = brick_mesh(2, 2, 2, 3, 0.05)
    gpu = Nekbone(m.E, m.N, m.coords, m.glo_num, np.zeros(m.L))
    xg, hg = gpu.cg(to_dev(rhs_unique(m, 3)), 5)
    assert not bool(xg.any()) and not bool(hg.any())
    # E = 1 at N = 5: only the 4^3 interior nodes are free
    m = brick_mesh(1, 1, 1, 5, 0.0)
    f = rhs_unique(m, 4)
    xo, ho = Oracle.from_mesh(m).cg(f, 30)
    _, hb = Oracle.from_mesh(m, fma=True).cg(f, 30)
    xg, hg = Nekbone.from_mesh(m).cg(to_dev(f), 30)
    # 64 free nodes: CG converges to rounding level well before iteration 30, after which the
    # recursive residual is rounding noise and no two fp64 implementations agree.  R15 protocol:
    # flat 1e-10 while the oracle's own band (contraction-on vs -off builds) is <= 1e-11;
    # past that point both sides must simply have converged (9 decades below hist[0]).
    band = np.maximum.accumulate(np.abs(hb - ho) / ho)      # rounding noise only grows
    ok = band <= 1e-11
    hg = to_np(hg)
    assert ok[:13].all()
    assert np.all(np.abs(hg[ok] - ho[ok]) <= TOL_CG * ho[ok])
    assert np.all(hg[~ok] <= 1e-9 * ho[0]) and np.all(ho[~ok] <= 1e-9 * ho[0])
    assert elem_err(to_np(xg), xo, 216) <= TOL_CG


def test_cg_argument_errors():
    from paper_2606_12650_b200 import NkError
    pr = pair_for_config("config1")
    f = to_dev(config_rhs("config1", pr.mesh))
    with pytest.raises(NkError):
        pr.gpu.cg(f, -1)
    with pytest.raises(NkError):
        pr.gpu.cg(f, 3, x=f)                     # f == x
    with pytest.raises(NkError):
        pr.gpu.ax_e(f, f)                        # u == w
    with pytest.raises(NkError):
        pr.gpu.set_option("no_such_option", 1)
    with pytest.raises(NkError):
        pr.gpu.set_option("fuse_pap", 7)
    with pytest.raises(ValueError):
        pr.gpu.ax_e(f[:-1].contiguous())


def test_graph_default_and_pointer_change():
    """"graph" = 2 is the default (replay a CUDA graph on small meshes); a cached graph must follow new
    f / x / history pointers (in-place update) and give bitwise the same result as direct launches."""
    import torch
    from paper_2606_12650_b200 import Nekbone
    pr = pair_for_config("config2")
    gpu = Nekbone.from_mesh(pr.mesh)                  # a fresh context: the shared one has had options set
    assert gpu.get_option("graph") == 2 and gpu.solve_path() == "cooperative"
    gpu.set_option("coop", 0)                         # below the cooperative launch the rule is: replay a graph
    assert gpu.solve_path() == "graph"
    f1 = to_dev(config_rhs("config2", pr.mesh))
    f2 = f1.clone()
    xa, ha = gpu.cg(f1, 25)
    xb, hb = gpu.cg(f2, 25)                        # new f, x, hist tensors -> graph update path
    xc, hc = gpu.cg(f2, 12)                        # different iteration count -> new topology
    gpu.set_option("graph", 0)
    xd, hd = gpu.cg(f1, 25)
    xe, he = gpu.cg(f1, 12)
    gpu.set_option("graph", 2)
    torch.cuda.synchronize()
    assert bool((xa == xd).all()) and bool((ha == hd).all())
    assert bool((xb == xd).all()) and bool((hb == hd).all())
    assert bool((xc == xe).all()) and bool((hc == he).all())


@pytest.mark.parametrize("name", ["config1", "config2", "config3"])
@pytest.mark.parametrize("fuse_p", [0, 1])
def test_programmatic_dependent_launch_is_bitwise_neutral(name, fuse_p):
    """"pdl" (default 3: gs too on meshes up to 2^24 points) overlaps each kernel's prologue with its predecessor's tail; every read of the
    predecessor's output sits behind griddepcontrol.wait, so x and the residual history must be bitwise those
    of plain launches, graphed or not, with p folded into ax_e or not."""
    import torch
    from paper_2606_12650_b200 import Nekbone
    from workloads import config_mesh
    mesh = config_mesh(name)
    gpu = Nekbone.from_mesh(mesh)
    assert gpu.get_option("pdl") == 3
    gpu.set_option("coop", 0)
    gpu.set_option("fuse_p", fuse_p)
    f = to_dev(config_rhs(name, mesh))
    out = {}
    for graph in (0, 1):
        for pdl in (0, 1, 2, 3):
            gpu.set_option("graph", graph)
            gpu.set_option("pdl", pdl)
            for rep in range(3):                       # replays too: the waits must hold on every run
                out[graph, pdl, rep] = gpu.cg(f, 40)
    torch.cuda.synchronize()
    x0, h0 = out[0, 0, 0]
    for key, (x, h) in out.items():
        assert bool((x == x0).all()) and bool((h == h0).all()), key
    gpu.close()


# ---- NEXT row f-3: Jacobi-preconditioned CG ------------------------------------------------------------
@pytest.mark.parametrize("name", ["config1", "config2"])
def test_jacobi_diag_and_pcg(name):
    from paper_2606_12650_b200 import Nekbone
    pr = pair_for_config(name)
    gpu = Nekbone.from_mesh(pr.mesh)
    niter = CONFIGS[name]["niter"]
    f = config_rhs(name, pr.mesh)
    assert elem_err(to_np(gpu.diag()), pr.orc.diag(), pr.P) <= TOL_OP
    xo, ho = pr.orc.pcg(f, niter)
    for fuse_pap in (1, 0):
        gpu.set_option("fuse_pap", fuse_pap)
        xg, hg = gpu.pcg(to_dev(f), niter)
        xg, hg = to_np(xg), to_np(hg)
        assert np.all(np.abs(hg - ho) <= TOL_CG * ho), np.abs(hg / ho - 1).max()
        assert elem_err(xg, xo, pr.P) <= TOL_CG
        assert np.all(xg[pr.mesh.mask == 0.0] == 0.0)
    # guards and reproducibility
    import torch
    x0, h0 = gpu.pcg(torch.zeros(pr.L, dtype=torch.float64, device="cuda"), 4)
    assert not bool(x0.any()) and not bool(h0.any())
    xa, ha = gpu.pcg(to_dev(f), 10)
    xb, hb = gpu.pcg(to_dev(f), 10)
    assert bool((xa == xb).all()) and bool((ha == hb).all())


@pytest.mark.parametrize("name", ["config1", "config2", "config3"])
@pytest.mark.parametrize("fuse_pap", [1, 0])
def test_pcg_programmatic_dependent_launch_is_bitwise_neutral(name, fuse_pap):
    """nk_pcg's loop launches ax_e, update_rz and update_pz as programmatic dependents too: same iterates,
    bit for bit, as plain launches, on repeated calls."""
    import torch
    from paper_2606_12650_b200 import Nekbone
    from workloads import config_mesh
    mesh = config_mesh(name)
    gpu = Nekbone.from_mesh(mesh)
    gpu.set_option("fuse_pap", fuse_pap)
    f = to_dev(config_rhs(name, mesh))
    out = {}
    for pdl in (0, 1, 2):
        gpu.set_option("pdl", pdl)
        for rep in range(3):
            x, h = gpu.pcg(f, 40)
            out[pdl, rep] = (x.clone(), h.clone())
    torch.cuda.synchronize()
    x0, h0 = out[0, 0]
    for key, (x, h) in out.items():
        assert bool((x == x0).all()) and bool((h == h0).all()), key
    gpu.close()


@pytest.mark.parametrize("N", [6, 10, 12, 14, 15])
def test_cg_high_and_odd_orders(N):
    """CG through the fused-pap path of every kernel configuration family: sync groups per slot (N = 10),
    one work-array pair (N = 11 is config 5), single-element batches (N = 12), and the warp-specialised
    register budget with the producer in its own warpgroup (N = 14, 15)."""
    pr = pair_for_brick(3, 2, 2, N, 0.1)
    f = rhs_unique(pr.mesh, 40 + N)
    xo, ho = pr.orc.cg(f, 12)
    for coop, graph in ((0, 0), (0, 1), (2, 2)):          # launches, graph replay, the default (cooperative up to N = 13)
        pr.gpu.set_option("coop", coop)
        pr.gpu.set_option("graph", graph)
        xg, hg = pr.gpu.cg(to_dev(f), 12)
        assert np.all(np.abs(to_np(hg) - ho) <= TOL_CG * ho), (N, coop, graph)
        assert elem_err(to_np(xg), xo, pr.P) <= TOL_CG, (N, coop, graph)
    assert pr.gpu.solve_path() == ("cooperative" if N <= 13 else "graph")


# ---- gs folded into the residual update ("fuse_gs") ------------------------------------------------------
@pytest.mark.parametrize("name", ["config1", "config2", "config3"])
@pytest.mark.parametrize("fuse_p", [0, 1])
def test_fused_gs_against_separate_gs(name, fuse_p):
    """The residual update that sums the copies of shared nodes from the unsummed ax_e output ("fuse_gs") gives,
    for the same alpha, r and x entry by entry as the separate gs kernel does (same order of addition per node);
    rho' adds the same terms in another fixed order, so the two solves agree to rounding (config 1 has converged
    nine decades by iteration 40, where rounding differences have grown to a few 1e-13: bound 1e-11).  Each is bitwise reproducible, launch by launch or graphed, with or without programmatic
    dependent launches."""
    import torch
    from paper_2606_12650_b200 import Nekbone
    from workloads import config_mesh
    mesh = config_mesh(name)
    gpu = Nekbone.from_mesh(mesh)
    assert gpu.get_option("fuse_gs") == 2
    gpu.set_option("coop", 0)
    gpu.set_option("fuse_p", fuse_p)
    f = to_dev(config_rhs(name, mesh))
    # one iteration from the same state: r, x bitwise equal (rho' and beta, hence p, only to rounding)
    state = {}
    for fuse_gs in (0, 1):
        gpu.set_option("fuse_gs", fuse_gs)
        x = gpu.empty()
        gpu.cg_init(f, x)
        gpu.cg_step(x)
        r, p, w = gpu.cg_get_state()
        state[fuse_gs] = (x.clone(), r.clone(), w.clone(), gpu.scalars())
    assert bool((state[0][0] == state[1][0]).all()) and bool((state[0][1] == state[1][1]).all())
    assert bool((state[0][2] == state[1][2]).all())
    assert abs(state[0][3]["rho_new"] - state[1][3]["rho_new"]) <= 1e-14 * abs(state[0][3]["rho_new"])
    out = {}
    for fuse_gs in (0, 1):
        for graph, pdl in ((0, 0), (0, 3), (1, 3)):
            gpu.set_option("fuse_gs", fuse_gs)
            gpu.set_option("graph", graph)
            gpu.set_option("pdl", pdl)
            for rep in range(2):
                out[fuse_gs, graph, pdl, rep] = gpu.cg(f, 40)
    torch.cuda.synchronize()
    for fuse_gs in (0, 1):
        x0, h0 = out[fuse_gs, 0, 0, 0]
        for key, (x, h) in out.items():
            if key[0] == fuse_gs:
                assert bool((x == x0).all()) and bool((h == h0).all()), key
    (xa, ha), (xb, hb) = out[0, 0, 0, 0], out[1, 0, 0, 0]
    assert float(((ha - hb).abs() / ha).max()) <= 1e-11
    assert elem_err(to_np(xb), to_np(xa), mesh.n ** 3) <= 1e-12
    gpu.close()


@pytest.mark.parametrize("brick", [(3, 2, 2, 4), (10, 8, 7, 4), (3, 3, 3, 2), (6, 1, 1, 2), (5, 3, 3, 6)])
def test_fused_gs_on_irregular_ids(brick):
    """Rows of 3, 5, 12 copies and scattered ids take the fused gather's CSR path; Dirichlet rows its zero path.
    1500 points: the cooperative solve runs on one cluster; 70 000 points: on the grid.  The last three meshes have
    729, 162 and 15435 points: one, two and three points past the last quad of the fused update's 256-bit loop."""
    from oracle.nko import Oracle
    from paper_2606_12650_b200 import Nekbone
    from workloads import brick_mesh
    m = brick_mesh(*brick, 0.05)
    rng = np.random.Generator(np.random.PCG64(12))
    glo = rng.integers(0, m.L // 4 + 25, m.L).astype(np.int64) * 1_000_003 + 17      # ~3.75 copies per id, scattered
    glo[:12] = 5                                                            # one row of >= 12 copies
    glo[m.L - 1] = 999_999_999_999                                          # the last point alone (odd L: 1500... even; harmless)
    mask = np.ones(m.L)
    mask[np.isin(glo, glo[100:110])] = 0.0
    orc, gpu = Oracle(m.E, m.N, m.coords, glo, mask), Nekbone(m.E, m.N, m.coords, glo, mask)
    _, inv = np.unique(glo, return_inverse=True)
    f = rng.uniform(-1, 1, inv.max() + 1)[inv]                              # consistent on every copy
    xo, ho = orc.cg(f, 15)
    res = {}
    # the cooperative whole-solve launch (one cluster at this size) takes the same rows through coop_row_update
    assert gpu.solve_path() == "cooperative"
    xc, hc = gpu.cg(to_dev(f), 15)
    assert np.all(np.abs(to_np(hc) - ho) <= TOL_CG * ho) and elem_err(to_np(xc), xo, m.n ** 3) <= TOL_CG
    gpu.set_option("coop", 0)
    for fuse_p in (0, 1):
        for fuse_gs in (0, 1):
            gpu.set_option("fuse_p", fuse_p)
            gpu.set_option("fuse_gs", fuse_gs)
            xg, hg = gpu.cg(to_dev(f), 15)
            res[fuse_p, fuse_gs] = (to_np(xg), to_np(hg))
            assert np.all(np.abs(res[fuse_p, fuse_gs][1] - ho) <= TOL_CG * ho), (fuse_p, fuse_gs)
            assert elem_err(res[fuse_p, fuse_gs][0], xo, m.n ** 3) <= TOL_CG, (fuse_p, fuse_gs)


# ---- the whole solve as one cooperative launch ("coop") -----------------------------------------------------
COOP_MESHES = [(2, 2, 2, 3), (5, 3, 3, 1), (3, 3, 3, 2), (7, 6, 5, 4), (6, 5, 5, 6), (8, 8, 8, 7), (6, 5, 4, 8), (5, 4, 4, 9),
               (4, 3, 3, 11), (3, 2, 2, 13), (300, 1, 1, 5)]


@pytest.mark.parametrize("nx,ny,nz,N", COOP_MESHES)
def test_cooperative_solve(nx, ny, nz, N):
    """One persistent cooperative launch for the whole solve: against the oracle at 1e-10 (history and
    x), against the launch-by-launch path to rounding, bitwise reproducible, context left as the other paths leave
    it.  Meshes: fewer elements than CTAs (CTAs with no element still take their share of the vector phases and
    of the barriers), more than one batch per CTA (300 elements at N = 5 on 148 CTAs... 2-3 elements each, the
    8^3 mesh of config 2), odd L (N = 2: 27 points per element, 27 elements)."""
    import torch
    from paper_2606_12650_b200 import Nekbone
    pr = pair_for_brick(nx, ny, nz, N, 0.05)
    gpu = Nekbone.from_mesh(pr.mesh)
    assert gpu.solve_path() == "cooperative"
    f = rhs_unique(pr.mesh, 300 + N)
    niter = 30
    xo, ho = pr.orc.cg(f, niter)
    fd = to_dev(f)
    runs = [gpu.cg(fd, niter) for _ in range(3)]
    torch.cuda.synchronize()
    x0, h0 = runs[0]
    for x, h in runs[1:]:
        assert bool((x == x0).all()) and bool((h == h0).all())
    xg, hg = to_np(x0), to_np(h0)
    if not (np.all(np.abs(hg - ho) <= TOL_CG * ho) and elem_err(xg, xo, pr.P) <= TOL_CG):
        from parity import history_parity, oracle_variants           # tiny meshes converge within the 30 iterations
        alts = oracle_variants(pr.mesh, f, niter)
        ok, worst, kstar = history_parity(hg, ho, [h for _, h in alts])
        assert ok and kstar >= 8, (N, worst, kstar)
        assert elem_err(xg, xo, pr.P) <= max(TOL_CG, 10.0 * max(elem_err(xb, xo, pr.P) for xb, _ in alts))
    assert np.all(xg[pr.mesh.mask == 0.0] == 0.0)
    # the context afterwards: r, p, w = M Q Q^T A_L p and the scalars of the last iteration, as the launch path leaves them
    rc, pc, wc = (to_np(t) for t in gpu.cg_get_state())
    sc = gpu.scalars()
    gpu.set_option("coop", 0)
    xl, hl = gpu.cg(fd, niter)
    rl, pl, wl = (to_np(t) for t in gpu.cg_get_state())
    sl = gpu.scalars()
    k = int(np.nonzero(to_np(hl) > 1e-8 * to_np(hl)[0])[0].max())          # compare where rounding has not taken over
    assert float(np.abs(hg[:k + 1] / to_np(hl)[:k + 1] - 1).max()) <= 1e-11
    if k == niter:
        assert elem_err(xg, to_np(xl), pr.P) <= 1e-11
        assert elem_err(rc, rl, pr.P) <= 1e-9 and elem_err(pc, pl, pr.P) <= 1e-9 and elem_err(wc, wl, pr.P) <= 1e-9
        for key in ("pap", "alpha", "rho_new", "beta"):
            assert abs(sc[key] - sl[key]) <= 1e-9 * abs(sl[key]), key
    # guards and degenerate calls on the cooperative path
    gpu.set_option("coop", 1)
    xz, hz = gpu.cg(torch.zeros(pr.L, dtype=torch.float64, device="cuda"), 5)
    assert not bool(xz.any()) and not bool(hz.any())
    x1, h1 = gpu.cg(fd, 1)
    xo1, ho1 = pr.orc.cg(f, 1)
    assert np.all(np.abs(to_np(h1) - ho1) <= TOL_OP * ho1) and elem_err(to_np(x1), xo1, pr.P) <= TOL_OP
    xh, hh = gpu.cg_host(f, niter)
    assert np.array_equal(xh, xg) and np.array_equal(hh, hg)
    gpu.close()


@pytest.mark.parametrize("fuse_p", [0, 1])
@pytest.mark.parametrize("graph", [0, 1])
def test_context_state_after_a_solve(graph, fuse_p):
    """r, p, w = M Q Q^T A_L p and the scalars a solve leaves in the context (the direction update of the last
    iteration applied) against the oracle's, on every launch path, with programmatic dependent launches on: the final
    p = r + beta p once read beta before its predecessor had written it (a `const __restrict__` load hoisted above
    griddepcontrol.wait)."""
    from paper_2606_12650_b200 import Nekbone
    pr = pair_for_config("config2")
    gpu = Nekbone.from_mesh(pr.mesh)
    gpu.set_option("coop", 0)
    gpu.set_option("graph", graph)
    gpu.set_option("fuse_p", fuse_p)
    f = config_rhs("config2", pr.mesh)
    x, r, p, rho = pr.orc.cg_init(f)
    for k in range(3):
        w, so = pr.orc.cg_step(x, r, p, rho)
        rho = so["rho_new"]
    for rep in range(3):
        xg, hg = gpu.cg(to_dev(f), 3)
        rg, pg, wg = (to_np(t) for t in gpu.cg_get_state())
        assert elem_err(to_np(xg), x, pr.P) <= TOL_OP and elem_err(rg, r, pr.P) <= TOL_OP
        assert elem_err(pg, p, pr.P) <= TOL_OP, rep
        assert elem_err(wg, w, pr.P) <= TOL_OP
        sg = gpu.scalars()
        for key in ("pap", "alpha", "rho_new", "beta"):
            assert abs(sg[key] - so[key]) <= TOL_OP * abs(so[key]), key
    gpu.close()
