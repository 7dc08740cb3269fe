"""-m gpu parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(default options, device-resident vectors): config 3 (E=4096, N=9) and config 5 (E=32768, N=11).

The oracle is affordable at these sizes (one operator application takes well under a second on the host
cores, a CG iteration of config 5 about 0.4 s), so everything is compared over the WHOLE vector:

* set-up: the six geometric factors, multiplicities, sizes;
* one application of ax_e, gs, ax on a field drawn per local point, and the weighted dot product
  (SURVEY.md 8(c) protocol part 1);
* lock-step CG iterations k = 1, 50, 100 from the oracle's state (protocol part 2);
* free-running CG: residual history and x (protocol parts 3-4; config 3 by the R15 band protocol:
  flat 1e-10 up to K*, the last iteration with oracle band <= 1e-11; max(1e-10, 10 x band) beyond);
* properties that hold at any size: symmetry, null space, analytic multiplicity counts.
"""
import numpy as np
import pytest

from parity import elem_err, scaled_err, gs_scale, history_parity, oracle_variants
from gpu_common import to_dev, to_np, TOL_OP, TOL_CG
from workloads import CONFIGS, config_mesh, config_rhs, brick_counts, field_local

pytestmark = pytest.mark.gpu


class Full:
    def __init__(self, name):
        from oracle.nko import Oracle
        from paper_2606_12650_b200 import Nekbone
        self.name = name
        self.mesh = config_mesh(name)
        self.gpu = Nekbone.from_mesh(self.mesh)
        self.orc = Oracle.from_mesh(self.mesh)
        self.P = self.mesh.n ** 3

    def close(self):
        self.gpu.close()
        self.orc.close()


@pytest.fixture(scope="module", params=["config3", "config5"])
def full(request):
    """One full-size context pair at a time; pytest runs all tests of one parameter before the next."""
    fx = Full(request.param)
    yield fx
    fx.close()


def test_setup_whole_mesh(full):
    mesh, gpu, orc, P = full.mesh, full.gpu, full.orc, full.P
    Go = orc.geom()[0]
    Gg = to_np(gpu.geom())
    sc = np.repeat(np.abs(Go.reshape(6, -1, P)).max(axis=(0, 2)), P)    # per element, over all six factors (R14):
    for a in range(6):                                                  # off-diagonals vanish on the boundary
        assert scaled_err(Gg[a], Go[a], sc) <= TOL_OP, a
    del Go, Gg
    assert np.array_equal(to_np(gpu.mult()), orc.mult())
    assert gpu.sizes() == orc.sizes()


def test_operators_whole_vector(full):
    mesh, gpu, orc, P = full.mesh, full.gpu, full.orc, full.P
    sched = gpu.ax_launch()
    assert sched["max_batches_per_cta"] >= 9          # the persistent loop wraps its ring at these sizes
    u = field_local(mesh, 1004)
    ud = to_dev(u)
    wo, wg = orc.ax_e(u), to_np(gpu.ax_e(ud))
    assert elem_err(wg, wo, P) <= TOL_OP
    go, gg = orc.gs(u), to_np(gpu.gs(ud.clone()))
    assert scaled_err(gg, go, gs_scale(u, mesh.glo_num)) <= TOL_OP
    single = orc.mult() == 1.0
    assert np.array_equal(gg[single], u[single])     # multiplicity-1 entries bitwise unchanged
    ao, ag = orc.ax(u), to_np(gpu.ax(ud))
    assert elem_err(ag, ao, P) <= TOL_OP
    assert np.all(ag[mesh.mask == 0.0] == 0.0)
    v = np.random.Generator(np.random.PCG64(78)).uniform(-1, 1, mesh.L)
    do = orc.dot(u, v)
    dg = float(to_np(gpu.dot(ud, to_dev(v)))[0])
    # condition of the sum: sum |c u v| ~ L/4 against |sum| ~ sqrt(L)
    assert abs(dg - do) <= 1e-15 * np.sum(np.abs(u * v) / orc.mult()), (dg, do)


def test_properties_full_size(full):
    import torch
    mesh, gpu = full.mesh, full.gpu
    c = CONFIGS[full.name]
    counts = brick_counts(*c["brick"], c["N"])
    s = gpu.sizes()
    assert s["n_local"] == counts["L"] and s["n_unique"] == counts["U"]
    assert s["n_shared_unique"] == counts["shared_unique"]
    assert s["n_masked_unique"] == counts["masked_unique"]
    mult = gpu.mult()
    assert set(torch.unique(mult).tolist()) <= {1.0, 2.0, 4.0, 8.0}
    assert float((1.0 / mult).sum()) == pytest.approx(counts["U"], rel=1e-12)
    # null space before masking: gs(ax_e(1)) = 0 relative to the size of the addends
    one = torch.ones(mesh.L, dtype=torch.float64, device="cuda")
    w = gpu.ax_e(one)
    scale = float(gpu.geom().abs().max()) * 6 * mesh.n
    gpu.gs(w)
    assert float(w.abs().max()) <= 1e-12 * scale
    # symmetry of the assembled, masked operator on consistent fields
    rng = np.random.Generator(np.random.PCG64(9))
    _, inv = np.unique(mesh.glo_num, return_inverse=True)       # consistent AND masked: M A M is symmetric
    uu = to_dev(rng.uniform(-1, 1, counts["U"])[inv] * mesh.mask)
    vv = to_dev(rng.uniform(-1, 1, counts["U"])[inv] * mesh.mask)
    a = float(gpu.dot(uu, gpu.ax(vv))[0])
    b = float(gpu.dot(vv, gpu.ax(uu))[0])
    assert abs(a - b) <= 1e-11 * max(abs(a), abs(b))


def _rel(a, b):
    return abs(a - b) / abs(b) if b != 0 else abs(a)


def test_lockstep_and_free_running_cg(full):
    """One pass over the oracle's trajectory serves both protocols: at k = 1, 50, 100 the ORACLE's state
    entering the iteration is loaded into the GPU, one GPU iteration runs, and (w, pap, alpha, x, r, rho',
    beta, p) are compared at 1e-12; the GPU's own free-running solve is compared at the end."""
    mesh, gpu, orc, P = full.mesh, full.gpu, full.orc, full.P
    name = full.name
    niter = CONFIGS[name]["niter"]
    f = config_rhs(name, mesh)
    xg, hg = gpu.cg(to_dev(f), niter)                         # free-running, default options
    xg, hg = to_np(xg), to_np(hg)
    x, r, p, rho = orc.cg_init(f)
    ho = [np.sqrt(rho)]
    checks = (1, 50, 100)
    for k in range(1, niter + 1):
        if k in checks:
            xd = to_dev(x)
            gpu.cg_load_state(to_dev(r), to_dev(p), rho)
            gpu.cg_step(xd)
            sg = gpu.scalars()
            rg, pg, wg = (to_np(t) for t in gpu.cg_get_state())
        w, so = orc.cg_step(x, r, p, rho)                     # advances x, r, p in place
        if k in checks:
            assert elem_err(wg, w, P) <= TOL_OP, k
            for key in ("pap", "alpha", "rho_new", "beta"):
                assert _rel(sg[key], so[key]) <= TOL_OP, (k, key, sg[key], so[key])
            assert elem_err(to_np(xd), x, P) <= TOL_OP, k
            assert elem_err(rg, r, P) <= TOL_OP, k
            assert elem_err(pg, p, P) <= TOL_OP, k
            del rg, pg, wg, xd
        rho = so["rho_new"]
        ho.append(np.sqrt(rho))
    ho, xo = np.array(ho), x
    if name == "config3":
        # the oracle's own rounding band decides how far the flat 1e-10 applies (R15)
        alts = oracle_variants(mesh, f, niter)
        ok, worst, kstar = history_parity(hg, ho, [h for _, h in alts])
        assert kstar >= 50, kstar
        assert ok, (kstar, worst, float(np.abs(hg / ho - 1).max()))
        assert elem_err(xg, xo, P) <= max(TOL_CG, 10.0 * max(elem_err(xb, xo, P) for xb, _ in alts))
    else:
        assert np.all(np.abs(hg - ho) <= TOL_CG * ho), float(np.abs(hg / ho - 1).max())
        assert elem_err(xg, xo, P) <= TOL_CG
    assert np.all(xg[mesh.mask == 0.0] == 0.0)


def test_jacobi_diag_and_pcg_early_iterations(full):
    """NEXT row f-3 at full size: the diagonal everywhere on both configs, and on config 3 PCG through
    iteration 60 (well inside the stable part of its trajectory, see the band protocol above)."""
    mesh, gpu, orc, P = full.mesh, full.gpu, full.orc, full.P
    assert elem_err(to_np(gpu.diag()), orc.diag(), P) <= TOL_OP
    if full.name == "config3":
        f = config_rhs("config3", mesh)
        xo, ho = orc.pcg(f, 60)
        xg, hg = gpu.pcg(to_dev(f), 60)
        assert np.all(np.abs(to_np(hg) - ho) <= TOL_CG * ho), float(np.abs(to_np(hg) / ho - 1).max())
        assert elem_err(to_np(xg), xo, P) <= TOL_CG


def test_device_plan_equals_host_plan_at_full_size(full):
    """The gather-scatter plan built on the device (radix sort over hundreds of blocks and thousands of tiles, scans,
    1728 gs chunks at config 5) against the host builder's, byte for byte, at the sizes the bench runs."""
    from paper_2606_12650_b200 import Nekbone
    from paper_2606_12650_b200.binding import set_plan_builder
    mesh = full.mesh
    assert full.gpu.setup_info()["plan_builder"] == "device"
    dev = {k: v.cpu().numpy().copy() for k, v in full.gpu.plan_arrays().items()}
    try:
        set_plan_builder("host")
        host = Nekbone.from_mesh(mesh)
        assert host.setup_info()["plan_builder"] == "host"
        assert host.sizes() == full.gpu.sizes() and host.gs_sizes() == full.gpu.gs_sizes()
        for k, v in host.plan_arrays().items():
            a = v.cpu().numpy()
            assert a.shape == dev[k].shape and np.array_equal(a, dev[k]), k
        host.close()
    finally:
        set_plan_builder("device")


def test_default_iteration_is_two_kernels(full):
    """At these sizes the default CG iteration is two launches -- ax_e with the direction update folded into its load
    and pap fused, and the fused gs + mask + residual update (which every second time also applies the x update of
    two iterations) -- plus cg_init at the start and the one pending direction update at the end."""
    gpu = full.gpu
    niter = CONFIGS[full.name]["niter"]
    for k, v in (("fuse_pap", 1), ("fuse_p", 2), ("fuse_gs", 2), ("defer_x", 1)):
        assert gpu.get_option(k) == v, k
    f = to_dev(config_rhs(full.name, full.mesh))
    n0 = gpu.launch_count()
    gpu.cg(f, niter)
    assert gpu.launch_count() - n0 == 1 + 2 * niter + 1
    assert gpu.solve_path() == ("graph" if full.mesh.L <= (1 << 24) else "launches")
