"""-m gpu parity where the kernels actually run at full size: the multi-batch persistent loop of ax_e.

ax_e launches min(batches, SMs) persistent CTAs, so a CTA runs more than one batch -- ring wrap, mbarrier
phase flips, next-pencil prefetch, work-array aliasing between batches -- only on meshes with more than
SMs x nk_ax_batch_elements(N) elements.  The order sweep of test_gpu_operators.py uses 6-45 elements
(every CTA runs ONE batch).  Here, for every order N = 1..15, the mesh is sized so that every CTA runs at
least 8 batches (the ring holds up to 3: each mbarrier flips its phase at least twice), with a ragged last
round and a ragged last batch, and ONE application of ax_e, gs and ax on a field drawn per LOCAL point
(copies differ: SURVEY.md 8(d) "do the parity check on a single application") is compared with the oracle
over the WHOLE vector at 1e-12 (metric: DESIGN.md R14 = tests/parity.py).  Two lock-step CG iterations
from the oracle's state then take the same loop through the fused variants (pap inside ax_e; p = r + beta p
folded into the load of the second iteration's ax_e), with fuse_p off and on.
"""
import numpy as np
import pytest

from parity import elem_err, scaled_err, gs_scale
from gpu_common import Pair, to_dev, to_np, TOL_OP
from workloads import brick_mesh, field_local, rhs_unique

pytestmark = pytest.mark.gpu

MIN_BATCHES_PER_CTA = 8


def _sm_count():
    import torch
    return int(torch.cuda.get_device_properties(0).multi_processor_count)


def multibatch_brick(N: int, sms: int):
    """Smallest near-cubic brick with >= 8 batches on every CTA, E not a multiple of the batch size
    (ragged last batch) and a number of batches that is not a multiple of the CTA count (ragged round)."""
    from paper_2606_12650_b200.binding import ax_batch_elements
    epb = ax_batch_elements(N)
    need = MIN_BATCHES_PER_CTA * sms * epb + 1
    a = max(2, int(round(need ** (1.0 / 3.0))))
    for nx in range(a, 4 * a + 64):
        for ny, nz in ((a, a), (a, a - 1), (a + 1, a - 1), (a + 1, a)):
            E = nx * ny * nz
            nb = -(-E // epb)
            if E >= need and (epb == 1 or E % epb) and nb % sms and nb // sms >= MIN_BATCHES_PER_CTA:
                return (nx, ny, nz), epb
    raise AssertionError("no brick found")


def _rel(a, b):
    return abs(a - b) / abs(b) if b != 0 else abs(a)


@pytest.mark.parametrize("N", range(1, 16))
def test_persistent_loop_every_order(N):
    sms = _sm_count()
    brick, epb = multibatch_brick(N, sms)
    pr = Pair(brick_mesh(*brick, N, 0.1))
    try:
        sched = pr.gpu.ax_launch()
        assert sched["batch_elements"] == epb and sched["ctas"] == sms
        assert sched["max_batches_per_cta"] > MIN_BATCHES_PER_CTA          # ragged: some CTAs run one more
        # ---- one application of each operator, whole vector -------------------------------------------
        u = field_local(pr.mesh, 1004)
        ud = to_dev(u)
        wo, wg = pr.orc.ax_e(u), to_np(pr.gpu.ax_e(ud))
        assert elem_err(wg, wo, pr.P) <= TOL_OP, (N, brick, elem_err(wg, wo, pr.P))
        go, gg = pr.orc.gs(u), to_np(pr.gpu.gs(ud.clone()))
        assert scaled_err(gg, go, gs_scale(u, pr.mesh.glo_num)) <= TOL_OP, (N, brick)
        ao, ag = pr.orc.ax(u), to_np(pr.gpu.ax(ud))
        assert elem_err(ag, ao, pr.P) <= TOL_OP, (N, brick)
        assert np.all(ag[pr.mesh.mask == 0.0] == 0.0)
        # ---- two lock-step CG iterations: fused pap, then the p update folded into ax_e's load ---------
        f = rhs_unique(pr.mesh, 2000 + N)
        x, r, p, rho = pr.orc.cg_init(f)
        states = []
        for _ in range(2):
            w, so = pr.orc.cg_step(x, r, p, rho)
            rho = so["rho_new"]
            states.append((w.copy(), dict(so), x.copy(), r.copy(), p.copy()))
        x0, r0, p0, rho0 = pr.orc.cg_init(f)
        for fuse_p in (0, 1):
            pr.gpu.set_option("fuse_p", fuse_p)
            for nsteps in (1, 2):
                # (reading the state back applies a pending p update, so the folded update only runs when the
                #  two steps follow one another without a read in between)
                xd = to_dev(x0)
                pr.gpu.cg_load_state(to_dev(r0), to_dev(p0), rho0)
                for _ in range(nsteps):
                    pr.gpu.cg_step(xd)
                sg = pr.gpu.scalars()
                rg, pg, wg = (to_np(t) for t in pr.gpu.cg_get_state())
                w, so, xo, ro, po = states[nsteps - 1]
                key = (N, fuse_p, nsteps)
                assert elem_err(wg, w, pr.P) <= TOL_OP, key
                for name in ("pap", "alpha", "rho_new", "beta"):
                    assert _rel(sg[name], so[name]) <= TOL_OP, (key, name, sg[name], so[name])
                assert elem_err(to_np(xd), xo, pr.P) <= TOL_OP, key
                assert elem_err(rg, ro, pr.P) <= TOL_OP, key
                assert elem_err(pg, po, pr.P) <= TOL_OP, key
        pr.gpu.set_option("fuse_p", 2)
    finally:
        pr.close()
