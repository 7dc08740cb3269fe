"""-m gpu parity of BASELINE.json configs[3] (the ax_e + gs roofline sweep) AT ITS OWN SIZES: every point
that `python -m paper_2606_12650_b200.sweep` times is a mesh the persistent ax_e loop and the chunked gs
run differently on (7 to 220 batches per CTA, 1 to 300 gs chunks), so the numbers in profiles/*sweep* rest
on these comparisons.  One application of ax_e, gs and ax on the sweep's own input (u uniform[-1,1) per
LOCAL point, seed 1004, amplitude 0.05: SURVEY.md 8(d) rows 4a/4b), whole vector against the oracle at
1e-12 in the R14 metric (tests/parity.py).
"""
import numpy as np
import pytest

from parity import elem_err, scaled_err, gs_scale
from gpu_common import Pair, to_dev, to_np, TOL_OP
from workloads import E_SWEEP, N_SWEEP, sweep_mesh, sweep_field, sweep_brick

pytestmark = pytest.mark.gpu


def _check_point(point):
    pr = Pair(sweep_mesh(point))
    try:
        u = sweep_field(pr.mesh)
        ud = to_dev(u)
        wo, wg = pr.orc.ax_e(u), to_np(pr.gpu.ax_e(ud))
        assert elem_err(wg, wo, pr.P) <= TOL_OP, (point, elem_err(wg, wo, pr.P))
        del wo, wg
        go, gg = pr.orc.gs(u), to_np(pr.gpu.gs(ud.clone()))
        assert scaled_err(gg, go, gs_scale(u, pr.mesh.glo_num)) <= TOL_OP, point
        del go, gg
        ao, ag = pr.orc.ax(u), to_np(pr.gpu.ax(ud))
        assert elem_err(ag, ao, pr.P) <= TOL_OP, point
        assert np.all(ag[pr.mesh.mask == 0.0] == 0.0)
        return pr.gpu.ax_launch(), pr.gpu.gs_sizes()
    finally:
        pr.close()


@pytest.mark.parametrize("k", [13, 15, 17])
def test_config4a_element_sweep_points(k):
    """4a: N = 7 at E = 2^13, 2^15, 2^17 (the three points the >= 70 % claim is quoted on)."""
    point = dict(brick=sweep_brick(k), N=7)
    assert point in E_SWEEP
    sched, gs = _check_point(point)
    assert sched["max_batches_per_cta"] >= (1 << k) // sched["batch_elements"] // sched["ctas"]
    assert sched["max_batches_per_cta"] >= 13
    assert gs["n_sum_rows"] > 32768                   # more than one gs chunk


@pytest.mark.parametrize("N", range(3, 16))
def test_config4b_order_sweep_points(N):
    """4b: all 13 orders N = 3..15 at E = 4096 (16^3)."""
    point = dict(brick=(16, 16, 16), N=N)
    assert point in N_SWEEP
    sched, _ = _check_point(point)
    assert sched["max_batches_per_cta"] >= 2                # every order wraps its ring at 16^3
