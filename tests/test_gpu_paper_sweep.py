"""-m gpu parity on the paper's own sweep: N in {4, 6, 8}, E = 2^k.

The paper's only correctness evidence is that the residual after 100 CG iterations agrees between its
implementations for every (N, E) (section VIII-B; section VIII-C).  Same
criterion here, GPU against the oracle, on the full residual HISTORY and on x, for a subset of the 42 sweep
points that spans every path nk_cg takes (a handful of elements on a few CTAs, graph replay, direct launches
on the 2^14-element meshes); `python tests/sweep_parity.py --which paper` does all 42 and writes the CSV
under profiles/.  Tiny meshes converge to rounding level before iteration 100, after which two correct fp64
implementations cannot agree digit by digit: the R15 band protocol (tests/parity.history_parity) applies.
"""
import numpy as np
import pytest

from parity import elem_err, history_parity, oracle_variants
from gpu_common import Pair, to_dev, to_np, TOL_CG
from workloads import brick_mesh, rhs_unique, sweep_brick
from workloads.configs import SWEEP_AMPLITUDE, SWEEP_SEED

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("k", [1, 4, 7, 10, 12, 14])
@pytest.mark.parametrize("N", [4, 6, 8])
def test_residual_agrees_with_oracle(N, k):
    mesh = brick_mesh(*sweep_brick(k), N, SWEEP_AMPLITUDE)
    pr = Pair(mesh)
    try:
        f = rhs_unique(mesh, SWEEP_SEED)
        xo, ho = pr.orc.cg(f, 100)
        xg, hg = pr.gpu.cg(to_dev(f), 100)
        xg, hg = to_np(xg), to_np(hg)
        if not (np.all(np.abs(hg - ho) <= TOL_CG * ho) and elem_err(xg, xo, pr.P) <= TOL_CG):
            # the flat 1e-10 fails somewhere (tiny meshes past convergence; x along directions the residual
            # norm barely sees): the oracle's own rounding band decides (R15)
            alts = oracle_variants(mesh, f, 100)
            ok, worst, kstar = history_parity(hg, ho, [h for _, h in alts])
            assert ok, (N, k, worst, kstar)
            assert kstar >= 10, (N, k, kstar)
            assert elem_err(xg, xo, pr.P) <= max(TOL_CG, 10.0 * max(elem_err(xb, xo, pr.P) for xb, _ in alts)), (N, k)
        assert np.all(xg[mesh.mask == 0.0] == 0.0)
    finally:
        pr.close()
