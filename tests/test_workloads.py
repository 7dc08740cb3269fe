"""The seeded input generator: shapes, counts, reproducibility, consistency of shared copies."""
import numpy as np

from workloads import (brick_mesh, config_mesh, config_rhs, brick_counts, sweep_brick,
                       field_local, CONFIGS, E_SWEEP, N_SWEEP)


def test_config1_shapes_and_determinism():
    m = config_mesh("config1")
    assert (m.E, m.N, m.L, m.U) == (8, 3, 512, 343)
    assert m.coords.shape == (3, 512) and m.glo_num.dtype == np.int64
    m2 = config_mesh("config1")
    assert np.array_equal(m.coords, m2.coords) and np.array_equal(m.glo_num, m2.glo_num)
    f, f2 = config_rhs("config1", m), config_rhs("config1", m2)
    assert np.array_equal(f, f2) and f.min() >= -1 and f.max() < 1
    # consistency: copies of a node carry identical coordinates and rhs values
    order = np.argsort(m.glo_num, kind="stable")
    g = m.glo_num[order]
    same = g[1:] == g[:-1]
    for a in (m.coords[0], m.coords[1], m.coords[2], f, m.mask):
        assert np.array_equal(a[order][1:][same], a[order][:-1][same])


def test_domain_stays_unit_cube_and_mask_is_boundary():
    m = config_mesh("config2")
    assert m.coords.min() == 0.0 and m.coords.max() == 1.0
    on_bnd = np.any((m.coords == 0.0) | (m.coords == 1.0), axis=0)
    assert np.array_equal(on_bnd, m.mask == 0.0)
    c = brick_counts(8, 8, 8, 7)
    assert int((m.mask == 0).sum()) == c["masked_local"]
    assert np.unique(m.glo_num).size == c["U"]


def test_element_and_point_ordering():
    # e = ex + nx*(ey + ny*ez); l = e*n^3 + i + n*j + n^2*k with i <-> x on an undeformed brick
    m = brick_mesh(3, 2, 2, 2, 0.0)
    n = m.n
    x, y, z = (a.reshape(m.E, n, n, n) for a in m.coords)
    assert np.all(np.diff(x, axis=3) > 0) and np.all(np.diff(y, axis=2) > 0) and np.all(np.diff(z, axis=1) > 0)
    assert x[1].min() > x[0].min() and np.isclose(x[1].min(), 1 / 3)       # ex fastest
    assert np.isclose(y[3].min(), 0.5) and np.isclose(z[6].min(), 0.5)


def test_sweep_bricks():
    shapes = [sweep_brick(k) for k in range(10, 18)]
    assert shapes == [(16, 8, 8), (16, 16, 8), (16, 16, 16), (32, 16, 16), (32, 32, 16),
                      (32, 32, 32), (64, 32, 32), (64, 64, 32)]
    assert [p["N"] for p in N_SWEEP] == list(range(3, 16))
    assert all(np.prod(p["brick"]) == 2 ** k for p, k in zip(E_SWEEP, range(10, 18)))


def test_field_local_differs_across_copies():
    m = config_mesh("config1")
    u = field_local(m, 1004)
    order = np.argsort(m.glo_num, kind="stable")
    g = m.glo_num[order]
    same = g[1:] == g[:-1]
    assert np.all(u[order][1:][same] != u[order][:-1][same])


def test_config_table():
    assert CONFIGS["config5"]["brick"] == (32, 32, 32) and CONFIGS["config5"]["N"] == 11
    assert CONFIGS["config3"]["amplitude"] == 0.1 and CONFIGS["config2"]["niter"] == 100


def test_history_parity_protocol():
    """The R15 protocol helper the GPU tests rely on: flat 1e-10 while the oracle's own band is small,
    band-scaled or 'both converged' beyond."""
    import sys, os
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    from parity import history_parity
    k = np.arange(40)
    ho = 10.0 ** (-0.5 * k)                                  # converges 20 decades in 40 iterations
    hb = ho * (1 + np.where(k < 25, 1e-15, 1e-3))            # the oracle's two builds part ways at k = 25
    good = ho * (1 + np.where(k < 25, 5e-12, 0.5))           # ... where everything is below 1e-9 h0
    ok, worst, kstar = history_parity(good, ho, hb)
    assert ok and kstar == 24 and 4e-12 < worst < 6e-12
    bad = good.copy(); bad[10] *= 1 + 1e-9                   # a real disagreement inside the flat part
    assert not history_parity(bad, ho, hb)[0]
    notconv = ho.copy(); notconv[30] = 1e-3                  # beyond the band, but one side did not converge
    assert not history_parity(notconv, ho, hb)[0]
