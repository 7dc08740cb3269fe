"""Pins for the oracle's operator (O3-O6): analytic -Laplace identities on the undeformed brick,
symmetry, null space, SPD, dense Kronecker assembly, dot-fusion identity.
BASELINE.json north_star pins 2-4; SURVEY.md §8(c) pins table."""
import numpy as np
import pytest

from oracle import nko
from workloads import brick_mesh, config_mesh, config_rhs
import sem_dense


def consistent_random(m, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.uniform(-1, 1, m.U)[m.glo_num]


def interior(m):
    return m.mask == 1.0


@pytest.mark.parametrize("brick,N", [((2, 2, 2), 3), ((3, 2, 1), 5), ((2, 2, 2), 2)])
def test_strong_form_minus_laplace_on_undeformed_brick(brick, N):
    """u polynomial of degree <= N in each variable => at every node off the boundary
    (QQ^T A_L u)_g = -B_g Lap u(x_g), B = QQ^T (w_i w_j w_k J)."""
    m = brick_mesh(*brick, N, 0.0)
    o = nko.Oracle.from_mesh(m)
    x, y, z = m.coords
    _, w, _ = o.basis()
    _, J = o.geom()
    n = m.n
    W3 = (w[:, None, None] * w[None, :, None] * w[None, None, :]).reshape(-1)
    B = o.gs(np.tile(W3, m.E) * J)
    p = N  # highest admissible degree per variable
    u = x ** p * y + 0.5 * y ** p * z ** (p - 1) - 2.0 * x * y * z ** p + 3 * x ** 2
    lap = (p * (p - 1) * x ** (p - 2) * y + 6.0
           + 0.5 * p * (p - 1) * y ** (p - 2) * z ** (p - 1)
           + (0.5 * (p - 1) * (p - 2) * y ** p * z ** (p - 3) if p >= 3 else 0.0)
           - 2.0 * p * (p - 1) * x * y * z ** (p - 2)) if p >= 2 else None
    lhs = o.gs(o.ax_e(u))
    rhs = -B * lap
    it = interior(m)
    scale = np.max(np.abs(rhs[it]))
    assert np.max(np.abs(lhs[it] - rhs[it])) < 2e-13 * scale


@pytest.mark.parametrize("N", [2, 3, 6])
def test_weak_form_value_23_over_24(N):
    """sum_l v_l (A_L u)_l = int grad u . grad v = 23/24 for u = x^2 y, v = xyz + x^2 on [0,1]^3."""
    m = brick_mesh(2, 3, 2, N, 0.0)
    o = nko.Oracle.from_mesh(m)
    x, y, z = m.coords
    u = x ** 2 * y
    v = x * y * z + x ** 2
    val = np.sum(v * o.ax_e(u))
    assert abs(val - 23.0 / 24.0) < 2e-14
    assert abs(np.sum(u * o.ax_e(v)) - 23.0 / 24.0) < 2e-14


@pytest.mark.parametrize("name", ["config1", "config2"])
def test_symmetry_nullspace_spd_on_deformed_mesh(name):
    m = config_mesh(name)
    o = nko.Oracle.from_mesh(m)
    u, v = consistent_random(m, 1), consistent_random(m, 2)
    Au, Av = o.gs(o.ax_e(u)), o.gs(o.ax_e(v))
    a, b = o.dot(u, Av), o.dot(v, Au)
    assert abs(a - b) < 1e-13 * max(abs(a), abs(b))
    G, _ = o.geom()
    one = o.gs(o.ax_e(np.ones(m.L)))
    assert np.max(np.abs(one)) < 1e-13 * np.abs(G).max() * m.n ** 2
    pm = o.mask(u)
    assert o.dot(pm, o.ax(pm)) > 0


def test_dense_kronecker_assembly_matches_matrix_free():
    m = config_mesh("config1")
    o = nko.Oracle.from_mesh(m)
    _, _, D = o.basis()
    G, _ = o.geom()
    A, inv = sem_dense.assemble(D, G, m.glo_num, m.E)
    assert np.max(np.abs(A - A.T)) < 1e-14 * np.abs(A).max()
    assert np.max(np.abs(A @ np.ones(m.U))) < 1e-13 * np.abs(A).max()
    rng = np.random.Generator(np.random.PCG64(3))
    for _ in range(3):
        uu = rng.uniform(-1, 1, m.U)
        ref = (A @ uu)[inv]
        got = o.gs(o.ax_e(uu[inv]))
        assert np.max(np.abs(got - ref)) < 1e-13 * np.max(np.abs(ref))
    # per-element (no assembly): matrix-free vs dense element matrix on a NON-consistent vector
    n3 = m.n ** 3
    ul = rng.uniform(-1, 1, m.L)
    wl = o.ax_e(ul)
    for e in (0, 5):
        Ae = sem_dense.element_matrix(D, G[:, e * n3:(e + 1) * n3])
        ref = Ae @ ul[e * n3:(e + 1) * n3]
        assert np.max(np.abs(wl[e * n3:(e + 1) * n3] - ref)) < 1e-13 * np.max(np.abs(ref))


def test_ax_is_mask_of_gs_of_ax_e():
    m = config_mesh("config1")
    o = nko.Oracle.from_mesh(m)
    u = consistent_random(m, 9)
    assert np.array_equal(o.ax(u), m.mask * o.gs(o.ax_e(u)))
    assert np.all(o.ax(u)[m.mask == 0.0] == 0.0)


@pytest.mark.parametrize("name", ["config1", "config2"])
def test_dot_fusion_identity(name):
    """For consistent masked p: <M QQ^T A_L p, p>_c = sum_l (A_L p)_l p_l  (pre-gs, unweighted)."""
    m = config_mesh(name)
    o = nko.Oracle.from_mesh(m)
    p = o.mask(consistent_random(m, 4))
    lhs = o.dot(o.ax(p), p)
    rhs = float(np.sum(o.ax_e(p).astype(np.longdouble) * p.astype(np.longdouble)))
    assert abs(lhs - rhs) < 1e-13 * abs(lhs)


def test_dot_counts_each_unique_node_once():
    m = config_mesh("config1")
    o = nko.Oracle.from_mesh(m)
    rng = np.random.Generator(np.random.PCG64(8))
    au, bu = rng.uniform(-1, 1, m.U), rng.uniform(-1, 1, m.U)
    assert abs(o.dot(au[m.glo_num], bu[m.glo_num]) - float(au @ bu)) < 1e-13 * m.U ** 0.5
    o.set_dot_mode(1)
    assert abs(o.dot(au[m.glo_num], bu[m.glo_num]) - float(au @ bu)) < 1e-12 * m.U ** 0.5
