"""Pins for the oracle's GLL basis (O1): closed forms, exactness degrees, library cross-checks.

SURVEY.md §8(c) pins "GLL nodes/weights" and "D"; BASELINE.json north_star pin 1
("GLL D differentiates polynomials of degree <= N exactly").  The paper itself says only that the
derivative matrices depend on the polynomial order.
"""
import numpy as np
import pytest
from numpy.polynomial import legendre as leg

from oracle import nko
from workloads import gll_abscissae

ALL_N = list(range(1, 16))


def test_closed_form_nodes_weights():
    s5, s37 = np.sqrt(1 / 5), np.sqrt(3 / 7)
    cases = {
        1: ([-1, 1], [1, 1]),
        2: ([-1, 0, 1], [1 / 3, 4 / 3, 1 / 3]),
        3: ([-1, -s5, s5, 1], [1 / 6, 5 / 6, 5 / 6, 1 / 6]),
        4: ([-1, -s37, 0, s37, 1], [1 / 10, 49 / 90, 32 / 45, 49 / 90, 1 / 10]),
    }
    for N, (x_ref, w_ref) in cases.items():
        xi, w, _ = nko.basis(N)
        np.testing.assert_allclose(xi, x_ref, rtol=0, atol=5e-16)
        np.testing.assert_allclose(w, w_ref, rtol=0, atol=5e-16)


@pytest.mark.parametrize("N", ALL_N)
def test_nodes_are_roots_of_PN_prime_and_symmetric(N):
    xi, w, _ = nko.basis(N)
    assert xi[0] == -1.0 and xi[-1] == 1.0
    assert np.all(np.diff(xi) > 0)
    assert np.array_equal(xi, -xi[::-1])          # exact symmetry
    assert np.array_equal(w, w[::-1])
    c = np.zeros(N + 1); c[N] = 1
    if N > 1:
        assert np.max(np.abs(leg.legval(xi[1:-1], leg.legder(c)))) < 1e-12 * N * N
    # independent route: numpy companion-matrix roots used by the mesh generator
    np.testing.assert_allclose(xi, gll_abscissae(N), rtol=0, atol=4e-16)


@pytest.mark.parametrize("N", ALL_N)
def test_quadrature_exact_to_degree_2N_minus_1(N):
    xi, w, _ = nko.basis(N)
    assert abs(w.sum() - 2.0) < 5e-16 * 4
    assert np.all(w > 0)
    for p in range(0, 2 * N):
        exact = 2.0 / (p + 1) if p % 2 == 0 else 0.0
        assert abs(np.sum(w * xi ** p) - exact) < 2e-15, (N, p)


def test_quadrature_not_exact_at_degree_2N():
    # negative test: GLL with N+1 points integrates degree 2N-1 exactly, not 2N
    for N in (2, 4, 7):
        xi, w, _ = nko.basis(N)
        err = abs(np.sum(w * xi ** (2 * N)) - 2.0 / (2 * N + 1))
        assert err > 1e-6, (N, err)
    xi, w, _ = nko.basis(7)
    assert abs(abs(np.sum(w * xi ** 14) - 2 / 15) - 2.1e-4) < 0.2e-4   # SURVEY: 2.1e-4 at N=7


def test_closed_form_D():
    _, _, D1 = nko.basis(1)
    np.testing.assert_allclose(D1, [[-0.5, 0.5], [-0.5, 0.5]], rtol=0, atol=1e-16)
    _, _, D2 = nko.basis(2)
    np.testing.assert_allclose(D2, [[-1.5, 2, -0.5], [-0.5, 0, 0.5], [0.5, -2, 1.5]], rtol=0, atol=1e-15)


@pytest.mark.parametrize("N", ALL_N)
def test_D_structure(N):
    _, _, D = nko.basis(N)
    assert D[0, 0] == -N * (N + 1) / 4 and D[N, N] == N * (N + 1) / 4
    for i in range(1, N):
        assert D[i, i] == 0.0
    # constants differentiate to zero
    assert np.max(np.abs(D.sum(axis=1))) < 2e-13 * max(1, N * N / 16)
    # centro-antisymmetry D[i,m] = -D[N-i,N-m]
    np.testing.assert_allclose(D, -D[::-1, ::-1], rtol=0, atol=1e-14 * N * N)


@pytest.mark.parametrize("N", ALL_N)
def test_D_differentiates_monomials_exactly(N):
    xi, _, D = nko.basis(N)
    tol = 1e-14 if N <= 8 else 3e-13
    for p in range(0, N + 1):
        u = xi ** p
        du = p * xi ** (p - 1) if p > 0 else np.zeros_like(xi)
        assert np.max(np.abs(D @ u - du)) < tol * max(1, N * N / 4), (N, p)


@pytest.mark.parametrize("N", [1, 2, 3, 5, 8, 12])
def test_D_is_derivative_of_lagrange_basis(N):
    # library route: l_m built from its roots with numpy.poly1d, differentiated by numpy
    xi, _, D = nko.basis(N)
    for m in range(N + 1):
        others = np.delete(xi, m)
        lm = np.poly1d(others, r=True)
        lm = lm / lm(xi[m])
        np.testing.assert_allclose(D[:, m], lm.deriv()(xi), rtol=0, atol=2e-11 * N)


def test_bad_arguments():
    with pytest.raises(nko.NkoError) as e:
        nko.basis(0)
    assert e.value.code == nko.NKO_ERR_ARG
