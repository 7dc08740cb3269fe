"""Pins for the oracle's geometric factors (O2).  SURVEY.md §8(c) pins "geometry" and
"geometry, deformed"; the paper is silent on G (BASELINE.json north_star: "6 symmetric
geometric factors G")."""
import numpy as np
import pytest

from oracle import nko
from workloads import brick_mesh, config_mesh

RR, RS, RT, SS, ST, TT = range(6)


def single_element(N, mapfun):
    """One element whose nodes are mapfun(r, s, t) at the GLL lattice, local layout i fastest."""
    xi, w, _ = nko.basis(N)
    n = N + 1
    T, S, R = np.meshgrid(xi, xi, xi, indexing="ij")        # axes k, j, i
    x, y, z = mapfun(R, S, T)
    coords = np.stack([np.asarray(a, dtype=float).reshape(-1) for a in (x, y, z)])
    glo = np.arange(n ** 3, dtype=np.int64)
    mask = np.ones(n ** 3)
    W3 = (w[:, None, None] * w[None, :, None] * w[None, None, :]).reshape(-1)
    return coords, glo, mask, (R.reshape(-1), S.reshape(-1), T.reshape(-1)), W3


def analytic_G(W3, Jac):
    """Jac[..., a, b] = d x_a / d r_b at every node -> (G6, J) through numpy.linalg."""
    J = np.linalg.det(Jac)
    inv = np.linalg.inv(Jac)                  # inv[..., b, a] = d r_b / d x_a
    M = inv @ np.swapaxes(inv, -1, -2)        # M[b, b'] = grad r_b . grad r_b'
    G = np.stack([M[:, 0, 0], M[:, 0, 1], M[:, 0, 2], M[:, 1, 1], M[:, 1, 2], M[:, 2, 2]]) * (W3 * J)
    return G, J


@pytest.mark.parametrize("N", [1, 2, 3, 7])
def test_stretched_box_closed_form(N):
    Lx, Ly, Lz = 1.7, 0.6, 2.9
    f = lambda R, S, T: ((R + 1) / 2 * Lx, (S + 1) / 2 * Ly, (T + 1) / 2 * Lz)
    coords, glo, mask, _, W3 = single_element(N, f)
    o = nko.Oracle(1, N, coords, glo, mask)
    G, J = o.geom()
    np.testing.assert_allclose(J, Lx * Ly * Lz / 8, rtol=3e-14)
    np.testing.assert_allclose(G[RR], W3 * Ly * Lz / (2 * Lx), rtol=3e-14)
    np.testing.assert_allclose(G[SS], W3 * Lx * Lz / (2 * Ly), rtol=3e-14)
    np.testing.assert_allclose(G[TT], W3 * Lx * Ly / (2 * Lz), rtol=3e-14)
    for a in (RS, RT, ST):
        assert np.max(np.abs(G[a])) < 1e-14 * np.max(G[RR])


@pytest.mark.parametrize("name", ["config1", "config2"])
def test_volume_is_one(name):
    m = config_mesh(name)
    o = nko.Oracle.from_mesh(m)
    _, w, _ = o.basis()
    _, J = o.geom()
    n = m.n
    W3 = (w[:, None, None] * w[None, :, None] * w[None, None, :]).reshape(-1)
    vol = np.sum(J.reshape(m.E, n ** 3) * W3[None, :])
    assert abs(vol - 1.0) < 2e-14
    assert J.min() > 0


@pytest.mark.parametrize("N", [1, 2, 4])
def test_trilinear_hex_matches_analytic_jacobian(N):
    rng = np.random.Generator(np.random.PCG64(7))
    V = np.array([[-1, -1, -1], [1, -1, -1], [-1, 1, -1], [1, 1, -1],
                  [-1, -1, 1], [1, -1, 1], [-1, 1, 1], [1, 1, 1]], dtype=float)
    Vp = V + 0.25 * rng.uniform(-1, 1, V.shape)       # moved vertices, still a valid hex

    def shape(R, S, T):
        return [(1 + V[a, 0] * R) * (1 + V[a, 1] * S) * (1 + V[a, 2] * T) / 8 for a in range(8)]

    def f(R, S, T):
        sh = shape(R, S, T)
        return tuple(sum(sh[a] * Vp[a, d] for a in range(8)) for d in range(3))

    coords, glo, mask, (R, S, T), W3 = single_element(N, f)
    Jac = np.zeros((R.size, 3, 3))
    for a in range(8):
        dN = np.stack([V[a, 0] * (1 + V[a, 1] * S) * (1 + V[a, 2] * T),
                       (1 + V[a, 0] * R) * V[a, 1] * (1 + V[a, 2] * T),
                       (1 + V[a, 0] * R) * (1 + V[a, 1] * S) * V[a, 2]], axis=-1) / 8
        Jac += Vp[a][None, :, None] * dN[:, None, :]
    Gref, Jref = analytic_G(W3, Jac)
    o = nko.Oracle(1, N, coords, glo, mask)
    G, J = o.geom()
    np.testing.assert_allclose(J, Jref, rtol=2e-13)
    scale = np.abs(Gref).max(axis=0)
    assert np.max(np.abs(G - Gref) / scale[None, :]) < 1e-12
    # off-diagonal planes really are exercised (non-zero, both signs)
    for a in (RS, RT, ST):
        assert np.abs(Gref[a]).max() > 1e-3 * np.abs(Gref[RR]).max()


@pytest.mark.parametrize("N", [2, 5])
def test_quadratic_map_matches_analytic_jacobian(N):
    a, b = 0.2, 0.15
    f = lambda R, S, T: (R + a * (1 - R * R) * S, S + b * T * T, T + 0.1 * R * S)
    coords, glo, mask, (R, S, T), W3 = single_element(N, f)
    Jac = np.zeros((R.size, 3, 3))
    Jac[:, 0, 0] = 1 - 2 * a * R * S; Jac[:, 0, 1] = a * (1 - R * R); Jac[:, 0, 2] = 0
    Jac[:, 1, 0] = 0;                 Jac[:, 1, 1] = 1;               Jac[:, 1, 2] = 2 * b * T
    Jac[:, 2, 0] = 0.1 * S;           Jac[:, 2, 1] = 0.1 * R;         Jac[:, 2, 2] = 1
    Gref, Jref = analytic_G(W3, Jac)
    o = nko.Oracle(1, N, coords, glo, mask)
    G, J = o.geom()
    np.testing.assert_allclose(J, Jref, rtol=2e-13)
    scale = np.abs(Gref).max(axis=0)
    assert np.max(np.abs(G - Gref) / scale[None, :]) < 1e-12


def _rotation():
    # proper rotation from a QR factorisation
    rng = np.random.Generator(np.random.PCG64(11))
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    return Q


def test_rotation_invariance_reflection_and_scaling():
    m = brick_mesh(2, 2, 2, 4, 0.05)
    o = nko.Oracle.from_mesh(m)
    G, J = o.geom()
    Q = _rotation()
    o_rot = nko.Oracle(m.E, m.N, Q @ m.coords, m.glo_num, m.mask)
    G_rot, J_rot = o_rot.geom()
    scale = np.abs(G).max()
    assert np.max(np.abs(G_rot - G)) < 1e-13 * scale
    np.testing.assert_allclose(J_rot, J, rtol=1e-12)
    # reflection: left-handed elements -> error
    refl = m.coords.copy(); refl[0] = -refl[0]
    with pytest.raises(nko.NkoError) as e:
        nko.Oracle(m.E, m.N, refl, m.glo_num, m.mask)
    assert e.value.code == nko.NKO_ERR_GEOM
    # scaling by lambda scales G by lambda and J by lambda^3
    lam = 3.0
    G_s, J_s = nko.Oracle(m.E, m.N, lam * m.coords, m.glo_num, m.mask).geom()
    assert np.max(np.abs(G_s - lam * G)) < 1e-13 * lam * scale
    np.testing.assert_allclose(J_s, lam ** 3 * J, rtol=1e-12)


def test_pointwise_spd():
    m = config_mesh("config1")
    G, _ = nko.Oracle.from_mesh(m).geom()
    M = np.empty((m.L, 3, 3))
    M[:, 0, 0], M[:, 0, 1], M[:, 0, 2] = G[RR], G[RS], G[RT]
    M[:, 1, 0], M[:, 1, 1], M[:, 1, 2] = G[RS], G[SS], G[ST]
    M[:, 2, 0], M[:, 2, 1], M[:, 2, 2] = G[RT], G[ST], G[TT]
    assert np.all(np.linalg.eigvalsh(M) > 0)


def test_cyclic_axis_relabelling_permutes_G():
    # new element axes (r',s',t') = (s,t,r): data transposed so that i' <-> old j, j' <-> old k,
    # k' <-> old i.  Then G'_{r'r'} = G_ss, G'_{r's'} = G_st, G'_{r't'} = G_sr, G'_{s's'} = G_tt,
    # G'_{s't'} = G_tr, G'_{t't'} = G_rr at the same physical point.
    m = brick_mesh(2, 1, 1, 3, 0.0)
    n = m.n
    c = m.coords.reshape(3, m.E, n, n, n).copy()          # axes e, k, j, i
    rng = np.random.Generator(np.random.PCG64(5))
    # smooth, orientation-preserving deformation
    x, y, z = c
    c = np.stack([x + 0.05 * np.sin(2 * y) * z, y + 0.04 * x * z, z + 0.03 * np.cos(x) * y])
    flat = c.reshape(3, -1)
    G = nko.Oracle(m.E, m.N, flat, m.glo_num, m.mask).geom()[0].reshape(6, m.E, n, n, n)
    # old [e,k,j,i] -> new [e,k'=i,j'=k,i'=j]
    perm = (0, 3, 1, 2)
    c_new = np.stack([np.transpose(c[d], perm) for d in range(3)]).reshape(3, -1)
    glo_new = np.transpose(m.glo_num.reshape(m.E, n, n, n), perm).reshape(-1)
    G_new = nko.Oracle(m.E, m.N, c_new, glo_new, np.ones(m.L)).geom()[0].reshape(6, m.E, n, n, n)
    expect = {RR: SS, RS: ST, RT: RS, SS: TT, ST: RT, TT: RR}
    scale = np.abs(G).max()
    for new, old in expect.items():
        assert np.max(np.abs(G_new[new] - np.transpose(G[old], perm))) < 1e-13 * scale, (new, old)
    # the off-diagonal planes are distinct, so a swapped pair would be caught
    assert np.max(np.abs(G[RS] - G[RT])) > 1e-4 * scale
    assert np.max(np.abs(G[RS] - G[ST])) > 1e-4 * scale


def test_fine_mesh_element_against_40_digit_arithmetic():
    """Conditioning pin (R22): on a fine, deformed mesh the derivative sums of absolute
    coordinates cancel ~10^3 leading digits, and a derivative matrix rounded to double (row sums
    ~1e-16 |D| instead of 0) alone costs G three digits.  O2 re-evaluated with mpmath at 40 digits
    (GLL nodes by Newton on P_N', D and weights from their closed forms, S 8(c) O1-O2) must agree
    with the oracle's G to a few ulp of the element scale."""
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 40
    N = 9
    m = brick_mesh(32, 2, 2, N, 0.1)
    n, P = m.n, m.n ** 3
    G, _ = nko.Oracle.from_mesh(m).geom()
    G = G.reshape(6, m.E, P)

    def leg(x):                      # P_N(x), P_{N-1}(x) by the three-term recurrence
        a, b = mp.mpf(1), x
        for k in range(1, N):
            a, b = b, ((2 * k + 1) * x * b - k * a) / (k + 1)
        return b, a

    xi, _, _ = nko.basis(N)
    xs = [mp.mpf(-1)] + [None] * (N - 1) + [mp.mpf(1)]
    for i in range(1, N):
        t = mp.mpf(float(xi[i]))
        for _ in range(60):          # Newton on q = P_{N+1} - P_{N-1}, q' = (2N+1) P_N
            pn, pm = leg(t)
            pp = ((2 * N + 1) * t * pn - N * pm) / (N + 1)
            t -= (pp - pm) / ((2 * N + 1) * pn)
        xs[i] = t
    pn = [leg(x)[0] for x in xs]
    D = [[(pn[i] / (pn[q] * (xs[i] - xs[q])) if i != q else
           (-mp.mpf(N * (N + 1)) / 4 if i == 0 else (mp.mpf(N * (N + 1)) / 4 if i == N else mp.mpf(0))))
          for q in range(n)] for i in range(n)]
    w = [2 / (N * (N + 1) * p * p) for p in pn]

    e = 31 + 32 * 3                  # last element along x: coordinates near 1, spacing 1/32
    X = [[mp.mpf(float(v)) for v in m.coords[c].reshape(m.E, P)[e]] for c in range(3)]
    idx = lambda i, j, k: i + n * j + n * n * k
    worst = 0.0
    scale = float(np.abs(G[:, e, :]).max())
    for (i, j, k) in [(0, 0, 0), (n - 1, n - 1, n - 1), (3, 5, 7), (n - 1, 0, 4), (4, 4, 4), (1, 8, 2)]:
        d = [[sum(D[i][q] * X[c][idx(q, j, k)] for q in range(n)),
              sum(D[j][q] * X[c][idx(i, q, k)] for q in range(n)),
              sum(D[k][q] * X[c][idx(i, j, q)] for q in range(n))] for c in range(3)]
        (xr, xs_, xt), (yr, ys, yt), (zr, zs, zt) = d
        r = (ys * zt - yt * zs, zs * xt - zt * xs_, xs_ * yt - xt * ys)
        s = (yt * zr - yr * zt, zt * xr - zr * xt, xt * yr - xr * yt)
        t = (yr * zs - ys * zr, zr * xs_ - zs * xr, xr * ys - xs_ * yr)
        J = xr * r[0] + yr * r[1] + zr * r[2]
        sc = w[i] * w[j] * w[k] / J
        dot = lambda a, b: a[0] * b[0] + a[1] * b[1] + a[2] * b[2]
        for c, (a, b) in enumerate([(r, r), (r, s), (r, t), (s, s), (s, t), (t, t)]):
            worst = max(worst, abs(float(sc * dot(a, b)) - G[c, e, idx(i, j, k)]) / scale)
    assert worst <= 4e-16, worst
