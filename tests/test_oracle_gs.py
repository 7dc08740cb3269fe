"""Pins for the oracle's gather-scatter (O4, O7): brute-force multiplicities, analytic node
counts, algebraic identities, id-relabelling invariance.  north_star pin 5."""
import numpy as np
import pytest

from oracle import nko
from workloads import brick_mesh, config_mesh, brick_counts


def test_multiplicity_by_brute_force_on_config1():
    m = config_mesh("config1")
    o = nko.Oracle.from_mesh(m)
    mult = o.mult()
    brute = (m.glo_num[:, None] == m.glo_num[None, :]).sum(axis=1)            # O(L^2)
    assert np.array_equal(mult, brute.astype(float))
    # same count from bitwise-equal coordinates (copies of a node share coordinates exactly)
    c = m.coords.T.copy().view([("x", "f8"), ("y", "f8"), ("z", "f8")]).reshape(-1)
    same = (c[:, None] == c[None, :]).sum(axis=1)
    assert np.array_equal(mult, same.astype(float))
    assert set(np.unique(mult)) <= {1.0, 2.0, 4.0, 8.0}
    assert np.sum(1.0 / mult) == m.U


@pytest.mark.parametrize("brick,N", [((2, 2, 2), 3), ((8, 8, 8), 7), ((3, 2, 1), 4), ((16, 8, 8), 2), ((1, 1, 1), 5)])
def test_counts_match_analytic_lattice_counts(brick, N):
    m = brick_mesh(*brick, N, 0.05)
    o = nko.Oracle.from_mesh(m)
    s = o.sizes()
    a = brick_counts(*brick, N)
    assert s["n_local"] == a["L"] == m.L
    assert s["n_unique"] == a["U"] == m.U
    assert s["n_shared_unique"] == a["shared_unique"]
    assert s["n_masked_unique"] == a["masked_unique"]
    mult = o.mult()
    assert int(np.sum(mult > 1)) == a["shared_local"]
    assert int(np.sum(m.mask == 0)) == a["masked_local"]
    assert int(np.sum((m.mask == 0) & (mult == 1))) == a["masked_single"]


def test_survey_size_table_rows():
    # SURVEY.md §8 size table, configs 1 and 2
    a = brick_counts(2, 2, 2, 3)
    assert (a["L"], a["U"], a["shared_unique"], a["shared_local"], a["masked_unique"],
            a["masked_local"], a["masked_single"]) == (512, 343, 127, 296, 218, 296, 152)
    a = brick_counts(8, 8, 8, 7)
    assert (a["L"], a["U"], a["shared_unique"], a["shared_local"], a["masked_unique"],
            a["masked_local"], a["masked_single"]) == (262144, 185193, 60193, 137144, 18818, 23816, 14408)
    a = brick_counts(32, 32, 32, 11)
    assert (a["L"], a["U"], a["shared_unique"], a["shared_local"], a["masked_unique"],
            a["masked_local"], a["masked_single"]) == (56623104, 43986977, 10600729, 23236856, 743426, 880136, 618248)


def test_gs_identities():
    m = config_mesh("config2")
    o = nko.Oracle.from_mesh(m)
    rng = np.random.Generator(np.random.PCG64(21))
    v = rng.uniform(-1, 1, m.L)
    g = o.gs(v)
    mult = o.mult()
    # library route: bincount over compressed ids
    _, inv = np.unique(m.glo_num, return_inverse=True)
    ref = np.bincount(inv, weights=v)[inv]
    assert np.max(np.abs(g - ref)) < 4e-16 * 8
    # single copies bitwise untouched
    assert np.array_equal(g[mult == 1], v[mult == 1])
    # all copies of a node carry the same value afterwards
    first = np.zeros(m.U); first[inv] = g
    assert np.array_equal(first[inv], g)
    # gs(gs(v)) = mult o gs(v)   (to rounding: the ordered sum s+s+s passes through 3s)
    assert np.max(np.abs(o.gs(g) - mult * g)) < 1e-15 * 8
    # sum over unique nodes preserved: sum_l c_l gs(v)_l = sum_l v_l
    assert abs(np.sum(g / mult) - np.sum(v)) < 1e-10


def test_gs_accepts_arbitrary_ids():
    m = config_mesh("config1")
    rng = np.random.Generator(np.random.PCG64(31))
    relabel = rng.permutation(10 * m.U)[:m.U].astype(np.int64) * 977 + 5     # sparse, unordered ids
    o1 = nko.Oracle.from_mesh(m)
    o2 = nko.Oracle(m.E, m.N, m.coords, relabel[m.glo_num], m.mask)
    v = rng.uniform(-1, 1, m.L)
    assert np.array_equal(o1.gs(v), o2.gs(v))
    assert o1.sizes() == o2.sizes()


def test_setup_errors():
    m = config_mesh("config1")
    bad = m.glo_num.copy(); bad[3] = -1
    with pytest.raises(nko.NkoError) as e:
        nko.Oracle(m.E, m.N, m.coords, bad, m.mask)
    assert e.value.code == nko.NKO_ERR_ID
    mk = m.mask.copy(); mk[0] = 0.5
    with pytest.raises(nko.NkoError) as e:
        nko.Oracle(m.E, m.N, m.coords, m.glo_num, mk)
    assert e.value.code == nko.NKO_ERR_MASK
    # copies of one node disagree
    mult = nko.Oracle.from_mesh(m).mult()
    l = int(np.nonzero((mult > 1) & (m.mask == 1))[0][0])
    mk = m.mask.copy(); mk[l] = 0.0
    with pytest.raises(nko.NkoError) as e:
        nko.Oracle(m.E, m.N, m.coords, m.glo_num, mk)
    assert e.value.code == nko.NKO_ERR_MASK
