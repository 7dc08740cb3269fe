"""-m gpu parity: set-up (basis, geometry, multiplicity, sizes), ax_e, gs, ax, dot -- CUDA path
through the C-ABI vs the oracle, element by element, on the same seeded inputs (SURVEY.md 8(c)
protocol part 1; tolerance metric DESIGN.md R14 = tests/parity.py)."""
import numpy as np
import pytest

from parity import elem_err, scaled_err, gs_scale, maxnorm_rel
from gpu_common import Pair, pair_for_brick, pair_for_config, to_dev, to_np, rng_field, TOL_OP
from workloads import brick_mesh, brick_counts, field_local

pytestmark = pytest.mark.gpu

# small bricks spanning every order; element counts chosen NOT to be multiples of the kernels'
# elements-per-block, so every launch has a ragged last block
ALL_N = [(3, 2, 1, N) if N > 8 else (3, 3, 2, N) if N > 3 else (5, 3, 3, N) for N in range(1, 16)]


def test_basis_matches_oracle():
    from oracle import nko
    for N in range(1, 16):
        pr = pair_for_brick(1, 1, 1, N, 0.0)
        xi, w, D = pr.gpu.basis()
        xo, wo, Do = nko.basis(N)
        assert np.abs(xi - xo).max() <= 1e-15
        assert np.abs(w - wo).max() <= 1e-15 * np.abs(wo).max()
        assert np.abs(D - Do).max() <= 1e-14 * np.abs(Do).max(), N


@pytest.mark.parametrize("nx,ny,nz,N", ALL_N)
def test_setup_geometry_mult_sizes(nx, ny, nz, N):
    pr = pair_for_brick(nx, ny, nz, N, 0.1)
    Go, _ = pr.orc.geom()
    Gg = to_np(pr.gpu.geom())
    for a in range(6):
        # off-diagonal planes hold exact zeros; scale by the element's largest |G| over all six
        sc = np.repeat(np.abs(Go.reshape(6, -1, pr.P)).max(axis=(0, 2)), pr.P)
        assert scaled_err(Gg[a], Go[a], sc) <= TOL_OP, (N, a)
    assert np.array_equal(to_np(pr.gpu.mult()), pr.orc.mult())
    assert pr.gpu.sizes() == pr.orc.sizes()
    cnt = brick_counts(nx, ny, nz, N)
    s = pr.gpu.sizes()
    assert (s["n_local"], s["n_unique"], s["n_shared_unique"], s["n_masked_unique"]) == \
        (cnt["L"], cnt["U"], cnt["shared_unique"], cnt["masked_unique"])


@pytest.mark.parametrize("nx,ny,nz,N", ALL_N)
def test_ax_e_every_order(nx, ny, nz, N):
    pr = pair_for_brick(nx, ny, nz, N, 0.1)
    u = rng_field(pr.L, 7 + N)
    wo = pr.orc.ax_e(u)
    wg = to_np(pr.gpu.ax_e(to_dev(u)))
    assert elem_err(wg, wo, pr.P) <= TOL_OP, (N, elem_err(wg, wo, pr.P), maxnorm_rel(wg, wo))


@pytest.mark.parametrize("nx,ny,nz,N", ALL_N)
def test_gs_and_ax_every_order(nx, ny, nz, N):
    pr = pair_for_brick(nx, ny, nz, N, 0.1)
    v = rng_field(pr.L, 100 + N)                     # copies differ: exercises gs fully
    go = pr.orc.gs(v)
    gg = to_np(pr.gpu.gs(to_dev(v)))
    assert scaled_err(gg, go, gs_scale(v, pr.mesh.glo_num)) <= TOL_OP
    single = pr.orc.mult() == 1.0
    assert np.array_equal(gg[single], v[single])     # multiplicity-1 entries bitwise unchanged
    wo = pr.orc.ax(v)
    wg = to_np(pr.gpu.ax(to_dev(v)))
    assert elem_err(wg, wo, pr.P) <= TOL_OP
    assert np.all(wg[pr.mesh.mask == 0.0] == 0.0)    # Dirichlet nodes exactly zero


@pytest.mark.parametrize("name", ["config1", "config2"])
def test_operators_on_configs(name):
    pr = pair_for_config(name)
    u = field_local(pr.mesh, 1004)
    ud = to_dev(u)
    wo, wg = pr.orc.ax_e(u), to_np(pr.gpu.ax_e(ud))
    assert elem_err(wg, wo, pr.P) <= TOL_OP
    go, gg = pr.orc.gs(u), to_np(pr.gpu.gs(ud.clone()))
    assert scaled_err(gg, go, gs_scale(u, pr.mesh.glo_num)) <= TOL_OP
    ao, ag = pr.orc.ax(u), to_np(pr.gpu.ax(ud))
    assert elem_err(ag, ao, pr.P) <= TOL_OP
    Go, _ = pr.orc.geom()
    Gg = to_np(pr.gpu.geom())
    sc = np.repeat(np.abs(Go.reshape(6, -1, pr.P)).max(axis=(0, 2)), pr.P)
    assert max(scaled_err(Gg[a], Go[a], sc) for a in range(6)) <= TOL_OP


def test_dot_weighted_by_inverse_multiplicity():
    pr = pair_for_config("config2")
    a, b = rng_field(pr.L, 1), rng_field(pr.L, 2)
    do = pr.orc.dot(a, b)
    dg = float(to_np(pr.gpu.dot(to_dev(a), to_dev(b)))[0])
    # condition of the sum: sum |c a b| ~ L/4 against |sum| ~ sqrt(L)
    bound = 1e-15 * np.sum(np.abs(a * b) / pr.orc.mult())
    assert abs(dg - do) <= bound, (dg, do)
    # odd L takes the scalar tail: 1 element at N=2 -> L = 27
    pr2 = pair_for_brick(1, 1, 1, 2, 0.0)
    a, b = rng_field(27, 3), rng_field(27, 4)
    assert abs(float(to_np(pr2.gpu.dot(to_dev(a), to_dev(b)))[0]) - pr2.orc.dot(a, b)) <= 1e-14


def test_bitwise_reproducible_run_to_run():
    pr = pair_for_config("config2")
    u = to_dev(field_local(pr.mesh, 5))
    w1 = pr.gpu.ax(u).clone()
    w2 = pr.gpu.ax(u).clone()
    assert bool((w1 == w2).all())
    d1 = pr.gpu.dot(u, w1).clone()
    d2 = pr.gpu.dot(u, w1).clone()
    assert float(d1) == float(d2)


def test_gs_arbitrary_ids_and_odd_multiplicities():
    """Ids need not be contiguous or lattice-like; rows of length 3, 5, 12 take the generic path."""
    from oracle.nko import Oracle
    from paper_2606_12650_b200 import Nekbone
    m = brick_mesh(2, 2, 1, 3, 0.0)
    rng = np.random.Generator(np.random.PCG64(11))
    glo = rng.integers(0, 60, m.L).astype(np.int64) * 1_000_003 + 17      # ~4.3 copies per id, scattered
    glo[:12] = 5                                                           # one row of >= 12 copies
    mask = np.ones(m.L)
    mask[np.isin(glo, glo[100:103])] = 0.0
    orc, gpu = Oracle(m.E, m.N, m.coords, glo, mask), Nekbone(m.E, m.N, m.coords, glo, mask)
    v = rng.uniform(-1, 1, m.L)
    go, gg = orc.gs(v), to_np(gpu.gs(to_dev(v)))
    assert scaled_err(gg, go, gs_scale(v, glo)) <= TOL_OP
    assert np.array_equal(to_np(gpu.mult()), orc.mult())
    ao, ag = orc.ax(v), to_np(gpu.ax(to_dev(v)))
    assert elem_err(ag, ao, m.n ** 3) <= TOL_OP
    assert gpu.sizes() == orc.sizes()


def test_single_element_and_order_one():
    for (nx, ny, nz, N) in [(1, 1, 1, 1), (1, 1, 1, 7), (2, 1, 1, 1)]:
        pr = pair_for_brick(nx, ny, nz, N, 0.0)
        u = rng_field(pr.L, 9)
        assert elem_err(to_np(pr.gpu.ax_e(to_dev(u))), pr.orc.ax_e(u), pr.P) <= TOL_OP
        assert elem_err(to_np(pr.gpu.ax(to_dev(u))), pr.orc.ax(u), pr.P) <= TOL_OP


def test_setup_errors():
    from paper_2606_12650_b200 import Nekbone, NkError, NK_ERR_GEOM, NK_ERR_ID, NK_ERR_MASK
    m = brick_mesh(2, 2, 2, 3, 0.05)
    co = m.coords.copy()
    co[0] = -co[0]                                   # reflection: left-handed elements, J < 0
    with pytest.raises(NkError) as ei:
        Nekbone(m.E, m.N, co, m.glo_num, m.mask)
    assert ei.value.code == NK_ERR_GEOM
    co = m.coords.copy()
    P = m.n ** 3
    co[:, 3 * P:4 * P] = co[:, 3 * P:4 * P][:, ::-1]  # one inverted element
    with pytest.raises(NkError) as ei:
        Nekbone(m.E, m.N, co, m.glo_num, m.mask)
    assert ei.value.code == NK_ERR_GEOM
    g = m.glo_num.copy(); g[5] = -1
    with pytest.raises(NkError) as ei:
        Nekbone(m.E, m.N, m.coords, g, m.mask)
    assert ei.value.code == NK_ERR_ID
    mk = m.mask.copy(); mk[7] = 0.5
    with pytest.raises(NkError) as ei:
        Nekbone(m.E, m.N, m.coords, m.glo_num, mk)
    assert ei.value.code == NK_ERR_MASK
    mk = m.mask.copy()
    shared = np.flatnonzero(m.glo_num == m.glo_num[m.n - 1])   # a node with >= 2 copies
    assert shared.size >= 2
    mk[shared[0]] = 1.0 - mk[shared[0]]                        # copies disagree
    with pytest.raises(NkError) as ei:
        Nekbone(m.E, m.N, m.coords, m.glo_num, mk)
    assert ei.value.code == NK_ERR_MASK


def test_rotation_invariance_through_the_gpu_path():
    """Rigid rotation leaves every G_ab unchanged (SURVEY 8(c) geometry pin ii) -- property at the
    GPU's own precision, independent of the oracle."""
    from paper_2606_12650_b200 import Nekbone
    m = brick_mesh(2, 2, 2, 5, 0.1)
    th = 0.7
    R = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1.0]])
    R = R @ np.array([[1, 0, 0], [0, np.cos(0.3), -np.sin(0.3)], [0, np.sin(0.3), np.cos(0.3)]])
    g0 = to_np(Nekbone.from_mesh(m).geom())
    g1 = to_np(Nekbone(m.E, m.N, R @ m.coords, m.glo_num, m.mask).geom())
    sc = np.repeat(np.abs(g0.reshape(6, -1, 216)).max(axis=(0, 2)), 216)
    assert max(scaled_err(g1[a], g0[a], sc) for a in range(6)) <= 1e-13


def test_plan_does_not_depend_on_host_threads():
    """nk_setup builds the gather-scatter plan on all host cores (parallel radix sort, group walk cut at group
    boundaries, chunked packing); the plan -- hence gs, ax and a CG solve with the fused gs, bit for bit -- must be
    the one a single thread builds.  Irregular ids (rows of 3, 5, 12 copies) and a brick with several gs chunks."""
    from paper_2606_12650_b200 import Nekbone
    from paper_2606_12650_b200.binding import set_host_threads, set_plan_builder
    set_plan_builder("host")                                  # the default builder runs on the device (test below)
    m1 = brick_mesh(3, 2, 2, 4, 0.05)
    rng = np.random.Generator(np.random.PCG64(13))
    glo = rng.integers(0, 400, m1.L).astype(np.int64) * 1_000_003 + 17
    glo[:12] = 5
    mask = np.ones(m1.L)
    mask[np.isin(glo, glo[100:110])] = 0.0
    m2 = brick_mesh(24, 20, 16, 3, 0.05)                      # 7680 elements, 116 K summed rows: four gs chunks
    cases = [(m1.E, m1.N, m1.coords, glo, mask), (m2.E, m2.N, m2.coords, m2.glo_num, m2.mask)]
    try:
        for E, N, co, g, mk in cases:
            L = E * (N + 1) ** 3
            v = to_dev(rng.uniform(-1, 1, L))
            _, inv = np.unique(g, return_inverse=True)
            f = to_dev(rng.uniform(-1, 1, inv.max() + 1)[inv])
            out = []
            for threads in (1, 3, 0):
                set_host_threads(threads)
                gpu = Nekbone(E, N, co, g, mk)
                gpu.set_option("coop", 0)
                gpu.set_option("fuse_gs", 1)
                x, h = gpu.cg(f, 10)
                assert gpu.setup_info()["plan_builder"] == "host"
                out.append((gpu.sizes(), gpu.gs_sizes(), to_np(gpu.gs(v.clone())), to_np(gpu.ax(v)), to_np(gpu.mult()),
                            to_np(x), to_np(h)) + tuple(a.cpu().numpy().copy() for a in gpu.plan_arrays().values()))
                gpu.close()
            for o in out[1:]:
                assert o[0] == out[0][0] and o[1] == out[0][1]
                for a, b in zip(o[2:], out[0][2:]):
                    assert np.array_equal(a, b)
    finally:
        set_host_threads(0)
        set_plan_builder("device")


def _irregular_case(rng):
    """Ids drawn at random (rows of many lengths, some longer than 8), a run of 12 equal ids, Dirichlet nodes."""
    m = brick_mesh(3, 2, 2, 4, 0.05)
    glo = rng.integers(0, 400, m.L).astype(np.int64) * 1_000_003 + 17
    glo[:12] = 5
    mask = np.ones(m.L)
    mask[np.isin(glo, glo[100:110])] = 0.0
    return m.E, m.N, m.coords, glo, mask


def test_device_plan_equals_host_plan():
    """nk_setup builds the gather-scatter plan on the device by default (csrc/nk_plan.cu: radix sort, scans, per-point
    kernels); every array of it -- codes, CSR, packed rows and descriptors, gather codes, gx rows and their per-block
    cut, multiplicity tables -- and every size must equal, byte for byte, what the host builder produces.  Cases: a
    single element (no shared node), irregular ids (rows of 3, 5, 12 copies, ids up to 4e8: four sort passes), all ids
    equal (one group of L copies), a brick with several gs chunks and an odd point count, ids above 2^40."""
    from paper_2606_12650_b200 import Nekbone
    from paper_2606_12650_b200.binding import set_plan_builder
    rng = np.random.Generator(np.random.PCG64(29))
    m0 = brick_mesh(1, 1, 1, 2, 0.0)
    m2 = brick_mesh(24, 20, 16, 3, 0.05)
    m3 = brick_mesh(5, 3, 3, 6, 0.05)
    m4 = brick_mesh(2, 2, 1, 2, 0.0)
    cases = {
        "single element": (m0.E, m0.N, m0.coords, m0.glo_num, m0.mask),
        "irregular ids": _irregular_case(rng),
        "all ids equal": (m4.E, m4.N, m4.coords, np.full(m4.L, 7, dtype=np.int64), np.ones(m4.L)),
        "all ids zero, masked": (m4.E, m4.N, m4.coords, np.zeros(m4.L, dtype=np.int64), np.zeros(m4.L)),
        "four gs chunks": (m2.E, m2.N, m2.coords, m2.glo_num, m2.mask),
        "odd point count": (m3.E, m3.N, m3.coords, m3.glo_num, m3.mask),
        "ids above 2^40": (m3.E, m3.N, m3.coords, m3.glo_num * 3 + (1 << 41), m3.mask),
    }
    try:
        for name, (E, N, co, g, mk) in cases.items():
            got = {}
            for which in ("host", "device"):
                set_plan_builder(which)
                gpu = Nekbone(E, N, co, g, mk)
                assert gpu.setup_info()["plan_builder"] == which
                got[which] = (gpu.sizes(), gpu.gs_sizes(), {k: v.cpu().numpy().copy() for k, v in gpu.plan_arrays().items()})
                gpu.close()
            assert got["host"][0] == got["device"][0], name
            assert got["host"][1] == got["device"][1], name
            for k, a in got["host"][2].items():
                b = got["device"][2][k]
                assert a.shape == b.shape, (name, k, a.shape, b.shape)
                assert np.array_equal(a, b), (name, k, int(np.flatnonzero(a != b)[0]))
    finally:
        set_plan_builder("device")


def test_device_plan_rejects_what_the_host_plan_rejects():
    from paper_2606_12650_b200 import Nekbone
    from paper_2606_12650_b200.binding import NkError
    m = brick_mesh(2, 2, 2, 3, 0.0)
    bad_id = m.glo_num.copy()
    bad_id[5] = -1
    bad_mask = m.mask.copy()
    bad_mask[7] = 0.5
    clash = m.mask.copy()
    shared = np.flatnonzero(np.bincount(m.glo_num)[m.glo_num] > 1)
    clash[shared[0]] = 1.0 - clash[shared[0]]
    for g, mk, code in ((bad_id, m.mask, -3), (m.glo_num, bad_mask, -4), (m.glo_num, clash, -4)):
        with pytest.raises(NkError) as e:
            Nekbone(m.E, m.N, m.coords, g, mk)
        assert e.value.code == code
