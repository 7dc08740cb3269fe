"""-m gpu: nk_dot_static, the entry point that allocates nothing (include/nk.h; csrc/nk_static.cu).

It is a variant of the weighted dot product nk_dot (S 8(a) a4) whose scratch -- per-block partials and the
ticket counter -- is a fixed __device__ array inside the library instead of the caller's workspace.  Checked against
the existing path, nk_dot, on the same vectors with c = 1/multiplicity, on two calls in a row (the second on other
data: the shared array still holds the first call's partials), at the tolerance the operator tests use for dot
products, 1e-15 x sum |c a b| (tests/test_gpu_fullsize.py).  This file sorts last on purpose: the suite runs with
pytest -x, so a failure here hides nothing after it.  It passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

from workloads import brick_mesh

pytestmark = pytest.mark.gpu


def _vectors(mesh, seed):
    import torch
    rng = np.random.Generator(np.random.PCG64(seed))
    a = torch.from_numpy(rng.uniform(-1, 1, mesh.L)).cuda()
    b = torch.from_numpy(rng.uniform(-1, 1, mesh.L)).cuda()
    return a, b


@pytest.mark.parametrize("brick,N", [((3, 2, 2), 4), ((12, 10, 9), 7), ((5, 3, 3), 6)])
def test_dot_static_matches_nk_dot_on_two_calls_in_a_row(brick, N):
    """Small (one block), 553 K points (68 blocks, ragged last one), and an odd point count."""
    import torch
    from paper_2606_12650_b200 import Nekbone
    from paper_2606_12650_b200.binding import dot_static
    mesh = brick_mesh(*brick, N, 0.05)
    gpu = Nekbone.from_mesh(mesh)
    try:
        c = 1.0 / gpu.mult()
        for seed in (3, 4):                                   # two calls in a row, different data
            a, b = _vectors(mesh, seed)
            want = float(gpu.dot(a, b)[0])
            got = float(dot_static(a, b, c)[0])
            tol = 1e-15 * float((c * a * b).abs().sum())
            assert abs(got - want) <= tol, (seed, got, want, tol)
            again = float(dot_static(a, b, c)[0])             # same inputs: bitwise reproducible
            assert again == got
        # plain dot product (c = NULL) against a float64 sum on the host, same tolerance
        a, b = _vectors(mesh, 5)
        got = float(dot_static(a, b)[0])
        an, bn = a.cpu().numpy(), b.cpu().numpy()
        assert abs(got - float(np.dot(an, bn))) <= 1e-15 * float(np.abs(an * bn).sum())
        # a misaligned view takes the scalar loads: same run of entries per block
        v = float(dot_static(a[1:], b[1:], c[1:])[0])
        w = float((c[1:] * a[1:] * b[1:]).sum())
        assert abs(v - w) <= 1e-15 * float((c[1:] * a[1:] * b[1:]).abs().sum())
    finally:
        gpu.close()


def test_dot_static_limits_and_degenerate_sizes():
    import torch
    from paper_2606_12650_b200 import NkError
    from paper_2606_12650_b200.binding import dot_static, dot_static_max_n, load, _check, _vp, _stream
    assert dot_static_max_n() == 1 << 27
    assert load().nk_static_setup() == 0
    a = torch.ones(16, dtype=torch.float64, device="cuda")
    out = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")
    dot_static(a, a, out=out, n=0)
    assert float(out[0]) == 0.0                               # n = 0 stores 0
    assert float(dot_static(a, a, n=1)[0]) == 1.0
    assert float(dot_static(a, a)[0]) == 16.0
    with pytest.raises(NkError) as e:                         # rejected before anything is launched or read
        _check(load().nk_dot_static(_vp(a.data_ptr()), _vp(a.data_ptr()), None, dot_static_max_n() + 1,
                                    _vp(out.data_ptr()), _stream()))
    assert e.value.code == -9
    assert load().nk_dot_static(None, None, None, 4, None, None) == -1
    assert float(out[0]) == 0.0


def test_dot_static_at_the_largest_size_it_serves():
    """n = 2^27 (1 GiB per vector, 16384 blocks: every slot of the scratch array in use), then a small call right
    after it on the same stream: stale partials of the big call must not leak into the small one."""
    import torch
    from paper_2606_12650_b200.binding import dot_static, dot_static_max_n
    n = dot_static_max_n()
    a = torch.full((n,), 0.5, dtype=torch.float64, device="cuda")
    b = torch.full((n,), 2.0, dtype=torch.float64, device="cuda")
    a[n - 1] = 3.0
    big = dot_static(a, b)
    small = dot_static(a[:1000], b[:1000])
    assert float(big[0]) == float(n - 1) + 6.0                # exact: integers below 2^53
    assert float(small[0]) == 1000.0
