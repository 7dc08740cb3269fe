"""Shared helpers of the -m gpu parity tests: build both sides on the same seeded mesh."""
import functools

import numpy as np

from workloads import brick_mesh, config_mesh, CONFIGS

TOL_OP = 1e-12     # BJ north_star: ax / gs relative 1e-12 per entry (metric: DESIGN.md R14)
TOL_CG = 1e-10     # BJ north_star: CG solution and residual history


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def to_np(t):
    return t.detach().cpu().numpy()


class Pair:
    """The oracle and the CUDA path set up on one mesh."""

    def __init__(self, mesh):
        from oracle.nko import Oracle
        from paper_2606_12650_b200 import Nekbone
        self.mesh = mesh
        self.orc = Oracle.from_mesh(mesh)
        self.gpu = Nekbone.from_mesh(mesh)
        self.P = mesh.n ** 3
        self.L = mesh.L

    def close(self):
        self.orc.close()
        self.gpu.close()


@functools.lru_cache(maxsize=4)
def pair_for_brick(nx, ny, nz, N, amplitude):
    return Pair(brick_mesh(nx, ny, nz, N, amplitude))


@functools.lru_cache(maxsize=2)
def pair_for_config(name):
    return Pair(config_mesh(name))


def rng_field(L, seed):
    return np.random.Generator(np.random.PCG64(seed)).uniform(-1.0, 1.0, L)
