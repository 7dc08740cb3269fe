"""The five BASELINE.json configs as concrete seeded inputs."""
from __future__ import annotations

from .mesh import brick_mesh, rhs_unique, field_local, sweep_brick

# name -> (nx, ny, nz), N, amplitude, niter, seed          (BASELINE.json configs[0..4])
CONFIGS = {
    "config1": dict(brick=(2, 2, 2), N=3, amplitude=0.05, niter=20, seed=1001),
    "config2": dict(brick=(8, 8, 8), N=7, amplitude=0.05, niter=100, seed=1002),
    "config3": dict(brick=(16, 16, 16), N=9, amplitude=0.1, niter=100, seed=1003),
    "config5": dict(brick=(32, 32, 32), N=11, amplitude=0.1, niter=100, seed=1005),
}

# config 4: ax_e + gs roofline sweep, amplitude 0.05, seed 1004, u per LOCAL point, 50 applications
SWEEP_AMPLITUDE = 0.05
SWEEP_SEED = 1004
SWEEP_REPEATS = 50
E_SWEEP = [dict(brick=sweep_brick(k), N=7) for k in range(10, 18)]          # 4a: E = 2^10..2^17
N_SWEEP = [dict(brick=(16, 16, 16), N=N) for N in range(3, 16)]             # 4b: N = 3..15


def config_mesh(name: str):
    c = CONFIGS[name]
    return brick_mesh(*c["brick"], c["N"], c["amplitude"])


def config_rhs(name: str, mesh=None):
    c = CONFIGS[name]
    if mesh is None:
        mesh = config_mesh(name)
    return rhs_unique(mesh, c["seed"])


def sweep_mesh(point: dict):
    return brick_mesh(*point["brick"], point["N"], SWEEP_AMPLITUDE)


def sweep_field(mesh):
    return field_local(mesh, SWEEP_SEED)
