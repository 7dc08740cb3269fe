"""Seeded synthetic inputs for the Nekbone CG hot path.

This package serves BOTH the oracle (`oracle/`) and the CUDA path (`paper_2606_12650_b200/`)
with bit-identical inputs.  It imports neither and holds none of the method's arithmetic: no
derivative matrix, no geometric factors, no gather-scatter, no CG.  The only mathematics in
here is where mesh nodes are placed (Gauss-Lobatto-Legendre abscissae, taken from numpy's
Legendre class) and the sine bump that deforms the brick.
"""
from .mesh import (BrickMesh, brick_mesh, gll_abscissae, rhs_unique, field_local,
                   brick_counts, sweep_brick)
from .configs import (CONFIGS, config_mesh, config_rhs, E_SWEEP, N_SWEEP, sweep_mesh, sweep_field,
                      SWEEP_REPEATS)

__all__ = ["BrickMesh", "brick_mesh", "gll_abscissae", "rhs_unique", "field_local",
           "brick_counts", "sweep_brick", "CONFIGS", "config_mesh", "config_rhs",
           "E_SWEEP", "N_SWEEP", "sweep_mesh", "sweep_field", "SWEEP_REPEATS"]
