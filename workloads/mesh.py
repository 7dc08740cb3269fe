"""Brick meshes of hexahedral spectral elements in Nekbone's element-local layout.

Recipe (SURVEY.md §8(c) readings R8-R11, §8(d); BASELINE.json `configs`):

* Box [0,1]^3 cut into nx*ny*nz elements, element order e = ex + nx*(ey + ny*ez)        (R9)
* Each element carries n^3 points, n = N+1, local index l = e*n^3 + i + n*j + n^2*k,
  i <-> r (fastest), j <-> s, k <-> t
* Unperturbed node position  x0 = (ex + (xi_i + 1)/2)/nx  with xi the GLL abscissae      (R9)
* Perturbation: the same scalar s = a*sin(2 pi x0) sin(2 pi y0) sin(2 pi z0), evaluated at the
  UNPERTURBED position, is added to all three coordinates                                  (R8)
* glo_num: lattice id g = gx + (nx*N+1)*(gy + (ny*N+1)*gz), gx = ex*N + i, 0-based int64  (R10)
* mask = 0.0 on every local copy of a node on the outer boundary of the box, else 1.0     (R11)

Coordinates are computed ONCE PER UNIQUE LATTICE NODE and then copied to the element-local
layout, so all copies of a shared node are bitwise equal.

Nothing in this module differentiates, integrates, assembles or solves anything.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
from numpy.polynomial import legendre as _leg


def gll_abscissae(N: int) -> np.ndarray:
    """Gauss-Lobatto-Legendre abscissae -1 = xi_0 < ... < xi_N = 1 for order N >= 1.

    Interior points are the roots of P_N'(x), taken from numpy's Legendre companion-matrix
    root finder and polished by two Newton steps; the set is symmetrised so xi_i = -xi_{N-i}
    exactly.  Used only to PLACE mesh nodes; the oracle and the CUDA library each compute
    their own basis.
    """
    if N < 1:
        raise ValueError("N must be >= 1")
    if N == 1:
        return np.array([-1.0, 1.0])
    cN = np.zeros(N + 1)
    cN[N] = 1.0
    d1 = _leg.legder(cN)
    d2 = _leg.legder(d1)
    x = np.sort(np.real(_leg.legroots(d1)))
    for _ in range(2):
        x = x - _leg.legval(x, d1) / _leg.legval(x, d2)
    xi = np.concatenate(([-1.0], x, [1.0]))
    xi = 0.5 * (xi - xi[::-1])
    return xi


@dataclass
class BrickMesh:
    nx: int
    ny: int
    nz: int
    N: int
    amplitude: float
    coords: np.ndarray    # (3, L) float64, planes x | y | z, element-local layout
    glo_num: np.ndarray   # (L,) int64
    mask: np.ndarray      # (L,) float64, exactly 0.0 or 1.0

    @property
    def E(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def n(self) -> int:
        return self.N + 1

    @property
    def L(self) -> int:
        return self.E * self.n ** 3

    @property
    def U(self) -> int:
        N = self.N
        return (self.nx * N + 1) * (self.ny * N + 1) * (self.nz * N + 1)


def _axis_positions(nel: int, N: int, xi: np.ndarray) -> np.ndarray:
    """Unperturbed 1-D lattice positions, one per lattice index g = e*N + i (length nel*N+1)."""
    pos = np.empty(nel * N + 1)
    half = (xi + 1.0) / 2.0
    for e in range(nel):
        pos[e * N:(e + 1) * N] = (e + half[:N]) / nel
    pos[nel * N] = 1.0
    return pos


def _local_lattice_index(nx, ny, nz, N):
    n = N + 1
    gx = np.arange(nx, dtype=np.int64)[:, None] * N + np.arange(n, dtype=np.int64)[None, :]
    gy = np.arange(ny, dtype=np.int64)[:, None] * N + np.arange(n, dtype=np.int64)[None, :]
    gz = np.arange(nz, dtype=np.int64)[:, None] * N + np.arange(n, dtype=np.int64)[None, :]
    mx, my = nx * N + 1, ny * N + 1
    # axes: ez, ey, ex, k, j, i
    GX = gx[None, None, :, None, None, :]
    GY = gy[None, :, None, None, :, None]
    GZ = gz[:, None, None, :, None, None]
    glo = GX + mx * (GY + my * GZ)
    return np.ascontiguousarray(glo).reshape(-1)


def brick_mesh(nx: int, ny: int, nz: int, N: int, amplitude: float) -> BrickMesh:
    xi = gll_abscissae(N)
    X1 = _axis_positions(nx, N, xi)
    Y1 = _axis_positions(ny, N, xi)
    Z1 = _axis_positions(nz, N, xi)
    two_pi = 2.0 * np.pi
    sx, sy, sz = np.sin(two_pi * X1), np.sin(two_pi * Y1), np.sin(two_pi * Z1)
    # one value per unique lattice node, array axes (gz, gy, gx)
    S = amplitude * (sz[:, None, None] * sy[None, :, None] * sx[None, None, :])
    glo = _local_lattice_index(nx, ny, nz, N)
    L = glo.shape[0]
    coords = np.empty((3, L))
    coords[0] = (X1[None, None, :] + S).reshape(-1)[glo]
    coords[1] = (Y1[None, :, None] + S).reshape(-1)[glo]
    coords[2] = (Z1[:, None, None] + S).reshape(-1)[glo]
    del S
    mx, my, mz = nx * N + 1, ny * N + 1, nz * N + 1
    bx = np.zeros(mx, dtype=bool); bx[[0, mx - 1]] = True
    by = np.zeros(my, dtype=bool); by[[0, my - 1]] = True
    bz = np.zeros(mz, dtype=bool); bz[[0, mz - 1]] = True
    bnd = bz[:, None, None] | by[None, :, None] | bx[None, None, :]
    mask = np.where(bnd.reshape(-1)[glo], 0.0, 1.0)
    return BrickMesh(nx, ny, nz, N, float(amplitude), coords, glo, mask)


def rhs_unique(mesh: BrickMesh, seed: int) -> np.ndarray:
    """f ~ uniform[-1,1) drawn once per UNIQUE node, copied to the local layout (R7)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    fu = rng.uniform(-1.0, 1.0, mesh.U)
    return fu[mesh.glo_num]


def field_local(mesh: BrickMesh, seed: int) -> np.ndarray:
    """u ~ uniform[-1,1) drawn per LOCAL point: copies of a shared node differ (config 4)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.uniform(-1.0, 1.0, mesh.L)


def brick_counts(nx: int, ny: int, nz: int, N: int) -> dict:
    """Exact node counts of a brick by counting lattice lines (no mesh is built).

    Along one axis with nel elements the lattice has nel*N+1 nodes; nel-1 of them sit on an
    interior element interface (1-D multiplicity 2), the rest have 1-D multiplicity 1, and the
    two end nodes are on the boundary.  3-D multiplicity is the product over the axes.
    """
    n = N + 1
    E = nx * ny * nz
    L = E * n ** 3
    tot = [a * N + 1 for a in (nx, ny, nz)]
    c2 = [a - 1 for a in (nx, ny, nz)]                    # 1-D multiplicity 2
    c1 = [t - c for t, c in zip(tot, c2)]                  # 1-D multiplicity 1
    U = tot[0] * tot[1] * tot[2]
    single = c1[0] * c1[1] * c1[2]                         # nodes of multiplicity 1
    interior_unique = (tot[0] - 2) * (tot[1] - 2) * (tot[2] - 2)
    interior_local = 1
    for a in range(3):
        interior_local *= (c1[a] - 2) + 2 * c2[a]
    single_interior = (c1[0] - 2) * (c1[1] - 2) * (c1[2] - 2)
    return dict(E=E, L=L, U=U,
                shared_unique=U - single, shared_local=L - single,
                masked_unique=U - interior_unique, masked_local=L - interior_local,
                masked_single=single - single_interior)


def sweep_brick(k: int):
    """nx >= ny >= nz, powers of two, nx*ny*nz = 2^k (reading R13)."""
    a = -(-k // 3)
    b = -(-(k - a) // 2)
    c = k - a - b
    return 2 ** a, 2 ** b, 2 ** c
