"""Dense (non sum-factorised) spectral-element assembly used by the oracle's pins.

Independent route to the operator: element matrix A_e = sum_ab D_a^T diag(G_ab) D_b with the
Kronecker forms D_r = I (x) I (x) D, D_s = I (x) D (x) I, D_t = D (x) I (x) I acting on the local
ordering l = i + n j + n^2 k, assembled by global id.  numpy only.  (SURVEY.md §8(c) pins,
"dense cross-check of ax".)
"""
import numpy as np


def kron_derivatives(D):
    n = D.shape[0]
    I = np.eye(n)
    Dr = np.kron(I, np.kron(I, D))
    Ds = np.kron(I, np.kron(D, I))
    Dt = np.kron(D, np.kron(I, I))
    return Dr, Ds, Dt


def element_matrix(D, G6e):
    """G6e: (6, n^3) planes rr rs rt ss st tt of one element."""
    Dr, Ds, Dt = kron_derivatives(D)
    d = (Dr, Ds, Dt)
    idx = {(0, 0): 0, (0, 1): 1, (0, 2): 2, (1, 1): 3, (1, 2): 4, (2, 2): 5}
    P = Dr.shape[0]
    A = np.zeros((P, P))
    for a in range(3):
        for b in range(3):
            g = G6e[idx[(min(a, b), max(a, b))]]
            A += d[a].T @ (g[:, None] * d[b])
    return A


def unique_ids(glo_num):
    """Map arbitrary ids to 0..U-1 (ascending id order)."""
    ids, inv = np.unique(glo_num, return_inverse=True)
    return ids, inv


def assemble(D, G6, glo_num, E):
    n = D.shape[0]
    P = n ** 3
    ids, inv = unique_ids(glo_num)
    U = ids.size
    A = np.zeros((U, U))
    for e in range(E):
        sl = slice(e * P, (e + 1) * P)
        Ae = element_matrix(D, G6[:, sl])
        g = inv[sl]
        np.add.at(A, np.ix_(g, g), Ae)
    return A, inv
