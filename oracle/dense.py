"""Brute-force dense assembly of the Wilson-Dirac operator -- TEST INFRASTRUCTURE (pins oracle.c).

Independent of the stencil in oracle.c: builds the forward-hop matrices
    H_mu[(x,a),(y,b)] = sigma+_mu(x) * U^R_mu(x)[a,b] * delta_{y, x+mu}
and assembles (BASELINE.json:north_star, SURVEY.md section 8(c) oracle step 4)
    D = (4+m0) * 1  -  1/2 * sum_mu [ (1-gamma_mu) (x) H_mu  +  (1+gamma_mu) (x) H_mu^dagger ]
with numpy Kronecker-style products; the backward term of the definition is exactly H_mu^dagger.
Rows/columns are ordered (site i lexicographic, spin alpha, colour a), i.e. the flattening of a
canonical [V][4][d] field.  Only usable on tiny lattices (the matrix is (4 d V)^2).
"""
from __future__ import annotations

import numpy as np


def hop_matrix(dims, bc, links_R: np.ndarray, mu: int) -> np.ndarray:
    """H_mu as a [V, d, V, d] array."""
    dims = [int(v) for v in dims]
    V = int(np.prod(dims))
    d = links_R.shape[-1]
    H = np.zeros((V, d, V, d), dtype=np.complex128)
    for i in range(V):
        x = list(np.unravel_index(i, dims))
        sgn = bc[mu] if x[mu] == dims[mu] - 1 else 1
        y = list(x)
        y[mu] = (x[mu] + 1) % dims[mu]
        j = int(np.ravel_multi_index(y, dims))
        H[i, :, j, :] += sgn * links_R[i, mu]
    return H


def dirac_matrix(dims, bc, links_R: np.ndarray, m0: float, gammas, hopping_only: bool = False) -> np.ndarray:
    """Dense D (or Dphi if hopping_only) of shape [4dV, 4dV]; gammas = [g0, g1, g2, g3] (4x4)."""
    V = int(np.prod([int(v) for v in dims]))
    d = links_R.shape[-1]
    n = V * 4 * d
    D = np.zeros((V, 4, d, V, 4, d), dtype=np.complex128)
    one = np.eye(4)
    for mu in range(4):
        H = hop_matrix(dims, bc, links_R, mu)
        Hd = np.conj(np.transpose(H, (2, 3, 0, 1)))
        D += -0.5 * np.einsum("st,iajb->isajtb", one - gammas[mu], H)
        D += -0.5 * np.einsum("st,iajb->isajtb", one + gammas[mu], Hd)
    D = D.reshape(n, n)
    if not hopping_only:
        D = D + (4.0 + m0) * np.eye(n)
    return D
