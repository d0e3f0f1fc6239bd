"""Oracle for SURVEY.md section 8(f) NEXT-4, the clover term -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md:70 lists "clover [17]" improvement of the Wilson-Dirac operator and prints no formula.  Reading C28 of
DESIGN.md (the Sheikholeslami-Wohlert term in the normalisation of north_star's D = (4+m0) + Dphi):

    D_sw psi(x) = D psi(x) + T(x) psi(x),      T(x) = -(c_sw / 2) sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}(x)
    sigma_{mu nu} = (i/2) [gamma_mu, gamma_nu]                       (acts on spin)
    F_{mu nu}(x)  = (Q_{mu nu}(x) - Q_{mu nu}(x)^dagger) / (8 i)     (Hermitian d_R x d_R, acts on colour)
    Q_{mu nu}(x)  = sum of the four plaquettes ("leaves") of the mu-nu plane that start and end at x, all taken
                    counter-clockwise (mu -> nu), built from the REPRESENTED links:
        U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
      + U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
      + U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
      + U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
With U = exp(i A) this gives F_{mu nu} = d_mu A_nu - d_nu A_mu + O(a^2) (pinned by the constant abelian field in
tests/test_oracle_clover.py).  Links are periodic; the fermionic boundary signs do not enter T (reading C9).

Written with whole-lattice numpy arrays and np.roll, one line per term, nothing blocked or fused; gamma matrices come
from oracle.gamma (the C tables of reading C1).  Imports nothing from paper_2405_19294_b200.
"""
from __future__ import annotations

import numpy as np

from . import dirac, eo_to_lex, gamma, lex_to_eo


def _at(field, dims, shifts):
    """field(x + sum_k shifts[k] e_k) for a lattice-shaped array [T,X,Y,Z,...]; periodic."""
    out = field
    for ax, s in enumerate(shifts):
        if s:
            out = np.roll(out, -s, axis=ax)
    return out


def _dag(m):
    return np.conj(np.swapaxes(m, -1, -2))


def field_strength(dims, links_R, mu, nu):
    """F_{mu nu}(x) for all sites, lexicographic [V, d, d] complex (Hermitian)."""
    dims = tuple(int(v) for v in dims)
    d = links_R.shape[-1]
    U = links_R.reshape(dims + (4, d, d))
    e = lambda k, s=1: tuple(s if a == k else 0 for a in range(4))
    add = lambda a, b: tuple(x + y for x, y in zip(a, b))
    Um = lambda sh: _at(U[..., mu, :, :], dims, sh)
    Un = lambda sh: _at(U[..., nu, :, :], dims, sh)
    z = (0, 0, 0, 0)
    q = Um(z) @ Un(e(mu)) @ _dag(Um(e(nu))) @ _dag(Un(z))
    q = q + Un(z) @ _dag(Um(add(e(mu, -1), e(nu)))) @ _dag(Un(e(mu, -1))) @ Um(e(mu, -1))
    q = q + _dag(Um(e(mu, -1))) @ _dag(Un(add(e(mu, -1), e(nu, -1)))) @ Um(add(e(mu, -1), e(nu, -1))) @ Un(e(nu, -1))
    q = q + _dag(Un(e(nu, -1))) @ Um(e(nu, -1)) @ Un(add(e(mu), e(nu, -1))) @ _dag(Um(z))
    f = (q - _dag(q)) / 8j
    return f.reshape(-1, d, d)


def sigma(mu, nu):
    g = [gamma(k) for k in range(4)]
    return 0.5j * (g[mu] @ g[nu] - g[nu] @ g[mu])


def clover_term(dims, links_R, csw):
    """T(x) as [V, 4, d, 4, d] (row spin, row colour, column spin, column colour), lexicographic sites."""
    d = links_R.shape[-1]
    V = int(np.prod([int(v) for v in dims]))
    T = np.zeros((V, 4, d, 4, d), dtype=np.complex128)
    for mu in range(4):
        for nu in range(mu + 1, 4):
            T += -0.5 * csw * np.einsum("st,xab->xsatb", sigma(mu, nu), field_strength(dims, links_R, mu, nu))
    return T


def apply_clover_lex(T, psi_lex):
    return np.einsum("xsatb,xtb->xsa", T, psi_lex)


def dirac_clover(dims, bc, links_R, m0, csw, psi_eo):
    """D_sw on a full field [even half | odd half]."""
    T = clover_term(dims, links_R, csw)
    tpsi = lex_to_eo(dims, apply_clover_lex(T, eo_to_lex(dims, psi_eo)))
    return dirac(dims, bc, links_R, m0, psi_eo) + tpsi


# ---- exponentiated clover ("exponentiated clover improvement [8]"; reading C31) -----------------------
def exp_clover_term(dims, links_R, m0, csw):
    """Reading C31: the site-diagonal part (4+m0) + T(x) of D_sw is replaced by (4+m0) exp(T(x) / (4+m0)), which is
    positive definite for every gauge field.  Returned is E(x) = (4+m0) [exp(T(x)/(4+m0)) - 1] as [V, 4, d, 4, d], so
    that D_exp = D + E; computed from the Hermitian eigendecomposition of the dense 4d x 4d matrix of every site."""
    m = 4.0 + m0
    T = clover_term(dims, links_R, csw)
    V, d = T.shape[0], T.shape[2]
    Tm = T.reshape(V, 4 * d, 4 * d)
    w, Q = np.linalg.eigh(Tm)
    E = (Q * (m * np.expm1(w / m))[:, None, :]) @ np.conj(np.swapaxes(Q, -1, -2))
    return E.reshape(V, 4, d, 4, d)


def dirac_expclover(dims, bc, links_R, m0, csw, psi_eo):
    """D_exp on a full field [even half | odd half]: Dphi psi + (4+m0) exp(T/(4+m0)) psi."""
    E = exp_clover_term(dims, links_R, m0, csw)
    epsi = lex_to_eo(dims, apply_clover_lex(E, eo_to_lex(dims, psi_eo)))
    return dirac(dims, bc, links_R, m0, psi_eo) + epsi


# ---- even-odd preconditioning WITH the clover term ("even-odd preconditioning, clover"; reading C32) ----
def site_term(dims, links_R, m0, csw, exponentiated=False):
    """The site-diagonal part A(x) of the improved operator as dense [V, 4d, 4d] matrices (lexicographic sites):
    A = (4+m0) + T (clover) or (4+m0) exp(T/(4+m0)) (exponentiated clover)."""
    m = 4.0 + m0
    X = exp_clover_term(dims, links_R, m0, csw) if exponentiated else clover_term(dims, links_R, csw)
    V, d = X.shape[0], X.shape[2]
    return X.reshape(V, 4 * d, 4 * d) + m * np.eye(4 * d)[None]


def _halves(dims, A_lex):
    """[V, n, n] lexicographic -> (even sites, odd sites) in canonical half-field order."""
    eo = lex_to_eo(dims, A_lex)
    vh = A_lex.shape[0] // 2
    return eo[:vh], eo[vh:]


def _blockmul(A_half, psi_half):
    n = A_half.shape[-1]
    return (A_half @ psi_half.reshape(psi_half.shape[0], n, 1)).reshape(psi_half.shape)


def dhat_clover(dims, bc, links_R, m0, csw, psi_e, exponentiated=False):
    """Reading C32: with D_sw = [[A_ee, Dphi_eo], [Dphi_oe, A_oo]] the even-odd preconditioned operator is the Schur
    complement on the even sites,  Dhat_sw = A_ee - Dphi_eo A_oo^{-1} Dphi_oe  (not multiplied by anything: A is a
    matrix now, not the number 4+m0 of reading C20)."""
    from . import dphi_eo
    Ae, Ao = _halves(dims, site_term(dims, links_R, m0, csw, exponentiated))
    t = dphi_eo(dims, bc, links_R, 1, psi_e)                                   # odd sites
    n = Ao.shape[-1]
    t = np.linalg.solve(Ao, t.reshape(t.shape[0], n, 1)).reshape(t.shape)       # A_oo^{-1}
    return _blockmul(Ae, psi_e) - dphi_eo(dims, bc, links_R, 0, t)


def dirac_clover_solve(dims, bc, links_R, m0, csw, b_eo, tol, maxiter, exponentiated=False):
    """x = D_sw^{-1} b through the preconditioned system (BiCGstab of oracle.solver on Dhat_sw):
    Dhat_sw x_e = b_e - Dphi_eo A_oo^{-1} b_o,   x_o = A_oo^{-1} (b_o - Dphi_oe x_e).  Returns (x_eo, iterations)."""
    from . import dphi_eo
    from .solver import bicgstab
    Ae, Ao = _halves(dims, site_term(dims, links_R, m0, csw, exponentiated))
    n = Ao.shape[-1]
    ainv = lambda v: np.linalg.solve(Ao, v.reshape(v.shape[0], n, 1)).reshape(v.shape)
    vh = b_eo.shape[0] // 2
    b_e, b_o = b_eo[:vh], b_eo[vh:]
    rhs = b_e - dphi_eo(dims, bc, links_R, 0, ainv(b_o))
    op = lambda v: dhat_clover(dims, bc, links_R, m0, csw, v, exponentiated)
    x_e, it, _ = bicgstab(op, rhs, tol, maxiter)
    x_o = ainv(b_o - dphi_eo(dims, bc, links_R, 1, x_e))
    return np.concatenate([x_e, x_o], axis=0), it
