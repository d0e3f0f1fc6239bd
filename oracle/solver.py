"""Oracle for the rows SURVEY.md section 8(f) NEXT-1 adds -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The paper names these operations but prints no formula for any of them: "even-odd preconditioning"
(PAPER.md:70), the spinor linear algebra "Copy spinor field", "g5 application", "g5 mulc add assign", inner
products and norms (Fig. 7) and "the Conjugate Gradient" inverter.  What is
written out below are their plain definitions under the readings C20-C24 of DESIGN.md:

  C20  even-odd preconditioned operator, on EVEN sites:   Dhat = (4+m0)^2 - Dphi_eo Dphi_oe
       (the Schur complement of D = [[m, Dphi_eo], [Dphi_oe, m]], m = 4+m0, times m).
  C21  Dhat^dagger = gamma5 Dhat gamma5 (gamma5-hermiticity); the CG runs on the normal equations
       Dhat^dagger Dhat x = Dhat^dagger b, started from x = 0, with the recursively updated residual and the
       stopping rule  |r_k|^2 <= tol^2 |rhs|^2  checked after every update.
  C22  <a, b> = sum conj(a) b (antilinear in the first slot); norm2(a) = <a, a>; sums in fp64.
  C23  "g5 mulc add assign":  out += c gamma5 in;  "mulc add assign": out += c in  (c complex).
  C24  full solve D x = b through the preconditioned system:
       Dhat x_e = m b_e - Dphi_eo b_o,   x_o = (b_o - Dphi_oe x_e) / m.

  C29  BiCGstab (below);  C33  gamma5-QMR (below): both written out at their definitions further down.

Every function is numpy on canonical half fields [V/2][4][d] complex128 and calls oracle.dphi_eo (the C
definition of the hopping term) as its only non-trivial step; the CG is the textbook algorithm, one line per
step, no fusion.  Pins: tests/test_oracle_solver.py (dense Schur complement and numpy.linalg.solve through
oracle.dense, CG's finite-termination property on matrices with k distinct eigenvalues, hermiticity of
gamma5 Dhat).  Imports nothing from paper_2405_19294_b200.
"""
from __future__ import annotations

import numpy as np

from . import dphi_eo

_G5 = np.array([1.0, 1.0, -1.0, -1.0])[None, :, None]  # gamma5 = diag(1,1,-1,-1), reading C1


# ---- spinor linear algebra (readings C22, C23) ----------------------------------
def g5(psi):
    return psi * _G5


def mulc_add_assign(out, c, psi):
    """out += c psi (returns the new out; no in-place aliasing games)."""
    return out + complex(c) * psi


def g5_mulc_add_assign(out, c, psi):
    """out += c gamma5 psi."""
    return out + complex(c) * g5(psi)


def dot(a, b):
    """<a, b> = sum conj(a) b, fp64 accumulation (math.fsum-free: numpy pairwise sum in complex128)."""
    return complex(np.sum(np.conj(a.astype(np.complex128)) * b.astype(np.complex128)))


def norm2(a):
    a = a.astype(np.complex128)
    return float(np.sum(a.real * a.real + a.imag * a.imag))


# ---- even-odd preconditioned operator (reading C20) ----------------------------------
def dhat(dims, bc, links_R, m0, psi_e):
    """Dhat psi_e = (4+m0)^2 psi_e - Dphi_eo(Dphi_oe psi_e); psi_e lives on the even sites."""
    m = 4.0 + m0
    odd = dphi_eo(dims, bc, links_R, 1, psi_e)       # output on odd sites
    return m * m * psi_e - dphi_eo(dims, bc, links_R, 0, odd)


def dhat_dagger(dims, bc, links_R, m0, psi_e):
    """Dhat^dagger = gamma5 Dhat gamma5 (reading C21)."""
    return g5(dhat(dims, bc, links_R, m0, g5(psi_e)))


# ---- conjugate gradient (reading C21) -----------------------------------------------
def cg(apply_A, b, tol, maxiter):
    """Textbook CG for a Hermitian positive definite A, x0 = 0.
    Returns (x, iterations, [|r_k|^2 / |b|^2 for k = 0..iterations])."""
    x = np.zeros_like(b)
    r = b.copy()
    p = r.copy()
    rr = norm2(r)
    bb = rr
    hist = [1.0 if bb > 0 else 0.0]
    if bb == 0.0:
        return x, 0, hist
    k = 0
    while k < maxiter and rr > tol * tol * bb:
        Ap = apply_A(p)
        alpha = rr / dot(p, Ap).real
        x = x + alpha * p
        r = r - alpha * Ap
        rr_new = norm2(r)
        beta = rr_new / rr
        p = r + beta * p
        rr = rr_new
        k += 1
        hist.append(rr / bb)
    return x, k, hist


def cg_dhat(dims, bc, links_R, m0, b_e, tol, maxiter):
    """Solve Dhat x = b_e on the even sites by CG on Dhat^dagger Dhat x = Dhat^dagger b_e."""
    A = lambda v: dhat_dagger(dims, bc, links_R, m0, dhat(dims, bc, links_R, m0, v))
    return cg(A, dhat_dagger(dims, bc, links_R, m0, b_e), tol, maxiter)


def dirac_solve(dims, bc, links_R, m0, b_eo, tol, maxiter):
    """x = D^{-1} b for full fields [even half | odd half] (reading C24).  Returns (x_eo, iterations)."""
    m = 4.0 + m0
    vh = b_eo.shape[0] // 2
    b_e, b_o = b_eo[:vh], b_eo[vh:]
    rhs = m * b_e - dphi_eo(dims, bc, links_R, 0, b_o)
    x_e, it, _ = cg_dhat(dims, bc, links_R, m0, rhs, tol, maxiter)
    x_o = (b_o - dphi_eo(dims, bc, links_R, 1, x_e)) / m
    return np.concatenate([x_e, x_o], axis=0), it


# ---- stabilised bi-conjugate gradient ("stabilized Bi-Conjugate Gradient [11, 19]"; reading C29) ----
def bicgstab(apply_A, b, tol, maxiter):
    """Textbook BiCGstab (van der Vorst) for a general non-singular A, x0 = 0, shadow residual rhat = r0 = b,
    no preconditioner, no half-step exit; the stopping rule |r_k|^2 <= tol^2 |b|^2 is tested after every full
    iteration (reading C29).  <.,.> is antilinear in its first slot (reading C22).
    Returns (x, iterations, [|r_k|^2 / |b|^2 for k = 0..iterations])."""
    x = np.zeros_like(b)
    r = b.copy()
    rhat = b.copy()
    bb = norm2(b)
    hist = [1.0 if bb > 0 else 0.0]
    if bb == 0.0:
        return x, 0, hist
    rho_old = alpha = omega = 1.0 + 0.0j
    v = np.zeros_like(b)
    p = np.zeros_like(b)
    rr = bb
    k = 0
    while k < maxiter and rr > tol * tol * bb:
        rho = dot(rhat, r)
        beta = (rho / rho_old) * (alpha / omega)
        p = r + beta * (p - omega * v)
        v = apply_A(p)
        alpha = rho / dot(rhat, v)
        s = r - alpha * v
        t = apply_A(s)
        omega = dot(t, s) / norm2(t)
        x = x + alpha * p + omega * s
        r = s - omega * t
        rho_old = rho
        rr = norm2(r)
        k += 1
        hist.append(rr / bb)
    return x, k, hist


def bicgstab_dhat(dims, bc, links_R, m0, b_e, tol, maxiter):
    """Solve Dhat x = b_e on the even sites with BiCGstab applied to Dhat itself (no normal equations)."""
    return bicgstab(lambda v: dhat(dims, bc, links_R, m0, v), b_e, tol, maxiter)


# ---- QMR for gamma5-hermitian operators ("QMR gamma_5 inverters"; reading C33) ------------------------------
def qmr_j(apply_A, apply_J, b, tol, maxiter, debug=False):
    """Quasi-minimal residual method without look-ahead for an operator that is self-adjoint in the indefinite inner
    product (x, y)_J = <x, J y>, J a Hermitian involution (gamma5 for the Wilson-Dirac operator and for Dhat, reading
    C21): A^dagger = J A J.  The paper names the method and prints nothing (reading C33); this is the method written out
    from its definition:

      Lanczos in the J-inner product (ONE operator application per step, no A^dagger): v_1 = b / rho_1, rho_1 = |b|,
          delta_k = (v_k, v_k)_J                                    (real)
          alpha_k = (v_k, A v_k)_J / delta_k                        (real)
          beta_k  = rho_k delta_k / delta_{k-1},  beta_1 = 0
          vt      = A v_k - alpha_k v_k - beta_k v_{k-1};   rho_{k+1} = |vt|;   v_{k+1} = vt / rho_{k+1}
      so that A V_k = V_{k+1} T_k with T_k tridiagonal: T[k-1,k] = beta_k, T[k,k] = alpha_k, T[k+1,k] = rho_{k+1},
      and V_k^dagger J V_k = diag(delta).
      Quasi-minimisation: x_k = V_k y_k with y_k = argmin | rho_1 e_1 - T_k y |, by Givens rotations (QR of T_k):
          theta_k = s_{k-2} beta_k;   t = c_{k-2} beta_k
          eps_k   = c_{k-1} t + s_{k-1} alpha_k;   zt = -s_{k-1} t + c_{k-1} alpha_k
          zeta_k  = sqrt(zt^2 + rho_{k+1}^2);   c_k = zt / zeta_k;   s_k = rho_{k+1} / zeta_k
          p_k = (v_k - eps_k p_{k-1} - theta_k p_{k-2}) / zeta_k
          x_k = x_{k-1} + c_k eta p_k;   eta <- -s_k eta             (eta starts at rho_1)
      |eta| is the norm of the QUASI-residual; |b - A x_k| <= sqrt(k+1) |eta| because the v_k are not orthonormal.
    Stopping (reading C33): x0 = 0; after step k, if |eta| <= tol |b| the TRUE residual b - A x_k is computed (one more
    operator application) and the iteration ends when |b - A x_k| <= tol |b|; it also ends at k = maxiter, at
    rho_{k+1} = 0 (Krylov space exhausted: x_k is exact) and at a Lanczos breakdown delta_k = 0.
    Returns (x, iterations, [|eta_k| / |b| for k = 0..iterations], |b - A x|^2 / |b|^2) -- plus the Lanczos data when debug."""
    x = np.zeros_like(b)
    bnorm = np.sqrt(norm2(b))
    hist = [1.0 if bnorm > 0 else 0.0]
    if bnorm == 0.0:
        return (x, 0, hist, 0.0) + (({},) if debug else ())
    v_prev = np.zeros_like(b)
    v = b / bnorm
    p1 = np.zeros_like(b)            # p_{k-1}
    p2 = np.zeros_like(b)            # p_{k-2}
    c1, s1, c2, s2 = 1.0, 0.0, 1.0, 0.0   # (c_{k-1}, s_{k-1}), (c_{k-2}, s_{k-2})
    eta = bnorm
    rho = bnorm
    delta_prev = 1.0
    delta = dot(v, apply_J(v)).real
    V, alphas, betas, rhos, deltas = [v], [], [], [rho], [delta]
    k = 0
    res2 = 1.0
    while k < maxiter:
        if delta == 0.0:
            break                                                   # Lanczos breakdown
        w = apply_A(v)
        alpha = dot(v, apply_J(w)).real / delta
        beta = rho * delta / delta_prev if k > 0 else 0.0
        vt = w - alpha * v - beta * v_prev
        rho_next = np.sqrt(norm2(vt))
        theta = s2 * beta
        t = c2 * beta
        eps = c1 * t + s1 * alpha
        zt = -s1 * t + c1 * alpha
        zeta = np.sqrt(zt * zt + rho_next * rho_next)
        if zeta == 0.0:
            break
        c, s = zt / zeta, rho_next / zeta
        p = (v - eps * p1 - theta * p2) / zeta
        x = x + (c * eta) * p
        eta = -s * eta
        k += 1
        hist.append(abs(eta) / bnorm)
        alphas.append(alpha); betas.append(beta); rhos.append(rho_next)
        p2, p1 = p1, p
        c2, s2, c1, s1 = c1, s1, c, s
        if rho_next == 0.0:
            res2 = norm2(b - apply_A(x)) / (bnorm * bnorm)
            break
        if abs(eta) <= tol * bnorm:
            res2 = norm2(b - apply_A(x)) / (bnorm * bnorm)
            if res2 <= tol * tol:
                break
        v_prev, v = v, vt / rho_next
        delta_prev, delta, rho = delta, dot(v, apply_J(v)).real, rho_next
        V.append(v); deltas.append(delta)
    else:
        res2 = norm2(b - apply_A(x)) / (bnorm * bnorm)
    if k == maxiter or delta == 0.0:
        res2 = norm2(b - apply_A(x)) / (bnorm * bnorm)
    if debug:
        return x, k, hist, res2, dict(V=V, alpha=alphas, beta=betas, rho=rhos, delta=deltas)
    return x, k, hist, res2


def qmr_dhat(dims, bc, links_R, m0, b_e, tol, maxiter):
    """Solve Dhat x = b_e on the even sites with the gamma5-QMR (Dhat^dagger = gamma5 Dhat gamma5, reading C21)."""
    return qmr_j(lambda v: dhat(dims, bc, links_R, m0, v), g5, b_e, tol, maxiter)
