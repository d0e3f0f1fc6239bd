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
