"""Pins of the oracle's hopping term against what the physics fixes (BASELINE.json:north_star;
SURVEY.md section 8(c) "Pins").  CPU only.  None of these compares the oracle with itself retyped:
they are closed forms, invariants and a brute-force dense assembly through numpy matmul."""
import itertools
import os

import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle import dense

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "gamma_chiral.txt")
BC_T = (-1, 1, 1, 1)


def gammas():
    return [oracle.gamma(mu) for mu in range(4)]


# ---------------------------------------------------------------------------------- gamma tables
def test_gamma_tables_match_printed_reading():
    want = {mu: np.zeros((4, 4), complex) for mu in (0, 1, 2, 3, 5)}
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        mu, r, c, re, im = line.split()
        want[int(mu)][int(r), int(c)] = float(re) + 1j * float(im)
    for mu in (0, 1, 2, 3, 5):
        assert np.array_equal(oracle.gamma(mu), want[mu]), mu


def test_clifford_algebra_hermiticity_gamma5():
    g = gammas()
    g5 = oracle.gamma(5)
    for mu in range(4):
        assert np.allclose(g[mu], g[mu].conj().T)
        assert np.allclose(g5 @ g[mu] + g[mu] @ g5, 0)
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2 * np.eye(4) * (mu == nu))
        for s in (+1, -1):
            assert np.linalg.matrix_rank(np.eye(4) + s * g[mu]) == 2
    assert np.allclose(g5, g[0] @ g[1] @ g[2] @ g[3])
    assert np.allclose(g5, np.diag([1, 1, -1, -1]))


# ---------------------------------------------------------------------------------- free field
def _coords(dims):
    return np.stack(np.meshgrid(*[np.arange(n) for n in dims], indexing="ij"), axis=-1).reshape(-1, 4)


@pytest.mark.parametrize("bc", [BC_T, (1, 1, 1, 1), (1, -1, 1, -1), (-1, -1, -1, -1)])
@pytest.mark.parametrize("d", [2, 3])
def test_free_field_plane_waves_every_momentum(bc, d):
    """U = 1, psi = u e^{ipx}:  D psi = [(4+m0) - sum cos p + i sum gamma_mu sin p_mu] psi, vector-wise."""
    dims = (4, 2, 6, 8)            # four different even extents: catches any direction swap
    m0 = -0.37
    V = li.volume(dims)
    links = li.unit_links(d, dims)
    xs = _coords(dims)
    g = gammas()
    rng = np.random.default_rng(7)
    par = li.parity_mask(dims)
    worst = 0.0
    for n in itertools.product(*[range(L) for L in dims]):
        p = np.array([2 * np.pi * (n[mu] + (0.5 if bc[mu] == -1 else 0.0)) / dims[mu] for mu in range(4)])
        u = rng.normal(size=(4, d)) + 1j * rng.normal(size=(4, d))
        phase = np.exp(1j * (xs @ p))
        psi = phase[:, None, None] * u[None]
        Dp = (4 + m0 - np.cos(p).sum()) * np.eye(4) + 1j * sum(np.sin(p[mu]) * g[mu] for mu in range(4))
        want = phase[:, None, None] * (Dp @ u)[None]
        got = oracle.dirac(dims, bc, links, m0, oracle.lex_to_eo(dims, psi))
        got = oracle.eo_to_lex(dims, got)
        worst = max(worst, np.linalg.norm(got - want) / np.linalg.norm(psi))
        if sum(n) % 7 == 0:  # the even-odd form on a subset of momenta (same closed form without 4+m0)
            Dh = Dp - (4 + m0) * np.eye(4)
            for parity in (0, 1):
                out = oracle.dphi_eo(dims, bc, links, parity, psi[par == 1 - parity])
                w = (phase[:, None, None] * (Dh @ u)[None])[par == parity]
                worst = max(worst, np.linalg.norm(out - w) / np.linalg.norm(psi))  # Dh u can vanish exactly
    assert worst < 5e-13, worst


# ---------------------------------------------------------------------------------- dense assembly
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 2, 2), (2, 2, 2, 4), (2, 4, 2, 2)])
@pytest.mark.parametrize("N,rep", [(2, oracle.REP_FUND), (3, oracle.REP_FUND), (2, oracle.REP_ADJ), (3, oracle.REP_SYM)])
def test_stencil_equals_dense_assembly(dims, N, rep):
    """Includes the extent-2 double hop (reading C10) and both seam hops."""
    m0 = -0.5
    V = li.volume(dims)
    U = li.haar_links(11, N, dims)
    R = oracle.represent(N, rep, U)
    d = R.shape[-1]
    psi = li.gaussian_spinor(12, V, d)
    D = dense.dirac_matrix(dims, BC_T, R, m0, gammas())
    Dh = dense.dirac_matrix(dims, BC_T, R, m0, gammas(), hopping_only=True)
    want = (D @ psi.reshape(-1)).reshape(psi.shape)
    got = oracle.eo_to_lex(dims, oracle.dirac(dims, BC_T, R, m0, oracle.lex_to_eo(dims, psi)))
    assert np.linalg.norm(got - want) / np.linalg.norm(want) < 1e-14
    got_h = oracle.dphi_lex(dims, BC_T, R, psi)
    want_h = (Dh @ psi.reshape(-1)).reshape(psi.shape)
    assert np.linalg.norm(got_h - want_h) / np.linalg.norm(want_h) < 1e-14

    # even-odd structure: zero EE/OO blocks, and Dphi_eo(p) = restriction of Dphi on a masked input
    par = li.parity_mask(dims)
    idx = np.arange(V * 4 * d).reshape(V, 4 * d)
    for p in (0, 1):
        rows = idx[par == p].reshape(-1)
        assert np.all(Dh[np.ix_(rows, rows)] == 0)
        cols = idx[par == 1 - p].reshape(-1)
        want_eo = (Dh[np.ix_(rows, cols)] @ psi[par == 1 - p].reshape(-1)).reshape(-1, 4, d)
        got_eo = oracle.dphi_eo(dims, BC_T, R, p, psi[par == 1 - p])
        assert np.linalg.norm(got_eo - want_eo) / np.linalg.norm(want_eo) < 1e-14
        # sampled-sites entry point gives the same rows
        hi = np.array([0, 1, V // 2 - 1, V // 4, 3])
        some = oracle.dphi_eo_sites(dims, BC_T, R, p, psi[par == 1 - p], hi)
        assert np.array_equal(some, got_eo[hi])


def test_gamma5_hermiticity_dense_and_stencil():
    dims = (4, 2, 4, 2)
    N, rep = 3, oracle.REP_FUND
    V = li.volume(dims)
    R = oracle.represent(N, rep, li.haar_links(21, N, dims))
    d = 3
    g5 = oracle.gamma(5)
    D = dense.dirac_matrix(dims, BC_T, R, -0.2, gammas())
    G5 = np.kron(np.eye(V), np.kron(g5, np.eye(d)))
    assert np.abs(G5 @ D @ G5 - D.conj().T).max() < 1e-15
    # stencil form on a bigger lattice: <phi, g5 D g5 psi> = <D phi, psi>
    dims = (6, 4, 4, 8)
    V = li.volume(dims)
    R = li.haar_links(22, N, dims)
    phi = li.gaussian_spinor(23, V, d)
    psi = li.gaussian_spinor(24, V, d)
    g5v = np.array([1, 1, -1, -1])[None, :, None]
    Dg5psi = oracle.dirac(dims, BC_T, R, -0.2, g5v * psi)
    lhs = np.vdot(phi, g5v * Dg5psi)
    rhs = np.vdot(oracle.dirac(dims, BC_T, R, -0.2, phi), psi)
    assert abs(lhs - rhs) / abs(rhs) < 1e-13
    # eo form: <phi_e, Dphi_eo psi_o> = <g5 Dphi_oe g5 phi_e, psi_o>
    vh = V // 2
    phi_e, psi_o = phi[:vh], psi[:vh]
    lhs = np.vdot(phi_e, oracle.dphi_eo(dims, BC_T, R, 0, psi_o))
    rhs = np.vdot(g5v * oracle.dphi_eo(dims, BC_T, R, 1, g5v * phi_e), psi_o)
    assert abs(lhs - rhs) / abs(rhs) < 1e-13


# ---------------------------------------------------------------------------------- gauge covariance
def _shift_plus(dims, field, mu):
    """field(x) -> field(x+mu) on a lexicographic [V,...] array (periodic)."""
    f = field.reshape(tuple(dims) + field.shape[1:])
    return np.roll(f, -1, axis=mu).reshape(field.shape)


@pytest.mark.parametrize("N,rep", [(2, oracle.REP_FUND), (3, oracle.REP_FUND), (2, oracle.REP_ADJ),
                                   (3, oracle.REP_SYM), (3, oracle.REP_ASYM), (3, oracle.REP_ADJ),
                                   (2, oracle.REP_SYM), (4, oracle.REP_ASYM)])
def test_gauge_covariance(N, rep):
    """D[R(U^g)] (R(g) psi) = R(g) D[R(U)] psi  with U^g_mu(x) = g(x) U_mu(x) g(x+mu)^dagger."""
    dims = (4, 2, 4, 6)
    V = li.volume(dims)
    U = li.haar_links(31, N, dims)
    g = li.haar_matrices(32, N, V)
    Ug = np.empty_like(U)
    for mu in range(4):
        gp = _shift_plus(dims, g, mu)
        Ug[:, mu] = g @ U[:, mu] @ np.conj(np.swapaxes(gp, -1, -2))
    R, Rg_links, Rg = oracle.represent(N, rep, U), oracle.represent(N, rep, Ug), oracle.represent(N, rep, g)
    d = R.shape[-1]
    psi = li.gaussian_spinor(33, V, d)
    psig = np.einsum("xab,xsb->xsa", Rg, psi)
    lhs = oracle.dphi_lex(dims, BC_T, Rg_links, psig)
    rhs = np.einsum("xab,xsb->xsa", Rg, oracle.dphi_lex(dims, BC_T, R, psi))
    assert np.linalg.norm(lhs - rhs) / np.linalg.norm(rhs) < 1e-13


def test_bad_arguments_rejected():
    R = li.unit_links(2, (2, 2, 2, 2))
    psi = li.gaussian_spinor(1, 16, 2)
    with pytest.raises(ValueError):
        oracle.dphi_lex((3, 2, 2, 2), BC_T, R, psi)          # odd extent (reading C11)
    with pytest.raises(ValueError):
        oracle.dphi_lex((2, 2, 2, 2), (0, 1, 1, 1), R, psi)  # bc not +-1
    with pytest.raises(ValueError):
        oracle.dphi_eo((2, 2, 2, 2), BC_T, R, 2, psi[:8])    # parity not 0/1
