"""Pins of the oracle's link map U -> U^R (BASELINE.json:north_star, configs[2], configs[3];
SURVEY.md section 8(c) readings C6-C8 and "Pins").  CPU only."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle

REPS = [oracle.REP_FUND, oracle.REP_ADJ, oracle.REP_SYM, oracle.REP_ASYM]


def dag(a):
    return np.conj(np.swapaxes(a, -1, -2))


@pytest.mark.parametrize("N", [2, 3, 4])
@pytest.mark.parametrize("rep", REPS)
def test_dimension_identity_unitarity_homomorphism(N, rep):
    d = oracle.rep_dim(N, rep)
    assert d == {oracle.REP_FUND: N, oracle.REP_ADJ: N * N - 1,
                 oracle.REP_SYM: N * (N + 1) // 2, oracle.REP_ASYM: N * (N - 1) // 2}[rep]
    U = li.haar_matrices(41, N, 64)
    Vv = li.haar_matrices(42, N, 64)
    RU, RV, RUV = oracle.represent(N, rep, U), oracle.represent(N, rep, Vv), oracle.represent(N, rep, U @ Vv)
    assert RU.shape == (64, d, d)
    eye = np.eye(d)
    assert np.abs(oracle.represent(N, rep, np.eye(N)[None]) - eye).max() < 1e-15
    assert np.abs(RU @ dag(RU) - eye).max() < 5e-15          # unitarity
    assert np.abs(RUV - RU @ RV).max() < 5e-15                # homomorphism
    if rep == oracle.REP_ADJ:                                 # real orthogonal, det +1 (reading C7)
        assert np.abs(RU.imag).max() < 1e-15
        assert np.abs(np.linalg.det(RU.real) - 1).max() < 1e-13


@pytest.mark.parametrize("N", [2, 3, 4])
def test_characters(N):
    """Compared as complex numbers: catches R <-> R* and wrong sqrt2 / sign factors."""
    U = li.haar_matrices(43, N, 200)
    tr = np.trace(U, axis1=-2, axis2=-1)
    tr2 = np.trace(U @ U, axis1=-2, axis2=-1)
    chi = lambda rep: np.trace(oracle.represent(N, rep, U), axis1=-2, axis2=-1)
    assert np.abs(chi(oracle.REP_FUND) - tr).max() < 1e-14
    assert np.abs(chi(oracle.REP_ADJ) - (np.abs(tr) ** 2 - 1)).max() < 1e-13
    assert np.abs(chi(oracle.REP_SYM) - (tr ** 2 + tr2) / 2).max() < 1e-13
    assert np.abs(chi(oracle.REP_ASYM) - (tr ** 2 - tr2) / 2).max() < 1e-13


@pytest.mark.parametrize("N", [2, 3, 4])
def test_diagonal_links_give_diagonal_two_index_reps(N):
    rng = np.random.default_rng(5)
    th = rng.uniform(0, 2 * np.pi, size=N)
    th[-1] = -th[:-1].sum()
    U = np.diag(np.exp(1j * th))[None]
    pairs_sym = [(i, j) for i in range(N) for j in range(i, N)]
    pairs_asym = [(i, j) for i in range(N) for j in range(i + 1, N)]
    for rep, pairs in ((oracle.REP_SYM, pairs_sym), (oracle.REP_ASYM, pairs_asym)):
        R = oracle.represent(N, rep, U)[0]
        want = np.diag([np.exp(1j * (th[i] + th[j])) for i, j in pairs])
        assert np.abs(R - want).max() < 1e-15


def test_su2_adjoint_closed_form():
    """U = a0 + i a.sigma  =>  R_ab = (a0^2 - a.a) delta_ab + 2 a_a a_b + 2 a0 eps_abc a_c (textbook SO(3))."""
    U = li.haar_matrices(44, 2, 100)
    a0 = U[:, 0, 0].real
    a = np.stack([U[:, 0, 1].imag, U[:, 0, 1].real, U[:, 0, 0].imag], axis=-1)
    eps = np.zeros((3, 3, 3))
    eps[0, 1, 2] = eps[1, 2, 0] = eps[2, 0, 1] = 1
    eps[0, 2, 1] = eps[2, 1, 0] = eps[1, 0, 2] = -1
    want = ((a0 ** 2 - (a * a).sum(-1))[:, None, None] * np.eye(3)
            + 2 * a[:, :, None] * a[:, None, :]
            + 2 * a0[:, None, None] * np.einsum("abc,nc->nab", eps, a))
    got = oracle.represent(2, oracle.REP_ADJ, U)
    assert np.abs(got - want).max() < 1e-15


def test_su3_antisymmetric_is_antifundamental():
    """In the pair order (01),(02),(12): R_asym(U) = P U* P^T, P = antidiag(1,-1,1)."""
    U = li.haar_matrices(45, 3, 100)
    P = np.array([[0, 0, 1], [0, -1, 0], [1, 0, 0]], dtype=float)
    got = oracle.represent(3, oracle.REP_ASYM, U)
    assert np.abs(got - P @ np.conj(U) @ P.T).max() < 1e-15


def test_su2_symmetric_equivalent_to_adjoint():
    U = li.haar_matrices(46, 2, 50)
    s = oracle.represent(2, oracle.REP_SYM, U)
    a = oracle.represent(2, oracle.REP_ADJ, U)
    for k in range(50):
        assert np.abs(np.poly(s[k]) - np.poly(a[k])).max() < 1e-13


def test_two_index_closed_form_su3():
    """R_{(ij),(kl)} = n_ij n_kl (U_ik U_jl +- U_il U_jk), n = 1/sqrt2 on diagonal pairs (reading C8)."""
    N = 3
    U = li.haar_matrices(47, N, 20)
    for rep, sign in ((oracle.REP_SYM, +1), (oracle.REP_ASYM, -1)):
        pairs = [(i, j) for i in range(N) for j in range(i, N) if not (i == j and sign < 0)]
        R = oracle.represent(N, rep, U)
        for a, (i, j) in enumerate(pairs):
            for b, (k, l) in enumerate(pairs):
                n = (2 ** -0.5 if i == j else 1.0) * (2 ** -0.5 if k == l else 1.0)
                want = n * (U[:, i, k] * U[:, j, l] + sign * U[:, i, l] * U[:, j, k])
                assert np.abs(R[:, a, b] - want).max() < 1e-15


def test_last_row_of_a_special_unitary_matrix_is_fixed_by_the_others():
    """Reading C30 (row-compressed links): for U in SU(3) the third row is conj(row0 x row1), for U in SU(2) the second
    row is (-conj u01, conj u00); and the SU(2) adjoint link is a function of the first row alone,
    R_ab = (a0^2 - a.a) delta_ab + 2 a_a a_b + 2 a0 eps_abc a_c with (a0, a3, a2, a1) = (Re u00, Im u00, Re u01, Im u01).
    Checked on the seeded generator's links against the oracle's trace definition."""
    U3 = li.haar_links(71, 3, (2, 2, 2, 2)).reshape(-1, 3, 3)
    assert np.abs(np.conj(np.cross(U3[:, 0], U3[:, 1])) - U3[:, 2]).max() < 1e-14
    U2 = li.haar_links(72, 2, (2, 2, 2, 2)).reshape(-1, 2, 2)
    assert np.abs(U2[:, 1, 0] + np.conj(U2[:, 0, 1])).max() < 1e-14 and np.abs(U2[:, 1, 1] - np.conj(U2[:, 0, 0])).max() < 1e-14
    R = oracle.represent(2, oracle.REP_ADJ, U2).real
    a0, a3, a2, a1 = U2[:, 0, 0].real, U2[:, 0, 0].imag, U2[:, 0, 1].real, U2[:, 0, 1].imag
    a = np.stack([a1, a2, a3], axis=-1)
    eps = np.zeros((3, 3, 3))
    eps[0, 1, 2] = eps[1, 2, 0] = eps[2, 0, 1] = 1
    eps[0, 2, 1] = eps[2, 1, 0] = eps[1, 0, 2] = -1
    want = (a0 ** 2 - np.sum(a * a, -1))[:, None, None] * np.eye(3) + 2 * a[:, :, None] * a[:, None, :] \
        + 2 * a0[:, None, None] * np.einsum("abc,xc->xab", eps, a)
    assert np.abs(R - want).max() < 1e-14
