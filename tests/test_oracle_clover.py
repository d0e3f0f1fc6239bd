"""Pins of oracle/clover.py (reading C28) against what the physics fixes.  CPU only.
Closed forms and invariants, none of them the oracle's formula retyped: the constant abelian field (fixes the
orientation of the leaves, the sign and the 1/8), pure-gauge fields, gauge covariance, antisymmetry in (mu, nu),
Hermiticity / gamma5-commutation / tracelessness / chiral block structure of T, gamma5-hermiticity of the dense
D_sw assembled with oracle.dense, and c_sw = 0."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle import clover, dense

BC_T = (-1, 1, 1, 1)


def _coords(dims):
    return np.stack(np.meshgrid(*[np.arange(n) for n in dims], indexing="ij"), axis=-1).reshape(-1, 4)


def _gauge_transform(dims, U, g):
    """U_mu(x) -> g(x) U_mu(x) g(x+mu)^dagger; U [V,4,N,N], g [V,N,N] lexicographic."""
    dims = tuple(dims)
    N = U.shape[-1]
    gl = g.reshape(dims + (N, N))
    out = np.empty_like(U)
    for mu in range(4):
        gs = np.roll(gl, -1, axis=mu).reshape(-1, N, N)
        out[:, mu] = g @ U[:, mu] @ np.conj(np.swapaxes(gs, -1, -2))
    return out


def test_unit_and_pure_gauge_fields_have_no_field_strength():
    dims = (4, 2, 4, 6)
    V = li.volume(dims)
    one = np.broadcast_to(np.eye(3, dtype=complex), (V, 4, 3, 3)).copy()
    g = li.haar_links(5, 3, dims)[:, 0]                     # a random SU(3) element per site
    pure = _gauge_transform(dims, one, g)
    for U in (one, pure):
        for mu in range(4):
            for nu in range(mu + 1, 4):
                assert np.abs(clover.field_strength(dims, U, mu, nu)).max() < 1e-13
    assert np.abs(clover.clover_term(dims, pure, 1.7)).max() < 1e-12


@pytest.mark.parametrize("mu,nu", [(0, 1), (1, 2), (0, 3), (2, 3)])
def test_constant_abelian_field_closed_form(mu, nu):
    """A_nu(x) = B q x_mu, all other A = 0, with B L_mu a multiple of 2 pi: every leaf is exp(i B q), so
    F_{mu nu} = diag(sin(B q_a)) = d_mu A_nu + O(B^3) exactly at every site, and F_{nu mu} = -F_{mu nu}."""
    dims = (8, 4, 6, 4)
    V = li.volume(dims)
    x = _coords(dims)
    q = np.array([1.0, -2.0, 3.0])
    B = 2 * np.pi / dims[mu]
    U = np.broadcast_to(np.eye(3, dtype=complex), (V, 4, 3, 3)).copy()
    U[:, nu] = np.exp(1j * B * x[:, mu, None] * q[None, :])[:, :, None] * np.eye(3)
    F = clover.field_strength(dims, U, mu, nu)
    want = np.broadcast_to(np.diag(np.sin(B * q)), (V, 3, 3))
    assert np.abs(F - want).max() < 1e-13
    assert np.abs(clover.field_strength(dims, U, nu, mu) + want).max() < 1e-13
    for a in range(4):
        for b in range(a + 1, 4):
            if (a, b) != (min(mu, nu), max(mu, nu)):
                assert np.abs(clover.field_strength(dims, U, a, b)).max() < 1e-13
    # T = -(c_sw/2) sigma_{mu nu} (x) F_{mu nu} for this field
    T = clover.clover_term(dims, U, 1.3)
    s = clover.sigma(mu, nu) if mu < nu else clover.sigma(nu, mu)
    sign = 1.0 if mu < nu else -1.0
    wantT = -0.65 * sign * np.einsum("st,ab->satb", s, np.diag(np.sin(B * q)))
    assert np.abs(T - wantT[None]).max() < 1e-13


@pytest.mark.parametrize("N,rep", [(3, "fund"), (2, "adj"), (3, "sym")])
def test_field_strength_hermitian_antisymmetric_and_gauge_covariant(N, rep):
    dims = (4, 4, 2, 4)
    rid = oracle.REP_NAMES[rep]
    U = li.haar_links(7, N, dims)
    g = li.haar_links(8, N, dims)[:, 1]
    R, Rg = oracle.represent(N, rid, U), oracle.represent(N, rid, g)
    Rt = oracle.represent(N, rid, _gauge_transform(dims, U, g))
    for mu in range(4):
        for nu in range(mu + 1, 4):
            F = clover.field_strength(dims, R, mu, nu)
            assert np.abs(F - np.conj(np.swapaxes(F, -1, -2))).max() < 1e-13
            assert np.abs(F + clover.field_strength(dims, R, nu, mu)).max() < 1e-13
            Ft = clover.field_strength(dims, Rt, mu, nu)
            assert np.abs(Ft - Rg @ F @ np.conj(np.swapaxes(Rg, -1, -2))).max() < 1e-12
    assert np.abs(F).max() > 0.1      # a Haar field is far from pure gauge


def test_clover_term_structure():
    dims = (4, 2, 4, 4)
    U = li.haar_links(9, 3, dims)
    V, d = li.volume(dims), 3
    T = clover.clover_term(dims, U, 1.0).reshape(V, 4 * d, 4 * d)
    assert np.abs(T - np.conj(np.swapaxes(T, -1, -2))).max() < 1e-13                   # Hermitian
    g5 = np.kron(np.diag([1, 1, -1, -1]), np.eye(d))
    assert np.abs(T @ g5 - g5 @ T).max() < 1e-13                                       # commutes with gamma5
    assert np.abs(T[:, :2 * d, 2 * d:]).max() == 0 and np.abs(T[:, 2 * d:, :2 * d]).max() == 0   # chiral blocks
    Tsc = T.reshape(V, 4, d, 4, d)
    assert np.abs(np.einsum("xsasb->xab", Tsc)).max() < 1e-13                          # tr_spin sigma = 0
    assert np.abs(clover.clover_term(dims, U, 0.0)).max() == 0
    assert np.allclose(clover.clover_term(dims, U, 2.0), 2 * clover.clover_term(dims, U, 1.0))
    for mu in range(4):                                                                # sigma: Hermitian, (i/2)[g,g]
        for nu in range(mu + 1, 4):
            s = clover.sigma(mu, nu)
            assert np.allclose(s, s.conj().T) and np.allclose(s @ s, np.eye(4))
            assert np.allclose(s, 1j * oracle.gamma(mu) @ oracle.gamma(nu))


def test_dirac_clover_is_gamma5_hermitian_and_reduces_to_dirac():
    dims = (2, 2, 4, 2)
    U = li.haar_links(10, 2, dims)
    R = oracle.represent(2, oracle.REP_ADJ, U)
    V, d = li.volume(dims), 3
    m0, csw = -0.4, 1.2
    g = [oracle.gamma(mu) for mu in range(4)]
    D = dense.dirac_matrix(dims, BC_T, R, m0, g)                                        # lexicographic (site, spin, colour)
    T = clover.clover_term(dims, R, csw).reshape(V, 4 * d, 4 * d)
    Dsw = D.copy()
    for x in range(V):
        Dsw[x * 4 * d:(x + 1) * 4 * d, x * 4 * d:(x + 1) * 4 * d] += T[x]
    G5 = np.kron(np.eye(V), np.kron(np.diag([1, 1, -1, -1]), np.eye(d)))
    assert np.abs(G5 @ Dsw @ G5 - Dsw.conj().T).max() < 1e-12
    psi = li.gaussian_spinor(11, V, d)
    want = oracle.lex_to_eo(dims, (Dsw @ oracle.eo_to_lex(dims, psi).reshape(-1)).reshape(V, 4, d))
    got = clover.dirac_clover(dims, BC_T, R, m0, csw, psi)
    assert np.linalg.norm(got - want) <= 1e-13 * np.linalg.norm(want)
    assert np.array_equal(clover.dirac_clover(dims, BC_T, R, m0, 0.0, psi), oracle.dirac(dims, BC_T, R, m0, psi))


# ------------------------------------------------------------------------------------------ exponentiated clover
def test_exp_clover_equals_its_power_series_and_is_positive():
    dims = (4, 2, 2, 4)
    U = li.haar_links(12, 3, dims)
    V, d = li.volume(dims), 3
    m0, csw = -0.5, 1.5
    m = 4 + m0
    T = clover.clover_term(dims, U, csw).reshape(V, 4 * d, 4 * d)
    E = clover.exp_clover_term(dims, U, m0, csw).reshape(V, 4 * d, 4 * d)
    series = np.zeros_like(T)
    term = np.broadcast_to(np.eye(4 * d, dtype=complex), T.shape).copy()
    for k in range(1, 40):                          # m (exp(T/m) - 1) = sum_{k>=1} T^k / (k! m^(k-1))
        term = term @ T / (k * m)
        series = series + m * term
    assert np.abs(E - series).max() < 1e-12
    assert np.abs(E - np.conj(np.swapaxes(E, -1, -2))).max() < 1e-13
    g5 = np.kron(np.diag([1, 1, -1, -1]), np.eye(d))
    assert np.abs(E @ g5 - g5 @ E).max() < 1e-13
    assert np.abs(E[:, :2 * d, 2 * d:]).max() < 1e-13
    # the whole point of the exponential: the diagonal term m + E = m exp(T/m) is positive definite, while m + T need not be
    assert np.linalg.eigvalsh(m * np.eye(4 * d) + E).min() > 0
    # small c_sw: E = T + T^2 / (2m) + O(c_sw^3)
    eps = 1e-3
    Ts = clover.clover_term(dims, U, eps).reshape(V, 4 * d, 4 * d)
    Es = clover.exp_clover_term(dims, U, m0, eps).reshape(V, 4 * d, 4 * d)
    fro = np.linalg.norm(Ts, axis=(1, 2)).max()                      # the remainder is T^3/(6 m^2) + ...: third order
    assert np.abs(Es - Ts - Ts @ Ts / (2 * m)).max() <= 1.05 * fro ** 3 / (6 * m * m)
    assert np.abs(Es - Ts).max() > 10 * fro ** 3                       # ... and the second-order term is really there


def test_exp_clover_closed_form_on_the_constant_abelian_field():
    """T = -(c/2) sigma_01 sin(B q): sigma^2 = 1, so exp(t sigma) = cosh t + sigma sinh t."""
    dims = (8, 4, 2, 2)
    V = li.volume(dims)
    x = _coords(dims)
    q = np.array([1.0, -2.0, 3.0])
    B = 2 * np.pi / dims[0]
    U = np.broadcast_to(np.eye(3, dtype=complex), (V, 4, 3, 3)).copy()
    U[:, 1] = np.exp(1j * B * x[:, 0, None] * q[None, :])[:, :, None] * np.eye(3)
    m0, csw = 0.2, 1.1
    m = 4 + m0
    E = clover.exp_clover_term(dims, U, m0, csw)
    t = -0.5 * csw * np.sin(B * q) / m
    s = clover.sigma(0, 1)
    want = m * (np.einsum("st,ab->satb", np.eye(4), np.diag(np.cosh(t) - 1)) + np.einsum("st,ab->satb", s, np.diag(np.sinh(t))))
    assert np.abs(E - want[None]).max() < 1e-13


def test_dirac_expclover_reduces_to_dirac_without_field_strength():
    dims = (2, 2, 2, 4)
    V = li.volume(dims)
    one = np.broadcast_to(np.eye(2, dtype=complex), (V, 4, 2, 2)).copy()
    psi = li.gaussian_spinor(13, V, 2)
    assert np.allclose(clover.dirac_expclover(dims, BC_T, one, -0.1, 1.3, psi), oracle.dirac(dims, BC_T, one, -0.1, psi), atol=1e-14)


# ------------------------------------------------------------------------------ even-odd preconditioning with clover
def _dense_dsw_eo(dims, bc, R, m0, csw, exponentiated):
    """Dense D_sw (oracle.dense + per-site blocks), rows/columns in [even sites | odd sites] order."""
    V, d = li.volume(dims), R.shape[-1]
    g = [oracle.gamma(mu) for mu in range(4)]
    D = dense.dirac_matrix(dims, bc, R, m0, g, hopping_only=True)
    A = clover.site_term(dims, R, m0, csw, exponentiated)
    for x in range(V):
        D[x * 4 * d:(x + 1) * 4 * d, x * 4 * d:(x + 1) * 4 * d] += A[x]
    site_eo = oracle.lex_to_eo(dims, np.arange(V))
    idx = (site_eo[:, None] * (4 * d) + np.arange(4 * d)[None, :]).reshape(-1)
    return D[np.ix_(idx, idx)]


@pytest.mark.parametrize("exponentiated", [False, True])
@pytest.mark.parametrize("dims,N,rep", [((2, 2, 2, 2), 2, "fund"), ((2, 2, 4, 2), 2, "adj"), ((2, 2, 2, 2), 3, "fund")])
def test_dhat_clover_is_the_dense_schur_complement_and_the_solve_is_the_dense_solve(dims, N, rep, exponentiated):
    U = li.haar_links(21, N, dims)
    R = oracle.represent(N, oracle.REP_NAMES[rep], U)
    d, V = R.shape[-1], li.volume(dims)
    m0, csw = -0.3, 1.2
    D = _dense_dsw_eo(dims, BC_T, R, m0, csw, exponentiated)
    n = D.shape[0] // 2
    schur = D[:n, :n] - D[:n, n:] @ np.linalg.inv(D[n:, n:]) @ D[n:, :n]
    psi = li.gaussian_spinor(22, V // 2, d)
    want = (schur @ psi.reshape(-1)).reshape(psi.shape)
    got = clover.dhat_clover(dims, BC_T, R, m0, csw, psi, exponentiated)
    assert np.linalg.norm(got - want) <= 1e-12 * np.linalg.norm(want)
    b = li.gaussian_spinor(23, V, d)
    x, it = clover.dirac_clover_solve(dims, BC_T, R, m0, csw, b, 1e-13, 500, exponentiated)
    xs = np.linalg.solve(D, b.reshape(-1)).reshape(b.shape)
    assert 0 < it < 500 and np.linalg.norm(x - xs) <= 1e-9 * np.linalg.norm(xs)
    # c_sw = 0: A = 4 + m0 and Dhat_sw = Dhat / (4 + m0) of reading C20
    from oracle import solver
    z = clover.dhat_clover(dims, BC_T, R, m0, 0.0, psi, exponentiated)
    assert np.allclose(z * (4 + m0), solver.dhat(dims, BC_T, R, m0, psi), atol=1e-12)
