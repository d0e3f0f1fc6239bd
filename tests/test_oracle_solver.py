"""Pins of oracle/solver.py (even-odd preconditioned operator, spinor linear
algebra, CG) against what the mathematics fixes.  CPU only.  The dense matrices come from oracle.dense
(numpy Kronecker assembly, independent of the stencil) and from numpy.linalg, never from solver.py itself."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle import dense, solver

BC_T = (-1, 1, 1, 1)


def _problem(dims, N, rep, seed):
    U = li.haar_links(seed, N, dims)
    R = oracle.represent(N, oracle.REP_NAMES[rep], U)
    return R, R.shape[-1]


def _dense_eo(dims, bc, R, m0):
    """Dense D with rows/columns permuted to [even sites | odd sites] (canonical half-field order)."""
    V = li.volume(dims)
    d = R.shape[-1]
    g = [oracle.gamma(mu) for mu in range(4)]
    D = dense.dirac_matrix(dims, bc, R, m0, g)
    site_eo = oracle.lex_to_eo(dims, np.arange(V))          # lexicographic site index of every eo position
    idx = (site_eo[:, None] * (4 * d) + np.arange(4 * d)[None, :]).reshape(-1)
    return D[np.ix_(idx, idx)]


@pytest.mark.parametrize("dims,N,rep", [((2, 2, 2, 2), 2, "fund"), ((4, 2, 2, 2), 2, "adj"), ((2, 2, 2, 4), 3, "fund"),
                                        ((2, 4, 2, 2), 3, "sym")])
def test_dhat_is_m_times_the_schur_complement(dims, N, rep):
    R, d = _problem(dims, N, rep, 11)
    m0 = -0.3
    m = 4 + m0
    D = _dense_eo(dims, BC_T, R, m0)
    n = D.shape[0] // 2
    Dee, Deo, Doe, Doo = D[:n, :n], D[:n, n:], D[n:, :n], D[n:, n:]
    assert np.allclose(Dee, m * np.eye(n)) and np.allclose(Doo, m * np.eye(n))   # the hopping term has no ee / oo block
    schur = Dee - Deo @ np.linalg.inv(Doo) @ Doe
    psi = li.gaussian_spinor(5, li.volume(dims) // 2, d)
    want = (m * schur @ psi.reshape(-1)).reshape(psi.shape)
    got = solver.dhat(dims, BC_T, R, m0, psi)
    assert np.linalg.norm(got - want) <= 1e-13 * np.linalg.norm(want)
    # dagger: dense conjugate transpose
    want_d = (m * schur.conj().T @ psi.reshape(-1)).reshape(psi.shape)
    got_d = solver.dhat_dagger(dims, BC_T, R, m0, psi)
    assert np.linalg.norm(got_d - want_d) <= 1e-13 * np.linalg.norm(want_d)


def test_gamma5_dhat_is_hermitian():
    dims = (4, 4, 2, 6)
    R, d = _problem(dims, 2, "adj", 3)
    vh = li.volume(dims) // 2
    a, b = li.gaussian_spinor(1, vh, d), li.gaussian_spinor(2, vh, d)
    Q = lambda v: solver.g5(solver.dhat(dims, BC_T, R, -0.8, v))
    lhs, rhs = solver.dot(a, Q(b)), np.conj(solver.dot(b, Q(a)))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_linear_algebra_definitions():
    vh, d = 64, 3
    a, b = li.gaussian_spinor(1, vh, d), li.gaussian_spinor(2, vh, d)
    g5m = np.kron(np.eye(vh), np.kron(np.diag([1, 1, -1, -1]), np.eye(d)))   # gamma5 as a dense matrix
    assert np.allclose(solver.g5(a).reshape(-1), g5m @ a.reshape(-1))
    c = 0.3 - 1.7j
    assert np.allclose(solver.g5_mulc_add_assign(b, c, a).reshape(-1), b.reshape(-1) + c * (g5m @ a.reshape(-1)))
    assert np.allclose(solver.mulc_add_assign(b, c, a), b + c * a)
    # <a,b> antilinear in the first slot, = numpy's vdot; norm2 = |a|^2; Cauchy-Schwarz; sesquilinearity
    assert np.isclose(solver.dot(a, b), np.vdot(a.reshape(-1), b.reshape(-1)))
    assert np.isclose(solver.dot(c * a, b), np.conj(c) * solver.dot(a, b))
    assert np.isclose(solver.dot(a, c * b), c * solver.dot(a, b))
    assert np.isclose(solver.norm2(a), np.linalg.norm(a.reshape(-1)) ** 2)
    assert abs(solver.dot(a, b)) ** 2 <= solver.norm2(a) * solver.norm2(b)
    # exactly representable case: 256 entries of (3 + 4i) -> norm2 = 25 * 256
    e = np.full((16, 4, 4), 3 + 4j)
    assert solver.norm2(e) == 25.0 * 256 and solver.dot(e, e) == 25.0 * 256


@pytest.mark.parametrize("k", [1, 3, 7])
def test_cg_terminates_in_k_steps_for_k_distinct_eigenvalues(k):
    """Finite termination: CG on a Hermitian positive definite matrix with k distinct eigenvalues reaches the
    exact solution in k iterations (textbook property; a wrong alpha or beta formula breaks it)."""
    rng = np.random.default_rng(7)
    n = 48
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n)))
    ev = np.array([1.0 + 2.5 * (i % k) for i in range(n)])
    A = (Q * ev) @ Q.conj().T
    b = (rng.normal(size=n) + 1j * rng.normal(size=n)).reshape(n // 12, 4, 3)
    apply_A = lambda v: (A @ v.reshape(-1)).reshape(v.shape)
    x, it, hist = solver.cg(apply_A, b, 1e-12, 100)
    assert it == k
    assert np.allclose(x.reshape(-1), np.linalg.solve(A, b.reshape(-1)), rtol=0, atol=1e-10)
    assert len(hist) == it + 1 and hist[0] == 1.0 and hist[-1] <= 1e-24
    # not converged before step k
    assert all(h > 1e-20 for h in hist[:k])


def test_cg_error_decreases_monotonically_in_the_A_norm():
    rng = np.random.default_rng(3)
    n = 60
    M = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    A = M.conj().T @ M + 0.5 * np.eye(n)
    b = (rng.normal(size=n) + 1j * rng.normal(size=n)).reshape(n // 12, 4, 3)
    xs = np.linalg.solve(A, b.reshape(-1))
    apply_A = lambda v: (A @ v.reshape(-1)).reshape(v.shape)
    errs = []
    for it in range(1, 12):
        x, k, _ = solver.cg(apply_A, b, 0.0, it)
        e = x.reshape(-1) - xs
        errs.append(np.real(np.vdot(e, A @ e)))
    assert all(errs[i + 1] < errs[i] for i in range(len(errs) - 1))


@pytest.mark.parametrize("dims,N,rep", [((2, 2, 2, 2), 2, "fund"), ((2, 2, 4, 2), 2, "adj"), ((2, 2, 2, 2), 3, "sym")])
def test_dirac_solve_equals_dense_solve(dims, N, rep):
    R, d = _problem(dims, N, rep, 21)
    m0 = -0.2
    V = li.volume(dims)
    b = li.gaussian_spinor(9, V, d)
    x, it = solver.dirac_solve(dims, BC_T, R, m0, b, 1e-13, 2000)
    D = _dense_eo(dims, BC_T, R, m0)
    want = np.linalg.solve(D, b.reshape(-1)).reshape(b.shape)
    assert 0 < it < 2000
    assert np.linalg.norm(x - want) <= 1e-10 * np.linalg.norm(want)
    # and it really solves the stencil operator
    assert np.linalg.norm(oracle.dirac(dims, BC_T, R, m0, x) - b) <= 1e-10 * np.linalg.norm(b)


# ------------------------------------------------------------------------------------------------- BiCGstab
def _rand_system(n, seed, shift):
    rng = np.random.default_rng(seed)
    A = (rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))) / np.sqrt(n) + shift * np.eye(n)   # non-Hermitian
    b = (rng.normal(size=n) + 1j * rng.normal(size=n)).reshape(n // 12, 4, 3)
    return A, b


def test_bicgstab_solves_a_non_hermitian_system_like_numpy():
    A, b = _rand_system(96, 1, 3.0)
    apply_A = lambda v: (A @ v.reshape(-1)).reshape(v.shape)
    x, it, hist = solver.bicgstab(apply_A, b, 1e-12, 200)
    assert 2 < it < 100 and hist[0] == 1.0 and len(hist) == it + 1 and hist[-1] <= 1e-24
    assert np.allclose(x.reshape(-1), np.linalg.solve(A, b.reshape(-1)), rtol=0, atol=1e-9)
    # the recursively updated residual is the true one
    assert abs(solver.norm2(b - apply_A(x)) / solver.norm2(b) - hist[-1]) <= 1e-20


@pytest.mark.parametrize("k", [2, 3, 5])
def test_bicgstab_terminates_within_k_steps_for_k_distinct_eigenvalues(k):
    """r_j = Q_j(A) P_j(A) r_0 with P_j the BiCG residual polynomial: for a diagonalisable A with k distinct
    eigenvalues P_k is the minimal polynomial, so BiCGstab is exact after at most k iterations (and, generically, not
    before: the history must still be far from zero at k-1)."""
    n = 24
    evs = [2.0 + 1.0j, 0.5 - 0.25j, -1.0 + 0.5j, 1.5 + 2.0j, 3.0 - 1.0j][:k]
    ev = np.array([evs[i % k] for i in range(n)])
    b = (np.arange(n) + 1.0 + 0.5j * np.arange(n)[::-1]).reshape(2, 4, 3)
    apply_A = lambda v: (ev * v.reshape(-1)).reshape(v.shape)
    x, it, hist = solver.bicgstab(apply_A, b, 1e-12, 20)
    assert it == k and hist[-1] <= 1e-24 and hist[k - 1] > 1e-12
    assert np.allclose(x.reshape(-1), b.reshape(-1) / ev, rtol=0, atol=1e-10)


def test_bicgstab_iterates_lie_in_the_krylov_spaces():
    """x_k is in K_{2k}(A, b) = span{b, A b, ..., A^{2k-1} b}: a wrong update formula leaves the space."""
    A, b = _rand_system(48, 5, 2.5)
    apply_A = lambda v: (A @ v.reshape(-1)).reshape(v.shape)
    for k in (1, 2, 3):
        x, it, _ = solver.bicgstab(apply_A, b, 0.0, k)
        assert it == k
        K = np.empty((48, 2 * k), dtype=complex)
        w = b.reshape(-1).copy()
        for j in range(2 * k):
            K[:, j] = w / np.linalg.norm(w)
            w = A @ K[:, j]
        coef, res, *_ = np.linalg.lstsq(K, x.reshape(-1), rcond=None)
        assert np.linalg.norm(K @ coef - x.reshape(-1)) <= 1e-9 * np.linalg.norm(x)


@pytest.mark.parametrize("dims,N,rep", [((2, 2, 2, 2), 2, "fund"), ((2, 2, 4, 2), 2, "adj")])
def test_bicgstab_dhat_equals_dense_schur_solve(dims, N, rep):
    R, d = _problem(dims, N, rep, 31)
    m0 = -0.2
    m = 4 + m0
    D = _dense_eo(dims, BC_T, R, m0)
    n = D.shape[0] // 2
    schur = m * (D[:n, :n] - D[:n, n:] @ np.linalg.inv(D[n:, n:]) @ D[n:, :n])
    b = li.gaussian_spinor(32, li.volume(dims) // 2, d)
    x, it, hist = solver.bicgstab_dhat(dims, BC_T, R, m0, b, 1e-13, 500)
    assert 0 < it < 500
    want = np.linalg.solve(schur, b.reshape(-1)).reshape(b.shape)
    assert np.linalg.norm(x - want) <= 1e-10 * np.linalg.norm(want)
