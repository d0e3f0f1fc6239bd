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


# ---- QMR for J-hermitian operators ("QMR gamma_5"; reading C33) -----------------------------------------
def _j_system(n, seed, shift):
    """A = J H with H Hermitian (so A^dagger = J A J), J = diag(+1 x n/2, -1 x n/2); b complex."""
    rng = np.random.default_rng(seed)
    J = np.diag([1.0] * (n // 2) + [-1.0] * (n - n // 2)).astype(complex)
    H = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    H = H + H.conj().T + shift * np.eye(n)
    b = (rng.normal(size=n) + 1j * rng.normal(size=n)).reshape(n // 4, 4, 1)
    return J @ H, J, b


def _ops(A, J):
    n = A.shape[0]
    return (lambda v: (A @ v.reshape(n)).reshape(v.shape)), (lambda v: (J @ v.reshape(n)).reshape(v.shape))


def test_qmr_solves_a_j_hermitian_indefinite_system_like_numpy():
    A, J, b = _j_system(40, 5, 9.0)
    assert np.allclose(A.conj().T, J @ A @ J) and not np.allclose(A, A.conj().T)
    apply_A, apply_J = _ops(A, J)
    x, it, hist, res2 = solver.qmr_j(apply_A, apply_J, b, 1e-11, 200)
    want = np.linalg.solve(A, b.reshape(-1))
    assert 0 < it < 200 and res2 <= 1e-22
    assert np.linalg.norm(x.reshape(-1) - want) <= 1e-9 * np.linalg.norm(want)
    # the reported residual is the true one
    assert np.isclose(res2, np.linalg.norm(b.reshape(-1) - A @ x.reshape(-1)) ** 2 / np.linalg.norm(b) ** 2, rtol=1e-6)


def test_qmr_lanczos_vectors_are_j_orthogonal_and_satisfy_the_three_term_relation():
    """A V_k = V_{k+1} T_k with the tridiagonal T of (beta, alpha, rho) and V^dagger J V = diag(delta): the two defining
    properties of the J-Lanczos process, checked on the vectors the solver actually built."""
    n = 24
    A, J, b = _j_system(n, 6, 7.0)
    apply_A, apply_J = _ops(A, J)
    x, it, hist, res2, dbg = solver.qmr_j(apply_A, apply_J, b, 1e-30, 10, debug=True)
    assert it == 10
    V = np.stack([v.reshape(n) for v in dbg["V"]], axis=1)          # n x (k+1)
    k = 10
    assert V.shape[1] == k + 1 or V.shape[1] == k                  # the last v_{k+1} is built only if the loop continues
    G = V.conj().T @ J @ V
    assert np.abs(G - np.diag(np.diag(G))).max() <= 1e-10
    assert np.allclose(np.diag(G).real, dbg["delta"][:V.shape[1]], atol=1e-12) and np.abs(np.diag(G).imag).max() <= 1e-12
    assert np.allclose(np.linalg.norm(V, axis=0), 1.0)
    kk = V.shape[1] - 1
    T = np.zeros((kk + 1, kk))
    for j in range(kk):
        T[j, j] = dbg["alpha"][j]
        T[j + 1, j] = dbg["rho"][j + 1]
        if j > 0:
            T[j - 1, j] = dbg["beta"][j]
    assert np.abs(A @ V[:, :kk] - V @ T).max() <= 1e-10


def test_qmr_with_j_identity_is_minres_and_eta_is_the_true_residual_norm():
    """J = 1, A Hermitian (indefinite): the Lanczos vectors are orthonormal, so the quasi-residual IS the residual:
    |eta_k| = |b - A x_k| at every k, and it never increases (minimal residual over the Krylov space)."""
    n = 32
    rng = np.random.default_rng(7)
    H = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    H = H + H.conj().T                                                        # indefinite
    b = (rng.normal(size=n) + 1j * rng.normal(size=n)).reshape(n // 4, 4, 1)
    apply_A = lambda v: (H @ v.reshape(n)).reshape(v.shape)
    ident = lambda v: v
    bn = np.linalg.norm(b)
    prev = 1.0
    for k in (1, 2, 5, 9, 17):
        x, it, hist, res2 = solver.qmr_j(apply_A, ident, b, 1e-30, k)
        assert it == k
        true = np.linalg.norm(b.reshape(-1) - H @ x.reshape(-1)) / bn
        assert np.isclose(hist[-1], true, rtol=1e-8)
        # minimal residual: no other vector of the Krylov space does better
        K = np.stack([np.linalg.matrix_power(H, j) @ b.reshape(-1) for j in range(k)], axis=1)
        Q, _ = np.linalg.qr(K)
        y = np.linalg.lstsq(H @ Q, b.reshape(-1), rcond=None)[0]
        assert np.isclose(true, np.linalg.norm(b.reshape(-1) - H @ Q @ y) / bn, rtol=1e-6)
        assert true <= prev * (1 + 1e-12)
        prev = true


def test_qmr_iterates_lie_in_the_krylov_space_and_bound_the_true_residual():
    n = 28
    A, J, b = _j_system(n, 8, 8.0)
    apply_A, apply_J = _ops(A, J)
    bn = np.linalg.norm(b)
    for k in (1, 3, 6):
        x, it, hist, res2 = solver.qmr_j(apply_A, apply_J, b, 1e-30, k)
        K = np.stack([np.linalg.matrix_power(A, j) @ b.reshape(-1) for j in range(k)], axis=1)
        Q, _ = np.linalg.qr(K)
        xv = x.reshape(-1)
        assert np.linalg.norm(xv - Q @ (Q.conj().T @ xv)) <= 1e-9 * np.linalg.norm(xv)
        assert np.sqrt(res2) <= np.sqrt(k + 1) * hist[-1] * (1 + 1e-9)       # |r_k| <= sqrt(k+1) |eta_k|


def test_qmr_terminates_when_the_krylov_space_is_exhausted():
    """k distinct eigenvalues of a J-hermitian diagonalisable A: rho_{k+1} = 0 and x_k is exact."""
    n = 16
    J = np.diag([1.0] * 8 + [-1.0] * 8)
    d = np.array([2.0, -1.5, 0.75] * 6)[:n]                    # A = J diag(J d) = diag(d): J-hermitian, 3 eigenvalues
    b = (np.arange(n) + 1.0 - 0.5j * np.arange(n)[::-1]).reshape(4, 4, 1)
    apply_A = lambda v: (d * v.reshape(-1)).reshape(v.shape)
    apply_J = lambda v: (np.diag(J) * v.reshape(-1)).reshape(v.shape)
    x, it, hist, res2 = solver.qmr_j(apply_A, apply_J, b, 1e-13, 50)
    assert it <= 4 and res2 <= 1e-24
    assert np.allclose(x.reshape(-1), b.reshape(-1) / d, atol=1e-10)


def test_qmr_zero_rhs_and_maxiter_zero():
    A, J, b = _j_system(8, 9, 5.0)
    apply_A, apply_J = _ops(A, J)
    x, it, hist, res2 = solver.qmr_j(apply_A, apply_J, 0 * b, 1e-10, 10)
    assert it == 0 and res2 == 0.0 and not x.any()
    x, it, hist, res2 = solver.qmr_j(apply_A, apply_J, b, 1e-10, 0)
    assert it == 0 and np.isclose(res2, 1.0) and not x.any()


@pytest.mark.parametrize("dims,N,rep", [((2, 2, 2, 2), 2, "fund"), ((2, 2, 4, 2), 2, "adj")])
def test_qmr_dhat_equals_dense_schur_solve(dims, N, rep):
    R, d = _problem(dims, N, rep, 41)
    m0 = -0.2
    m = 4 + m0
    D = _dense_eo(dims, BC_T, R, m0)
    n = D.shape[0] // 2
    schur = m * (D[:n, :n] - D[:n, n:] @ np.linalg.inv(D[n:, n:]) @ D[n:, :n])
    b = li.gaussian_spinor(42, li.volume(dims) // 2, d)
    x, it, hist, res2 = solver.qmr_dhat(dims, BC_T, R, m0, b, 1e-12, 500)
    assert 0 < it < 500 and res2 <= 1e-24
    want = np.linalg.solve(schur, b.reshape(-1)).reshape(b.shape)
    assert np.linalg.norm(x - want) <= 1e-9 * np.linalg.norm(want)
