"""GPU parity of the rows SURVEY.md section 8(f) NEXT-1 adds, through the C ABI, against oracle/solver.py on
the same seeded inputs: spinor linear algebra, the even-odd preconditioned operator
(PAPER.md:70), the CG and the full solve.  Tolerances: BASELINE.json:north_star's relative L2
(1e-13 fp64 / 2e-6 fp32 vs the fp64 oracle) for every operator application; solver tolerances are stated
at each test and derived in DESIGN.md section 12."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle import solver
from gpu_common import BC_T, TOL, GpuProblem, oracle_rep_id, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available()
    from paper_2405_19294_b200 import build
    build.build()
    import paper_2405_19294_b200 as hr
    return hr


class Fields:
    """Half-field helpers on top of GpuProblem (marshalling only)."""

    def __init__(self, hr, prob):
        self.hr, self.prob, self.lat, self.P = hr, prob, prob.lat, prob.prec

    def put(self, canon, parity=0):
        t = self.lat.spinor(self.P)
        self.lat.import_spinor(t, self.P, canon, parity)
        return t

    def get(self, t, parity=0):
        return self.lat.export_spinor(t, self.P, parity)

    def new(self):
        t = self.lat.spinor(self.P)
        t.fill_(0xFF)
        return t


# dims chosen so that V/2 * (16-byte vectors per site) is NOT a multiple of the 1024-vector CTA tile (ragged
# tail) and spans several CTAs
LA_CASES = [((4, 2, 6, 2), 2, "fund"), ((4, 6, 6, 10), 3, "fund"), ((6, 4, 2, 10), 2, "adj"), ((4, 4, 6, 2), 3, "sym"),
            ((2, 2, 2, 2), 3, "adj"), ((4, 2, 2, 6), 4, "sym"), ((2, 4, 2, 6), 4, "adj")]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,N,rep", LA_CASES)
def test_linear_algebra_matches_oracle(hr, dims, N, rep, prec):
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    vh = li.volume(dims) // 2
    a, b = li.gaussian_spinor(101, vh, d), li.gaussian_spinor(102, vh, d)
    prob = GpuProblem(hr, dims, N, rep, prec, li.haar_links(1, N, dims))
    f = Fields(hr, prob)
    ctx, P, st = prob.lat.ctx, f.P, prob.lat.stream()
    tol = TOL[prec]
    ga, gb = f.put(a), f.put(b)
    out = f.new()
    hr.hr_spinor_copy(ctx, P, out, ga, st)
    assert np.array_equal(f.get(out), f.get(ga))
    hr.hr_spinor_g5(ctx, P, out, ga, st)
    assert rel_l2(f.get(out), solver.g5(a)) <= tol
    assert np.array_equal(f.get(out), solver.g5(f.get(ga)))          # a pure sign pattern: exact on the stored values
    c = 0.3 - 1.7j
    hr.hr_spinor_copy(ctx, P, out, gb, st)
    hr.hr_spinor_mulc_add_assign(ctx, P, out, c, ga, st)
    assert rel_l2(f.get(out), solver.mulc_add_assign(b, c, a)) <= tol
    hr.hr_spinor_copy(ctx, P, out, gb, st)
    hr.hr_spinor_g5_mulc_add_assign(ctx, P, out, c, ga, st)
    assert rel_l2(f.get(out), solver.g5_mulc_add_assign(b, c, a)) <= tol
    ca, cb = -0.9 + 0.2j, 1.1 + 0.4j
    hr.hr_spinor_lincomb(ctx, P, out, ca, 1, ga, cb, gb, st)
    assert rel_l2(f.get(out), ca * solver.g5(a) + cb * b) <= tol
    hr.hr_spinor_lincomb(ctx, P, ga, ca, 0, ga, cb, gb, st)          # out aliases x
    assert rel_l2(f.get(ga), ca * a + cb * b) <= tol
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,N,rep", LA_CASES + [((16, 16, 16, 16), 3, "fund")])
def test_reductions_match_oracle_and_are_deterministic(hr, dims, N, rep, prec):
    import torch
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    vh = li.volume(dims) // 2
    a, b = li.gaussian_spinor(103, vh, d), li.gaussian_spinor(104, vh, d)
    prob = GpuProblem(hr, dims, N, rep, prec, li.haar_links(1, N, dims))
    f = Fields(hr, prob)
    ctx, P, st = prob.lat.ctx, f.P, prob.lat.stream()
    ga, gb = f.put(a), f.put(b)
    # sums in fp64 on both sides; fp32 fields carry the input rounding 2^-24 per element (reading C13)
    rtol = 1e-13 if prec == "f64" else 2e-6
    scale = np.sqrt(solver.norm2(a) * solver.norm2(b))
    got = hr.hr_spinor_dot(ctx, P, ga, gb, st)
    assert abs(got - solver.dot(a, b)) <= rtol * scale
    n2 = hr.hr_spinor_norm2(ctx, P, ga, st)
    assert abs(n2 - solver.norm2(a)) <= rtol * solver.norm2(a)
    same = hr.hr_spinor_dot(ctx, P, ga, ga, st)
    assert same.imag == 0.0 and same.real == n2
    # exact check on the values the GPU actually holds (no input-rounding slack): fp64 sums of the stored field
    ha = f.get(ga)
    assert abs(n2 - solver.norm2(ha)) <= 1e-13 * n2 if prec == "f64" else abs(n2 - solver.norm2(ha)) <= 1e-6 * n2
    # bitwise run-to-run determinism (reading C15) and the device-result path
    for _ in range(3):
        assert hr.hr_spinor_dot(ctx, P, ga, gb, st) == got
    res = torch.zeros(2, dtype=torch.float64, device="cuda")
    hr.hr_spinor_dot(ctx, P, ga, gb, st, result=res)
    torch.cuda.synchronize()
    assert complex(res[0].item(), res[1].item()) == got
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("g5", [0, 1])
@pytest.mark.parametrize("dims,N,rep", [((4, 4, 6, 8), 3, "fund"), ((6, 4, 4, 4), 2, "adj"), ((4, 4, 4, 6), 3, "sym"),
                                        ((2, 2, 2, 2), 2, "fund"), ((4, 2, 6, 4), 3, "asym"), ((4, 2, 4, 6), 4, "sym"), ((2, 4, 6, 2), 4, "adj")])
def test_dhat_matches_oracle(hr, dims, N, rep, g5, prec):
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(111, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    psi = li.gaussian_spinor(112, li.volume(dims) // 2, d)
    m0 = -0.45
    want = solver.dhat(dims, BC_T, R, m0, psi)
    if g5:
        want = solver.g5(want)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    f = Fields(hr, prob)
    gin, out, tmp = f.put(psi), f.new(), f.new()
    n0 = hr.hr_launch_count()
    prob.lat.dhat(m0, bool(g5), out, gin, tmp, prob.links)
    assert hr.hr_launch_count() == n0 + 2          # two Dphi launches, diagonal term and gamma5 fused
    assert rel_l2(f.get(out), want) <= TOL[prec]
    # every kernel variant computes the same operator
    for variant in (0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11):
        try:
            prob.lat.set_tuning("variant", variant)
            out2 = f.new()
            prob.lat.dhat(m0, bool(g5), out2, gin, tmp, prob.links)
        except hr.HrError:
            continue
        assert rel_l2(f.get(out2), want) <= TOL[prec], variant
    with pytest.raises(hr.HrError):
        prob.lat.dhat(m0, bool(g5), out, gin, gin, prob.links)     # tmp aliases in
    prob.close()


# ---------------------------------------------------------------------------------------------- CG
CG_CASES = [((4, 4, 4, 8), 3, "fund", -0.3), ((4, 4, 6, 4), 2, "adj", -0.5), ((4, 4, 4, 4), 3, "sym", -0.2),
            ((4, 2, 4, 6), 4, "sym", -0.25)]          # d_R = 10: the colour-parallel kernel with the fused reduction


@pytest.mark.parametrize("dims,N,rep,m0", CG_CASES)
def test_cg_dhat_fp64_follows_the_oracle_iteration_by_iteration(hr, dims, N, rep, m0):
    """Same algorithm, same start, same stopping rule (reading C21): the residual history of the GPU CG tracks
    the oracle's (rounding differences grow slowly with k), the iteration counts agree to +-1 and the
    solutions agree to the solver tolerance times a modest condition-number factor."""
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(121, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    b = li.gaussian_spinor(122, li.volume(dims) // 2, d)
    tol, maxiter = 1e-10, 500
    x_want, it_want, hist_want = solver.cg_dhat(dims, BC_T, R, m0, b, tol, maxiter)
    assert 5 < it_want < maxiter
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    f = Fields(hr, prob)
    gb, gx = f.put(b), f.new()
    ws = prob.lat.cg_workspace(f.P, maxiter)
    it, res2, hist = prob.lat.cg_dhat(m0, gx, gb, prob.links, tol, maxiter, ws, want_hist=True)
    assert abs(it - it_want) <= 1
    assert hist[0] == 1.0 and len(hist) == it + 1 and res2 == hist[-1] <= tol * tol
    n = min(it, it_want) + 1
    assert np.allclose(hist[:n], hist_want[:n], rtol=1e-6, atol=0)
    x = f.get(gx)
    assert rel_l2(x, x_want) <= 1e-8
    # and it solves the oracle's operator: |Dhat x - b| / |b|
    assert rel_l2(solver.dhat(dims, BC_T, R, m0, x), b) <= 1e-8
    # bitwise reproducible (device-resident scalars, ordered reductions)
    gx2 = f.new()
    it2, res2b, _ = prob.lat.cg_dhat(m0, gx2, gb, prob.links, tol, maxiter, ws)
    assert it2 == it and res2b == res2 and np.array_equal(f.get(gx2), x)
    prob.close()


def test_cg_dhat_fp32_reaches_single_precision(hr):
    dims, N, rep, m0 = (4, 4, 4, 8), 3, "fund", -0.3
    U = li.haar_links(121, N, dims)
    b = li.gaussian_spinor(122, li.volume(dims) // 2, 3)
    x_want, it_want, _ = solver.cg_dhat(dims, BC_T, U, m0, b, 1e-5, 500)
    prob = GpuProblem(hr, dims, N, rep, "f32", U)
    f = Fields(hr, prob)
    gb, gx = f.put(b), f.new()
    ws = prob.lat.cg_workspace(f.P, 500)
    it, res2, _ = prob.lat.cg_dhat(m0, gx, gb, prob.links, 1e-5, 500, ws)
    assert abs(it - it_want) <= 2 and res2 <= 1e-10
    assert rel_l2(f.get(gx), x_want) <= 1e-4
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_cg_dhat_dist_single_rank_follows_the_oracle_and_its_edge_cases(hr, prec):
    """hr_cg_dhat_dist (the CG with the operator and the all-reduce as callbacks; every recurrence in libhr) on ONE rank,
    where the distributed Dphi_eo is the plain hr_dphi_eo: iteration by iteration the oracle's CG (reading C21)."""
    import torch
    dims, N, m0 = (4, 4, 4, 8), 3, -0.3
    U = li.haar_links(131, N, dims)
    vh = li.volume(dims) // 2
    b = li.gaussian_spinor(132, vh, 3)
    prob = GpuProblem(hr, dims, N, "fund", prec, U)
    f = Fields(hr, prob)
    gb, gx = f.put(b), f.new()
    ws = torch.empty(hr.hr_cg_dist_workspace_bytes(prob.lat.ctx, f.P), dtype=torch.uint8, device="cuda")
    calls = []

    def dphi(out, inp, parity):
        calls.append(parity)
        hr.hr_dphi_eo(out, inp, prob.links, parity, prob.lat.stream())

    tol, maxit = (1e-10, 400) if prec == "f64" else (1e-5, 400)
    x_o, it_o, hist_o = solver.cg_dhat(dims, BC_T, U, m0, b, tol, maxit)
    it, hist = hr.hr_cg_dhat_dist(prob.lat.ctx, f.P, m0, gx, gb, tol, maxit, ws, dphi, None, prob.lat.stream())
    assert abs(it - it_o) <= (1 if prec == "f64" else 2)
    n = min(it, it_o, 8)
    assert np.allclose(hist[:n + 1], hist_o[:n + 1], rtol=1e-6 if prec == "f64" else 1e-2)
    assert rel_l2(f.get(gx), x_o) <= (1e-8 if prec == "f64" else 1e-3)
    assert len(calls) == 2 + 4 * it and calls[:4] == [1, 0, 1, 0]        # rhs: one gamma5 Dhat (two Dphi_eo); per iteration two
    # an all-reduce that doubles every sum is what two identical ranks would see: |rhs|^2, <p, Ap>, |r|^2 all scale, the
    # iterates do not
    it2, hist2 = hr.hr_cg_dhat_dist(prob.lat.ctx, f.P, m0, gx, gb, tol, maxit, ws, dphi, lambda v: [2.0 * t for t in v], prob.lat.stream())
    assert it2 == it and np.allclose(hist2, hist, rtol=1e-12)
    # edge cases: maxiter = 0, b = 0, tol >= 1
    it0, h0 = hr.hr_cg_dhat_dist(prob.lat.ctx, f.P, m0, gx, gb, tol, 0, ws, dphi, None, prob.lat.stream())
    assert it0 == 0 and h0 == [1.0] and not f.get(gx).any()
    gz = f.put(np.zeros_like(b))
    it0, h0 = hr.hr_cg_dhat_dist(prob.lat.ctx, f.P, m0, gx, gz, tol, 50, ws, dphi, None, prob.lat.stream())
    assert it0 == 0 and h0 == [0.0] and not f.get(gx).any()
    it0, _ = hr.hr_cg_dhat_dist(prob.lat.ctx, f.P, m0, gx, gb, 1.0, 50, ws, dphi, None, prob.lat.stream())
    assert it0 == 0
    # a failing callback surfaces as the Python exception, not as a crash across the C frames
    def broken(out, inp, parity):
        raise RuntimeError("exchange failed")
    with pytest.raises(RuntimeError):
        hr.hr_cg_dhat_dist(prob.lat.ctx, f.P, m0, gx, gb, tol, 5, ws, broken, None, prob.lat.stream())
    with pytest.raises(hr.HrError):
        hr.hr_cg_dhat_dist(prob.lat.ctx, f.P, m0, gb, gb, tol, 5, ws, dphi, None, prob.lat.stream())      # x aliases b
    prob.close()


def test_cg_edge_cases(hr):
    dims, N, m0 = (4, 4, 4, 4), 2, -0.4
    U = li.haar_links(5, N, dims)
    vh = li.volume(dims) // 2
    b = li.gaussian_spinor(6, vh, 2)
    prob = GpuProblem(hr, dims, N, "fund", "f64", U)
    f = Fields(hr, prob)
    ws = prob.lat.cg_workspace(f.P, 50)
    gb, gx = f.put(b), f.new()
    # maxiter = 0: x = 0, no iteration
    it, res2, hist = prob.lat.cg_dhat(m0, gx, gb, prob.links, 1e-10, 0, ws, want_hist=True)
    assert it == 0 and res2 == 1.0 and not f.get(gx).any()
    # b = 0: x = 0 at once (oracle: 0 iterations)
    gz = f.put(np.zeros_like(b))
    it, res2, _ = prob.lat.cg_dhat(m0, gx, gz, prob.links, 1e-10, 50, ws)
    assert it == 0 and res2 == 0.0 and not f.get(gx).any()
    assert solver.cg_dhat(dims, BC_T, U, m0, np.zeros_like(b), 1e-10, 50)[1] == 0
    # tol >= 1: satisfied by x0 = 0
    it, _, _ = prob.lat.cg_dhat(m0, gx, gb, prob.links, 1.0, 50, ws)
    assert it == 0 == solver.cg_dhat(dims, BC_T, U, m0, b, 1.0, 50)[1]
    # maxiter hit before convergence: stops exactly there, same history as the oracle
    it, res2, hist = prob.lat.cg_dhat(m0, gx, gb, prob.links, 1e-14, 7, ws, want_hist=True)
    x_o, it_o, hist_o = solver.cg_dhat(dims, BC_T, U, m0, b, 1e-14, 7)
    assert it == it_o == 7 and np.allclose(hist, hist_o, rtol=1e-9) and rel_l2(f.get(gx), x_o) <= 1e-11
    # argument errors
    with pytest.raises(hr.HrError):
        prob.lat.cg_dhat(m0, gb, gb, prob.links, 1e-10, 50, ws)          # x aliases b
    with pytest.raises(hr.HrError):
        prob.lat.cg_dhat(m0, gx, gb, prob.links, 1e-10, -1, ws)          # negative maxiter
    with pytest.raises(hr.HrError):
        prob.lat.cg_dhat(m0, gx, gb, prob.links, -1.0, 50, ws)
    prob.close()


@pytest.mark.parametrize("dims,N,rep,m0", CG_CASES)
def test_dirac_solve_matches_oracle_and_inverts_hr_dirac(hr, dims, N, rep, m0):
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(131, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    b = li.gaussian_spinor(132, V, d)
    x_want, it_want = solver.dirac_solve(dims, BC_T, R, m0, b, 1e-11, 1000)
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    lat, P = prob.lat, prob.prec
    half = hr.hr_spinor_bytes(lat.ctx, P)
    gb, gx, gy = lat.spinor(P, full=True), lat.spinor(P, full=True), lat.spinor(P, full=True)
    for p in (0, 1):
        lat.import_spinor(gb[p * half:(p + 1) * half], P, b[p * (V // 2):(p + 1) * (V // 2)], p)
    ws = lat.cg_workspace(P, 1000)
    it, res2 = lat.dirac_solve(m0, gx, gb, prob.links, 1e-11, 1000, ws)
    assert abs(it - it_want) <= 1 and res2 <= 1e-22
    x = np.concatenate([lat.export_spinor(gx[p * half:(p + 1) * half], P, p) for p in (0, 1)])
    assert rel_l2(x, x_want) <= 1e-9
    assert rel_l2(oracle.dirac(dims, BC_T, R, m0, x), b) <= 1e-9       # the oracle's D applied to the GPU's x
    lat.dirac(m0, gy, gx, prob.links)                                   # and the GPU's own D
    y = np.concatenate([lat.export_spinor(gy[p * half:(p + 1) * half], P, p) for p in (0, 1)])
    assert rel_l2(y, b) <= 1e-9
    prob.close()


def test_cg_at_config2_volume_converges_and_satisfies_the_equation(hr):
    """SU(3) fundamental 32^3 x 64 (BASELINE.json:configs[1]), near-identity links so that the system is well
    conditioned: the oracle cannot iterate at this size in seconds, so the check is the property
    |Dhat x - b| <= tol-ish, with Dhat applied by the ORACLE on a sample of sites after the solve."""
    dims, N, m0 = (64, 32, 32, 32), 3, 0.1
    U = li.near_identity_links(141, N, dims, 0.3)
    vh = li.volume(dims) // 2
    b = li.gaussian_spinor(142, vh, 3)
    prob = GpuProblem(hr, dims, N, "fund", "f64", U)
    f = Fields(hr, prob)
    gb, gx = f.put(b), f.new()
    ws = prob.lat.cg_workspace(f.P, 400)
    it, res2, hist = prob.lat.cg_dhat(m0, gx, gb, prob.links, 1e-9, 400, ws, want_hist=True)
    assert 3 < it < 400 and res2 <= 1e-18
    assert all(h > 0 for h in hist)
    x = f.get(gx)
    hidx = np.unique(np.random.Generator(np.random.Philox(7)).integers(0, vh, size=1 << 16))
    odd = oracle.dphi_eo(dims, BC_T, U, 1, x)                              # oracle, full odd field
    dd = oracle.dphi_eo_sites(dims, BC_T, U, 0, odd, hidx)
    dhat_x = (4 + m0) ** 2 * x[hidx] - dd
    assert rel_l2(dhat_x, b[hidx]) <= 1e-7
    prob.close()


def test_cg_graph_replay_is_bitwise_the_plain_launch_sequence(hr):
    """tuning key "cg_graph": one CG iteration captured as a CUDA graph and replayed (default) vs the same six kernels
    launched one by one -- same kernels, same order, same device-resident scalars: identical bits, identical history."""
    dims, N, m0 = (4, 4, 4, 8), 3, -0.3
    U = li.haar_links(121, N, dims)
    b = li.gaussian_spinor(122, li.volume(dims) // 2, 3)
    prob = GpuProblem(hr, dims, N, "fund", "f64", U)
    f = Fields(hr, prob)
    gb = f.put(b)
    ws = prob.lat.cg_workspace(f.P, 200)
    res = {}
    for mode in (2, 1, 0):
        prob.lat.set_tuning("cg_graph", mode)
        gx = f.new()
        n0 = hr.hr_launch_count()
        it, res2, hist = prob.lat.cg_dhat(m0, gx, gb, prob.links, 1e-10, 200, ws, want_hist=True)
        res[mode] = (it, res2, hist.copy(), f.get(gx), hr.hr_launch_count() - n0)
    assert res[0][0] == res[1][0] and res[0][1] == res[1][1]
    assert np.array_equal(res[0][2], res[1][2]) and np.array_equal(res[0][3], res[1][3])
    assert res[0][4] == res[1][4]                     # the launch counter counts replayed kernels too
    assert res[2][0] == res[0][0] and np.array_equal(res[2][3], res[0][3])
    with pytest.raises(hr.HrError):
        prob.lat.set_tuning("cg_graph", 3)
    prob.close()


# ---------------------------------------------------------------------------------------------- BiCGstab
@pytest.mark.parametrize("dims,N,rep,m0", CG_CASES)
def test_bicgstab_dhat_fp64_follows_the_oracle(hr, dims, N, rep, m0):
    """PAPER.md:124 "stabilized Bi-Conjugate Gradient"; reading C29.  Same algorithm and stopping rule on both sides:
    the residual histories agree while they are well above rounding (BiCGstab amplifies rounding differences faster
    than CG, so the history is compared for the first iterations and down to 1e-12 only), iteration counts to +-2,
    solutions to the solver tolerance x condition number."""
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(121, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    b = li.gaussian_spinor(122, li.volume(dims) // 2, d)
    tol, maxiter = 1e-10, 300
    x_want, it_want, hist_want = solver.bicgstab_dhat(dims, BC_T, R, m0, b, tol, maxiter)
    assert 3 < it_want < maxiter
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    f = Fields(hr, prob)
    gb, gx = f.put(b), f.new()
    import torch
    ws = torch.empty(hr.hr_bicgstab_workspace_bytes(prob.lat.ctx, f.P, maxiter), dtype=torch.uint8, device="cuda")
    it, res2, hist = hr.hr_bicgstab_dhat(prob.lat.ctx, m0, gx, gb, prob.links, tol, maxiter, ws, prob.lat.stream(), want_hist=True)
    assert abs(it - it_want) <= 2 and hist[0] == 1.0 and len(hist) == it + 1 and res2 == hist[-1] <= tol * tol
    n = min(it, it_want, 8) + 1
    assert np.allclose(hist[:n], hist_want[:n], rtol=1e-5, atol=1e-14)
    x = f.get(gx)
    assert rel_l2(x, x_want) <= 1e-8
    assert rel_l2(solver.dhat(dims, BC_T, R, m0, x), b) <= 1e-8         # it solves the oracle's operator
    # fewer operator applications than the CG on the normal equations for the same accuracy
    _, it_cg, _ = solver.cg_dhat(dims, BC_T, R, m0, b, tol, 500)
    assert it <= it_cg
    # bitwise reproducible
    gx2 = f.new()
    it2, res2b, _ = hr.hr_bicgstab_dhat(prob.lat.ctx, m0, gx2, gb, prob.links, tol, maxiter, ws, prob.lat.stream())
    assert it2 == it and res2b == res2 and np.array_equal(f.get(gx2), x)
    prob.close()


def test_bicgstab_fp32_and_edge_cases(hr):
    import torch
    dims, N, m0 = (4, 4, 4, 8), 3, -0.3
    U = li.haar_links(121, N, dims)
    b = li.gaussian_spinor(122, li.volume(dims) // 2, 3)
    x_want, it_want, _ = solver.bicgstab_dhat(dims, BC_T, U, m0, b, 1e-5, 300)
    prob = GpuProblem(hr, dims, N, "fund", "f32", U)
    f = Fields(hr, prob)
    ctx, st = prob.lat.ctx, prob.lat.stream()
    ws = torch.empty(hr.hr_bicgstab_workspace_bytes(ctx, f.P, 300), dtype=torch.uint8, device="cuda")
    gb, gx = f.put(b), f.new()
    it, res2, _ = hr.hr_bicgstab_dhat(ctx, m0, gx, gb, prob.links, 1e-5, 300, ws, st)
    assert abs(it - it_want) <= 2 and res2 <= 1e-10 and rel_l2(f.get(gx), x_want) <= 1e-4
    it, res2, hist = hr.hr_bicgstab_dhat(ctx, m0, gx, gb, prob.links, 1e-5, 0, ws, st, want_hist=True)     # maxiter = 0
    assert it == 0 and res2 == 1.0 and not f.get(gx).any()
    it, res2, _ = hr.hr_bicgstab_dhat(ctx, m0, gx, f.put(np.zeros_like(b)), prob.links, 1e-5, 50, ws, st)  # b = 0
    assert it == 0 and res2 == 0.0 and not f.get(gx).any()
    it, res2, hist = hr.hr_bicgstab_dhat(ctx, m0, gx, gb, prob.links, 1e-12, 3, ws, st, want_hist=True)    # maxiter hit
    assert it == 3 and len(hist) == 4
    with pytest.raises(hr.HrError):
        hr.hr_bicgstab_dhat(ctx, m0, gb, gb, prob.links, 1e-5, 10, ws, st)
    prob.close()


@pytest.mark.parametrize("dims,N,rep,m0", CG_CASES)
def test_dirac_solve_bicgstab_inverts_the_oracles_dirac_operator(hr, dims, N, rep, m0):
    import torch
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(131, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    b = li.gaussian_spinor(132, V, d)
    x_want, _ = solver.dirac_solve(dims, BC_T, R, m0, b, 1e-11, 1000)
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    lat, P = prob.lat, prob.prec
    half = hr.hr_spinor_bytes(lat.ctx, P)
    gb, gx = lat.spinor(P, full=True), lat.spinor(P, full=True)
    for p in (0, 1):
        lat.import_spinor(gb[p * half:(p + 1) * half], P, b[p * (V // 2):(p + 1) * (V // 2)], p)
    ws = torch.empty(hr.hr_bicgstab_workspace_bytes(lat.ctx, P, 500), dtype=torch.uint8, device="cuda")
    it, res2 = hr.hr_dirac_solve_bicgstab(lat.ctx, m0, gx, gb, prob.links, 1e-11, 500, ws, lat.stream())
    assert 0 < it < 500 and res2 <= 1e-22
    x = np.concatenate([lat.export_spinor(gx[p * half:(p + 1) * half], P, p) for p in (0, 1)])
    assert rel_l2(x, x_want) <= 1e-9
    assert rel_l2(oracle.dirac(dims, BC_T, R, m0, x), b) <= 1e-9
    prob.close()


@pytest.mark.parametrize("dims,N,rep,m0", CG_CASES)
def test_mixed_precision_bicgstab_reaches_fp64_accuracy(hr, dims, N, rep, m0):
    """hr_bicgstab_dhat_mixed: fp32 inner solves + fp64 true residual.  What it reaches has a plain definition, the
    solution of Dhat x = b: compared with the oracle's fp64 solution, and its true residual with the oracle's Dhat."""
    import torch
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(121, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    b = li.gaussian_spinor(122, li.volume(dims) // 2, d)
    x_want, _, _ = solver.bicgstab_dhat(dims, BC_T, R, m0, b, 1e-12, 500)
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    lat = prob.lat
    l32 = lat.gauge(True, hr.HR_F32)
    lat.represent_links(l32, prob.fund)                     # fp64 fundamental -> fp32 represented (one rounding on store)
    f = Fields(hr, prob)
    gb, gx = f.put(b), f.new()
    ws = torch.empty(hr.hr_mixed_workspace_bytes(lat.ctx, 500), dtype=torch.uint8, device="cuda")
    it, outer, res2 = hr.hr_bicgstab_dhat_mixed(lat.ctx, m0, gx, gb, prob.links, l32, 1e-10, 1e-4, 500, ws, lat.stream())
    assert 0 < it < 500 and 2 <= outer <= 6 and res2 <= 1e-20
    x = f.get(gx)
    assert rel_l2(x, x_want) <= 1e-8
    assert rel_l2(solver.dhat(dims, BC_T, R, m0, x), b) <= 2e-10        # TRUE residual, oracle's operator
    # argument errors: precisions swapped
    with pytest.raises(hr.HrError):
        hr.hr_bicgstab_dhat_mixed(lat.ctx, m0, gx, gb, l32, prob.links, 1e-10, 1e-4, 500, ws, lat.stream())
    with pytest.raises(hr.HrError):
        hr.hr_bicgstab_dhat_mixed(lat.ctx, m0, gx, gb, prob.links, l32, 1e-10, 1.5, 500, ws, lat.stream())
    prob.close()


def test_bicgstab_graph_replay_is_bitwise_the_plain_launch_sequence(hr):
    import torch
    dims, N, m0 = (4, 4, 4, 8), 3, -0.3
    U = li.haar_links(121, N, dims)
    b = li.gaussian_spinor(122, li.volume(dims) // 2, 3)
    prob = GpuProblem(hr, dims, N, "fund", "f64", U)
    f = Fields(hr, prob)
    gb = f.put(b)
    ws = torch.empty(hr.hr_bicgstab_workspace_bytes(prob.lat.ctx, f.P, 200), dtype=torch.uint8, device="cuda")
    res = {}
    for mode in (2, 0):
        prob.lat.set_tuning("cg_graph", mode)
        gx = f.new()
        n0 = hr.hr_launch_count()
        it, res2, hist = hr.hr_bicgstab_dhat(prob.lat.ctx, m0, gx, gb, prob.links, 1e-10, 200, ws, prob.lat.stream(), want_hist=True)
        res[mode] = (it, res2, hist.copy(), f.get(gx), hr.hr_launch_count() - n0)
    assert res[0][0] == res[2][0] and res[0][1] == res[2][1] and res[0][4] == res[2][4]
    assert np.array_equal(res[0][2], res[2][2]) and np.array_equal(res[0][3], res[2][3])
    prob.close()


# ---------------------------------------------------------------------------------------------
# gamma5-QMR ("QMR gamma_5 inverters"; reading C33)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims,N,rep,m0", CG_CASES)
def test_qmr_dhat_fp64_follows_the_oracle(hr, dims, N, rep, m0):
    """Same Lanczos process, same rotations, same stopping rule on both sides: the quasi-residual history |eta_k| / |b|
    agrees while it is well above rounding, iteration counts to +-1, the reported residual is the true one, the solution
    solves the oracle's operator."""
    import torch
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(121, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    b = li.gaussian_spinor(122, li.volume(dims) // 2, d)
    tol, maxiter = 1e-10, 300
    x_want, it_want, hist_want, res2_want = solver.qmr_dhat(dims, BC_T, R, m0, b, tol, maxiter)
    assert 3 < it_want < maxiter and res2_want <= tol * tol
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    f = Fields(hr, prob)
    gb, gx = f.put(b), f.new()
    ws = torch.empty(hr.hr_qmr_workspace_bytes(prob.lat.ctx, f.P), dtype=torch.uint8, device="cuda")
    ws.fill_(0xFF)
    it, res2, hist = hr.hr_qmr_dhat(prob.lat.ctx, m0, gx, gb, prob.links, tol, maxiter, ws, prob.lat.stream(), want_hist=True)
    assert abs(it - it_want) <= 1 and hist[0] == 1.0 and len(hist) == it + 1 and res2 <= tol * tol
    n = min(it, it_want) + 1
    assert np.allclose(hist[:n], hist_want[:n], rtol=1e-5, atol=1e-13)
    x = f.get(gx)
    assert rel_l2(x, x_want) <= 1e-8
    r = b - solver.dhat(dims, BC_T, R, m0, x)
    assert np.isclose(res2, solver.norm2(r) / solver.norm2(b), rtol=1e-3, atol=1e-26)   # the TRUE residual
    # one operator application per iteration: no more iterations than twice the CG's on the normal equations
    _, it_cg, _ = solver.cg_dhat(dims, BC_T, R, m0, b, tol, 500)
    assert it <= 2 * it_cg
    # bitwise reproducible
    gx2 = f.new()
    it2, res2b, _ = hr.hr_qmr_dhat(prob.lat.ctx, m0, gx2, gb, prob.links, tol, maxiter, ws, prob.lat.stream())
    assert it2 == it and res2b == res2 and np.array_equal(f.get(gx2), x)
    prob.close()


def test_qmr_fp32_on_the_fly_links_and_edge_cases(hr):
    import torch
    dims, N, m0 = (4, 4, 4, 8), 3, -0.3
    U = li.haar_links(121, N, dims)
    R = oracle.represent(N, oracle.REP_SYM, U)
    b = li.gaussian_spinor(122, li.volume(dims) // 2, 6)
    x_want, it_want, _, _ = solver.qmr_dhat(dims, BC_T, R, m0, b, 1e-5, 300)
    prob = GpuProblem(hr, dims, N, "sym", "f32", U)
    f = Fields(hr, prob)
    ctx, st = prob.lat.ctx, prob.lat.stream()
    ws = torch.empty(hr.hr_qmr_workspace_bytes(ctx, f.P), dtype=torch.uint8, device="cuda")
    gb, gx = f.put(b), f.new()
    for links in (prob.links, prob.fund):                                                     # represented / on the fly
        it, res2, _ = hr.hr_qmr_dhat(ctx, m0, gx, gb, links, 1e-5, 300, ws, st)
        assert abs(it - it_want) <= 2 and res2 <= 1e-10 and rel_l2(f.get(gx), x_want) <= 1e-4
    it, res2, hist = hr.hr_qmr_dhat(ctx, m0, gx, gb, prob.links, 1e-5, 0, ws, st, want_hist=True)        # maxiter = 0
    assert it == 0 and abs(res2 - 1.0) <= 1e-6 and not f.get(gx).any()
    it, res2, _ = hr.hr_qmr_dhat(ctx, m0, gx, f.put(np.zeros_like(b)), prob.links, 1e-5, 50, ws, st)     # b = 0
    assert it == 0 and res2 == 0.0 and not f.get(gx).any()
    it, res2, hist = hr.hr_qmr_dhat(ctx, m0, gx, gb, prob.links, 1e-12, 3, ws, st, want_hist=True)       # maxiter hit
    assert it == 3 and len(hist) == 4 and res2 > 1e-12
    with pytest.raises(hr.HrError):
        hr.hr_qmr_dhat(ctx, m0, gb, gb, prob.links, 1e-5, 10, ws, st)
    prob.close()
