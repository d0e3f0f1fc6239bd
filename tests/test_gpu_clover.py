"""GPU parity of SURVEY.md section 8(f) NEXT-4, the clover term (include/hr.h fourth part; reading C28),
through the C ABI against oracle/clover.py on the same seeded inputs.  The clover field itself is private (packed
Hermitian blocks), so what is compared is what is unique: T psi, obtained as hr_dirac_clover - hr_dirac, and the full
D_sw psi.  Tolerances: BASELINE.json:north_star (1e-13 fp64 / 2e-6 fp32, relative L2 vs the fp64 oracle); T alone is a
sum of 24 products of four links, checked to 20x those."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle import clover
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


def _full(prob, psi_eo):
    lat, P = prob.lat, prob.prec
    vh = lat.vh
    half = prob.hr.hr_spinor_bytes(lat.ctx, P)
    t = lat.spinor(P, full=True)
    for p in (0, 1):
        lat.import_spinor(t[p * half:(p + 1) * half], P, psi_eo[p * vh:(p + 1) * vh], p)
    return t


def _get_full(prob, t):
    lat, P = prob.lat, prob.prec
    half = prob.hr.hr_spinor_bytes(lat.ctx, P)
    return np.concatenate([lat.export_spinor(t[p * half:(p + 1) * half], P, p) for p in (0, 1)])


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(2, "fund"), (3, "fund"), (2, "adj"), (3, "sym"), (3, "adj"), (4, "fund")])
@pytest.mark.parametrize("dims", [(4, 4, 6, 8), (2, 2, 2, 2), (6, 2, 4, 2)])
def test_dirac_clover_matches_oracle(hr, dims, N, rep, prec):
    import torch
    if rep in ("sym", "adj") and N == 3 and dims != (4, 4, 6, 8) and prec == "f32":
        pytest.skip("covered by the other sizes")
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(401, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    psi = li.gaussian_spinor(402, V, d)
    m0, csw = -0.3, 1.4
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    lat, P = prob.lat, prob.prec
    cl = torch.empty(hr.hr_clover_bytes(lat.ctx, P), dtype=torch.uint8, device="cuda")
    cl.fill_(0xFF)
    n0 = hr.hr_launch_count()
    hr.hr_clover_build(cl, prob.links, csw, lat.stream())
    two = d >= 4 or (d == 3 and rep != "adj")                     # plane- or row-parallel Q kernel + packing kernel; else one kernel
    assert hr.hr_launch_count() == n0 + (2 if two else 1)
    gin = _full(prob, psi)
    gout, gref = lat.spinor(P, full=True), lat.spinor(P, full=True)
    gout.fill_(0xFF)
    n0 = hr.hr_launch_count()
    hr.hr_dirac_clover(m0, gout, gin, prob.links, cl, lat.stream())
    assert hr.hr_launch_count() - n0 in (2, 4)                          # fused into the Dphi epilogues where d_R <= 4
    got = _get_full(prob, gout)
    want = clover.dirac_clover(dims, BC_T, R, m0, csw, psi)
    assert rel_l2(got, want) <= TOL[prec]
    # the clover part alone: (D_sw - D) psi = T psi
    lat.dirac(m0, gref, gin, prob.links)
    tpsi = got - _get_full(prob, gref)
    T = clover.clover_term(dims, R, csw)
    want_t = oracle.lex_to_eo(dims, clover.apply_clover_lex(T, oracle.eo_to_lex(dims, psi)))
    assert np.linalg.norm(tpsi - want_t) <= 20 * TOL[prec] * np.linalg.norm(want)
    prob.close()


def test_clover_vanishes_on_pure_gauge_and_scales_with_csw(hr):
    import torch
    dims, N = (4, 4, 4, 4), 3
    V = li.volume(dims)
    g = li.haar_links(403, N, dims)[:, 0].reshape(dims + (N, N))
    pure = np.empty((V, 4, N, N), dtype=complex)
    for mu in range(4):                                                 # U_mu(x) = g(x) g(x+mu)^dagger
        gs = np.roll(g, -1, axis=mu)
        pure[:, mu] = (g @ np.conj(np.swapaxes(gs, -1, -2))).reshape(V, N, N)
    psi = li.gaussian_spinor(404, V, 3)
    prob = GpuProblem(hr, dims, N, "fund", "f64", pure)
    lat, P = prob.lat, prob.prec
    cl = torch.empty(hr.hr_clover_bytes(lat.ctx, P), dtype=torch.uint8, device="cuda")
    hr.hr_clover_build(cl, prob.links, 1.9, lat.stream())
    gin = _full(prob, psi)
    a, b = lat.spinor(P, full=True), lat.spinor(P, full=True)
    hr.hr_dirac_clover(0.1, a, gin, prob.links, cl, lat.stream())
    lat.dirac(0.1, b, gin, prob.links)
    assert rel_l2(_get_full(prob, a), _get_full(prob, b)) <= 1e-13      # F = 0 on a pure-gauge field
    prob.close()
    U = li.haar_links(405, N, dims)
    prob = GpuProblem(hr, dims, N, "fund", "f64", U)
    lat = prob.lat
    gin = _full(prob, psi)
    outs = []
    for csw in (0.0, 1.0, 2.0):
        hr.hr_clover_build(cl, prob.links, csw, lat.stream())
        o = lat.spinor(P, full=True)
        hr.hr_dirac_clover(0.1, o, gin, prob.links, cl, lat.stream())
        outs.append(_get_full(prob, o))
    lat.dirac(0.1, b, gin, prob.links)
    assert np.array_equal(outs[0], _get_full(prob, b))                  # c_sw = 0: exactly D
    assert rel_l2(outs[2] - outs[0], 2 * (outs[1] - outs[0])) <= 1e-12  # linear in c_sw
    with pytest.raises(hr.HrError):
        hr.hr_clover_build(cl, prob.fund, 1.0, lat.stream())            # needs the represented field
    with pytest.raises(hr.HrError):
        hr.hr_dirac_clover(0.1, gin, gin, prob.links, cl, lat.stream())
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_clover_on_a_131072_site_lattice(hr, prec):
    """SU(3) fundamental 16^3 x 32 (1024 CTAs of the apply kernel, 2048 of the build kernel): every site against the
    oracle (its whole-lattice numpy arrays take seconds here; at 32^3 x 64 they need minutes and 5 GB)."""
    import torch
    dims, N = (32, 16, 16, 16), 3
    U = li.near_identity_links(406, N, dims, 0.3)
    V = li.volume(dims)
    psi = li.gaussian_spinor(407, V, 3)
    prob = GpuProblem(hr, dims, N, "fund", prec, U)
    lat, P = prob.lat, prob.prec
    cl = torch.empty(hr.hr_clover_bytes(lat.ctx, P), dtype=torch.uint8, device="cuda")
    hr.hr_clover_build(cl, prob.links, 1.0, lat.stream())
    gin = _full(prob, psi)
    o = lat.spinor(P, full=True)
    hr.hr_dirac_clover(-0.2, o, gin, prob.links, cl, lat.stream())
    got = _get_full(prob, o)
    want = clover.dirac_clover(dims, BC_T, U, -0.2, 1.0, psi)
    assert rel_l2(got, want) <= TOL[prec]
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(2, "fund"), (3, "fund"), (2, "adj"), (3, "sym"), (3, "adj")])
def test_dirac_expclover_matches_oracle(hr, N, rep, prec):
    """PAPER.md:70 "exponentiated clover"; reading C31: hr_clover_build + hr_clover_exp + hr_dirac_clover = D_exp."""
    import torch
    dims = (4, 4, 2, 6)
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(411, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    psi = li.gaussian_spinor(412, V, d)
    m0, csw = -0.6, 1.7
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    lat, P = prob.lat, prob.prec
    cl = torch.empty(hr.hr_clover_bytes(lat.ctx, P), dtype=torch.uint8, device="cuda")
    hr.hr_clover_build(cl, prob.links, csw, lat.stream())
    n0 = hr.hr_launch_count()
    hr.hr_clover_exp(lat.ctx, P, cl, m0, lat.stream())
    assert hr.hr_launch_count() == n0 + 1
    gin = _full(prob, psi)
    gout, gref = lat.spinor(P, full=True), lat.spinor(P, full=True)
    hr.hr_dirac_clover(m0, gout, gin, prob.links, cl, lat.stream())
    got = _get_full(prob, gout)
    want = clover.dirac_expclover(dims, BC_T, R, m0, csw, psi)
    assert rel_l2(got, want) <= TOL[prec]
    # the exponential part alone, E psi = (D_exp - D) psi, and that it differs from the plain clover term at second order
    lat.dirac(m0, gref, gin, prob.links)
    epsi = got - _get_full(prob, gref)
    E = clover.exp_clover_term(dims, R, m0, csw)
    want_e = oracle.lex_to_eo(dims, clover.apply_clover_lex(E, oracle.eo_to_lex(dims, psi)))
    assert np.linalg.norm(epsi - want_e) <= 20 * TOL[prec] * np.linalg.norm(want)
    T = clover.clover_term(dims, R, csw)
    want_t = oracle.lex_to_eo(dims, clover.apply_clover_lex(T, oracle.eo_to_lex(dims, psi)))
    assert np.linalg.norm(epsi - want_t) > 1e-3 * np.linalg.norm(want_t)
    with pytest.raises(hr.HrError):
        hr.hr_clover_exp(lat.ctx, P, cl, -4.5, lat.stream())            # 4 + m0 <= 0
    prob.close()


@pytest.mark.parametrize("m0", [-0.3, -8.0])       # -8: A = -4 + T is negative definite -> the pivoted fallback of hr_clover_finalize
@pytest.mark.parametrize("exponentiated", [False, True])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(3, "fund"), (2, "adj"), (3, "sym"), (2, "fund"), (4, "fund"), (3, "adj")])
def test_dhat_clover_matches_oracle(hr, N, rep, prec, exponentiated, m0):
    """Reading C32: Dhat_sw = A_ee - Dphi_eo A_oo^{-1} Dphi_oe with A from hr_clover_build [+ hr_clover_exp] +
    hr_clover_finalize, against the oracle (dense per-site blocks, numpy.linalg.solve for A^{-1}).  hr_clover_finalize
    inverts positive definite blocks by a Cholesky factorisation (in registers for d_R <= 4, one warp per block in shared
    memory above) and everything else by Gauss-Jordan with partial pivoting: both paths here."""
    import torch
    dims = (4, 4, 2, 6)
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(421, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    psi = li.gaussian_spinor(422, V // 2, d)
    csw = 1.1
    if exponentiated and m0 < -4:
        pytest.skip("the exponentiated clover term is defined for 4 + m0 > 0")
    want = clover.dhat_clover(dims, BC_T, R, m0, csw, psi, exponentiated)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    lat, P = prob.lat, prob.prec
    nb = hr.hr_clover_bytes(lat.ctx, P)
    A = torch.empty(nb, dtype=torch.uint8, device="cuda")
    Ainv = torch.empty(nb, dtype=torch.uint8, device="cuda")
    Ainv.fill_(0xFF)
    hr.hr_clover_build(A, prob.links, csw, lat.stream())
    if exponentiated:
        hr.hr_clover_exp(lat.ctx, P, A, m0, lat.stream())
    hr.hr_clover_finalize(lat.ctx, P, A, Ainv, m0, lat.stream())
    gin = lat.spinor(P)
    lat.import_spinor(gin, P, psi, 0)
    out, t1, t2 = lat.spinor(P), lat.spinor(P), lat.spinor(P)
    out.fill_(0xFF)
    n0 = hr.hr_launch_count()
    hr.hr_dhat_clover(out, gin, t1, t2, prob.links, A, Ainv, lat.stream())
    assert hr.hr_launch_count() - n0 in (2, 4)
    # fp32: A^{-1} amplifies the input rounding by the condition number of the blocks (a few units here)
    assert rel_l2(lat.export_spinor(out, P, 0), want) <= (TOL[prec] if prec == "f64" else 5 * TOL[prec])
    with pytest.raises(hr.HrError):
        hr.hr_dhat_clover(out, gin, t1, t1, prob.links, A, Ainv, lat.stream())
    prob.close()


@pytest.mark.parametrize("exponentiated", [False, True])
@pytest.mark.parametrize("N,rep", [(3, "fund"), (2, "adj")])
def test_dirac_clover_solve_inverts_the_oracles_operator(hr, N, rep, exponentiated):
    import torch
    dims = (4, 4, 4, 4)
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(431, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    b = li.gaussian_spinor(432, V, d)
    m0, csw = -0.2, 1.0
    x_want, it_want = clover.dirac_clover_solve(dims, BC_T, R, m0, csw, b, 1e-11, 500, exponentiated)
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    lat, P = prob.lat, prob.prec
    nb = hr.hr_clover_bytes(lat.ctx, P)
    A = torch.empty(nb, dtype=torch.uint8, device="cuda")
    Ainv = torch.empty(nb, dtype=torch.uint8, device="cuda")
    hr.hr_clover_build(A, prob.links, csw, lat.stream())
    if exponentiated:
        hr.hr_clover_exp(lat.ctx, P, A, m0, lat.stream())
    hr.hr_clover_finalize(lat.ctx, P, A, Ainv, m0, lat.stream())
    gb = _full(prob, b)
    gx = lat.spinor(P, full=True)
    gx.fill_(0xFF)
    ws = torch.empty(hr.hr_clover_solve_workspace_bytes(lat.ctx, P, 500), dtype=torch.uint8, device="cuda")
    it, res2 = hr.hr_dirac_clover_solve(lat.ctx, gx, gb, prob.links, A, Ainv, 1e-11, 500, ws, lat.stream())
    assert abs(it - it_want) <= 2 and res2 <= 1e-22
    x = _get_full(prob, gx)
    assert rel_l2(x, x_want) <= 1e-9
    # the oracle's full operator applied to the GPU's solution gives back b
    Dx = clover.dirac_expclover(dims, BC_T, R, m0, csw, x) if exponentiated else clover.dirac_clover(dims, BC_T, R, m0, csw, x)
    assert rel_l2(Dx, b) <= 1e-9
    prob.close()


@pytest.mark.parametrize("variant", [0, 1, 6, 7])
def test_fused_and_unfused_clover_paths_agree(hr, variant):
    """hr_dirac_clover / hr_dhat_clover fuse the site-diagonal matrix into the Dphi epilogue for the `site` / `site_ef`
    kernels (d_R <= 4) and fall back to separate site-local launches otherwise: same operator either way."""
    import torch
    dims, N, rep, m0, csw = (4, 4, 2, 6), 3, "fund", -0.3, 1.1
    U = li.haar_links(441, N, dims)
    V = li.volume(dims)
    psi = li.gaussian_spinor(442, V, 3)
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    lat, P = prob.lat, prob.prec
    lat.set_tuning("variant", variant)
    nb = hr.hr_clover_bytes(lat.ctx, P)
    T = torch.empty(nb, dtype=torch.uint8, device="cuda")
    A = torch.empty(nb, dtype=torch.uint8, device="cuda")
    Ainv = torch.empty(nb, dtype=torch.uint8, device="cuda")
    hr.hr_clover_build(T, prob.links, csw, lat.stream())
    A.copy_(T)
    hr.hr_clover_finalize(lat.ctx, P, A, Ainv, m0, lat.stream())
    gin = _full(prob, psi)
    gout = lat.spinor(P, full=True)
    n0 = hr.hr_launch_count()
    hr.hr_dirac_clover(m0, gout, gin, prob.links, T, lat.stream())
    assert hr.hr_launch_count() - n0 == (2 if variant in (0, 1) else 4)
    assert rel_l2(_get_full(prob, gout), clover.dirac_clover(dims, BC_T, U, m0, csw, psi)) <= TOL["f64"]
    half = hr.hr_spinor_bytes(lat.ctx, P)
    out, t1, t2 = lat.spinor(P), lat.spinor(P), lat.spinor(P)
    n0 = hr.hr_launch_count()
    hr.hr_dhat_clover(out, gin[:half], t1, t2, prob.links, A, Ainv, lat.stream())
    assert hr.hr_launch_count() - n0 == (2 if variant in (0, 1) else 4)
    assert rel_l2(lat.export_spinor(out, P, 0), clover.dhat_clover(dims, BC_T, U, m0, csw, psi[:V // 2])) <= TOL["f64"]
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(3, "fund"), (4, "fund"), (3, "sym"), (3, "adj")])
def test_clover_setup_kernels_are_bitwise_repeatable(hr, N, rep, prec):
    """hr_clover_build / hr_clover_exp / hr_clover_finalize run the same arithmetic in the same order every time -- in
    registers (d_R <= 3 / 4), or shared out over the lanes of a warp or the row-threads of a CTA through shared memory
    (d_R >= 4 / 6): a missing barrier in those would show up as bytes that change from run to run (compute-sanitizer's
    racecheck is not available on this pool).  Ragged sizes: the last CTA / warp group is partial."""
    import torch
    dims = (6, 2, 6, 2)                                        # 72 sites per parity: no multiple of 32, 4 or 2 warps' worth
    prob = GpuProblem(hr, dims, N, rep, prec, li.haar_links(451, N, dims))
    lat, P, st = prob.lat, prob.prec, prob.lat.stream()
    nb = hr.hr_clover_bytes(lat.ctx, P)
    runs = []
    for _ in range(3):
        T = torch.full((nb,), 0xFF, dtype=torch.uint8, device="cuda")
        Ainv = torch.full((nb,), 0xFF, dtype=torch.uint8, device="cuda")
        hr.hr_clover_build(T, prob.links, 1.2, st)
        E = T.clone()
        hr.hr_clover_exp(lat.ctx, P, E, -0.25, st)
        A = E.clone()
        hr.hr_clover_finalize(lat.ctx, P, A, Ainv, -0.25, st)
        torch.cuda.synchronize()
        runs.append((T, E, A, Ainv))
    for k in (1, 2):
        for a, b in zip(runs[0], runs[k]):
            assert torch.equal(a, b)
    for t in runs[0]:                                          # every byte was written (0xFF.. is a NaN pattern in both precisions)
        v = t.view(torch.float64 if prec == "f64" else torch.float32)
        assert not torch.isnan(v).any()
    prob.close()
