"""GPU parity of SURVEY.md section 8(f) NEXT-3, "on-the-fly representation": every compute call accepts the
FUNDAMENTAL link field for the two-index representations and applies R(U) inside the kernel as
U Psi U^T / U^dagger Psi U^* (no represented field is ever read; 144 B instead of 576 B per SU(3) sextet link in
fp64).  The result is by definition the same operator, so the oracle is unchanged: represent (trace
definition, reading C8) followed by the stencil.  Tolerances: BASELINE.json:north_star."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle import solver
from gpu_common import BC_T, TOL, GpuProblem, oracle_rep_id, rel_l2

pytestmark = pytest.mark.gpu

OTF_COMBOS = [(2, "sym"), (3, "sym"), (3, "asym"), (4, "asym"), (3, "adj")]


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available()
    from paper_2405_19294_b200 import build
    build.build()
    import paper_2405_19294_b200 as hr
    return hr


def _put(prob, canon, parity):
    t = prob.lat.spinor(prob.prec)
    prob.lat.import_spinor(t, prob.prec, canon, parity)
    return t


def _new(prob, full=False):
    t = prob.lat.spinor(prob.prec, full=full)
    t.fill_(0xFF)
    return t


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", OTF_COMBOS)
@pytest.mark.parametrize("dims", [(4, 4, 6, 8), (2, 2, 2, 2), (6, 2, 4, 10)])
def test_dphi_eo_from_fundamental_links_matches_oracle(hr, dims, N, rep, prec):
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(201, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    vh = li.volume(dims) // 2
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    for parity in (0, 1):
        psi = li.gaussian_spinor(202 + parity, vh, d)
        want = oracle.dphi_eo(dims, BC_T, R, parity, psi)
        gin = _put(prob, psi, 1 - parity)
        for variant in (0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11):
            try:
                prob.lat.set_tuning("variant", variant)
                out = _new(prob)
                prob.lat.dphi_eo(out, gin, prob.fund, parity)        # FUNDAMENTAL links
            except hr.HrError as e:
                assert e.status in (hr.HR_EUNSUPPORTED, hr.HR_EINVAL)
                continue
            got = prob.lat.export_spinor(out, prob.prec, parity)
            assert rel_l2(got, want) <= TOL[prec], (variant, parity)
        prob.lat.set_tuning("variant", -1)
        # and the explicit-link path gives the same operator
        out = _new(prob)
        prob.lat.dphi_eo(out, gin, prob.links, parity)
        assert rel_l2(prob.lat.export_spinor(out, prob.prec, parity), want) <= TOL[prec]
    prob.close()


@pytest.mark.parametrize("bc", [(1, 1, 1, 1), (-1, -1, 1, -1)])
def test_otf_boundary_signs(hr, bc):
    dims, N, rep = (4, 2, 6, 4), 3, "sym"
    U = li.haar_links(203, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    psi = li.gaussian_spinor(204, li.volume(dims) // 2, 6)
    prob = GpuProblem(hr, dims, N, rep, "f64", U, bc=bc)
    out = _new(prob)
    prob.lat.dphi_eo(out, _put(prob, psi, 1), prob.fund, 0)
    assert rel_l2(prob.lat.export_spinor(out, prob.prec, 0), oracle.dphi_eo(dims, bc, R, 0, psi)) <= TOL["f64"]
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", OTF_COMBOS)
def test_dirac_and_dhat_from_fundamental_links(hr, N, rep, prec):
    dims, m0 = (4, 4, 4, 6), -0.35
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(205, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    psi = li.gaussian_spinor(206, V, d)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    lat, P = prob.lat, prob.prec
    half = hr.hr_spinor_bytes(lat.ctx, P)
    gin, gout = lat.spinor(P, full=True), _new(prob, full=True)
    for p in (0, 1):
        lat.import_spinor(gin[p * half:(p + 1) * half], P, psi[p * (V // 2):(p + 1) * (V // 2)], p)
    lat.dirac(m0, gout, gin, prob.fund)
    got = np.concatenate([lat.export_spinor(gout[p * half:(p + 1) * half], P, p) for p in (0, 1)])
    assert rel_l2(got, oracle.dirac(dims, BC_T, R, m0, psi)) <= TOL[prec]
    out, tmp = _new(prob), _new(prob)
    for g5 in (0, 1):
        lat.dhat(m0, bool(g5), out, gin[:half], tmp, prob.fund)
        want = solver.dhat(dims, BC_T, R, m0, psi[:V // 2])
        assert rel_l2(lat.export_spinor(out, P, 0), solver.g5(want) if g5 else want) <= TOL[prec]
    prob.close()


def test_cg_from_fundamental_links_follows_the_oracle(hr):
    dims, N, rep, m0 = (4, 4, 4, 4), 3, "sym", -0.2
    U = li.haar_links(121, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    b = li.gaussian_spinor(122, li.volume(dims) // 2, 6)
    x_want, it_want, hist_want = solver.cg_dhat(dims, BC_T, R, m0, b, 1e-10, 500)
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    gx = _new(prob)
    ws = prob.lat.cg_workspace(prob.prec, 500)
    it, res2, hist = prob.lat.cg_dhat(m0, gx, _put(prob, b, 0), prob.fund, 1e-10, 500, ws, want_hist=True)
    assert abs(it - it_want) <= 1 and res2 <= 1e-20
    n = min(it, it_want) + 1
    assert np.allclose(hist[:n], hist_want[:n], rtol=1e-6, atol=0)
    assert rel_l2(prob.lat.export_spinor(gx, prob.prec, 0), x_want) <= 1e-8
    prob.close()


def test_fundamental_rep_accepts_either_field_and_adjoint_rejects_fundamental_links(hr):
    dims = (4, 4, 4, 4)
    U = li.haar_links(207, 3, dims)
    psi = li.gaussian_spinor(208, li.volume(dims) // 2, 3)
    prob = GpuProblem(hr, dims, 3, "fund", "f64", U)
    a, b = _new(prob), _new(prob)
    gin = _put(prob, psi, 1)
    prob.lat.dphi_eo(a, gin, prob.links, 0)
    prob.lat.dphi_eo(b, gin, prob.fund, 0)       # FUND: the two fields are the same N x N links (reading C19)
    assert np.array_equal(prob.lat.export_spinor(a, prob.prec, 0), prob.lat.export_spinor(b, prob.prec, 0))
    prob.close()
    U2 = li.haar_links(209, 2, dims)
    prob = GpuProblem(hr, dims, 2, "adj", "f64", U2)
    with pytest.raises(hr.HrError) as e:
        prob.lat.dphi_eo(_new(prob), _new(prob), prob.fund, 0)
    assert e.value.status == hr.HR_EINVAL
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_config4_sextet_full_size_from_fundamental_links(hr, prec):
    """BASELINE.json:configs[3] (SU(3) two-index symmetric, 24^3 x 48) in the launch configuration bench.py
    times for the on-the-fly path, every output site against the oracle."""
    dims = (48, 24, 24, 24)
    U = li.haar_links(1004, 3, dims)
    R = oracle.represent(3, oracle.REP_SYM, U)
    vh = li.volume(dims) // 2
    prob = GpuProblem(hr, dims, 3, "sym", prec, U)
    for parity in (0, 1):
        psi = li.gaussian_spinor(2004 + 10 * parity, vh, 6)
        want = oracle.dphi_eo(dims, BC_T, R, parity, psi)
        out = _new(prob)
        prob.lat.dphi_eo(out, _put(prob, psi, 1 - parity), prob.fund, parity)
        got = prob.lat.export_spinor(out, prob.prec, parity)
        assert rel_l2(got, want) <= TOL[prec]
        scale = np.sqrt(np.mean(np.abs(want) ** 2))
        assert np.abs(got - want).max() <= 50 * TOL[prec] * scale
    prob.close()
