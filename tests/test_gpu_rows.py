"""GPU parity of the row-compressed fundamental links (hr_gauge_alloc(kind 2) + hr_gauge_compress; reading C30): the
fundamental representation of SU(2) / SU(3) with the last row rebuilt in the kernel, and the SU(2) adjoint built from
the four reals of the first row.  Same operator as with full links, so the oracle is unchanged; tolerances
BASELINE.json:north_star (the inputs are special unitary to 1e-16)."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle import solver
from gpu_common import BC_T, TOL, GpuProblem, oracle_rep_id, rel_l2

pytestmark = pytest.mark.gpu
COMBOS = [(2, "fund"), (3, "fund"), (2, "adj"), (3, "adj")]


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available()
    from paper_2405_19294_b200 import build
    build.build()
    import paper_2405_19294_b200 as hr
    return hr


def _rows(hr, prob):
    g = prob.lat.gauge(2, prob.prec)
    n0 = hr.hr_launch_count()
    prob.lat.compress_links(g, prob.fund)
    assert hr.hr_launch_count() == n0 + 1
    return g


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", COMBOS)
@pytest.mark.parametrize("dims,bc", [((4, 4, 6, 8), BC_T), ((2, 2, 2, 2), (-1, 1, -1, 1)), ((6, 2, 4, 10), (1, 1, 1, 1))])
def test_dphi_eo_from_row_compressed_links(hr, dims, bc, N, rep, prec):
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(601, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    vh = li.volume(dims) // 2
    prob = GpuProblem(hr, dims, N, rep, prec, U, bc=bc)
    rows = _rows(hr, prob)
    assert hr.hr_gauge_bytes(prob.lat.ctx, 2, prob.prec) * N == hr.hr_gauge_bytes(prob.lat.ctx, 0, prob.prec) * (N - 1)
    for parity in (0, 1):
        psi = li.gaussian_spinor(602 + parity, vh, d)
        want = oracle.dphi_eo(dims, bc, R, parity, psi)
        gin = prob.lat.spinor(prob.prec)
        prob.lat.import_spinor(gin, prob.prec, psi, 1 - parity)
        for variant in (-1, 0, 1, 2, 3, 4, 5, 7, 9, 10, 11):
            try:
                prob.lat.set_tuning("variant", variant)
                out = prob.lat.spinor(prob.prec)
                out.fill_(0xFF)
                prob.lat.dphi_eo(out, gin, rows, parity)
            except hr.HrError as e:
                assert e.status in (hr.HR_EUNSUPPORTED, hr.HR_EINVAL)
                continue
            assert rel_l2(prob.lat.export_spinor(out, prob.prec, parity), want) <= TOL[prec], (variant, parity)
        prob.lat.set_tuning("variant", -1)
    prob.close()


@pytest.mark.parametrize("N,rep", COMBOS)
def test_dirac_dhat_cg_and_slabs_from_row_compressed_links(hr, N, rep):
    from paper_2405_19294_b200 import halo
    dims, m0 = (4, 4, 4, 6), -0.3
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(603, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    psi = li.gaussian_spinor(604, V, d)
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    lat, P = prob.lat, prob.prec
    rows = _rows(hr, prob)
    half = hr.hr_spinor_bytes(lat.ctx, P)
    gin, gout = lat.spinor(P, full=True), lat.spinor(P, full=True)
    for p in (0, 1):
        lat.import_spinor(gin[p * half:(p + 1) * half], P, psi[p * (V // 2):(p + 1) * (V // 2)], p)
    lat.dirac(m0, gout, gin, rows)
    got = np.concatenate([lat.export_spinor(gout[p * half:(p + 1) * half], P, p) for p in (0, 1)])
    assert rel_l2(got, oracle.dirac(dims, BC_T, R, m0, psi)) <= TOL["f64"]
    out, tmp = lat.spinor(P), lat.spinor(P)
    lat.dhat(m0, True, out, gin[:half], tmp, rows)
    assert rel_l2(lat.export_spinor(out, P, 0), solver.g5(solver.dhat(dims, BC_T, R, m0, psi[:V // 2]))) <= TOL["f64"]
    x_want, it_want, _ = solver.cg_dhat(dims, BC_T, R, m0, psi[:V // 2], 1e-10, 500)
    gx = lat.spinor(P)
    it, res2, _ = lat.cg_dhat(m0, gx, gin[:half], rows, 1e-10, 500, lat.cg_workspace(P, 500))
    assert abs(it - it_want) <= 1 and rel_l2(lat.export_spinor(gx, P, 0), x_want) <= 1e-8
    slab = halo.SlabDphi(lat, P, halo.slab_plan(0, 1, dims[0]))
    o = lat.spinor(P)
    slab.dphi_eo(o, gin[half:], rows, 0)
    assert rel_l2(lat.export_spinor(o, P, 0), oracle.dphi_eo(dims, BC_T, R, 0, psi[V // 2:])) <= TOL["f64"]
    prob.close()


def test_row_compressed_field_rules(hr):
    dims = (4, 4, 4, 4)
    prob = GpuProblem(hr, dims, 3, "sym", "f64", li.haar_links(605, 3, dims))
    rows = _rows(hr, prob)
    with pytest.raises(hr.HrError) as e:                       # two-index representations: no kernel from rows
        prob.lat.dphi_eo(prob.lat.spinor(prob.prec), prob.lat.spinor(prob.prec), rows, 0)
    assert e.value.status == hr.HR_EINVAL
    with pytest.raises(hr.HrError):
        prob.lat.export_gauge(rows, False)
    with pytest.raises(hr.HrError):
        prob.lat.compress_links(prob.links, prob.fund)         # destination must be a rows field
    import torch
    with pytest.raises(hr.HrError):
        hr.hr_clover_build(torch.empty(hr.hr_clover_bytes(prob.lat.ctx, prob.prec), dtype=torch.uint8, device="cuda"), rows, 1.0, 0)
    prob.close()
    p4 = GpuProblem(hr, dims, 4, "fund", "f64", li.haar_links(606, 4, dims))
    with pytest.raises(hr.HrError) as e:
        p4.lat.gauge(2, p4.prec)
    assert e.value.status == hr.HR_EUNSUPPORTED
    p4.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_config2_from_row_compressed_links_full_size(hr, prec):
    """BASELINE.json:configs[1] (SU(3) fundamental 32^3 x 64) with 12-real links, every output site vs the oracle."""
    dims = (64, 32, 32, 32)
    U = li.haar_links(1002, 3, dims)
    vh = li.volume(dims) // 2
    prob = GpuProblem(hr, dims, 3, "fund", prec, U)
    rows = _rows(hr, prob)
    for parity in (0, 1):
        psi = li.gaussian_spinor(2002 + 10 * parity, vh, 3)
        want = oracle.dphi_eo(dims, BC_T, U, parity, psi)
        gin, out = prob.lat.spinor(prob.prec), prob.lat.spinor(prob.prec)
        prob.lat.import_spinor(gin, prob.prec, psi, 1 - parity)
        prob.lat.dphi_eo(out, gin, rows, parity)
        got = prob.lat.export_spinor(out, prob.prec, parity)
        assert rel_l2(got, want) <= TOL[prec]
        scale = np.sqrt(np.mean(np.abs(want) ** 2))
        assert np.abs(got - want).max() <= 50 * TOL[prec] * scale
    prob.close()
