"""GPU parity of SURVEY.md section 8(e)/(f) NEXT-2: Dphi_eo on slabs along t with half-spinor messages
(include/hr.h third part).  One GPU only, kernels launched one after the other (no rank waits on
another): (a) one rank whose neighbour is itself must reproduce hr_dphi_eo and the oracle; (b) a GLOBAL lattice
cut into 2 or 4 slabs, every slab run in turn on this GPU with the messages handed over by pointer, stitched
together, must equal the oracle on the global lattice -- this checks the decomposition (which slice, which link,
which projector, where the antiperiodic seam sits).  The two-process routing is tested on CPU (gloo) in
tests/test_multi_rank.py.  Tolerances: BASELINE.json:north_star."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
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


def _bufs(hr, prob, n=4):
    import torch
    nb = hr.hr_halo_bytes(prob.lat.ctx, prob.prec)
    out = []
    for _ in range(n):
        t = torch.empty(nb, dtype=torch.uint8, device="cuda")
        t.fill_(0xFF)
        out.append(t)
    return out


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep,fundlinks", [(3, "fund", False), (2, "adj", False), (3, "sym", False), (3, "sym", True), (4, "asym", True),
                                            (4, "adj", False)])      # SU(4) adjoint: link records with padded rows
@pytest.mark.parametrize("dims,bc", [((4, 4, 6, 8), BC_T), ((2, 2, 4, 2), (-1, 1, -1, 1)), ((6, 2, 2, 10), (1, 1, 1, 1))])
def test_single_rank_slab_reproduces_dphi_eo(hr, dims, bc, N, rep, fundlinks, prec):
    from paper_2405_19294_b200 import halo
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(301, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    vh = li.volume(dims) // 2
    prob = GpuProblem(hr, dims, N, rep, prec, U, bc=bc)
    links = prob.fund if fundlinks else prob.links
    plan = halo.slab_plan(0, 1, dims[0])
    assert plan["first_rank"] and plan["last_rank"] and plan["prev"] == plan["next"] == 0
    slab = halo.SlabDphi(prob.lat, prob.prec, plan)
    for parity in (0, 1):
        psi = li.gaussian_spinor(302 + parity, vh, d)
        gin = prob.lat.spinor(prob.prec)
        prob.lat.import_spinor(gin, prob.prec, psi, 1 - parity)
        out = prob.lat.spinor(prob.prec)
        out.fill_(0xFF)
        n0 = hr.hr_launch_count()
        slab.dphi_eo(out, gin, links, parity)
        assert hr.hr_launch_count() == n0 + 3                      # pack, interior, apply
        got = prob.lat.export_spinor(out, prob.prec, parity)
        assert rel_l2(got, oracle.dphi_eo(dims, bc, R, parity, psi)) <= TOL[prec]
    prob.close()


def _split_eo(dims, field_half, parity, nslab):
    """Canonical half field of the global lattice -> list of the slabs' canonical half fields (t-slabs are
    contiguous in the canonical half index, reading C4)."""
    per = field_half.shape[0] // nslab
    return [np.ascontiguousarray(field_half[r * per:(r + 1) * per]) for r in range(nslab)]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("nslab", [2, 4])
@pytest.mark.parametrize("N,rep,fundlinks", [(3, "fund", False), (2, "adj", False), (3, "sym", True)])
def test_slabs_stitched_equal_the_global_oracle(hr, N, rep, fundlinks, nslab, prec):
    from paper_2405_19294_b200 import halo
    dims = (8, 4, 2, 6)
    bc = BC_T                                                       # antiperiodic in t: the seam sign must sit on one face only
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(311, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    Tl = dims[0] // nslab
    ldims = (Tl,) + dims[1:]
    # gauge field: canonical order is lexicographic with t slowest -> slabs are contiguous blocks of sites
    Us = [np.ascontiguousarray(U[r * (V // nslab):(r + 1) * (V // nslab)]) for r in range(nslab)]
    probs = [GpuProblem(hr, ldims, N, rep, prec, Us[r], bc=bc) for r in range(nslab)]
    plans = [halo.slab_plan(r, nslab, dims[0]) for r in range(nslab)]
    for parity in (0, 1):
        psi = li.gaussian_spinor(312 + parity, V // 2, d)
        want = oracle.dphi_eo(dims, bc, R, parity, psi)
        psis = _split_eo(dims, psi, 1 - parity, nslab)
        gin, gout, bufs = [], [], []
        for r, prob in enumerate(probs):
            t = prob.lat.spinor(prob.prec)
            prob.lat.import_spinor(t, prob.prec, psis[r], 1 - parity)
            gin.append(t)
            o = prob.lat.spinor(prob.prec)
            o.fill_(0xFF)
            gout.append(o)
            bufs.append(_bufs(hr, prob, 2))                         # (send_up, send_dn) of rank r
        for r, prob in enumerate(probs):                            # 1. every rank packs
            lk = prob.fund if fundlinks else prob.links
            hr.hr_dphi_eo_halo_pack(bufs[r][0], bufs[r][1], gin[r], lk, parity, prob.lat.stream())
        for r, prob in enumerate(probs):                            # 2.-4. messages handed over by pointer
            lk = prob.fund if fundlinks else prob.links
            st = prob.lat.stream()
            hr.hr_dphi_eo_interior(gout[r], gin[r], lk, parity, st)
            recv_prev = bufs[plans[r]["prev"]][0]                   # the previous rank's send_up
            recv_next = bufs[plans[r]["next"]][1]                   # the next rank's send_dn
            hr.hr_dphi_eo_halo_apply(gout[r], recv_prev, recv_next, lk, parity, plans[r]["first_rank"], plans[r]["last_rank"], st)
        got = np.concatenate([probs[r].lat.export_spinor(gout[r], probs[r].prec, parity) for r in range(nslab)])
        assert rel_l2(got, want) <= TOL[prec], (parity, nslab)
        scale = np.sqrt(np.mean(np.abs(want) ** 2))
        assert np.abs(got - want).max() <= 50 * TOL[prec] * scale
    for p in probs:
        p.close()


def test_interior_alone_is_dphi_with_open_time_boundary(hr):
    """hr_dphi_eo_interior = Dphi_eo with the hops across the slab boundary removed: equal to the oracle's operator
    minus its t-boundary terms, obtained from two oracle calls with bc_t = +1 and -1 (their mean kills the seam)."""
    dims = (4, 4, 4, 6)
    U = li.haar_links(321, 3, dims)
    psi = li.gaussian_spinor(322, li.volume(dims) // 2, 3)
    want = 0.5 * (oracle.dphi_eo(dims, (1, 1, 1, 1), U, 0, psi) + oracle.dphi_eo(dims, (-1, 1, 1, 1), U, 0, psi))
    prob = GpuProblem(hr, dims, 3, "fund", "f64", U)
    gin, out = prob.lat.spinor(prob.prec), prob.lat.spinor(prob.prec)
    prob.lat.import_spinor(gin, prob.prec, psi, 1)
    hr.hr_dphi_eo_interior(out, gin, prob.links, 0, prob.lat.stream())
    assert rel_l2(prob.lat.export_spinor(out, prob.prec, 0), want) <= TOL["f64"]
    prob.close()


def test_halo_argument_errors(hr):
    dims = (4, 4, 4, 4)
    U = li.haar_links(331, 3, dims)
    prob = GpuProblem(hr, dims, 3, "fund", "f64", U)
    a, b = _bufs(hr, prob, 2)
    s, o = prob.lat.spinor(prob.prec), prob.lat.spinor(prob.prec)
    assert hr.hr_halo_bytes(prob.lat.ctx, hr.HR_F64) == 4 * 4 * 2 * 4 * 3 * 8      # X Y Z/2 sites x 2 d_R complex
    with pytest.raises(hr.HrError):
        hr.hr_dphi_eo_halo_pack(a, a, s, prob.links, 0, 0)          # send buffers alias
    with pytest.raises(hr.HrError):
        hr.hr_dphi_eo_halo_pack(a, b, s, prob.links, 3, 0)          # parity
    with pytest.raises(hr.HrError):
        hr.hr_dphi_eo_interior(o, o, prob.links, 0, 0)              # out aliases in
    with pytest.raises(hr.HrError):
        hr.hr_dphi_eo_halo_apply(o, None, b, prob.links, 0, True, True, 0)
    prob.close()
