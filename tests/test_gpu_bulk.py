"""GPU parity of kernel variant 7 `bulk` (csrc/dphi_bulk_kernel.cuh): persistent CTAs, the operands of every hop staged in
shared memory by TMA bulk copies behind an mbarrier ring (north_star: "TMA or shared-memory staging of neighbour spinors
along the fastest lattice direction").  Same operator, so the oracle is unchanged; tolerances BASELINE.json:north_star.
What can go wrong that the site kernel cannot get wrong: tile geometry (rows per tile, ragged consumer warps, tiles that
touch the y boundary -> two runs per plane), the ring (depth, phase wrap across tiles and across launches), tail planes of
records that are no multiple of 16 bytes, CTAs per SM, more tiles than CTAs and fewer."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle import solver
from gpu_common import BC_T, TOL, GpuProblem, oracle_rep_id, rel_l2

pytestmark = pytest.mark.gpu
BULK = 7


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


def _bulk_or_skip(hr, prob, links, gin, parity):
    """One launch of the bulk kernel; skips when this lattice cannot be tiled (tail planes need 16-byte runs)."""
    out = _new(prob)
    try:
        prob.lat.dphi_eo(out, gin, links, parity)
    except hr.HrError as e:
        assert e.status == hr.HR_EUNSUPPORTED
        return None
    return prob.lat.export_spinor(out, prob.prec, parity)


# every representation the kernel is compiled for, lattices with Zh = 1 ... 16 (one tile per CTA and many), all four
# boundary patterns in turn
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(2, "fund"), (3, "fund"), (4, "fund"), (2, "adj"), (2, "sym"), (3, "sym"), (3, "asym"), (3, "adj"), (4, "asym")])
@pytest.mark.parametrize("dims,bc", [((4, 4, 6, 8), BC_T), ((2, 2, 2, 2), (-1, -1, -1, -1)), ((6, 2, 4, 12), (1, -1, 1, -1)),
                                     ((4, 6, 8, 32), (1, 1, -1, 1)), ((2, 4, 2, 4), (-1, 1, 1, -1))])
@pytest.mark.parametrize("variant", [7, 8, 9, 10])
def test_bulk_kernel_matches_oracle(hr, dims, bc, N, rep, prec, variant):
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(701, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    vh = li.volume(dims) // 2
    prob = GpuProblem(hr, dims, N, rep, prec, U, bc=bc)
    try:
        prob.lat.set_tuning("variant", variant)
    except hr.HrError:
        prob.close()
        pytest.skip("this variant is not compiled for this d_R / precision")
    assert hr.hr_dphi_variant_name(prob.lat.ctx, prob.prec) == {7: "bulk", 8: "bulk2", 9: "bulkx", 10: "bulkx2"}[variant]
    ran = 0
    for parity in (0, 1):
        psi = li.gaussian_spinor(702 + parity, vh, d)
        want = oracle.dphi_eo(dims, bc, R, parity, psi)
        got = _bulk_or_skip(hr, prob, prob.links, _put(prob, psi, 1 - parity), parity)
        if got is None:
            continue
        ran += 1
        assert np.isfinite(got.view(np.float64 if got.dtype == np.complex128 else np.float32)).all()
        assert rel_l2(got, want) <= TOL[prec], parity
    prob.close()
    if not ran:
        pytest.skip("tail planes of this record cannot be aligned on this lattice")


# tile geometry and ring: rows per tile, stages, CTAs per SM -- the result may not depend on any of them (bitwise)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_bulk_tile_and_ring_geometry_do_not_change_the_result(hr, prec):
    dims, N, rep = (6, 4, 12, 8), 3, "fund"
    U = li.haar_links(711, N, dims)
    vh = li.volume(dims) // 2
    psi = li.gaussian_spinor(712, vh, 3)
    want = oracle.dphi_eo(dims, BC_T, U, 1, psi)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    prob.lat.set_tuning("variant", BULK)
    gin = _put(prob, psi, 0)
    ref = None
    for rows in (0, 1, 2, 3, 4, 6, 12):
        for stages in (0, 2, 3, 5):
            for ctas in (0, 1, 2, 4):
                prob.lat.set_tuning("bulk_rows", rows)
                prob.lat.set_tuning("bulk_stages", stages)
                prob.lat.set_tuning("bulk_ctas", ctas)
                out = _new(prob)
                prob.lat.dphi_eo(out, gin, prob.links, 1)
                got = prob.lat.export_spinor(out, prob.prec, 1)
                assert rel_l2(got, want) <= TOL[prec], (rows, stages, ctas)
                if ref is None:
                    ref = got
                assert np.array_equal(got.view(np.uint8), ref.view(np.uint8)), (rows, stages, ctas)
    prob.close()


@pytest.mark.parametrize("variant", [9, 10])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_bulkx_strip_and_tile_geometry_do_not_change_the_result(hr, prec, variant):
    """bulkx: rows per tile, tiles per strip and the x-block of the strip order are scheduling only (bitwise)."""
    dims, N, rep = (4, 12, 8, 8), 3, "fund"
    U = li.haar_links(713, N, dims)
    vh = li.volume(dims) // 2
    psi = li.gaussian_spinor(714, vh, 3)
    want = oracle.dphi_eo(dims, (-1, -1, 1, -1), U, 0, psi)
    prob = GpuProblem(hr, dims, N, rep, prec, U, bc=(-1, -1, 1, -1))
    try:
        prob.lat.set_tuning("variant", variant)
    except hr.HrError:
        prob.close()
        pytest.skip("bulkx2 needs vector-aligned spin components")
    gin = _put(prob, psi, 1)
    if _bulk_or_skip(hr, prob, prob.links, gin, 0) is None:
        prob.close()
        pytest.skip("bulkx2 needs vector-aligned spin components (fp32: even d_R)")
    ref = None
    for xblock in (0, 12, 6, 4, 1):
        for strip in (0, 1, 2, 3, 4, 6, 12):
            for rows in (0, 1, 2, 4, 8):
                prob.lat.set_tuning("xblock", xblock)
                prob.lat.set_tuning("bulk_strip", strip)
                prob.lat.set_tuning("bulk_rows", rows)
                out = _new(prob)
                prob.lat.dphi_eo(out, gin, prob.links, 0)
                got = prob.lat.export_spinor(out, prob.prec, 0)
                assert rel_l2(got, want) <= TOL[prec], (xblock, strip, rows)
                if ref is None:
                    ref = got
                assert np.array_equal(got.view(np.uint8), ref.view(np.uint8)), (xblock, strip, rows)
    prob.close()


# many launches back to back on one stream: the ring's phase bits start afresh in every launch; repeated = bitwise equal
def test_bulk_repeated_launches_are_bitwise_identical(hr):
    dims, N = (8, 8, 8, 16), 3
    U = li.haar_links(721, N, dims)
    vh = li.volume(dims) // 2
    prob = GpuProblem(hr, dims, N, "fund", "f64", U)
    prob.lat.set_tuning("variant", BULK)
    psi = li.gaussian_spinor(722, vh, 3)
    gin = _put(prob, psi, 1)
    outs = []
    for k in range(6):
        out = _new(prob)
        prob.lat.dphi_eo(out, gin, prob.links, 0)
        outs.append(prob.lat.export_spinor(out, prob.prec, 0))
    for o in outs[1:]:
        assert np.array_equal(o.view(np.uint8), outs[0].view(np.uint8))
    assert rel_l2(outs[0], oracle.dphi_eo(dims, BC_T, U, 0, psi)) <= TOL["f64"]
    prob.close()


# fundamental links applied on the fly (two-index, SU(3) adjoint) and row-compressed links through the bulk kernel
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep,src", [(3, "sym", "fund"), (2, "sym", "fund"), (3, "asym", "fund"), (4, "asym", "fund"), (3, "adj", "fund"),
                                       (3, "fund", "rows"), (2, "fund", "rows"), (2, "adj", "rows"), (3, "adj", "rows")])
@pytest.mark.parametrize("variant", [7, 8, 9, 10])
def test_bulk_kernel_with_on_the_fly_and_row_compressed_links(hr, N, rep, src, prec, variant):
    dims = (4, 4, 6, 8)
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(731, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    vh = li.volume(dims) // 2
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    if src == "rows":
        links = prob.lat.gauge(2, prob.prec)
        prob.lat.compress_links(links, prob.fund)
    else:
        links = prob.fund
    try:
        prob.lat.set_tuning("variant", variant)
    except hr.HrError:
        prob.close()
        pytest.skip("bulk2 is not compiled for this representation")
    for parity in (0, 1):
        psi = li.gaussian_spinor(732 + parity, vh, d)
        want = oracle.dphi_eo(dims, BC_T, R, parity, psi)
        got = _bulk_or_skip(hr, prob, links, _put(prob, psi, 1 - parity), parity)
        if got is None and variant != 7:
            prob.close()
            pytest.skip("this variant is not compiled for this link kind / precision")
        assert got is not None
        assert rel_l2(got, want) <= TOL[prec], parity
    prob.close()


# the epilogues: hr_dirac (self term), hr_dhat with and without gamma5, the CG (fused reduction + skip flag)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep,variant", [(3, "fund", 7), (2, "adj", 7), (3, "sym", 7), (3, "sym", 8), (3, "fund", 9), (3, "fund", 10), (2, "adj", 9), (2, "fund", 10)])
def test_bulk_kernel_dirac_dhat_and_cg(hr, N, rep, prec, variant):
    dims, m0 = (4, 4, 4, 8), -0.3
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(741, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    vh = V // 2
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    prob.lat.set_tuning("variant", variant)
    if variant in (8, 10) and prec == "f32" and d % 2:
        prob.close()
        pytest.skip("two consumer threads per site need vector-aligned spin components (fp32: even d_R)")
    psi = li.gaussian_spinor(742, V, d)
    got = prob.dirac(m0, psi)
    assert rel_l2(got, oracle.dirac(dims, BC_T, R, m0, psi)) <= TOL[prec]
    b = li.gaussian_spinor(743, vh, d)
    gb, tmp = _put(prob, b, 0), _new(prob)
    for g5 in (0, 1):
        out = _new(prob)
        prob.lat.dhat(m0, bool(g5), out, gb, tmp, prob.links)
        want = solver.dhat(dims, BC_T, R, m0, b)
        if g5:
            want = solver.g5(want)
        assert rel_l2(prob.lat.export_spinor(out, prob.prec, 0), want) <= TOL[prec], g5
    # CG on Dhat^dag Dhat with the device-resident scalars (RED epilogue, skip flag)
    tol = 1e-9 if prec == "f64" else 1e-5
    x = _new(prob)
    ws = prob.lat.cg_workspace(prob.prec, 500)
    iters, res2, hist = prob.lat.cg_dhat(0.2, x, gb, prob.links, tol, 500, ws, want_hist=True)
    xo, ko, ho = solver.cg_dhat(dims, BC_T, R, 0.2, b, tol, 500)
    assert abs(iters - ko) <= 1
    assert rel_l2(prob.lat.export_spinor(x, prob.prec, 0), xo) <= (1e-7 if prec == "f64" else 1e-3)
    prob.close()
