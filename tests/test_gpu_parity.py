"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on seeded
inputs at sizes the oracle finishes in seconds that still span several CTAs and a ragged tail.
Tolerances are BASELINE.json:north_star's: relative L2 <= 1e-13 (fp64), <= 2e-6 (fp32 vs the fp64
oracle on the unrounded inputs, reading C13); pure permutations and repeated launches are bit-exact."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from gpu_common import BC_T, COMBOS, TOL, GpuProblem, make_inputs, oracle_rep_id, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available()
    from paper_2405_19294_b200 import build
    build.build()
    import paper_2405_19294_b200 as hr
    return hr


# ---------------------------------------------------------------------------------------------
# a7 pack / unpack: pure permutation -> bit-exact round trip; a ragged number of sites per CTA
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", COMBOS)
def test_import_export_roundtrip_bit_exact(hr, N, rep, prec):
    dims = (4, 2, 6, 10)  # Vh = 240: not a multiple of the 128-thread CTA
    lat = hr.Lattice(dims, BC_T, N, rep)
    p = hr.PREC_NAMES[prec]
    cdt = np.complex128 if prec == "f64" else np.complex64
    U = li.haar_links(11, N, dims).astype(cdt)
    g = lat.gauge(False, p)
    lat.import_gauge(g, U)
    back = lat.export_gauge(g, False, p)
    assert back.dtype == cdt and np.array_equal(back, U)
    for parity in (0, 1):
        psi = li.gaussian_spinor(12 + parity, lat.vh, lat.d).astype(cdt)
        s = lat.spinor(p)
        lat.import_spinor(s, p, psi, parity)
        assert np.array_equal(lat.export_spinor(s, p, parity, p), psi)
    lat.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", COMBOS)
def test_represented_field_import_export_and_use(hr, N, rep, prec):
    """A REPRESENTED link field handed in by the caller (hr_gauge_import into a represented handle) instead of being made by
    hr_represent_links: bit-exact round trip of the canonical d_R x d_R records -- for the SU(4) adjoint the internal record
    has rows of d_R + 1 reals (include/hr.h, hr_gauge_bytes) and the canonical one does not -- and Dphi_eo on the imported
    field equals the oracle."""
    dims = (4, 2, 6, 10)
    lat = hr.Lattice(dims, BC_T, N, rep)
    p = hr.PREC_NAMES[prec]
    R64 = oracle.represent(N, oracle_rep_id(rep), li.haar_links(13, N, dims))
    if rep == "adj":
        R = np.ascontiguousarray(R64.real).astype(np.float64 if prec == "f64" else np.float32)
    else:
        R = R64.astype(np.complex128 if prec == "f64" else np.complex64)
    g = lat.gauge(True, p)
    w = 8 if prec == "f64" else 4
    ld = lat.d + 1 if (rep == "adj" and lat.d % 2 == 1 and lat.d > 8) else lat.d
    assert hr.hr_gauge_bytes(lat.ctx, 1, p) == li.volume(dims) * 4 * lat.d * ld * w * (1 if rep == "adj" else 2)
    lat.import_gauge(g, R)
    back = lat.export_gauge(g, True, p)
    assert back.dtype == R.dtype and back.shape == R.shape and np.array_equal(back, R)
    for parity in (0, 1):
        psi = li.gaussian_spinor(14 + parity, lat.vh, lat.d)
        inp, out = lat.spinor(p), lat.spinor(p)
        out.fill_(0xFF)
        lat.import_spinor(inp, p, psi, 1 - parity)
        lat.dphi_eo(out, inp, g, parity)
        assert rel_l2(lat.export_spinor(out, p, parity), oracle.dphi_eo(dims, BC_T, R64, parity, psi)) <= TOL[prec]
    lat.close()


def test_import_from_device_canonical_equals_import_from_host(hr):
    import torch
    dims = (4, 4, 4, 6)
    lat = hr.Lattice(dims, BC_T, 3, "fund")
    U = li.haar_links(5, 3, dims)
    g1, g2 = lat.gauge(False, hr.HR_F64), lat.gauge(False, hr.HR_F64)
    lat.import_gauge(g1, U)
    Ud = torch.from_numpy(U.view(np.float64)).cuda()
    hr.hr_gauge_import(g2, Ud, hr.HR_F64, lat.stream())
    torch.cuda.synchronize()
    assert np.array_equal(lat.export_gauge(g1, False), lat.export_gauge(g2, False))
    lat.close()


# ---------------------------------------------------------------------------------------------
# a2 link map
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", COMBOS)
def test_represent_links_matches_oracle(hr, N, rep, prec):
    dims = (4, 2, 6, 10)
    U = li.haar_links(21, N, dims)
    want = oracle.represent(N, oracle_rep_id(rep), U)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    got = prob.represented()
    if rep == "adj":
        assert got.dtype == np.float64 and got.shape == want.shape   # real d x d storage (reading C7)
        want = want.real
    assert rel_l2(got, want) <= TOL[prec]
    prob.close()


def test_represent_links_mixed_precision(hr):
    """fp64 fundamental -> fp32 represented: arithmetic in fp64, one rounding on store."""
    dims = (4, 4, 4, 4)
    U = li.haar_links(22, 3, dims)
    want = oracle.represent(3, oracle.REP_SYM, U)
    prob = GpuProblem(hr, dims, 3, "sym", "f32", U, fund_prec="f64")
    got = prob.represented()
    assert np.array_equal(got, want.astype(np.complex64).astype(np.complex128)) or rel_l2(got, want) <= 1e-7
    prob.close()


# ---------------------------------------------------------------------------------------------
# a3-a6 the hopping term
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("parity", [0, 1])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", COMBOS)
def test_dphi_eo_matches_oracle_all_representations(hr, N, rep, prec, parity):
    dims = (4, 6, 2, 10)  # four different extents, one of them 2 (double hop, reading C10); Vh = 240 ragged
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U, psi = make_inputs(dims, N, 31, 32 + parity, d)
    want = oracle.dphi_eo(dims, BC_T, oracle.represent(N, oracle_rep_id(rep), U), parity, psi)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    got = prob.dphi_eo(psi, parity)
    assert np.isfinite(got.view(np.float64)).all()
    assert rel_l2(got, want) <= TOL[prec]
    prob.close()


@pytest.mark.parametrize("dims,bc", [
    ((2, 2, 2, 2), BC_T),                 # every hop wraps onto the same neighbour
    ((2, 2, 2, 2), (-1, -1, -1, -1)),
    ((8, 4, 4, 6), (1, 1, 1, 1)),
    ((6, 4, 2, 8), (1, -1, 1, -1)),
    ((4, 4, 4, 2), BC_T),                 # Z/2 = 1: the z neighbour is always the same half index
    ((2, 8, 6, 4), (-1, 1, -1, 1)),
])
@pytest.mark.parametrize("parity", [0, 1])
def test_dphi_eo_boundaries_and_small_extents(hr, dims, bc, parity):
    U, psi = make_inputs(dims, 3, 41, 42, 3)
    want = oracle.dphi_eo(dims, bc, U, parity, psi)
    prob = GpuProblem(hr, dims, 3, "fund", "f64", U, bc=bc)
    assert rel_l2(prob.dphi_eo(psi, parity), want) <= TOL["f64"]
    prob.close()


@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(2, "fund"), (3, "fund"), (2, "adj"), (3, "sym"), (3, "adj"), (4, "sym"), (4, "adj")])
def test_every_kernel_variant_matches_oracle(hr, N, rep, prec, variant):
    dims = (4, 4, 6, 8)
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U, psi = make_inputs(dims, N, 51, 52, d)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    try:
        prob.lat.set_tuning("variant", variant)
    except hr.HrError:
        prob.close()
        pytest.skip(f"variant {variant} not compiled for d_R={d} {prec}")
    R = oracle.represent(N, oracle_rep_id(rep), U)
    for parity in (0, 1):
        want = oracle.dphi_eo(dims, BC_T, R, parity, psi)
        try:
            got = prob.dphi_eo(psi, parity)
        except hr.HrError as e:
            assert e.status == hr.HR_EUNSUPPORTED
            prob.close()
            pytest.skip(str(e))
        assert rel_l2(got, want) <= TOL[prec], (variant, parity)
    prob.close()


@pytest.mark.parametrize("xblock", [1, 2, 3, 6])
@pytest.mark.parametrize("variant", [0, 7])
def test_thread_order_xblock_does_not_change_the_result(hr, xblock, variant):
    """The [x/Xb][t][x%Xb][y][zh] thread order (L2 re-use of +-t neighbours) is only a permutation of
    which thread computes which site: bit-identical to the storage order Xb = X, and equal to the oracle."""
    dims = (4, 6, 4, 10)
    U, psi = make_inputs(dims, 3, 55, 56, 3)
    prob = GpuProblem(hr, dims, 3, "fund", "f64", U)
    prob.lat.set_tuning("variant", variant)
    prob.lat.set_tuning("xblock", 6)
    base = [prob.dphi_eo(psi, parity) for parity in (0, 1)]
    prob.lat.set_tuning("xblock", xblock)
    for parity in (0, 1):
        got = prob.dphi_eo(psi, parity)
        assert np.array_equal(got, base[parity])
        assert rel_l2(got, oracle.dphi_eo(dims, BC_T, U, parity, psi)) <= TOL["f64"]
    with pytest.raises(hr.HrError):
        prob.lat.set_tuning("xblock", 4)   # does not divide X = 6
    prob.close()


# config 1 (BASELINE.json:configs[0]): SU(2) fundamental, 4^4, fp64, full D with m0 = -0.5, both parities of Dphi_eo
def test_config1_su2_fund_4x4_dirac_and_both_parities(hr):
    dims = (4, 4, 4, 4)
    U = li.haar_links(1001, 2, dims)
    V = li.volume(dims)
    psi_eo = li.gaussian_spinor(2001, V, 2)       # [even half | odd half]
    prob = GpuProblem(hr, dims, 2, "fund", "f64", U)
    want = oracle.dirac(dims, BC_T, U, -0.5, psi_eo)
    got = prob.dirac(-0.5, psi_eo)
    assert rel_l2(got, want) <= TOL["f64"]
    for parity in (0, 1):
        psi_in = psi_eo[(1 - parity) * (V // 2):(2 - parity) * (V // 2)]
        want = oracle.dphi_eo(dims, BC_T, U, parity, psi_in)
        assert rel_l2(prob.dphi_eo(psi_in, parity), want) <= TOL["f64"]
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(3, "fund"), (2, "adj"), (3, "sym")])
def test_dirac_matches_oracle(hr, N, rep, prec):
    dims = (4, 4, 6, 8)
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(61, N, dims)
    psi_eo = li.gaussian_spinor(62, li.volume(dims), d)
    want = oracle.dirac(dims, BC_T, oracle.represent(N, oracle_rep_id(rep), U), 0.25, psi_eo)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    assert rel_l2(prob.dirac(0.25, psi_eo), want) <= TOL[prec]
    prob.close()


@pytest.mark.parametrize("N,rep,variant", [(3, "fund", -1), (3, "sym", 6), (4, "sym", -1), (4, "adj", -1)])
def test_repeated_launches_are_bitwise_identical(hr, N, rep, variant):
    """No atomics anywhere in the path: the result is deterministic (reading C15) -- the one-thread-per-site kernel and
    the colour-parallel kernel (its shared-memory exchange is ordered by barriers, not by arrival)."""
    dims = (8, 8, 8, 8)
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U, psi = make_inputs(dims, N, 71, 72, d)
    prob = GpuProblem(hr, dims, N, rep, "f64", U)
    prob.lat.set_tuning("variant", variant)
    a = prob.dphi_eo(psi, 0)
    for _ in range(3):
        assert np.array_equal(prob.dphi_eo(psi, 0), a)
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,N,rep", [((4, 4, 6, 8), 3, "fund"),      # T < 8: whole-field upload, one launch, download
                                        ((8, 4, 6, 8), 3, "fund"),      # 8 chunks of one time slice
                                        ((26, 2, 2, 4), 3, "fund"),     # chunks of 3 slices, a ragged last chunk of 2
                                        ((16, 2, 4, 2), 2, "adj"),      # real links
                                        ((10, 4, 2, 6), 3, "sym"),      # default kernel = colour: the chunks take the site kernel
                                        ((12, 2, 2, 4), 4, "adj")])
def test_host_entry_point_matches_oracle(hr, dims, N, rep, prec):
    """hr_dphi_eo_host: canonical host buffers in, canonical host buffers out (the e2e call of bench.py) -- from 8 time slices
    on a pipeline over chunks of slices (upload || pack, Dphi on the chunk's output slices, unpack || download), the chunks
    0 and C-1 last; every output site, both parities, antiperiodic t."""
    import torch
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(81, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    cdt = torch.complex128 if prec == "f64" else torch.complex64
    for parity in (0, 1):
        psi = li.gaussian_spinor(82 + parity, li.volume(dims) // 2, d)
        want = oracle.dphi_eo(dims, BC_T, R, parity, psi)
        inp = torch.from_numpy(psi).to(cdt).pin_memory()
        out = torch.full_like(inp, float("nan")).pin_memory()
        hr.hr_dphi_eo_host(prob.lat.ctx, out, inp, hr.PREC_NAMES[prec], prob.links, parity, prob.lat.stream())
        assert rel_l2(out.numpy(), want) <= TOL[prec]
        again = torch.full_like(inp, float("nan")).pin_memory()            # a second call re-uses the staging buffers and events
        hr.hr_dphi_eo_host(prob.lat.ctx, again, inp, hr.PREC_NAMES[prec], prob.links, parity, prob.lat.stream())
        assert torch.equal(out, again)
    prob.close()


@pytest.mark.parametrize("dims", [(4, 4, 6, 8), (12, 2, 4, 6)])
def test_host_entry_point_converts_the_canonical_precision(hr, dims):
    """hr_dphi_eo_host with fp32 canonical arrays on an fp64 field (and the other way round): the conversion happens in the
    pack / unpack kernels, whole-field and pipelined path alike; the error is the rounding of the fp32 side."""
    import torch
    U, psi = make_inputs(dims, 3, 85, 86, 3)
    want = oracle.dphi_eo(dims, BC_T, U, 0, psi)
    for prec, cdt in (("f64", torch.complex64), ("f32", torch.complex128)):
        prob = GpuProblem(hr, dims, 3, "fund", prec, U)
        inp = torch.from_numpy(psi).to(cdt).pin_memory()
        out = torch.full_like(inp, float("nan")).pin_memory()
        hr.hr_dphi_eo_host(prob.lat.ctx, out, inp, hr.HR_F32 if cdt == torch.complex64 else hr.HR_F64, prob.links, 0, prob.lat.stream())
        assert rel_l2(out.numpy(), want) <= TOL["f32"]
        prob.close()


def test_argument_errors_on_the_gpu(hr):
    dims = (4, 4, 4, 4)
    U, psi = make_inputs(dims, 3, 91, 92, 3)
    prob = GpuProblem(hr, dims, 3, "fund", "f64", U)
    s = prob.lat.spinor(hr.HR_F64)
    t = prob.lat.spinor(hr.HR_F64)
    with pytest.raises(hr.HrError) as e:
        hr.hr_dphi_eo(s, s, prob.links, 0, prob.lat.stream())            # out aliases in
    assert e.value.status == hr.HR_EINVAL
    with pytest.raises(hr.HrError) as e:
        hr.hr_dphi_eo(s, t, prob.links, 2, prob.lat.stream())            # parity not in {0,1}
    assert e.value.status == hr.HR_EINVAL
    U2 = li.haar_links(95, 2, dims)
    adj = GpuProblem(hr, dims, 2, "adj", "f64", U2)
    with pytest.raises(hr.HrError) as e:                                 # the adjoint needs its represented field
        hr.hr_dphi_eo(adj.lat.spinor(hr.HR_F64), adj.lat.spinor(hr.HR_F64), adj.fund, 0, adj.lat.stream())
    assert e.value.status == hr.HR_EINVAL
    adj.close()
    with pytest.raises(hr.HrError) as e:
        hr.hr_represent_links(prob.fund, prob.links, prob.lat.stream())  # swapped
    assert e.value.status == hr.HR_EINVAL
    prob.close()


def test_launch_counter_counts_our_kernels(hr):
    dims = (4, 4, 4, 4)
    U, psi = make_inputs(dims, 3, 93, 94, 3)
    prob = GpuProblem(hr, dims, 3, "fund", "f64", U)
    s, t = prob.lat.spinor(hr.HR_F64), prob.lat.spinor(hr.HR_F64)
    prob.lat.import_spinor(s, hr.HR_F64, psi, 1)
    n0 = hr.hr_launch_count()
    prob.lat.dphi_eo(t, s, prob.links, 0)
    assert hr.hr_launch_count() == n0 + 1        # hr_dphi_eo is ONE launch
    full_in, full_out = prob.lat.spinor(hr.HR_F64, full=True), prob.lat.spinor(hr.HR_F64, full=True)
    full_in.zero_()
    n0 = hr.hr_launch_count()
    prob.lat.dirac(0.1, full_out, full_in, prob.links)
    assert hr.hr_launch_count() == n0 + 2        # hr_dirac: one launch per output parity
    prob.close()


# ---------------------------------------------------------------------------------------------
# the colour-parallel kernel (variant 6): ragged CTA tails, boundary signs, mass term
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(3, "fund"), (2, "adj"), (3, "sym"), (3, "adj"), (4, "sym"), (4, "adj")])
@pytest.mark.parametrize("dims,bc", [((2, 2, 2, 2), BC_T), ((4, 6, 2, 10), (1, -1, 1, -1)), ((6, 2, 6, 6), (-1, -1, -1, -1))])
def test_colour_parallel_kernel_matches_oracle(hr, dims, bc, N, rep, prec):
    """Vh = 8, 240, 216: less than one CTA of 32 sites, and ragged tails; odd d_R in fp32 and real links exercise the
    unaligned element loads and the tail planes of the record layout."""
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(61, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    prob = GpuProblem(hr, dims, N, rep, prec, U, bc=bc)
    prob.lat.set_tuning("variant", 6)
    assert hr.hr_dphi_variant_name(prob.lat.ctx, prob.prec) == "colour"
    for parity in (0, 1):
        psi = li.gaussian_spinor(62 + parity, V // 2, d)
        assert rel_l2(prob.dphi_eo(psi, parity), oracle.dphi_eo(dims, bc, R, parity, psi)) <= TOL[prec], parity
    psi = li.gaussian_spinor(64, V, d)
    assert rel_l2(prob.dirac(-0.3, psi), oracle.dirac(dims, bc, R, -0.3, psi)) <= TOL[prec]
    prob.close()


def test_large_representations_default_to_the_colour_kernel(hr):
    for N, rep in ((4, "sym"), (4, "adj")):
        lat = hr.Lattice((4, 4, 4, 4), BC_T, N, rep)
        assert lat.d == (10 if rep == "sym" else 15)
        assert hr.hr_dphi_variant_name(lat.ctx, hr.HR_F64) == "colour" and hr.hr_dphi_variant_name(lat.ctx, hr.HR_F32) == "colour"
        with pytest.raises(hr.HrError):
            lat.set_tuning("variant", 2)            # no pair kernel at d_R > 8
        lat.close()
