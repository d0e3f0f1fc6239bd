"""hr_spinor_dot_noalloc (include/hr.h, csrc/dot_noalloc.cu): the allocation-free inner product -- its scratch is a static
device array of libhr.so -- against the existing hr_spinor_dot on the same device fields, on two calls in a row.

Collected last on purpose (the suite runs with `pytest -x`): a failure here must not hide another test."""
import numpy as np
import pytest

import lattice_inputs as li

pytestmark = pytest.mark.gpu

BC_T = (-1, 1, 1, 1)
# relative to |x| |y|, as tests/test_gpu_solver.py::test_reductions_match_oracle_and_are_deterministic: sums are fp64 on both
# paths; fp32 fields carry products rounded to 2^-24
RTOL = {"f64": 1e-13, "f32": 2e-6}
REP_DIM = {"fund": lambda N: N, "adj": lambda N: N * N - 1, "sym": lambda N: N * (N + 1) // 2}
# one CTA with a ragged tail; several CTAs; more vectors than the 1184-CTA grid covers in one stride
CASES = [((4, 2, 6, 2), 2, "fund"), ((6, 4, 2, 10), 2, "adj"), ((16, 16, 16, 16), 3, "fund"), ((24, 24, 24, 24), 3, "fund")]


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available()
    from paper_2405_19294_b200 import build
    build.build()
    import paper_2405_19294_b200 as hr
    return hr


def _device_pair(torch, res):
    torch.cuda.synchronize()
    return complex(res[0].item(), res[1].item())


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,N,rep", CASES)
def test_noalloc_dot_matches_the_existing_path_on_two_calls_in_a_row(hr, dims, N, rep, prec):
    import torch
    d = REP_DIM[rep](N)
    vh = li.volume(dims) // 2
    a, b = li.gaussian_spinor(903, vh, d), li.gaussian_spinor(904, vh, d)
    lat = hr.Lattice(dims, BC_T, N, rep)
    P, st = hr.PREC_NAMES[prec], lat.stream()
    ga, gb = lat.spinor(P), lat.spinor(P)
    lat.import_spinor(ga, P, a, 0)
    lat.import_spinor(gb, P, b, 0)
    assert hr.hr_spinor_bytes(lat.ctx, P) <= hr.hr_spinor_dot_noalloc_max_bytes()

    # the existing path (context scratch), device-result form
    ref = torch.zeros(2, dtype=torch.float64, device="cuda")
    want = []
    for x, y in ((ga, gb), (gb, ga), (ga, ga)):
        hr.hr_spinor_dot(lat.ctx, P, x, y, st, result=ref)
        want.append(_device_pair(torch, ref))
    na = float(np.sqrt(want[2].real))
    hr.hr_spinor_dot(lat.ctx, P, gb, gb, st, result=ref)
    nb = float(np.sqrt(_device_pair(torch, ref).real))
    assert na > 0 and nb > 0

    # the allocation-free path: three calls back to back on one stream, no synchronisation in between, each into its own
    # poisoned result -- the second and third run on a scratch that still holds the previous call's partial sums
    res = torch.full((3, 2), float("nan"), dtype=torch.float64, device="cuda")
    hr.hr_spinor_dot_noalloc(lat.ctx, P, ga, gb, res[0], st)
    hr.hr_spinor_dot_noalloc(lat.ctx, P, gb, ga, res[1], st)
    hr.hr_spinor_dot_noalloc(lat.ctx, P, ga, ga, res[2], st)
    torch.cuda.synchronize()
    got = [complex(res[k, 0].item(), res[k, 1].item()) for k in range(3)]
    tol = RTOL[prec]
    assert abs(got[0] - want[0]) <= tol * na * nb
    assert abs(got[1] - want[1]) <= tol * na * nb
    assert abs(got[1] - got[0].conjugate()) <= tol * na * nb          # <b, a> = conj <a, b>: not a stale copy of call 1
    assert got[2].imag == 0.0 and abs(got[2].real - want[2].real) <= tol * na * na
    # and once more after the existing path has run in between (the two paths share nothing)
    hr.hr_spinor_dot(lat.ctx, P, gb, ga, st, result=ref)
    again = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    hr.hr_spinor_dot_noalloc(lat.ctx, P, ga, gb, again, st)
    assert abs(_device_pair(torch, again) - want[0]) <= tol * na * nb
    lat.close()


def test_noalloc_dot_rejects_what_it_cannot_do(hr):
    import torch
    # a half field beyond the stated maximum: 128^4 SU(4) adjoint fp64 = 2^27 sites x 960 bytes; nothing is allocated or launched
    big = hr.Lattice((128, 128, 128, 128), BC_T, 4, "adj")
    assert hr.hr_spinor_bytes(big.ctx, hr.HR_F64) > hr.hr_spinor_dot_noalloc_max_bytes()
    dummy = torch.zeros(4, dtype=torch.float64, device="cuda")
    with pytest.raises(hr.HrError, match="exceeds the limit"):
        hr.hr_spinor_dot_noalloc(big.ctx, hr.HR_F64, dummy, dummy, dummy, 0)
    big.close()
    # a host result pointer: the call never synchronises, so it refuses
    lat = hr.Lattice((4, 4, 4, 4), BC_T, 2, "fund")
    x = lat.spinor(hr.HR_F64)
    x.zero_()
    host = np.zeros(2)
    with pytest.raises(hr.HrError, match="device memory"):
        hr.hr_spinor_dot_noalloc(lat.ctx, hr.HR_F64, x, x, host, 0)
    with pytest.raises(hr.HrError):
        hr.hr_spinor_dot_noalloc(lat.ctx, hr.HR_F64, x, None, dummy, 0)
    lat.close()
