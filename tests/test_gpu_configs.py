"""GPU parity at BASELINE.json's full sizes (configs[1..4]), in the launch configuration bench.py times
(default kernel variant and block size).  Configs 2-4 are compared with the oracle on EVERY output
site; config 5 (64^4, 8.4M output sites per parity) on the deterministic sample SURVEY.md section 8(d)
names -- all sites of the time-slices t in {0, 1, T/2, T-1} plus 2^20 seeded random sites -- and via a
property that holds at any size (gamma5-hermiticity evaluated from the GPU's own outputs).
Inputs: the seeded recipes of DESIGN.md "Input recipe" (seeds 100k / 200k as in SURVEY.md section 8(d))."""
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


_cache = {}


def inputs(tag, dims, N, d, seed_l, seed_s, kind="haar"):
    if tag not in _cache:
        _cache.clear()  # one config's fields at a time (config 5 fp64 links are 9 GiB)
        U = li.haar_links(seed_l, N, dims) if kind == "haar" else li.near_identity_links(seed_l, N, dims, 0.3)
        psi = [li.gaussian_spinor(seed_s + 10 * p, li.volume(dims) // 2, d) for p in (0, 1)]
        _cache[tag] = (U, psi)
    return _cache[tag]


def check_full(hr, dims, N, rep, prec, U, psi, check_links=False):
    R = oracle.represent(N, oracle_rep_id(rep), U)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    if check_links:
        got = prob.represented()
        assert rel_l2(got, R.real if rep == "adj" else R) <= TOL[prec]
    for parity in (0, 1):
        want = oracle.dphi_eo(dims, BC_T, R, parity, psi[parity])
        got = prob.dphi_eo(psi[parity], parity)
        assert rel_l2(got, want) <= TOL[prec], (prec, parity)
        # element-wise as well: no single site may be off while the norm hides it
        scale = np.sqrt(np.mean(np.abs(want) ** 2))
        assert np.abs(got - want).max() <= 50 * TOL[prec] * scale
    prob.close()


# configs[1]: SU(3) fundamental, 32^3 x 64, fp64 and fp32, Haar links, parity 0 and 1
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_config2_su3_fund_32x32x32x64(hr, prec):
    dims = (64, 32, 32, 32)
    U, psi = inputs("cfg2", dims, 3, 3, 1002, 2002)
    check_full(hr, dims, 3, "fund", prec, U, psi)


# configs[2]: SU(2) adjoint (real d_R = 3 links computed from the fundamental ones), 32^4, fp64
def test_config3_su2_adjoint_32x32x32x32(hr):
    dims = (32, 32, 32, 32)
    U, psi = inputs("cfg3", dims, 2, 3, 1003, 2003)
    check_full(hr, dims, 2, "adj", "f64", U, psi, check_links=True)


# configs[3]: SU(3) two-index symmetric (d_R = 6), 24^3 x 48, fp64 and fp32
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_config4_su3_sextet_24x24x24x48(hr, prec):
    dims = (48, 24, 24, 24)
    U, psi = inputs("cfg4", dims, 3, 6, 1004, 2004)
    check_full(hr, dims, 3, "sym", prec, U, psi, check_links=True)


# the large representations at the sizes bench_large_n times (the paper's Fig. 6 experiment), default
# kernel = colour-parallel or, for d_R = 8 in fp32, bulk2: every output site against the oracle
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep,dims", [(3, "adj", (48, 24, 24, 24)), (4, "sym", (56, 16, 16, 16)), (4, "adj", (48, 16, 16, 16))])
def test_large_representations_at_the_benchmarked_sizes(hr, N, rep, dims, prec):
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U, psi = inputs(f"large{N}{rep}", dims, N, d, 1006, 2006)
    import paper_2405_19294_b200 as lib
    lat = lib.Lattice(dims, BC_T, N, rep)
    # fp32 SU(3) adjoint on 24^3 x 48: the TMA-staged two-threads-per-site kernel since round 2 (tiles of 8 rows x 12 sites)
    want_kernel = "colour" if (prec == "f64" or d > 8) else "bulk2"
    assert lib.hr_dphi_variant_name(lat.ctx, lib.PREC_NAMES[prec]) == want_kernel
    lat.close()
    check_full(hr, dims, N, rep, prec, U, psi, check_links=True)


# configs[4]: SU(3) fundamental, 64^4, fp32 and fp64, near-identity links exp(0.3 i H)
def _sample_half_indices(dims, seed):
    T, X, Y, Z = dims
    per_t = X * Y * Z // 2
    slabs = [np.arange(t * per_t, (t + 1) * per_t, dtype=np.int64) for t in (0, 1, T // 2, T - 1)]
    rng = np.random.Generator(np.random.Philox(seed))
    rand = rng.integers(0, T * per_t, size=1 << 20, dtype=np.int64)
    return np.unique(np.concatenate(slabs + [rand]))


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_config5_su3_fund_64x64x64x64_sampled(hr, prec):
    import psutil
    dims = (64, 64, 64, 64)
    need = 22 << 30
    assert psutil.virtual_memory().available > need, "host needs ~22 GiB for the canonical 64^4 fp64 fields"
    U, psi = inputs("cfg5", dims, 3, 3, 1005, 2005, kind="near")
    prob = GpuProblem(hr, dims, 3, "fund", prec, U)
    hidx = _sample_half_indices(dims, 3005)
    outs = []
    for parity in (0, 1):
        got = prob.dphi_eo(psi[parity], parity)
        outs.append(got)
        want = oracle.dphi_eo_sites(dims, BC_T, U, parity, psi[parity], hidx)
        assert rel_l2(got[hidx], want) <= TOL[prec], (prec, parity)
        scale = np.sqrt(np.mean(np.abs(want) ** 2))
        assert np.abs(got[hidx] - want).max() <= 50 * TOL[prec] * scale
    # gamma5-hermiticity at full volume from the GPU's own outputs (BASELINE.json:north_star):
    #   <phi_e, Dphi_eo psi_o> = <gamma5 Dphi_oe gamma5 phi_e, psi_o>,  gamma5 = diag(1,1,-1,-1) (reading C1)
    # here: out0 = Dphi_eo(parity 0) psi[0] (psi[0] lives on odd sites), out1 = Dphi_eo(parity 1) psi[1] (even sites).
    g5 = np.array([1, 1, -1, -1], dtype=np.float64)[None, :, None]
    phi_e, psi_o = psi[1], psi[0]
    lhs = np.vdot(phi_e, outs[0])                       # <phi_e, D_eo psi_o>
    g5phi = phi_e * g5
    d_oe_g5phi = prob.dphi_eo(g5phi, 1)                 # D_oe gamma5 phi_e (output on odd sites)
    rhs = np.vdot(d_oe_g5phi * g5, psi_o)
    nrm = np.linalg.norm(phi_e) * np.linalg.norm(outs[0])
    assert abs(lhs - rhs) / nrm <= (1e-13 if prec == "f64" else 1e-6)
    prob.close()
