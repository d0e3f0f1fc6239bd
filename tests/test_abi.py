"""The C-ABI library loads and exports every symbol include/hr.h declares; host-side argument logic
(no compute calls, no GPU needed).  CPU only."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "hr.h")


@pytest.fixture(scope="module")
def hr():
    from paper_2405_19294_b200 import build
    build.build()
    import paper_2405_19294_b200 as hr
    return hr


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hr_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_all_exported(hr):
    names = declared_symbols()
    assert {"hr_gauge_alloc", "hr_represent_links", "hr_dphi_eo", "hr_dirac"} <= set(names)  # north_star's four
    lib = ctypes.CDLL(hr.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in hr.h but not exported by libhr.so"
    # and the binding wraps every one of them under the same name
    for n in names:
        assert hasattr(hr, n), f"python binding lacks {n}"
    assert set(hr._SIGNATURES) == set(names)


def test_version_string(hr):
    assert "sm_100a" in hr.hr_version()


@pytest.mark.parametrize("N,rep,d,real", [
    (2, "fund", 2, 0), (2, "adj", 3, 1), (2, "sym", 3, 0),
    (3, "fund", 3, 0), (3, "adj", 8, 1), (3, "sym", 6, 0), (3, "asym", 3, 0),
    (4, "fund", 4, 0), (4, "asym", 6, 0), (4, "sym", 10, 0), (4, "adj", 15, 1)])
def test_ctx_geometry_and_sizes(hr, N, rep, d, real):
    dims = (4, 2, 6, 8)
    ctx = hr.hr_ctx_create(dims, (-1, 1, 1, 1), N, hr.REP_NAMES[rep], 0)
    try:
        V = 4 * 2 * 6 * 8
        assert hr.hr_rep_dim(ctx) == d
        assert hr.hr_links_are_real(ctx) == real
        assert hr.hr_half_volume(ctx) == V // 2
        for prec, w in ((hr.HR_F64, 8), (hr.HR_F32, 4)):
            assert hr.hr_spinor_bytes(ctx, prec) == (V // 2) * 4 * d * 2 * w          # S = 4 d_R complex per site
            assert hr.hr_gauge_bytes(ctx, 0, prec) == V * 4 * N * N * 2 * w            # F = N^2 complex
            ld = d + 1 if (real and d % 2 == 1 and d > 8) else d                        # SU(4) adjoint: internal rows of 16 reals
            L = d * ld * w * (1 if real else 2)                                        # real adjoint: half the bytes (C7)
            assert hr.hr_gauge_bytes(ctx, 1, prec) == V * 4 * L
    finally:
        hr.hr_ctx_destroy(ctx)


@pytest.mark.parametrize("dims,bc,N,rep,status", [
    ((4, 4, 4, 3), (1, 1, 1, 1), 3, 0, -1),     # odd extent (reading C11)
    ((4, 4, 0, 4), (1, 1, 1, 1), 3, 0, -1),
    ((4, 4, 4, 4), (1, 1, 2, 1), 3, 0, -1),     # bc not +-1
    ((4, 4, 4, 4), (1, 1, 1, 1), 3, 7, -1),     # unknown rep
    ((4, 4, 4, 4), (1, 1, 1, 1), 2, 3, -2),     # SU(2) antisymmetric: d_R = 1, not instantiated
    ((4, 4, 4, 4), (1, 1, 1, 1), 5, 0, -2),     # SU(5) not instantiated
    ((4, 4, 4, 4), (1, 1, 1, 1), 6, 2, -2),     # SU(6) symmetric (d_R = 21) not instantiated
])
def test_ctx_create_rejects_bad_arguments(hr, dims, bc, N, rep, status):
    with pytest.raises(hr.HrError) as e:
        hr.hr_ctx_create(dims, bc, N, rep, 0)
    assert e.value.status == status
    assert hr.hr_last_error() != ""


@pytest.mark.parametrize("dims,N,rep,f64,f32", [
    ((64, 64, 64, 64), 3, "fund", "site", "site"),          # config 5
    ((64, 32, 32, 32), 3, "fund", "bulk", "site"),          # config 2: Z <= 32
    ((32, 32, 32, 32), 2, "adj", "bulk", "site_ef"),        # config 3
    ((48, 24, 24, 24), 3, "sym", "colour", "bulk2"),        # config 4: bulk2's tile is 8 rows x 12 sites
    ((32, 32, 32, 32), 3, "sym", "colour", "bulk"),         # Zh = 16: bulk2's tile would have 64 sites -> bulk
    ((48, 24, 24, 24), 3, "adj", "colour", "bulk2"),
    ((32, 32, 32, 32), 3, "adj", "colour", "bulk"),
    ((40, 32, 32, 32), 4, "fund", "bulk", "site"),
    ((16, 32, 64, 64), 4, "fund", "site", "site"),          # Z = 64: the site kernel stays
    ((56, 16, 16, 16), 4, "sym", "colour", "colour"),
    ((48, 16, 16, 16), 4, "adj", "colour", "colour"),
    ((8, 8, 8, 8), 3, "sym", "colour", "site_ef"),          # below 2^17 sites per parity: no persistent kernel
    ((4, 4, 4, 4), 3, "fund", "site", "site")])
def test_default_kernel_table(hr, dims, N, rep, f64, f32):
    """The measured default kernel per (d_R, link type, precision, lattice shape): DESIGN.md "Kernels", profiles/r2_staging.md."""
    ctx = hr.hr_ctx_create(dims, (-1, 1, 1, 1), N, hr.REP_NAMES[rep], 0)
    try:
        assert hr.hr_dphi_variant_name(ctx, hr.HR_F64) == f64
        assert hr.hr_dphi_variant_name(ctx, hr.HR_F32) == f32
    finally:
        hr.hr_ctx_destroy(ctx)


def test_tuning_keys_validated(hr):
    ctx = hr.hr_ctx_create((4, 4, 4, 4), (-1, 1, 1, 1), 3, hr.HR_REP_FUND, 0)
    try:
        hr.hr_ctx_set_tuning(ctx, "variant", 0)
        hr.hr_ctx_set_tuning(ctx, "variant", -1)
        hr.hr_ctx_set_tuning(ctx, "block", 64)
        for key, val in (("variant", 99), ("block", 33), ("nonsense", 1)):
            with pytest.raises(hr.HrError):
                hr.hr_ctx_set_tuning(ctx, key, val)
        assert hr.hr_dphi_variant_name(ctx, hr.HR_F64) != "?"
    finally:
        hr.hr_ctx_destroy(ctx)


def test_compute_calls_check_arguments_before_touching_the_gpu(hr):
    # NULL handles are rejected with HR_EINVAL whether or not a device exists
    with pytest.raises(hr.HrError) as e:
        hr.hr_dphi_eo(16, 32, 0, 0, 0)
    assert e.value.status == hr.HR_EINVAL
    with pytest.raises(hr.HrError) as e:
        hr.hr_represent_links(0, 0, 0)
    assert e.value.status == hr.HR_EINVAL


def test_no_cpu_fallback_without_a_device(hr):
    """On a box without CUDA the product path fails loudly (HR_ECUDA); it never computes on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    ctx = hr.hr_ctx_create((4, 4, 4, 4), (-1, 1, 1, 1), 3, hr.HR_REP_FUND, 0)
    try:
        with pytest.raises(hr.HrError) as e:
            hr.hr_gauge_alloc(ctx, 1, hr.HR_F64, None)
        assert e.value.status in (hr.HR_ECUDA, hr.HR_ENOMEM)
    finally:
        hr.hr_ctx_destroy(ctx)
