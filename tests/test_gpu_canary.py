"""Out-of-bounds WRITE guard for every call that writes a caller buffer (compute-sanitizer is not available on the
GPU pool): each output sits between two 4 KiB canary zones inside one allocation; after the call every canary byte
must be intact.  Lattices are chosen with ragged CTA tails (V/2 not a multiple of 128)."""
import numpy as np
import pytest

import lattice_inputs as li
from gpu_common import GpuProblem

pytestmark = pytest.mark.gpu
PAD = 4096


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available()
    from paper_2405_19294_b200 import build
    build.build()
    import paper_2405_19294_b200 as hr
    return hr


class Guarded:
    def __init__(self, nbytes):
        import torch
        self.buf = torch.empty(nbytes + 2 * PAD, dtype=torch.uint8, device="cuda")
        self.buf.fill_(0xA5)
        self.t = self.buf[PAD:PAD + nbytes]

    def intact(self):
        import torch
        torch.cuda.synchronize()
        return bool((self.buf[:PAD] == 0xA5).all().item()) and bool((self.buf[-PAD:] == 0xA5).all().item())


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(3, "fund"), (2, "adj"), (3, "sym"), (3, "adj"), (4, "fund"), (4, "adj")])
def test_no_call_writes_outside_its_output(hr, N, rep, prec):
    dims = (6, 2, 6, 10)                       # V/2 = 360: 2 full CTAs + a ragged tail of 104 sites
    U = li.haar_links(501, N, dims)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    lat, P = prob.lat, prob.prec
    ctx, st = lat.ctx, lat.stream()
    d = lat.d
    sb = hr.hr_spinor_bytes(ctx, P)
    psi = li.gaussian_spinor(502, lat.vh, d)
    gin = lat.spinor(P)
    lat.import_spinor(gin, P, psi, 1)
    full_in = lat.spinor(P, full=True)
    full_in.zero_()
    checks = []

    def guarded(n):
        g = Guarded(n)
        checks.append(g)
        return g

    for variant in (0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11):
        try:
            lat.set_tuning("variant", variant)
            o = guarded(sb)
            lat.dphi_eo(o.t, gin, prob.links, 0)
        except hr.HrError:
            continue
    lat.set_tuning("variant", -1)
    o = guarded(2 * sb); lat.dirac(0.1, o.t, full_in, prob.links)
    o = guarded(sb); tmp = guarded(sb); lat.dhat(0.1, True, o.t, gin, tmp.t, prob.links)
    o = guarded(sb); hr.hr_spinor_lincomb(ctx, P, o.t, 1 + 2j, 1, gin, 0.5j, gin, st)
    o = guarded(sb); hr.hr_spinor_copy(ctx, P, o.t, gin, st)
    ws = guarded(hr.hr_cg_workspace_bytes(ctx, P, 20)); x = guarded(sb)
    # the workspace must be 256-byte aligned: PAD is a multiple of 256 and torch allocations are 512-byte aligned
    hr.hr_cg_dhat(ctx, 0.2, x.t, gin, prob.links, 1e-6, 20, ws.t, st)
    xs = guarded(2 * sb); hr.hr_dirac_solve(ctx, 0.2, xs.t, full_in, prob.links, 1e-6, 20, ws.t, st)
    hb = hr.hr_halo_bytes(ctx, P)
    up, dn = guarded(hb), guarded(hb)
    hr.hr_dphi_eo_halo_pack(up.t, dn.t, gin, prob.links, 0, st)
    o = guarded(sb); hr.hr_dphi_eo_interior(o.t, gin, prob.links, 0, st)
    hr.hr_dphi_eo_halo_apply(o.t, up.t, dn.t, prob.links, 0, True, True, st)
    if d <= 8:                                  # the clover kernels stop at d_R = 8
        cl = guarded(hr.hr_clover_bytes(ctx, P)); hr.hr_clover_build(cl.t, prob.links, 1.0, st)
        o = guarded(2 * sb); hr.hr_dirac_clover(0.1, o.t, full_in, prob.links, cl.t, st)
        hr.hr_clover_exp(ctx, P, cl.t, 0.1, st)                      # in place
        inv = guarded(hr.hr_clover_bytes(ctx, P)); hr.hr_clover_finalize(ctx, P, cl.t, inv.t, 0.1, st)
        bad = guarded(hr.hr_clover_bytes(ctx, P)); hr.hr_clover_build(bad.t, prob.links, 1.0, st)
        inv2 = guarded(hr.hr_clover_bytes(ctx, P)); hr.hr_clover_finalize(ctx, P, bad.t, inv2.t, -8.0, st)   # the pivoted path
    # the faces of all four directions in one launch each (round 2), the rank being its own neighbour
    fb = {mu: hr.hr_face_bytes(ctx, P, mu) for mu in range(4)}
    fu = {mu: guarded(fb[mu]) for mu in range(4)}
    fd = {mu: guarded(fb[mu]) for mu in range(4)}
    hr.hr_dphi_eo_faces_pack(15, {mu: g.t for mu, g in fu.items()}, {mu: g.t for mu, g in fd.items()}, gin, prob.links, 0, st)
    o = guarded(sb); hr.hr_dphi_eo_interior_mask(o.t, gin, prob.links, 0, 15, st)
    hr.hr_dphi_eo_faces_apply(15, o.t, {mu: g.t for mu, g in fu.items()}, {mu: g.t for mu, g in fd.items()}, prob.links, 0, 15, 15, st)
    r2 = guarded(16); hr.hr_spinor_dot_noalloc(ctx, P, gin, gin, r2.t, st)
    g = guarded(hr.hr_gauge_bytes(ctx, 1, P))
    h = hr.hr_gauge_alloc(ctx, 1, P, g.t)
    hr.hr_represent_links(h, prob.fund, st)
    hr.hr_gauge_free(h)
    s = guarded(sb); lat.import_spinor(s.t, P, psi, 0)
    for k, c in enumerate(checks):
        assert c.intact(), f"call #{k} wrote outside its output buffer"
    prob.close()
