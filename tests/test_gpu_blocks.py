"""GPU parity of the 4-D block decomposition (include/hr.h third part: hr_face_bytes, hr_dphi_eo_face_pack,
hr_dphi_eo_interior_mask, hr_dphi_eo_face_apply; halo.block_plan / BlockDphi).
One GPU, kernels launched one after the other: a GLOBAL lattice is cut into a grid of blocks, every block is run in turn
with the messages handed over by pointer (the sender's buffer of direction mu becomes the receiver's), the results are
stitched and must equal the oracle on the global lattice -- for every direction alone, for several at once (edge and
corner sites get a term from each), with every boundary sign.  Tolerances: BASELINE.json:north_star."""
import itertools

import numpy as np
import pytest

import lattice_inputs as li
import oracle
from gpu_common import TOL, GpuProblem, oracle_rep_id, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available()
    from paper_2405_19294_b200 import build
    build.build()
    import paper_2405_19294_b200 as hr
    return hr


def _block(arr_lex, dims, plan):
    """Block of a lexicographic site array [V, ...] -> lexicographic array of the local lattice."""
    a = arr_lex.reshape(tuple(dims) + arr_lex.shape[1:])
    o, l = plan["origin"], plan["dims_local"]
    b = a[o[0]:o[0] + l[0], o[1]:o[1] + l[1], o[2]:o[2] + l[2], o[3]:o[3] + l[3]]
    return np.ascontiguousarray(b).reshape((-1,) + arr_lex.shape[1:])


def _half_to_lex(dims, half, parity):
    """Canonical half field of parity `parity` -> lexicographic full field with zeros on the other parity."""
    vh = half.shape[0]
    full = np.zeros((2 * vh,) + half.shape[1:], dtype=half.dtype)
    full[parity * vh:(parity + 1) * vh] = half
    return oracle.eo_to_lex(dims, full)


def _lex_to_half(dims, lex, parity):
    vh = lex.shape[0] // 2
    return np.ascontiguousarray(oracle.lex_to_eo(dims, lex)[parity * vh:(parity + 1) * vh])


CASES = [((1, 2, 1, 1), (4, 8, 4, 4)), ((1, 1, 2, 1), (4, 4, 8, 4)), ((1, 1, 1, 2), (4, 4, 4, 8)), ((2, 1, 1, 1), (8, 4, 4, 4)),
         ((2, 2, 1, 1), (4, 4, 2, 6)), ((1, 2, 2, 2), (2, 4, 4, 8)), ((2, 2, 2, 2), (4, 4, 4, 4)), ((1, 3, 1, 2), (2, 6, 2, 4))]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep,fundlinks", [(3, "fund", False), (2, "adj", False), (3, "sym", True)])
@pytest.mark.parametrize("grid,dims", CASES)
def test_blocks_stitched_equal_the_global_oracle(hr, grid, dims, N, rep, fundlinks, prec):
    from paper_2405_19294_b200 import halo
    bc = (-1, 1, -1, -1)                                       # a seam sign in t, y and z: each must land on exactly one face
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(361, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    V = li.volume(dims)
    world = int(np.prod(grid))
    plans = [halo.block_plan(r, grid, dims) for r in range(world)]
    probs = [GpuProblem(hr, plans[r]["dims_local"], N, rep, prec, _block(U, dims, plans[r]), bc=bc) for r in range(world)]
    blocks = [halo.BlockDphi(probs[r].lat, probs[r].prec, plans[r]) for r in range(world)]
    for parity in (0, 1):
        psi = li.gaussian_spinor(362 + parity, V // 2, d)
        want = oracle.dphi_eo(dims, bc, R, parity, psi)
        psi_lex = _half_to_lex(dims, psi, 1 - parity)
        gin, gout = [], []
        for r, prob in enumerate(probs):
            ld = plans[r]["dims_local"]
            t = prob.lat.spinor(prob.prec)
            prob.lat.import_spinor(t, prob.prec, _lex_to_half(ld, _block(psi_lex, dims, plans[r]), 1 - parity), 1 - parity)
            gin.append(t)
            o = prob.lat.spinor(prob.prec)
            o.fill_(0xFF)
            gout.append(o)
        lks = [p.fund if fundlinks else p.links for p in probs]
        for r in range(world):                                  # 1. every rank packs every split direction
            blocks[r].pack(gin[r], lks[r], parity)
        for r in range(world):                                  # 2. interior
            blocks[r].interior(gout[r], gin[r], lks[r], parity)
        for r in range(world):                                  # 3. messages handed over by pointer
            for mu in plans[r]["split"]:
                blocks[r].buf[mu][2].copy_(blocks[plans[r]["prev"][mu]].buf[mu][0])     # recv_prev <- prev's send_up
                blocks[r].buf[mu][3].copy_(blocks[plans[r]["next"][mu]].buf[mu][1])     # recv_next <- next's send_dn
        got_lex = np.zeros((V, 4, d), dtype=np.complex128)
        gl = got_lex.reshape(tuple(dims) + (4, d))
        for r, prob in enumerate(probs):                        # 4. apply, export, stitch
            blocks[r].apply(gout[r], lks[r], parity)
            ld, o = plans[r]["dims_local"], plans[r]["origin"]
            loc = _half_to_lex(ld, prob.lat.export_spinor(gout[r], prob.prec, parity).astype(np.complex128), parity)
            gl[o[0]:o[0] + ld[0], o[1]:o[1] + ld[1], o[2]:o[2] + ld[2], o[3]:o[3] + ld[3]] = loc.reshape(tuple(ld) + (4, d))
        got = _lex_to_half(dims, got_lex, parity)
        assert rel_l2(got, want) <= TOL[prec], (parity, grid)
        scale = np.sqrt(np.mean(np.abs(want) ** 2))
        assert np.abs(got - want).max() <= 50 * TOL[prec] * scale
    for p in probs:
        p.close()


@pytest.mark.parametrize("mu", [0, 1, 2, 3])
def test_single_rank_block_in_one_direction_reproduces_dphi_eo(hr, mu):
    """One rank whose neighbour in direction mu is itself (grid 1 in every direction, the direction forced through the
    face kernels): pack + interior with that direction masked + apply = hr_dphi_eo = the oracle, seam sign included."""
    dims, bc = (4, 6, 4, 8), (-1, -1, -1, -1)
    U = li.haar_links(371, 3, dims)
    prob = GpuProblem(hr, dims, 3, "fund", "f64", U, bc=bc)
    import torch
    nb = hr.hr_face_bytes(prob.lat.ctx, prob.prec, mu)
    assert nb == li.volume(dims) // 2 // dims[mu] * 2 * 3 * 16
    up, dn = (torch.empty(nb, dtype=torch.uint8, device="cuda") for _ in range(2))
    for parity in (0, 1):
        psi = li.gaussian_spinor(372 + parity, li.volume(dims) // 2, 3)
        gin, out = prob.lat.spinor(prob.prec), prob.lat.spinor(prob.prec)
        prob.lat.import_spinor(gin, prob.prec, psi, 1 - parity)
        out.fill_(0xFF)
        st = prob.lat.stream()
        hr.hr_dphi_eo_face_pack(mu, up, dn, gin, prob.links, parity, st)
        hr.hr_dphi_eo_interior_mask(out, gin, prob.links, parity, 1 << mu, st)
        hr.hr_dphi_eo_face_apply(mu, out, up, dn, prob.links, parity, True, True, st)
        assert rel_l2(prob.lat.export_spinor(out, prob.prec, parity), oracle.dphi_eo(dims, bc, U, parity, psi)) <= TOL["f64"]
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(3, "fund"), (2, "adj"), (3, "sym")])
@pytest.mark.parametrize("mask", [1, 6, 9, 15])
def test_fused_pack_of_all_directions_is_bitwise_the_per_direction_packs(hr, N, rep, mask, prec):
    """hr_dphi_eo_faces_pack (one launch for every split direction) against hr_dphi_eo_face_pack direction by direction:
    the same bytes in every message buffer, with ragged face counts (faces that are no multiple of the CTA size)."""
    import torch
    dims = (4, 6, 4, 10)
    U = li.haar_links(901, N, dims)
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    vh = li.volume(dims) // 2
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    lat, P, st = prob.lat, prob.prec, prob.lat.stream()
    for parity in (0, 1):
        gin = lat.spinor(P)
        lat.import_spinor(gin, P, li.gaussian_spinor(902 + parity, vh, d), 1 - parity)
        split = [mu for mu in range(4) if mask & (1 << mu)]
        one = {mu: [torch.full((hr.hr_face_bytes(lat.ctx, P, mu),), 0xFF, dtype=torch.uint8, device="cuda") for _ in range(2)] for mu in split}
        all_ = {mu: [torch.full((hr.hr_face_bytes(lat.ctx, P, mu),), 0xFF, dtype=torch.uint8, device="cuda") for _ in range(2)] for mu in split}
        for mu in split:
            hr.hr_dphi_eo_face_pack(mu, one[mu][0], one[mu][1], gin, prob.links, parity, st)
        n0 = hr.hr_launch_count()
        hr.hr_dphi_eo_faces_pack(mask, {mu: all_[mu][0] for mu in split}, {mu: all_[mu][1] for mu in split}, gin, prob.links, parity, st)
        assert hr.hr_launch_count() == n0 + 1
        for mu in split:
            for k in (0, 1):
                assert torch.equal(one[mu][k], all_[mu][k]), (mu, k)
    with pytest.raises(hr.HrError):
        hr.hr_dphi_eo_faces_pack(0, {}, {}, gin, prob.links, 0, st)                       # nothing to pack
    with pytest.raises(hr.HrError):
        hr.hr_dphi_eo_faces_pack(2, {}, {}, gin, prob.links, 0, st)                       # NULL buffers of a split direction
    prob.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep", [(3, "fund"), (2, "adj"), (3, "sym")])
@pytest.mark.parametrize("dims,mask", [((4, 6, 4, 10), 1), ((4, 6, 4, 10), 6), ((4, 6, 4, 10), 9), ((4, 6, 4, 10), 15), ((4, 6, 4, 10), 8),
                                       ((2, 2, 2, 2), 15), ((2, 4, 2, 4), 11), ((6, 2, 4, 2), 14)])
def test_fused_apply_of_all_directions_is_bitwise_the_per_direction_applies(hr, N, rep, dims, mask, prec):
    """hr_dphi_eo_faces_apply (one launch; every boundary site updated by one thread, its faces in ascending mu) against
    hr_dphi_eo_face_apply direction by direction in ascending mu: the same bytes in `out` -- edge and corner sites, extents
    of 2 (a site's two neighbours in a direction are both off the block), ragged face counts, every mix of seam flags."""
    import torch
    bc = (-1, 1, -1, -1)
    U = li.haar_links(911, N, dims)
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    vh = li.volume(dims) // 2
    prob = GpuProblem(hr, dims, N, rep, prec, U, bc=bc)
    lat, P, st = prob.lat, prob.prec, prob.lat.stream()
    split = [mu for mu in range(4) if mask & (1 << mu)]
    for parity, (first, last) in itertools.product((0, 1), ((mask, mask), (0, mask), (mask & 5, mask & 10))):
        gin = lat.spinor(P)
        lat.import_spinor(gin, P, li.gaussian_spinor(912 + parity, vh, d), 1 - parity)
        msg = {mu: [torch.empty(hr.hr_face_bytes(lat.ctx, P, mu), dtype=torch.uint8, device="cuda") for _ in range(2)] for mu in split}
        hr.hr_dphi_eo_faces_pack(mask, {mu: m[0] for mu, m in msg.items()}, {mu: m[1] for mu, m in msg.items()}, gin, prob.links, parity, st)
        base = lat.spinor(P)
        hr.hr_dphi_eo_interior_mask(base, gin, prob.links, parity, mask, st)
        one, fused = base.clone(), base.clone()
        for mu in split:                                            # the rank is its own neighbour in every direction
            hr.hr_dphi_eo_face_apply(mu, one, msg[mu][0], msg[mu][1], prob.links, parity, bool(first & (1 << mu)), bool(last & (1 << mu)), st)
        n0 = hr.hr_launch_count()
        hr.hr_dphi_eo_faces_apply(mask, fused, {mu: m[0] for mu, m in msg.items()}, {mu: m[1] for mu, m in msg.items()}, prob.links, parity,
                                  first, last, st)
        assert hr.hr_launch_count() == n0 + 1
        torch.cuda.synchronize()
        assert torch.equal(one, fused), (parity, first, last)
        assert not torch.equal(fused, base)
        if first == mask and last == mask:                          # and the whole sequence is hr_dphi_eo
            full = lat.spinor(P)
            lat.dphi_eo(full, gin, prob.links, parity)
            a, b = lat.export_spinor(fused, P, parity), lat.export_spinor(full, P, parity)
            assert rel_l2(a, b) <= TOL[prec]
    with pytest.raises(hr.HrError):
        hr.hr_dphi_eo_faces_apply(0, fused, {}, {}, prob.links, 0, 0, 0, st)
    with pytest.raises(hr.HrError):
        hr.hr_dphi_eo_faces_apply(2, fused, {}, {}, prob.links, 0, 0, 0, st)
    prob.close()
