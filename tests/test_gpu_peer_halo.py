"""GPU parity of the peer-memory halo path (include/hr.h third part: hr_halo_buffers_alloc / hr_ipc_*; halo.PeerSlabDphi;
PAPER.md:46-64): the pack kernel of one PROCESS stores its half-spinor messages straight into the receive buffers of
its neighbours, mapped with CUDA IPC.  (a) one rank (neighbour = itself) against the oracle; (b) TWO processes, each
owning one slab of a global lattice, both on cuda:0 -- IPC works inside one GPU as it does over NVLink -- with the
ordering done on the host (synchronize + gloo barrier; no kernel of one rank waits on a kernel of the other), results
stitched and compared with the oracle on the global lattice.  Tolerances: BASELINE.json:north_star."""
import os
import socket
import sys

import numpy as np
import pytest

import lattice_inputs as li
import oracle
from gpu_common import BC_T, TOL, GpuProblem, oracle_rep_id, rel_l2

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available()
    from paper_2405_19294_b200 import build
    build.build()
    import paper_2405_19294_b200 as hr
    return hr


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,rep,fundlinks", [(3, "fund", False), (3, "sym", True)])
def test_single_rank_peer_buffers_reproduce_the_oracle(hr, N, rep, fundlinks, prec):
    from paper_2405_19294_b200 import halo
    dims = (4, 4, 6, 8)
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    U = li.haar_links(341, N, dims)
    R = oracle.represent(N, oracle_rep_id(rep), U)
    prob = GpuProblem(hr, dims, N, rep, prec, U)
    slab = halo.PeerSlabDphi(prob.lat, prob.prec, halo.slab_plan(0, 1, dims[0]))
    for rounds in range(2):                                          # both halves of the double buffer
        for parity in (0, 1):
            psi = li.gaussian_spinor(342 + parity + 2 * rounds, li.volume(dims) // 2, d)
            gin, out = prob.lat.spinor(prob.prec), prob.lat.spinor(prob.prec)
            prob.lat.import_spinor(gin, prob.prec, psi, 1 - parity)
            out.fill_(0xFF)
            slab.dphi_eo(out, gin, prob.fund if fundlinks else prob.links, parity)
            assert rel_l2(prob.lat.export_spinor(out, prob.prec, parity), oracle.dphi_eo(dims, BC_T, R, parity, psi)) <= TOL[prec]
    slab.close()
    prob.close()


def test_ipc_handle_round_trip_inside_one_process_is_refused_or_maps(hr):
    """cudaIpcOpenMemHandle of an allocation of the SAME process is an error in CUDA; the binding must surface it as an
    HrError (not crash), and export must give a 64-byte handle."""
    prob = GpuProblem(hr, (4, 4, 4, 4), 3, "fund", "f64", li.haar_links(343, 3, (4, 4, 4, 4)))
    base = hr.hr_halo_buffers_alloc(prob.lat.ctx, hr.HR_F64)
    h = hr.hr_ipc_export(prob.lat.ctx, base)
    assert isinstance(h, bytes) and len(h) == 64
    try:
        p = hr.hr_ipc_open(prob.lat.ctx, h)
        hr.hr_ipc_close(prob.lat.ctx, p)
    except hr.HrError as e:
        assert e.status == hr.HR_ECUDA
    hr.hr_halo_buffers_free(prob.lat.ctx, base)
    prob.close()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _peer_worker(rank, world, port, q, case):
    try:
        _peer_worker_body(rank, world, port, q, case)
    except BaseException as e:                                       # the parent must not wait for a dead rank
        q.put((rank, {"error": repr(e)}))
        raise


def _peer_worker_body(rank, world, port, q, case):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import torch.distributed as dist
    import paper_2405_19294_b200 as hr
    from paper_2405_19294_b200 import halo
    from gpu_common import GpuProblem
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dims, N, rep, fundlinks, prec = case
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    V = li.volume(dims)
    U = li.haar_links(351, N, dims)
    ldims = (dims[0] // world,) + tuple(dims[1:])
    Ul = np.ascontiguousarray(U[rank * (V // world):(rank + 1) * (V // world)])       # t slowest: slabs are contiguous
    prob = GpuProblem(hr, ldims, N, rep, prec, Ul)
    slab = halo.PeerSlabDphi(prob.lat, prob.prec, halo.slab_plan(rank, world, dims[0]))
    lk = prob.fund if fundlinks else prob.links
    res = {}
    for rounds in range(2):
        for parity in (0, 1):
            psi = li.gaussian_spinor(352 + parity + 2 * rounds, V // 2, d)
            per = (V // 2) // world
            gin, out = prob.lat.spinor(prob.prec), prob.lat.spinor(prob.prec)
            prob.lat.import_spinor(gin, prob.prec, np.ascontiguousarray(psi[rank * per:(rank + 1) * per]), 1 - parity)
            out.fill_(0xFF)
            slab.dphi_eo(out, gin, lk, parity)
            res[(rounds, parity)] = prob.lat.export_spinor(out, prob.prec, parity)
    if case[2] == "fund" or world == 1:                              # distributed CG on the slabs (SlabCG)
        m0 = -0.2
        b = li.gaussian_spinor(361, V // 2, d)
        per = (V // 2) // world
        gb, gx = prob.lat.spinor(prob.prec), prob.lat.spinor(prob.prec)
        prob.lat.import_spinor(gb, prob.prec, np.ascontiguousarray(b[rank * per:(rank + 1) * per]), 0)
        gx.fill_(0xFF)
        it, hist = halo.SlabCG(slab, lk, m0).solve(gx, gb, 1e-10, 400)
        res["cg"] = (it, hist, prob.lat.export_spinor(gx, prob.prec, 0))
    dist.barrier()
    slab.close()
    prob.close()
    q.put((rank, res))
    dist.destroy_process_group()


@pytest.mark.parametrize("case", [((8, 4, 2, 6), 3, "fund", False, "f64"), ((8, 4, 2, 6), 3, "sym", True, "f32"),
                                  ((4, 4, 4, 4), 2, "adj", False, "f64")])
def test_two_processes_store_into_each_others_buffers(case):
    import torch
    import torch.multiprocessing as mp
    assert torch.cuda.is_available()
    from paper_2405_19294_b200 import build
    build.build()
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_peer_worker, args=(r, world, port, q, case)) for r in range(world)]
    for p in procs:
        p.start()
    got = {}
    for _ in range(world):
        r, res = q.get(timeout=240)
        if "error" in res:
            for p in procs:
                p.join(timeout=5)
                if p.is_alive():
                    p.terminate()                                    # the surviving rank sits in a barrier
            pytest.fail(f"rank {r}: {res['error']}")
        got[r] = res
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    dims, N, rep, _, prec = case
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    R = oracle.represent(N, oracle_rep_id(rep), li.haar_links(351, N, dims))
    for rounds in range(2):
        for parity in (0, 1):
            psi = li.gaussian_spinor(352 + parity + 2 * rounds, li.volume(dims) // 2, d)
            want = oracle.dphi_eo(dims, BC_T, R, parity, psi)
            stitched = np.concatenate([got[r][(rounds, parity)] for r in range(world)])
            assert rel_l2(stitched, want) <= TOL[prec], (rounds, parity)
    if "cg" in got[0]:
        from oracle import solver
        b = li.gaussian_spinor(361, li.volume(dims) // 2, d)
        x_want, it_want, hist_want = solver.cg_dhat(dims, BC_T, R, -0.2, b, 1e-10, 400)
        assert got[0]["cg"][0] == got[1]["cg"][0] and abs(got[0]["cg"][0] - it_want) <= 1
        n = min(got[0]["cg"][0], it_want) + 1
        assert np.allclose(got[0]["cg"][1][:n], hist_want[:n], rtol=1e-6, atol=0)
        assert got[0]["cg"][1] == got[1]["cg"][1]                    # both ranks saw the same all-reduced scalars
        x = np.concatenate([got[r]["cg"][2] for r in range(world)])
        assert rel_l2(x, x_want) <= 1e-8


# ---- 4-D blocks over peer memory: two processes, split in x, in z or in t ----------------------------------------------
def _block_worker(rank, world, port, q, case):
    try:
        sys.path.insert(0, ROOT)
        sys.path.insert(0, os.path.join(ROOT, "tests"))
        import torch.distributed as dist
        import paper_2405_19294_b200 as hr
        from paper_2405_19294_b200 import halo
        from gpu_common import GpuProblem
        from test_gpu_blocks import _block, _half_to_lex, _lex_to_half
        os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
        dist.init_process_group("gloo", rank=rank, world_size=world)
        grid, dims, N, rep, prec, bc = case
        d = oracle.rep_dim(N, oracle_rep_id(rep))
        V = li.volume(dims)
        U = li.haar_links(381, N, dims)
        plan = halo.block_plan(rank, grid, dims)
        ld = plan["dims_local"]
        prob = GpuProblem(hr, ld, N, rep, prec, _block(U, dims, plan), bc=bc)
        blk = halo.PeerBlockDphi(prob.lat, prob.prec, plan)
        res = {}
        for rounds in range(2):
            for parity in (0, 1):
                psi = li.gaussian_spinor(382 + parity + 2 * rounds, V // 2, d)
                loc = _lex_to_half(ld, _block(_half_to_lex(dims, psi, 1 - parity), dims, plan), 1 - parity)
                gin, out = prob.lat.spinor(prob.prec), prob.lat.spinor(prob.prec)
                prob.lat.import_spinor(gin, prob.prec, loc, 1 - parity)
                out.fill_(0xFF)
                blk.dphi_eo(out, gin, prob.links, parity)
                res[(rounds, parity)] = prob.lat.export_spinor(out, prob.prec, parity)
        # distributed CG on the blocks
        m0 = -0.2
        b = li.gaussian_spinor(391, V // 2, d)
        gb, gx = prob.lat.spinor(prob.prec), prob.lat.spinor(prob.prec)
        prob.lat.import_spinor(gb, prob.prec, _lex_to_half(ld, _block(_half_to_lex(dims, b, 0), dims, plan), 0), 0)
        gx.fill_(0xFF)
        it, hist = halo.SlabCG(blk, prob.links, m0).solve(gx, gb, 1e-10, 400)
        res["cg"] = (it, hist, prob.lat.export_spinor(gx, prob.prec, 0))
        res["plan"] = plan
        dist.barrier()
        blk.close()
        prob.close()
        q.put((rank, res))
        dist.destroy_process_group()
    except BaseException as e:
        q.put((rank, {"error": repr(e)}))
        raise


@pytest.mark.parametrize("case", [((1, 2, 1, 1), (4, 8, 4, 4), 3, "fund", "f64", (-1, -1, 1, 1)),
                                  ((1, 1, 1, 2), (4, 4, 4, 8), 3, "fund", "f64", (-1, 1, 1, -1)),
                                  ((2, 1, 1, 1), (8, 4, 4, 4), 2, "adj", "f64", (-1, 1, 1, 1))])
def test_two_processes_blocks_over_peer_memory(case):
    import torch
    import torch.multiprocessing as mp
    from test_gpu_blocks import _half_to_lex, _lex_to_half
    assert torch.cuda.is_available()
    from paper_2405_19294_b200 import build
    build.build()
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_block_worker, args=(r, world, port, q, case)) for r in range(world)]
    for p in procs:
        p.start()
    got = {}
    for _ in range(world):
        r, res = q.get(timeout=240)
        if "error" in res:
            for p in procs:
                p.join(timeout=5)
                if p.is_alive():
                    p.terminate()
            pytest.fail(f"rank {r}: {res['error']}")
        got[r] = res
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    grid, dims, N, rep, prec, bc = case
    d = oracle.rep_dim(N, oracle_rep_id(rep))
    R = oracle.represent(N, oracle_rep_id(rep), li.haar_links(381, N, dims))
    V = li.volume(dims)

    def stitch(key, parity):
        lex = np.zeros((V, 4, d), dtype=np.complex128)
        gl = lex.reshape(tuple(dims) + (4, d))
        for r in range(world):
            pl = got[r]["plan"]
            ld, o = pl["dims_local"], pl["origin"]
            val = got[r][key] if key != "cg" else got[r]["cg"][2]
            loc = _half_to_lex(ld, val.astype(np.complex128), parity)
            gl[o[0]:o[0] + ld[0], o[1]:o[1] + ld[1], o[2]:o[2] + ld[2], o[3]:o[3] + ld[3]] = loc.reshape(tuple(ld) + (4, d))
        return _lex_to_half(dims, lex, parity)

    for rounds in range(2):
        for parity in (0, 1):
            psi = li.gaussian_spinor(382 + parity + 2 * rounds, V // 2, d)
            assert rel_l2(stitch((rounds, parity), parity), oracle.dphi_eo(dims, bc, R, parity, psi)) <= TOL[prec], (rounds, parity)
    from oracle import solver
    b = li.gaussian_spinor(391, V // 2, d)
    x_want, it_want, hist_want = solver.cg_dhat(dims, bc, R, -0.2, b, 1e-10, 400)
    assert got[0]["cg"][0] == got[1]["cg"][0] and abs(got[0]["cg"][0] - it_want) <= 1
    n = min(got[0]["cg"][0], it_want) + 1
    assert np.allclose(got[0]["cg"][1][:n], hist_want[:n], rtol=1e-6, atol=0)
    assert rel_l2(stitch("cg", 0), x_want) <= 1e-8
