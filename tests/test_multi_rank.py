"""N > 1 host logic of bench.py on CPU (gloo, world size 2): DESIGN.md section 9 -- the path as specified
has no exchange step, so ranks are independent replicas; the only collectives are the timing barrier and the
MAX over ranks of the measured time.  Checked here: replica seeds differ per rank and give different fields,
max_over_ranks returns the slowest rank's time on every rank, value = units of all ranks / that time, and
`bench.py --impl reference` lets rank 0 alone print a line."""
import json
import itertools
import os
import socket
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    import lattice_inputs as li
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seeds = bench.replica_seeds(bench.CONFIGS[1]["seeds"], rank)
    U = li.haar_links(seeds[0], 2, (4, 4, 4, 4))
    dist.barrier()
    local_ms = 1.0 + 2.0 * rank            # rank 1 is the slow one
    ms = bench.max_over_ranks(local_ms, world, "cpu")
    val = bench.whole_job_value(1e9, world, ms * 1e-3)
    allU = [torch.zeros(U.size * 2, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(allU, torch.from_numpy(np.ascontiguousarray(U).view(np.float64).reshape(-1).copy()))
    q.put((rank, seeds, ms, val, bool(torch.equal(allU[0], allU[1]))))
    dist.destroy_process_group()


def test_replicas_max_over_ranks_gloo_world2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, ms0, v0, same0), (r1, s1, ms1, v1, same1) = res
    assert s0 != s1 and s0 == (1001, 2001) and s1 == (101001, 102001)
    assert not same0 and not same1                      # different replicas really hold different fields
    assert ms0 == ms1 == 3.0                            # the slowest rank's time, on every rank
    assert v0 == v1 == 2 * 1e9 / 3e-3 / 1e9             # units of all ranks / max time


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                        "--steps", "1", "--warmup", "0", "--gpus", "2"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                        "--steps", "1", "--warmup", "0", "--gpus", "2"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2


# ------------------------------------------------------------------------------------------------------------
# NEXT-2: routing of the half-spinor messages between t-slabs, world size 2 over gloo.
def _halo_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    from paper_2405_19294_b200 import halo
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    plan = halo.slab_plan(rank, world, 8)
    send_up = torch.full((16,), 10.0 * rank + 1)       # "for the next rank"
    send_dn = torch.full((16,), 10.0 * rank + 2)       # "for the previous rank"
    recv_prev, recv_next = torch.zeros(16), torch.zeros(16)
    halo.exchange(send_up, send_dn, recv_prev, recv_next, plan)
    q.put((rank, plan, float(recv_prev[0]), float(recv_next[0])))
    dist.destroy_process_group()


def test_halo_exchange_routing_gloo_world2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_halo_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=120) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, plan0, rp0, rn0), (_, plan1, rp1, rn1) = res
    assert plan0 == {"T_local": 4, "t0": 0, "prev": 1, "next": 1, "first_rank": True, "last_rank": False}
    assert plan1 == {"T_local": 4, "t0": 4, "prev": 0, "next": 0, "first_rank": False, "last_rank": True}
    # recv_prev = the previous rank's send_up, recv_next = the next rank's send_dn
    assert rp0 == 11.0 and rn0 == 12.0       # rank 0's neighbours are both rank 1
    assert rp1 == 1.0 and rn1 == 2.0


def test_slab_plan_rejects_bad_splits():
    import pytest
    sys.path.insert(0, ROOT)
    from paper_2405_19294_b200 import halo
    for T, world in ((8, 3), (12, 4), (4, 4)):      # not divisible / odd local extent / local extent 1
        with pytest.raises(ValueError):
            halo.slab_plan(0, world, T)
    assert halo.slab_plan(2, 4, 16) == {"T_local": 4, "t0": 8, "prev": 1, "next": 3, "first_rank": False, "last_rank": False}


def test_block_plan_neighbours_and_errors():
    import pytest
    sys.path.insert(0, ROOT)
    from paper_2405_19294_b200 import halo
    p = halo.block_plan(5, (2, 2, 2, 1), (8, 8, 8, 4))          # rank 5 = coords (1, 0, 1, 0)
    assert p["coords"] == (1, 0, 1, 0) and p["dims_local"] == (4, 4, 4, 4) and p["origin"] == (4, 0, 4, 0)
    assert p["prev"] == [1, 7, 4, 5] and p["next"] == [1, 7, 4, 5] and p["split"] == [0, 1, 2] and p["mask"] == 7
    assert p["first"] == [False, True, False, True] and p["last"] == [True, False, True, True]
    for grid, dims in (((3, 1, 1, 1), (8, 4, 4, 4)), ((2, 1, 1, 1), (6, 4, 4, 4)), ((1, 1, 1, 4), (4, 4, 4, 4))):
        with pytest.raises(ValueError):
            halo.block_plan(0, grid, dims)
    ranks = {tuple(halo.block_plan(r, (2, 1, 2, 2), (4, 4, 4, 4))["coords"]) for r in range(8)}
    assert ranks == set(itertools.product((0, 1), (0,), (0, 1), (0, 1)))
