#!/usr/bin/env python
"""bench.py -- one JSON line for the Dphi hot path (BASELINE.json:metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 2|3|4|5] [--prec f64|f32] [--no-table] [--no-cpu-baseline] [--no-e2e]
                    [--sharded]

HEADLINE (the timed region of K steps): config 5, SU(3) fundamental 64^4 fp64 -- the largest single-GPU workload of
BASELINE.json:configs and its "bandwidth run" (kernel time follows the memory moved, so the biggest
volume is the one to time).  A STEP is one pass of the whole hot path over one batch of seeded
synthetic fields: hr_represent_links (fundamental -> represented links) + hr_dphi_eo(parity 0) + hr_dphi_eo(parity 1),
spinor buffers rotating through 4 sets.
value    = north_star's contract bytes of the step / device time (GB/s), inputs resident in HBM:
           4V (F + L) for the link map + V (8L + 9S) for the two Dphi_eo calls.  The contract counts the 8 neighbour
           spinors of a site once each although 7 of them are served on chip, so `value` may exceed the HBM peak;
           the DRAM-side figure is value_compulsory (every byte once: 8L + 2S per site).
roofline = the dominant kernel (the Dphi_eo launch) alone: COMPULSORY bytes per launch / its average launch duration
           (CUDA events inside the timed region) against MEASURED_PEAKS.json; the contract-byte rate is contract_gbs.
configs  = SURVEY.md section 8(d)'s table, measured in the same run (N = 1): the seven (config, precision) datapoints
           and the timed link maps, each with 10 warm-up launches, 5 brackets of >= 100 back-to-back launches
           (alternating parity, rotating buffers; median and min per launch) and one cold-cache single call.
e2e      = the headline step through the C-ABI host entry points (hr_gauge_import from pinned host memory,
           hr_represent_links, hr_dphi_eo_host x2), host<->device copies inside the timed region.
cpu_baseline / --impl reference = the oracle (oracle/, as it stands) on this box's host cores, all threads and one.
N > 1 (torchrun): independent replicas, one per GPU, no data-path collective ("scaling": "weak");
--sharded: ONE 64^4 lattice cut into t-slabs over the ranks, half-spinor messages over peer memory,
value = the same contract bytes of the global lattice / max-over-ranks time ("scaling": "strong").
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Dphi_eo GB/s and GFLOP/s per B200, fraction of HBM roofline (fp64, fp32)"
BC = (-1, 1, 1, 1)
# BASELINE.json:configs[k-1]; seeds as SURVEY.md section 8(d)
CONFIGS = {
    1: dict(name="SU(2) fund 4^4", dims=(4, 4, 4, 4), N=2, rep="fund", kind="haar", seeds=(1001, 2001)),
    2: dict(name="SU(3) fund 32^3x64", dims=(64, 32, 32, 32), N=3, rep="fund", kind="haar", seeds=(1002, 2002)),
    3: dict(name="SU(2) adjoint 32^4", dims=(32, 32, 32, 32), N=2, rep="adj", kind="haar", seeds=(1003, 2003)),
    4: dict(name="SU(3) sextet 24^3x48", dims=(48, 24, 24, 24), N=3, rep="sym", kind="haar", seeds=(1004, 2004)),
    5: dict(name="SU(3) fund 64^4", dims=(64, 64, 64, 64), N=3, rep="fund", kind="near", seeds=(1005, 2005)),
    # not a BASELINE.json config: the local slab of config 5 on 8 GPUs split along t (NEXT-2)
    6: dict(name="SU(3) fund 64^3x8 slab", dims=(8, 64, 64, 64), N=3, rep="fund", kind="near", seeds=(1006, 2006)),
}
# the seven bandwidth datapoints (config 1 is correctness only), headline first
DATAPOINTS = [(5, "f64"), (5, "f32"), (2, "f64"), (2, "f32"), (3, "f64"), (4, "f64"), (4, "f32")]
REP_DIM = {"fund": lambda N: N, "adj": lambda N: N * N - 1, "sym": lambda N: N * (N + 1) // 2, "asym": lambda N: N * (N - 1) // 2}
NSET = 4          # rotating spinor buffer sets (section 8(d): consecutive calls must not re-read a hot output)
STEP_TEXT = "hr_represent_links + hr_dphi_eo(parity 0) + hr_dphi_eo(parity 1)"


def byte_model(cfg, prec):
    """Per-site algorithmic bytes / flops (SURVEY.md section 8(a),(d))."""
    w = 8 if prec == "f64" else 4
    N, rep = cfg["N"], cfg["rep"]
    d = REP_DIM[rep](N)
    real = rep == "adj"
    S = 4 * d * 2 * w
    L = d * d * w * (1 if real else 2)
    F = N * N * 2 * w
    V = int(np.prod(cfg["dims"]))
    return dict(d=d, S=S, L=L, F=F, V=V, dphi_bytes_per_site=8 * L + 9 * S, compulsory_bytes_per_site=8 * L + 2 * S,
                dphi_flops_per_site=(64 if real else 128) * d * d + 56 * d, represent_bytes_per_link=F + L)


def config_keys(cfg, world=1, sharded=False):
    """The `config` object: identical for --impl ours and --impl reference."""
    bm = byte_model(cfg, "f64")
    return {"workload": cfg["name"], "dims": list(cfg["dims"]), "bc": list(BC), "N": cfg["N"], "rep": cfg["rep"],
            "d_R": bm["d"], "step": STEP_TEXT, "l2": "inputs exceed L2 (no flush)",
            "parallelism": "single" if world == 1 else (f"t-slabs x{world}" if sharded else "replicas")}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(workload, prec):
    """dram bytes per Dphi launch from the committed ncu capture summary (profiles/dram_traffic.csv), or None.
    A constant read from the repository, NOT a measurement of this run (the JSON line says so)."""
    p = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    try:
        for line in open(p):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 4 and f[0] == workload and f[1] == prec:
                return float(f[3])
    except Exception:
        pass
    return None


def make_fields(cfg):
    import lattice_inputs as li
    d = REP_DIM[cfg["rep"]](cfg["N"])
    sl, ss = cfg["seeds"]
    U = li.haar_links(sl, cfg["N"], cfg["dims"]) if cfg["kind"] == "haar" else li.near_identity_links(sl, cfg["N"], cfg["dims"], 0.3)
    vh = li.volume(cfg["dims"]) // 2
    psi = [li.gaussian_spinor(ss + 10 * p, vh, d) for p in (0, 1)]
    return U, psi


def replica_seeds(seeds, rank):
    """Independent replica per rank (replicas only, no data-path collective)."""
    return (seeds[0] + 100000 * rank, seeds[1] + 100000 * rank)


def max_over_ranks(x, world, device):
    """MAX over ranks of a locally measured duration (the only collective besides the timing barrier)."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(step_bytes, world, seconds_per_step):
    """value = the units all ranks processed / the max-over-ranks time (GB/s)."""
    return world * step_bytes / seconds_per_step / 1e9


class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU during the timed region (NVML)."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.005)

    def __enter__(self):
        if self.nv:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"], "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline of the headline line, and --impl reference)
# ---------------------------------------------------------------------------------------------------------------
def oracle_sample_step(cfg, U, R, psi, n):
    """One sampled pass of the oracle over the step: the link map on the links of the first 2n lattice sites and Dphi_eo
    on the first n output sites of each parity (n = Vh: the whole step).  Returns seconds."""
    import oracle
    rid = oracle.REP_NAMES[cfg["rep"]]
    vh = int(np.prod(cfg["dims"])) // 2
    t0 = time.perf_counter()
    oracle.represent(cfg["N"], rid, U[:2 * n])
    if n == vh:
        for parity in (0, 1):
            oracle.dphi_eo(cfg["dims"], BC, R, parity, psi[parity])
    else:
        hidx = np.arange(n, dtype=np.int64)
        for parity in (0, 1):
            oracle.dphi_eo_sites(cfg["dims"], BC, R, parity, psi[parity], hidx)
    return time.perf_counter() - t0


def oracle_links(cfg, U):
    """R(U) on the whole lattice for the sampled Dphi (untimed set-up).  FUND: R(U) = U, no copy of a 9 GiB field."""
    import oracle
    if cfg["rep"] == "fund":
        return U
    return oracle.represent(cfg["N"], oracle.REP_NAMES[cfg["rep"]], U)


def sample_bytes(cfg, n):
    bm = byte_model(cfg, "f64")  # the oracle computes in fp64
    return 2 * n * 4 * bm["represent_bytes_per_link"] + 2 * n * bm["dphi_bytes_per_site"]


def sample_text(cfg, n):
    vh = int(np.prod(cfg["dims"])) // 2
    if n == vh:
        return f"the whole step of {cfg['name']} (all {vh} output sites of each parity and every link), fp64"
    return (f"a SAMPLE of {cfg['name']}: per step the link map on the first {2 * n} lattice sites and Dphi_eo on the first "
            f"{n} output sites of each parity (of {vh}), fp64; bytes counted for the sample only")


def run_reference(args, cfg):
    """--impl reference: the oracle, as it stands, on this box's host cores; same metric / config / unit.
    Each step is a bounded sample of the workload (args.sample_sites output sites per parity + their links)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    bm = byte_model(cfg, "f64")
    U, psi = make_fields(cfg)
    R = oracle_links(cfg, U)
    n = min(bm["V"] // 2, args.sample_sites)
    for _ in range(args.warmup):
        oracle_sample_step(cfg, U, R, psi, n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_sample_step(cfg, U, R, psi, n)
    dt = (time.perf_counter() - t0) / args.steps
    val = sample_bytes(cfg, n) / dt / 1e9
    threads = oracle.num_threads()
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": config_keys(cfg),
        "cpu_baseline": {"value": val, "unit": "GB/s", "cores": threads, "kind": "oracle", "sample": sample_text(cfg, n)},
        "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gflops": 2 * n * bm["dphi_flops_per_site"] / dt / 1e9,
    }))


def omp_set_threads(n):
    """Set the OpenMP team size of this process through the OpenMP runtime itself (libgomp, the runtime oracle.c's
    `-fopenmp` links): the oracle is timed as it stands, its source and build are not touched."""
    import ctypes
    ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))


def cpu_baseline(cfg, U, psi):
    """The oracle on this box's host cores, all threads and ONE thread.
    About 10-30 s of CPU work in total."""
    import oracle
    vh = int(np.prod(cfg["dims"])) // 2
    R = oracle_links(cfg, U)
    all_threads = oracle.num_threads()
    n = min(vh, 1 << 21)
    oracle_sample_step(cfg, U, R, psi, min(vh, 1 << 16))  # page in
    dt = min(oracle_sample_step(cfg, U, R, psi, n) for _ in range(3))
    out = {"value": sample_bytes(cfg, n) / dt / 1e9, "unit": "GB/s", "cores": all_threads, "kind": "oracle",
           "sample": sample_text(cfg, n) + ", best of 3", "ms_per_sample": dt * 1e3, "sites_per_s": 2 * n / dt}
    try:
        omp_set_threads(1)
        n1 = min(vh, 1 << 18)
        dt1 = min(oracle_sample_step(cfg, U, R, psi, n1) for _ in range(2))
        out["one_thread"] = {"value": sample_bytes(cfg, n1) / dt1 / 1e9, "unit": "GB/s", "cores": oracle.num_threads(),
                             "sample": sample_text(cfg, n1) + ", best of 2", "ms_per_sample": dt1 * 1e3,
                             "sites_per_s": 2 * n1 / dt1}
    except Exception as exc:  # the one-thread leg is a report, not a gate
        out["one_thread"] = {"unavailable": repr(exc)[:200]}
    finally:
        try:
            omp_set_threads(all_threads)
        except Exception:
            pass
    return out


# ---------------------------------------------------------------------------------------------------------------
# ours
# ---------------------------------------------------------------------------------------------------------------
class Problem:
    """One (config, precision) on the device: fundamental + represented links, NSET rotating spinor sets."""

    def __init__(self, hr, cfg, prec, U, psi, device, links="repr", tuning=None):
        self.hr, self.cfg, self.prec, self.P = hr, cfg, prec, hr.PREC_NAMES[prec]
        self.bm = byte_model(cfg, prec)
        self.lat = hr.Lattice(cfg["dims"], BC, cfg["N"], cfg["rep"], device=device)
        self.fund = self.lat.gauge(False, self.P)
        self.links = self.lat.gauge(True, self.P)
        self.lat.import_gauge(self.fund, U)
        self.lat.represent_links(self.links, self.fund)
        # what hr_dphi_eo reads: the represented field (north_star's contract), the FUNDAMENTAL field (representation applied
        # on the fly) or its row-compressed form (section 16); the last two move fewer link bytes
        self.src = links
        w = 8 if prec == "f64" else 4
        if links == "rows":
            self.dlinks = self.lat.gauge(2, self.P)
            self.lat.compress_links(self.dlinks, self.fund)
            self.link_bytes = 2 * cfg["N"] * (cfg["N"] - 1) * w
        else:
            self.dlinks = self.fund if links == "fund" else self.links
            self.link_bytes = self.bm["F"] if links == "fund" else self.bm["L"]
        self.needed_bytes_per_site = 8 * self.link_bytes + 2 * self.bm["S"]
        for key, val in (tuning or {}).items():
            self.lat.set_tuning(key, val)
        # set k: in[k] holds psi[k & 1] (the parity-(1 - (k&1)) half field), out[k] receives Dphi_eo(parity k & 1)
        self.inp = [self.lat.spinor(self.P) for _ in range(NSET)]
        self.out = [self.lat.spinor(self.P) for _ in range(NSET)]
        for k in range(NSET):
            self.lat.import_spinor(self.inp[k], self.P, psi[k & 1], 1 - (k & 1))

    def dphi(self, k):
        self.lat.dphi_eo(self.out[k % NSET], self.inp[k % NSET], self.dlinks, k & 1)

    def represent(self):
        self.lat.represent_links(self.links, self.fund)

    def close(self):
        self.lat.close()


def flush_l2(torch, scratch):
    scratch.zero_()  # 512 MiB written: 4x the 126 MB L2


def bracket_protocol(torch, fn, scratch, launches, brackets=5, warm=10, clocks=None):
    """`warm` warm-up launches, then `brackets` CUDA-event brackets of `launches` back-to-back
    launches each; returns (median ms, min ms, cold-cache single-launch ms).  clocks (a dict, optional) receives the SM
    clock / throttle reasons sampled during the brackets and `burst_ms`: 8 launches timed after 0.3 s of idle, i.e. at
    boost clocks -- back to back this operator sits at the 1 kW power cap near 1.4-1.7 GHz and runs 5-10 % slower."""
    for k in range(warm):
        fn(k)
    torch.cuda.synchronize()
    if clocks is not None:
        time.sleep(0.3)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for k in range(8):
            fn(k)
        e1.record()
        torch.cuda.synchronize()
        clocks["burst_ms"] = e0.elapsed_time(e1) / 8
    per = []
    with ClockSampler(torch.cuda.current_device()) as clk:
        for _ in range(brackets):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for k in range(launches):
                fn(k)
            e1.record()
            torch.cuda.synchronize()
            per.append(e0.elapsed_time(e1) / launches)
    if clocks is not None:
        clocks.update(clk.summary())
    flush_l2(torch, scratch)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    fn(0)
    e1.record()
    torch.cuda.synchronize()
    return statistics.median(per), min(per), e0.elapsed_time(e1)


def datapoint(torch, prob, scratch, peak, launches):
    """One row of section 8(d)'s table."""
    bm, cfg = prob.bm, prob.cfg
    vh = bm["V"] // 2
    clocks = {}
    med, mn, cold = bracket_protocol(torch, prob.dphi, scratch, launches, clocks=clocks)
    comp = vh * bm["compulsory_bytes_per_site"]
    contract = vh * bm["dphi_bytes_per_site"]
    row = {"workload": cfg["name"], "dtype": prob.prec, "d_R": bm["d"], "sites_per_launch": vh,
           "kernel_variant": prob.lat.variant_name(prob.P),
           "ms_per_launch_median": med, "ms_per_launch_min": mn, "ms_cold_single": cold, "launches_per_bracket": launches,
           "brackets": 5, "sites_per_s": vh / (med * 1e-3),
           "compulsory_gbs": comp / (med * 1e-3) / 1e9, "frac": comp / (med * 1e-3) / 1e9 / peak,
           "contract_gbs": contract / (med * 1e-3) / 1e9, "contract_frac_of_8TBs_nominal": contract / (med * 1e-3) / 1e9 / 8000.0,
           "gflops": vh * bm["dphi_flops_per_site"] / (med * 1e-3) / 1e9,
           "ms_per_launch_burst": clocks["burst_ms"], "frac_burst": comp / (clocks["burst_ms"] * 1e-3) / 1e9 / peak,
           "clocks": {k: clocks[k] for k in ("sm_mhz", "sm_max_mhz", "reasons")},
           "traffic": ncu_traffic(cfg["name"], prob.prec)}
    if cfg["rep"] != "fund":  # the timed link maps of configs 3 and 4
        rmed, rmn, rcold = bracket_protocol(torch, lambda k: prob.represent(), scratch, max(20, launches // 2))
        rb = 4 * bm["V"] * bm["represent_bytes_per_link"]
        row["represent"] = {"ms_median": rmed, "ms_min": rmn, "ms_cold_single": rcold, "bytes": rb,
                            "gbs": rb / (rmed * 1e-3) / 1e9, "frac": rb / (rmed * 1e-3) / 1e9 / peak}
    return row


def register_host(torch, arr):
    """Page-lock a numpy array in place (no second copy of a 9 GiB field); returns True if it is now pinned."""
    try:
        rc = torch.cuda.cudart().cudaHostRegister(arr.ctypes.data, arr.nbytes, 0)
        return int(rc) == 0
    except Exception:
        return False


def unregister_host(torch, arr):
    try:
        torch.cuda.cudart().cudaHostUnregister(arr.ctypes.data)
    except Exception:
        pass


def run_sharded(args, hr, world, rank, local):
    """--sharded: ONE lattice cut into t-slabs over the ranks: every rank owns T/N
    time-slices of the seeded global fields; a step is the link map on the slab + two distributed Dphi_eo -- half-spinor
    faces projected and written straight into the neighbours' receive buffers by the pack kernel (CUDA IPC peer memory
    over NVLink; --sharded-nccl: ncclSend/Recv on a side stream), interior launch meanwhile, apply after one fence.
    value = contract bytes of the GLOBAL lattice / max-over-ranks time: "scaling": "strong"."""
    import torch
    import torch.distributed as dist
    import lattice_inputs as li
    from paper_2405_19294_b200 import halo

    cfg, prec = CONFIGS[args.config], args.prec
    P = hr.PREC_NAMES[prec]
    bm = byte_model(cfg, prec)
    plan = halo.slab_plan(rank, world, cfg["dims"][0])
    ldims = (plan["T_local"],) + tuple(cfg["dims"][1:])
    vl = li.volume(ldims)
    sl, ss = cfg["seeds"]
    gen = li.haar_links if cfg["kind"] == "haar" else (lambda s, N, dm, **kw: li.near_identity_links(s, N, dm, 0.3, **kw))
    U = gen(sl, cfg["N"], ldims, first_site=rank * vl, nsites=vl)
    psi = [li.gaussian_spinor(ss + 10 * p, vl // 2, bm["d"], first_site=rank * (vl // 2)) for p in (0, 1)]
    lat = hr.Lattice(ldims, BC, cfg["N"], cfg["rep"], device=local)
    fund, links = lat.gauge(False, P), lat.gauge(True, P)
    lat.import_gauge(fund, U)
    lat.represent_links(links, fund)
    inp = [lat.spinor(P) for _ in range(NSET)]
    out = [lat.spinor(P) for _ in range(NSET)]
    for k in range(NSET):
        lat.import_spinor(inp[k], P, psi[k & 1], 1 - (k & 1))
    slab = (halo.SlabDphi if args.sharded_nccl else halo.PeerSlabDphi)(lat, P, plan)

    def step(k):
        lat.represent_links(links, fund)
        slab.dphi_eo(out[(2 * k) % NSET], inp[(2 * k) % NSET], links, 0)
        slab.dphi_eo(out[(2 * k + 1) % NSET], inp[(2 * k + 1) % NSET], links, 1)

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for k in range(args.warmup):
        step(k)
    sync_all()
    n0 = hr.hr_launch_count()
    with ClockSampler(local) as clk:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for k in range(args.steps):
            step(k)
        e1.record()
        sync_all()
    launches = hr.hr_launch_count() - n0
    ms_step = max_over_ranks(e0.elapsed_time(e1), world, "cuda") / args.steps
    # the same slab WITHOUT the decomposition (periodic in t inside the rank): what the faces cost
    med, _, _ = bracket_protocol(torch, lambda k: lat.dphi_eo(out[k % NSET], inp[k % NSET], links, k & 1),
                                 torch.empty(512 << 20, dtype=torch.uint8, device="cuda"), max(20, args.steps), brackets=3)
    dmed, _, _ = bracket_protocol(torch, lambda k: slab.dphi_eo(out[k % NSET], inp[k % NSET], links, k & 1),
                                  torch.empty(1, dtype=torch.uint8, device="cuda"), max(20, args.steps), brackets=3)
    med, dmed = max_over_ranks(med, world, "cuda"), max_over_ranks(dmed, world, "cuda")
    if rank == 0:
        step_bytes = 4 * bm["V"] * bm["represent_bytes_per_link"] + bm["V"] * bm["dphi_bytes_per_site"]
        comp = 4 * bm["V"] * bm["represent_bytes_per_link"] + bm["V"] * bm["compulsory_bytes_per_site"]
        peak, peak_src = measured_peak()
        print(json.dumps({
            "metric": METRIC, "value": step_bytes / (ms_step * 1e-3) / 1e9, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": prec, "data": "synthetic", "config": config_keys(cfg, world, sharded=True),
            "value_compulsory": comp / (ms_step * 1e-3) / 1e9, "clocks": clk.summary(), "gpu_launches": int(launches),
            "e2e": None,
            "sharded": {"exchange": "nccl send/recv on a side stream" if args.sharded_nccl else "peer stores from the pack kernel (CUDA IPC)",
                        "local_dims": list(ldims), "halo_bytes_per_message": hr.hr_halo_bytes(lat.ctx, P),
                        "dphi_eo_ms_distributed": dmed, "dphi_eo_ms_same_slab_undistributed": med,
                        "decomposition_overhead": dmed / med - 1.0},
            "roofline": {"bound": "hbm", "kernel": "interior Dphi launch + face pack / apply", "achieved": world * (vl // 2) * bm["compulsory_bytes_per_site"] / (dmed * 1e-3) / 1e9,
                         "peak": peak * world, "unit": "GB/s", "frac": (vl // 2) * bm["compulsory_bytes_per_site"] / (dmed * 1e-3) / 1e9 / peak,
                         "traffic": None, "peak_source": peak_src + " x n_gpus"}}))
    if hasattr(slab, "close"):
        slab.close()
    lat.close()
    if world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    from paper_2405_19294_b200 import build
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    import paper_2405_19294_b200 as hr

    if args.sharded:
        return run_sharded(args, hr, world, rank, local)

    cfg = CONFIGS[args.config]
    prec = args.prec
    peak, peak_src = measured_peak()
    scratch = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    cfg_r = dict(cfg, seeds=replica_seeds(cfg["seeds"], rank))
    U, psi = make_fields(cfg_r)
    tuning = {kv.split("=")[0]: int(kv.split("=")[1]) for kv in args.tuning.split(",") if kv}
    prob = Problem(hr, cfg, prec, U, psi, local, links=args.links, tuning=tuning)
    bm, lat, P = prob.bm, prob.lat, prob.P
    torch.cuda.synchronize()

    def step(k, events=None):
        if events is not None:
            events[0].record()
        prob.represent()
        if events is not None:
            events[1].record()
        prob.dphi(2 * k)
        if events is not None:
            events[2].record()
        prob.dphi(2 * k + 1)
        if events is not None:
            events[3].record()

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for k in range(args.warmup):
        step(k)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    sync_all()
    n0 = hr.hr_launch_count()
    with ClockSampler(local) as clk:
        t_begin = torch.cuda.Event(enable_timing=True)
        t_end = torch.cuda.Event(enable_timing=True)
        t_begin.record()
        for k in range(args.steps):
            step(k, ev[k])
        t_end.record()
        sync_all()
    launches = hr.hr_launch_count() - n0
    ms_total = t_begin.elapsed_time(t_end)
    rep_ms = statistics.mean(e[0].elapsed_time(e[1]) for e in ev)
    dphi_all = [e[1].elapsed_time(e[2]) for e in ev] + [e[2].elapsed_time(e[3]) for e in ev]
    dphi_ms, dphi_ms_min = statistics.mean(dphi_all), min(dphi_all)
    ms_total = max_over_ranks(ms_total, world, "cuda")
    ms_step = ms_total / args.steps
    vh = bm["V"] // 2
    step_bytes = 4 * bm["V"] * bm["represent_bytes_per_link"] + bm["V"] * bm["dphi_bytes_per_site"]
    step_bytes_compulsory = 4 * bm["V"] * bm["represent_bytes_per_link"] + bm["V"] * bm["compulsory_bytes_per_site"]
    value = whole_job_value(step_bytes, world, ms_step * 1e-3)

    # companion (NOT part of `value`): the same Dphi_eo reading row-compressed fundamental links --
    # fewer bytes than north_star's contract counts, so it is reported beside the headline, with its own byte count
    rows_info = None
    if args.links == "repr" and not tuning and cfg["N"] <= 3 and (cfg["rep"] == "fund" or (cfg["rep"] == "adj" and cfg["N"] == 2)):
        rows = lat.gauge(2, P)
        lat.compress_links(rows, prob.fund)
        fn = lambda k: lat.dphi_eo(prob.out[k % NSET], prob.inp[k % NSET], rows, k & 1)
        med, mn, _ = bracket_protocol(torch, fn, scratch, max(20, 2 * args.steps), brackets=3)
        med = max_over_ranks(med, world, "cuda")
        w = 8 if prec == "f64" else 4
        lrows = 2 * cfg["N"] * (cfg["N"] - 1) * w
        need = 8 * lrows + 2 * bm["S"]
        rows_info = {"ms_per_launch": med, "link_bytes": lrows, "needed_bytes_per_site": need,
                     "needed_gbs": vh * need / (med * 1e-3) / 1e9, "frac_of_needed": vh * need / (med * 1e-3) / 1e9 / peak,
                     "speedup_vs_full_links": dphi_ms / med}

    # end to end through the host entry points (page-locked host buffers; copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        cdt = np.complex128 if prec == "f64" else np.complex64
        hU = np.ascontiguousarray(U, dtype=cdt)
        hin = [np.ascontiguousarray(psi[p], dtype=cdt) for p in (0, 1)]
        hout = [np.empty_like(hin[p]) for p in (0, 1)]
        pinned = all([register_host(torch, a) for a in [hU] + hin + hout])
        st = lat.stream()

        def e2e_step():
            hr.hr_gauge_import(prob.fund, hU, P, st)
            hr.hr_represent_links(prob.links, prob.fund, st)
            for p in (0, 1):
                hr.hr_dphi_eo_host(lat.ctx, hout[p], hin[p], P, prob.links, p, st)

        ke = 3
        e2e_step()
        sync_all()
        t0 = time.perf_counter()
        for _ in range(ke):
            e2e_step()
        sync_all()
        dt = (time.perf_counter() - t0) / ke
        dt = max_over_ranks(dt, world, "cuda")
        h2d = hU.nbytes + sum(h.nbytes for h in hin)
        d2h = sum(h.nbytes for h in hout)
        e2e = {"value": whole_job_value(step_bytes, world, dt), "unit": "GB/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "ms_per_step": dt * 1e3, "steps": ke, "host_memory": "page-locked (cudaHostRegister)" if pinned else "pageable",
               "pcie_gbs": (h2d + d2h) / dt / 1e9}
        for a in [hU] + hin + hout:
            unregister_host(torch, a)
        del hU, hin, hout

    if rank != 0:
        prob.close()
        if world > 1:
            dist.destroy_process_group()
        return

    comp_launch = vh * prob.needed_bytes_per_site     # = Vh (8L + 2S) with the represented links of the contract
    contract_launch = vh * bm["dphi_bytes_per_site"]
    achieved = comp_launch / (dphi_ms * 1e-3) / 1e9
    traffic = ncu_traffic(cfg["name"], prec)
    out = {
        "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": prec,
        "data": "synthetic",
        "config": config_keys(cfg, world),
        "value_definition": "north_star contract bytes (4V(F+L) + V(8L+9S)) / device time; may exceed the HBM peak because "
                            "7 of a site's 8 neighbour-spinor reads are served on chip -- see value_compulsory and roofline",
        "value_compulsory": whole_job_value(step_bytes_compulsory, world, ms_step * 1e-3),
        "kernel_variant": lat.variant_name(P), "links_read_by_dphi": args.links, "tuning": tuning or None,
        "clocks": clk.summary(),
        "e2e": e2e,
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "kernel": "dphi (hr_dphi_eo launch, variant " + lat.variant_name(P) + ")",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "bytes_model": "compulsory DRAM bytes per launch: Vh (8L + 2S), every link / input spinor / output once",
                     "traffic": traffic,
                     "traffic_source": "profiles/dram_traffic.csv (ncu --set full capture of an earlier run; a constant, not measured here)"
                     if traffic is not None else None,
                     "peak_source": peak_src, "bytes_per_launch": comp_launch, "ms_per_launch": dphi_ms,
                     "ms_per_launch_min": dphi_ms_min,
                     "contract_gbs": contract_launch / (dphi_ms * 1e-3) / 1e9,
                     "contract_frac": contract_launch / (dphi_ms * 1e-3) / 1e9 / peak,
                     "contract_frac_of_8TBs_nominal": contract_launch / (dphi_ms * 1e-3) / 1e9 / 8000.0},
        "dphi_gflops": vh * bm["dphi_flops_per_site"] / (dphi_ms * 1e-3) / 1e9,
        "rows_links": rows_info,
        "represent_ms": rep_ms,
        "represent_gbs": 4 * bm["V"] * bm["represent_bytes_per_link"] / (rep_ms * 1e-3) / 1e9,
    }
    if not args.no_cpu_baseline and world == 1:
        out["cpu_baseline"] = cpu_baseline(cfg, U, psi)

    # section 8(d)'s table: every (config, precision) datapoint in the same run
    if not args.no_table and world == 1:
        rows = []
        cur_id, fields = args.config, (U, psi)
        del U, psi
        for cid, pr in DATAPOINTS:
            c = CONFIGS[cid]
            if prob is not None and cid == args.config and pr == prec:
                rows.append(datapoint(torch, prob, scratch, peak, 100))
                continue
            if cid != cur_id:
                if prob is not None:   # the headline problem's fields are no longer needed
                    prob.close()
                    prob = None
                    torch.cuda.empty_cache()
                fields = None          # one config's host fields at a time (64^4 fp64 links are 9 GiB)
                fields = make_fields(c)
                cur_id = cid
            p2 = Problem(hr, c, pr, fields[0], fields[1], local)
            rows.append(datapoint(torch, p2, scratch, peak, 100))
            p2.close()
            del p2
            torch.cuda.empty_cache()
        out["configs"] = rows
        out["protocol"] = ("SURVEY.md section 8(d): 10 warm-up launches, 5 CUDA-event brackets of 100 back-to-back hr_dphi_eo "
                           "launches alternating parity over 4 rotating buffer sets, median and min per launch; one single "
                           "launch after writing 512 MiB (cold L2); frac = Vh(8L+2S) / median / measured copy peak")
    if prob is not None:
        prob.close()
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, choices=sorted(CONFIGS))
    ap.add_argument("--prec", default="f64", choices=["f64", "f32"])
    ap.add_argument("--no-table", action="store_true", help="skip the per-config table (configs[])")
    ap.add_argument("--links", default="repr", choices=["repr", "fund", "rows"],
                    help="link field hr_dphi_eo reads in the headline step (default: the represented field of the contract)")
    ap.add_argument("--tuning", default="", help="hr_ctx_set_tuning keys for the headline problem, e.g. variant=7,bulk_ctas=2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--sharded", action="store_true", help="N > 1: one lattice on t-slabs instead of replicas")
    ap.add_argument("--sharded-nccl", action="store_true", help="--sharded with NCCL send/recv instead of peer stores")
    ap.add_argument("--sample-sites", type=int, default=1 << 18, help="--impl reference: output sites per parity and step")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args, CONFIGS[args.config])
    else:
        args.warmup = max(args.warmup, 3)
        run_ours(args)


if __name__ == "__main__":
    main()
