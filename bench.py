#!/usr/bin/env python
"""bench.py -- one JSON line for the Dphi hot path (BASELINE.json:metric, workload configs[1]).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 2|3|4|5] [--prec f64|f32] [--no-cpu-baseline] [--no-e2e]

A STEP is one pass of the whole hot path over one batch of seeded synthetic
fields: hr_represent_links (fundamental -> represented links) + hr_dphi_eo(parity 0) + hr_dphi_eo(parity 1).
value  = algorithmic bytes of the step / device time (GB/s), inputs resident in HBM:
         4V (F + L)  for the link map  +  V (8L + 9S)  for the two Dphi_eo calls  (north_star byte contract).
e2e    = the same, through the C-ABI host entry points (hr_gauge_import from pinned host memory,
         hr_represent_links, hr_dphi_eo_host x2), host<->device copies inside the timed region.
roofline = the dominant kernel (dphi_kernel) alone: contract bytes per launch / its average launch
         duration measured with CUDA events inside the timed region, against MEASURED_PEAKS.json.
cpu_baseline / --impl reference = the oracle (oracle/, as it stands) on this box's host cores.
N > 1 (torchrun): independent replicas, one per GPU, no data-path collective ("scaling": "weak").
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
REP_DIM = {"fund": lambda N: N, "adj": lambda N: N * N - 1, "sym": lambda N: N * (N + 1) // 2, "asym": lambda N: N * (N - 1) // 2}


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


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(workload, prec):
    """dram bytes per dphi launch from the committed ncu capture summary (profiles/dram_traffic.csv), or None."""
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


def oracle_step(cfg, U, psi, reps, nsample=None):
    """The oracle's pass over the same step (nsample: only the first nsample output sites of each parity
    and the links of the first 2*nsample lattice sites); returns seconds per step (best of reps), threads."""
    import oracle
    rid = oracle.REP_NAMES[cfg["rep"]]
    best = float("inf")
    for _ in range(reps):
        t0 = time.perf_counter()
        if nsample is None:
            R = oracle.represent(cfg["N"], rid, U)
            for parity in (0, 1):
                oracle.dphi_eo(cfg["dims"], BC, R, parity, psi[parity])
        else:
            oracle.represent(cfg["N"], rid, U[:2 * nsample])
            hidx = np.arange(nsample, dtype=np.int64)
            for parity in (0, 1):
                oracle.dphi_eo_sites(cfg["dims"], BC, oracle_step.R, parity, psi[parity], hidx)
        best = min(best, time.perf_counter() - t0)
    return best, oracle.num_threads()


def run_reference(args, cfg, prec):
    """--impl reference: the oracle, as it stands, on this box's host cores; same metric / config / unit.
    Each step is a bounded sample of the workload (2^16 output sites per parity + their links)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    bm = byte_model(cfg, "f64")  # the oracle computes in fp64
    U, psi = make_fields(cfg)
    oracle_step.R = oracle.represent(cfg["N"], oracle.REP_NAMES[cfg["rep"]], U)  # untimed set-up for the sampled Dphi
    n = min(bm["V"] // 2, 1 << 16)
    step_bytes = 2 * n * 4 * bm["represent_bytes_per_link"] + 2 * n * bm["dphi_bytes_per_site"]
    for _ in range(args.warmup):
        oracle_step(cfg, U, psi, 1, n)
    t0 = time.perf_counter()
    threads = 1
    for _ in range(args.steps):
        _, threads = oracle_step(cfg, U, psi, 1, n)
    dt = (time.perf_counter() - t0) / args.steps
    val = step_bytes / dt / 1e9
    sample = (f"{cfg['name']}: per step the link map on the first {2 * n} lattice sites and Dphi_eo on the first {n} "
              f"output sites of each parity (of {bm['V'] // 2}), fp64")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": cfg["name"], "dims": list(cfg["dims"]), "bc": list(BC)},
        "cpu_baseline": {"value": val, "unit": "GB/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gflops": 2 * n * bm["dphi_flops_per_site"] / dt / 1e9,
    }))


def run_ours(args, cfg, prec):
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

    bm = byte_model(cfg, prec)
    P = hr.PREC_NAMES[prec]
    cfg_r = dict(cfg, seeds=replica_seeds(cfg["seeds"], rank))
    U, psi = make_fields(cfg_r)
    lat = hr.Lattice(cfg["dims"], BC, cfg["N"], cfg["rep"], device=local)
    fund = lat.gauge(False, P)
    links = lat.gauge(True, P)
    lat.import_gauge(fund, U)
    sp_in = [lat.spinor(P) for _ in (0, 1)]
    sp_out = [lat.spinor(P) for _ in (0, 1)]
    for p in (0, 1):
        lat.import_spinor(sp_in[p], P, psi[p], 1 - p)
    torch.cuda.synchronize()

    def step(events=None):
        if events is not None:
            events[0].record()
        lat.represent_links(links, fund)
        if events is not None:
            events[1].record()
        lat.dphi_eo(sp_out[0], sp_in[0], links, 0)
        if events is not None:
            events[2].record()
        lat.dphi_eo(sp_out[1], sp_in[1], links, 1)
        if events is not None:
            events[3].record()

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    sync_all()
    n0 = hr.hr_launch_count()
    with ClockSampler(local) as clk:
        t_begin = torch.cuda.Event(enable_timing=True)
        t_end = torch.cuda.Event(enable_timing=True)
        t_begin.record()
        for k in range(args.steps):
            step(ev[k])
        t_end.record()
        sync_all()
    launches = hr.hr_launch_count() - n0
    ms_total = t_begin.elapsed_time(t_end)
    rep_ms = statistics.mean(e[0].elapsed_time(e[1]) for e in ev)
    dphi_ms = statistics.mean([e[1].elapsed_time(e[2]) for e in ev] + [e[2].elapsed_time(e[3]) for e in ev])
    dphi_ms_min = min([e[1].elapsed_time(e[2]) for e in ev] + [e[2].elapsed_time(e[3]) for e in ev])
    ms_total = max_over_ranks(ms_total, world, "cuda")
    ms_step = ms_total / args.steps
    step_bytes = 4 * bm["V"] * bm["represent_bytes_per_link"] + bm["V"] * bm["dphi_bytes_per_site"]
    value = whole_job_value(step_bytes, world, ms_step * 1e-3)

    # companion measurement (NOT part of `value`): the same two Dphi_eo calls reading row-compressed fundamental links
    # (SU(3) 12 of 18 reals, SU(2) 4 of 8, SU(2) adjoint built from 4 reals) -- fewer bytes than
    # north_star's contract counts, so it is reported beside the headline, with its own byte count
    rows_info = None
    if cfg["N"] <= 3 and (cfg["rep"] == "fund" or (cfg["rep"] == "adj" and cfg["N"] == 2)):
        rows = lat.gauge(2, P)
        lat.compress_links(rows, fund)
        for _ in range(args.warmup):
            lat.dphi_eo(sp_out[0], sp_in[0], rows, 0)
            lat.dphi_eo(sp_out[1], sp_in[1], rows, 1)
        sync_all()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        for _ in range(args.steps):
            lat.dphi_eo(sp_out[0], sp_in[0], rows, 0)
            lat.dphi_eo(sp_out[1], sp_in[1], rows, 1)
        r1.record()
        sync_all()
        rows_ms = max_over_ranks(r0.elapsed_time(r1) / (2 * args.steps), world, "cuda")
        w = 8 if prec == "f64" else 4
        lrows = 2 * cfg["N"] * (cfg["N"] - 1) * w
        need = 8 * lrows + 2 * bm["S"]
        rows_info = {"ms_per_launch": rows_ms, "link_bytes": lrows, "needed_bytes_per_site": need,
                     "needed_gbs": bm["V"] // 2 * need / (rows_ms * 1e-3) / 1e9,
                     "contract_gbs": bm["V"] // 2 * bm["dphi_bytes_per_site"] / (rows_ms * 1e-3) / 1e9,
                     "speedup_vs_full_links": dphi_ms / rows_ms}

    # end to end through the host entry points (pinned host buffers; copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        cdt = torch.complex128 if prec == "f64" else torch.complex64
        hU = torch.from_numpy(U).to(cdt).pin_memory()
        hin = [torch.from_numpy(psi[p]).to(cdt).pin_memory() for p in (0, 1)]
        hout = [torch.empty_like(hin[p]).pin_memory() for p in (0, 1)]
        st = lat.stream()

        def e2e_step():
            hr.hr_gauge_import(fund, hU, P, st)
            hr.hr_represent_links(links, fund, st)
            for p in (0, 1):
                hr.hr_dphi_eo_host(lat.ctx, hout[p], hin[p], P, links, p, st)

        ke = max(3, min(args.steps, 5))
        for _ in range(2):
            e2e_step()
        sync_all()
        t0 = time.perf_counter()
        for _ in range(ke):
            e2e_step()
        sync_all()
        dt = (time.perf_counter() - t0) / ke
        dt = max_over_ranks(dt, world, "cuda")
        h2d = hU.numel() * hU.element_size() + sum(h.numel() * h.element_size() for h in hin)
        d2h = sum(h.numel() * h.element_size() for h in hout)
        e2e = {"value": whole_job_value(step_bytes, world, dt), "unit": "GB/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "ms_per_step": dt * 1e3, "steps": ke}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak()
    dphi_bytes = bm["V"] // 2 * bm["dphi_bytes_per_site"]
    achieved = dphi_bytes / (dphi_ms * 1e-3) / 1e9
    traffic = ncu_traffic(cfg["name"], prec)
    out = {
        "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": prec,
        "data": "synthetic",
        "config": {"workload": cfg["name"], "dims": list(cfg["dims"]), "bc": list(BC), "N": cfg["N"], "rep": cfg["rep"],
                   "d_R": bm["d"], "step": "hr_represent_links + hr_dphi_eo(parity 0) + hr_dphi_eo(parity 1)",
                   "l2": "inputs exceed L2 (no flush)", "kernel_variant": lat.variant_name(P),
                   "parallelism": "replicas" if world > 1 else "single"},
        "clocks": clk.summary(),
        "e2e": e2e,
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "kernel": "dphi_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                     "bytes_per_launch": dphi_bytes, "ms_per_launch": dphi_ms, "ms_per_launch_min": dphi_ms_min,
                     "frac_of_8TBs_nominal": achieved / 8000.0,
                     "compulsory_gbs": bm["V"] // 2 * bm["compulsory_bytes_per_site"] / (dphi_ms * 1e-3) / 1e9},
        "dphi_gflops": bm["V"] // 2 * bm["dphi_flops_per_site"] / (dphi_ms * 1e-3) / 1e9,
        "rows_links": rows_info,
        "represent_ms": rep_ms,
        "represent_gbs": 4 * bm["V"] * bm["represent_bytes_per_link"] / (rep_ms * 1e-3) / 1e9,
    }
    if not args.no_cpu_baseline and world == 1:
        reps = 3
        dt, threads = oracle_step(cfg, U, psi, reps)
        bm64 = byte_model(cfg, "f64")
        sb64 = 4 * bm64["V"] * bm64["represent_bytes_per_link"] + bm64["V"] * bm64["dphi_bytes_per_site"]
        out["cpu_baseline"] = {"value": sb64 / dt / 1e9, "unit": "GB/s", "cores": threads, "kind": "oracle",
                               "sample": f"full {cfg['name']} volume, fp64, one step (represent + both parities), best of {reps}",
                               "ms_per_step": dt * 1e3}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=sorted(CONFIGS))
    ap.add_argument("--prec", default="f64", choices=["f64", "f32"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    cfg = CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg, args.prec)
    else:
        args.warmup = max(args.warmup, 3)
        run_ours(args, cfg, args.prec)


if __name__ == "__main__":
    main()
