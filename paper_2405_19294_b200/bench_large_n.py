#!/usr/bin/env python
"""Dphi_eo against the dimension d_R of the fermion representation, memory moved held about constant by shrinking the
lattice -- the experiment of the paper's Fig. 6 ("unimproved kernel blows up; improved is stable"),
here for every kernel flavour the library compiles for that d_R:

    site / site_ef   one thread per site (the paper's default kernel)
    pair / pair_ef   two threads per site (d_R <= 8)
    colour           one thread per (site, colour row): the large-d_R kernel (csrc/dphi_cp_kernel.cuh)

    python -m paper_2405_19294_b200.bench_large_n [--reps 50]

Haar links, gaussian spinors, represented link field.  One JSON line per (representation, precision, variant): time per
hr_dphi_eo launch (CUDA events, back to back, alternating parity, rotating buffer sets), compulsory GB/s (every byte
once) and GFLOP/s with bench.py's per-site model."""
from __future__ import annotations

import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

# (N, rep, dims): compulsory bytes 1.6-1.9 GB in fp64 for every row
CASES = [(2, "fund", (128, 32, 32, 32)), (3, "fund", (64, 32, 32, 32)), (4, "fund", (40, 32, 32, 32)),
         (3, "sym", (48, 24, 24, 24)), (3, "adj", (48, 24, 24, 24)), (4, "sym", (56, 16, 16, 16)), (4, "adj", (48, 16, 16, 16))]
NAMES = ["site", "site_ef", "pair", "pair_ef", "site_l1", "site_pf", "colour"]


def main():
    import torch
    import bench as B
    import lattice_inputs as li
    import paper_2405_19294_b200 as hr

    ap = argparse.ArgumentParser()
    ap.add_argument("--reps", type=int, default=50)
    ap.add_argument("--variants", default="0,1,2,3,6")
    ap.add_argument("--cases", default="", help="comma list of d_R values to run (default: all)")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("bench_large_n: no CUDA device; the product path has no CPU fallback")
    peak, _ = B.measured_peak()
    only = [int(x) for x in args.cases.split(",") if x]
    for N, rep, dims in CASES:
        if only and B.REP_DIM[rep](N) not in only:
            continue
        U = li.haar_links(1006, N, dims)
        vh = li.volume(dims) // 2
        for prec in ("f64", "f32"):
            P = hr.PREC_NAMES[prec]
            bm = B.byte_model({"N": N, "rep": rep, "dims": dims}, prec)
            lat = hr.Lattice(dims, B.BC, N, rep)
            fund = lat.gauge(False, P)
            lat.import_gauge(fund, U)
            links = lat.gauge(True, P)
            lat.represent_links(links, fund)
            psi = li.gaussian_spinor(2006, vh, bm["d"])
            a = [lat.spinor(P) for _ in range(2)]
            o = [lat.spinor(P) for _ in range(2)]
            for k in range(2):
                lat.import_spinor(a[k], P, psi, 0)
            st = lat.stream()
            default = hr.hr_dphi_variant_name(lat.ctx, P)
            for v in [int(x) for x in args.variants.split(",")]:
                try:
                    lat.set_tuning("variant", v)
                    hr.hr_dphi_eo(o[0], a[0], links, 0, st)
                except hr.HrError:
                    continue
                for k in range(5):
                    hr.hr_dphi_eo(o[k % 2], a[k % 2], links, k & 1, st)
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for k in range(args.reps):
                    hr.hr_dphi_eo(o[k % 2], a[k % 2], links, k & 1, st)
                e1.record()
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1) / args.reps
                cg = vh * bm["compulsory_bytes_per_site"] / (ms * 1e-3) / 1e9
                print(json.dumps({"workload": f"SU({N}) {rep} {dims[1]}^3x{dims[0]}", "d_R": bm["d"], "dtype": prec,
                                  "variant": NAMES[v], "default": NAMES[v] == default, "ms": ms,
                                  "compulsory_mb": vh * bm["compulsory_bytes_per_site"] / 1e6, "compulsory_gbs": cg,
                                  "compulsory_frac_of_copy_peak": cg / peak,
                                  "gflops": vh * bm["dphi_flops_per_site"] / (ms * 1e-3) / 1e9}), flush=True)
            lat.close()
            torch.cuda.empty_cache()


if __name__ == "__main__":
    main()
