#!/usr/bin/env python
"""Volume dependence of Dphi_eo and of a streaming copy ("add 16^4, 32^4, 48^4 points
for the curve, cf. Fig. 7's volume dependence, PAPER.md:116"; at small local lattices "the execution time
is dominated by the kernel call overheads").

    python -m paper_2405_19294_b200.bench_volume [--reps 200]

SU(3) fundamental, near-identity links (config 5's recipe), L^4 lattices, fp64 and fp32.  One JSON line per point:
time per hr_dphi_eo launch (CUDA events, back to back, alternating parity, 4 rotating buffer sets), contract and
compulsory GB/s, and hr_spinor_copy on the same half field."""
from __future__ import annotations

import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    import torch
    import bench as B
    import lattice_inputs as li
    import paper_2405_19294_b200 as hr

    ap = argparse.ArgumentParser()
    ap.add_argument("--reps", type=int, default=200)
    ap.add_argument("--sizes", default="8,12,16,24,32,48,64")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("bench_volume: no CUDA device; the product path has no CPU fallback")
    peak, _ = B.measured_peak()
    for L in [int(x) for x in args.sizes.split(",")]:
        dims = (L, L, L, L)
        U = li.near_identity_links(1005, 3, dims, 0.3)
        vh = li.volume(dims) // 2
        psi = li.gaussian_spinor(2005, vh, 3)
        for prec in ("f64", "f32"):
            P = hr.PREC_NAMES[prec]
            w = 8 if prec == "f64" else 4
            S, Lb = 24 * w, 18 * w
            lat = hr.Lattice(dims, B.BC, 3, "fund")
            links = lat.gauge(True, P)
            lat.import_gauge(links, U)
            a = [lat.spinor(P) for _ in range(4)]
            o = [lat.spinor(P) for _ in range(4)]
            for k in range(4):
                lat.import_spinor(a[k], P, psi, 0)
            st = lat.stream()

            def timed(fn):
                for k in range(10):
                    fn(k)
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for k in range(args.reps):
                    fn(k)
                e1.record()
                torch.cuda.synchronize()
                return e0.elapsed_time(e1) / args.reps

            ms = timed(lambda k: hr.hr_dphi_eo(o[k % 4], a[k % 4], links, k & 1, st))
            msc = timed(lambda k: hr.hr_spinor_copy(lat.ctx, P, o[k % 4], a[k % 4], st))
            print(json.dumps({"workload": f"SU(3) fund {L}^4", "dtype": prec, "sites": vh, "dphi_us": ms * 1e3,
                              "contract_gbs": vh * (8 * Lb + 9 * S) / (ms * 1e-3) / 1e9,
                              "compulsory_gbs": vh * (8 * Lb + 2 * S) / (ms * 1e-3) / 1e9,
                              "compulsory_frac_of_copy_peak": vh * (8 * Lb + 2 * S) / (ms * 1e-3) / 1e9 / peak,
                              "copy_us": msc * 1e3, "copy_gbs": vh * 2 * S / (msc * 1e-3) / 1e9,
                              "field_mb": (8 * Lb + 2 * S) * vh / 1e6}))
            lat.close()


if __name__ == "__main__":
    main()
