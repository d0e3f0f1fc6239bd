#!/usr/bin/env python
"""Measurement of the NEXT-1 rows: the paper's second benchmark, the spinor linear
algebra of PAPER.md:108-120 / Fig. 7 ("Copy spinor field", "g5 application", "g5 mulc add assign", norms and
inner products; SU(3) fundamental), plus hr_dhat and one CG iteration.

    python -m paper_2405_19294_b200.bench_solver [--config 2|3|4|5] [--prec f64|f32] [--reps 50]

Prints one JSON line per operation: algorithmic bytes (S = spinor bytes per site, Vh sites: copy/g5 2S,
g5_mulc_add_assign 3S, norm2 1S, dot 2S; Dhat 2(8L+2S)+S; CG iteration 4(8L+2S) + 2S + 8S), the time per call
from CUDA events on the launching stream (back to back, fields larger than L2 rotate through 4 buffer sets),
GB/s and the fraction of the measured copy peak (MEASURED_PEAKS.json).  Inputs: the seeded synthetic fields
of bench.py's configs.  bench.py stays the headline; this script is the Fig. 7 companion."""
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
    import paper_2405_19294_b200 as hr

    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--prec", default="f64", choices=["f64", "f32"])
    ap.add_argument("--reps", type=int, default=50)
    ap.add_argument("--m0", type=float, default=0.1)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("bench_solver: no CUDA device; the product path has no CPU fallback")
    cfg = B.CONFIGS[args.config]
    bm = B.byte_model(cfg, args.prec)
    P = hr.PREC_NAMES[args.prec]
    peak, peak_src = B.measured_peak()
    U, psi = B.make_fields(cfg)
    lat = hr.Lattice(cfg["dims"], B.BC, cfg["N"], cfg["rep"])
    fund, links = lat.gauge(False, P), lat.gauge(True, P)
    lat.import_gauge(fund, U)
    lat.represent_links(links, fund)
    nset = 4
    sets = []
    for k in range(nset):
        a, b, c = lat.spinor(P), lat.spinor(P), lat.spinor(P)
        lat.import_spinor(a, P, psi[0], 0)
        lat.import_spinor(b, P, psi[1], 0)
        c.zero_()
        sets.append((a, b, c))
    ctx, st = lat.ctx, lat.stream()
    res = torch.zeros(2, dtype=torch.float64, device="cuda")
    S, L, vh = bm["S"], bm["L"], bm["V"] // 2
    dphi_c = 8 * L + 2 * S

    def timed(fn, reps):
        for k in range(5):
            fn(k)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for k in range(reps):
            fn(k)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    ops = [
        ("copy", 2 * S, lambda k: hr.hr_spinor_copy(ctx, P, sets[k % nset][2], sets[k % nset][0], st)),
        ("g5", 2 * S, lambda k: hr.hr_spinor_g5(ctx, P, sets[k % nset][2], sets[k % nset][0], st)),
        ("g5_mulc_add_assign", 3 * S, lambda k: hr.hr_spinor_g5_mulc_add_assign(ctx, P, sets[k % nset][2], 0.3 - 0.2j, sets[k % nset][0], st)),
        ("norm2", S, lambda k: hr.hr_spinor_norm2(ctx, P, sets[k % nset][0], st, result=res)),
        ("dot", 2 * S, lambda k: hr.hr_spinor_dot(ctx, P, sets[k % nset][0], sets[k % nset][1], st, result=res)),
        ("dhat", 2 * dphi_c + S, lambda k: hr.hr_dhat(args.m0, 1, sets[k % nset][2], sets[k % nset][0], sets[k % nset][1], links, st)),
    ]
    ops.append(("dphi_eo (represented links, compulsory bytes 8L+2S)", dphi_c,
                lambda k: hr.hr_dphi_eo(sets[k % nset][2], sets[k % nset][0], links, k & 1, st)))
    if cfg["rep"] in ("sym", "asym"):
        # NEXT-3: the same operator from the FUNDAMENTAL links (8F+2S bytes per site actually needed)
        F = bm["F"]
        ops.append(("dphi_eo on-the-fly (fundamental links, bytes 8F+2S)", 8 * F + 2 * S,
                    lambda k: hr.hr_dphi_eo(sets[k % nset][2], sets[k % nset][0], fund, k & 1, st)))
        ops.append(("dhat on-the-fly", 2 * (8 * F + 2 * S) + S,
                    lambda k: hr.hr_dhat(args.m0, 1, sets[k % nset][2], sets[k % nset][0], sets[k % nset][1], fund, st)))
    if cfg["N"] <= 3 and (cfg["rep"] == "fund" or (cfg["rep"] == "adj" and cfg["N"] == 2)):
        # row-compressed fundamental links: bytes 8 Lrows + 2S actually needed
        rows = lat.gauge(2, P)
        lat.compress_links(rows, fund)
        lrows = 2 * cfg["N"] * (cfg["N"] - 1) * (8 if args.prec == "f64" else 4)
        ops.append(("dphi_eo from row-compressed links (bytes 8 Lrows + 2S)", 8 * lrows + 2 * S,
                    lambda k: hr.hr_dphi_eo(sets[k % nset][2], sets[k % nset][0], rows, k & 1, st)))
        ops.append(("dhat from row-compressed links", 2 * (8 * lrows + 2 * S) + S,
                    lambda k: hr.hr_dhat(args.m0, 1, sets[k % nset][2], sets[k % nset][0], sets[k % nset][1], rows, st)))
    # NEXT-2: the slab pipeline of ONE rank (its neighbour is itself): what the decomposition costs on top of
    # a plain Dphi_eo of the same local volume.  Algorithmic bytes: pack reads 2 slices of spinors and 1 of links
    # and writes 2 half-spinor faces; apply reads them back, 1 slice of links, and read-modify-writes 2 slices.
    nface = vh // cfg["dims"][0]
    nb = hr.hr_halo_bytes(ctx, P)
    hb = [torch.empty(nb, dtype=torch.uint8, device="cuda") for _ in range(2)]
    Lk = bm["L"]
    ops.append(("halo_pack", None, lambda k: hr.hr_dphi_eo_halo_pack(hb[0], hb[1], sets[k % nset][0], links, k & 1, st)))
    ops.append(("dphi_eo_interior", dphi_c, lambda k: hr.hr_dphi_eo_interior(sets[k % nset][2], sets[k % nset][0], links, k & 1, st)))
    ops.append(("halo_apply", None, lambda k: hr.hr_dphi_eo_halo_apply(sets[k % nset][2], hb[0], hb[1], links, k & 1, True, True, st)))
    face_bytes = {"halo_pack": nface * (2 * S + Lk + S), "halo_apply": nface * (S + Lk + 4 * S)}
    face_sites = {"halo_pack": nface, "halo_apply": nface}
    # 4-D block decomposition: the face kernels of the other directions (strided faces) and the interior launch with all
    # four directions masked
    fb = {}
    for mu, nm in ((1, "x"), (2, "y"), (3, "z")):
        nf_mu = vh // cfg["dims"][mu]
        fb[mu] = [torch.empty(hr.hr_face_bytes(ctx, P, mu), dtype=torch.uint8, device="cuda") for _ in range(2)]
        ops.append((f"face_pack {nm}", None, lambda k, mu=mu: hr.hr_dphi_eo_face_pack(mu, fb[mu][0], fb[mu][1], sets[k % nset][0], links, k & 1, st)))
        ops.append((f"face_apply {nm}", None, lambda k, mu=mu: hr.hr_dphi_eo_face_apply(mu, sets[k % nset][2], fb[mu][0], fb[mu][1], links, k & 1, True, True, st)))
        face_bytes[f"face_pack {nm}"] = nf_mu * (2 * S + Lk + S)
        face_bytes[f"face_apply {nm}"] = nf_mu * (S + Lk + 4 * S)
        face_sites[f"face_pack {nm}"] = face_sites[f"face_apply {nm}"] = nf_mu
    ops.append(("dphi_eo_interior, all four directions masked", dphi_c,
                lambda k: hr.hr_dphi_eo_interior_mask(sets[k % nset][2], sets[k % nset][0], links, k & 1, 15, st)))
    # NEXT-4: clover term.  build: reads the represented links (each link is used by many leaves; algorithmic bytes
    # 4L + C per site), apply as part of hr_dirac_clover: two Dphi launches with the mass term + two site-local launches
    # (C + 3S per site each); bytes per site of the full lattice: 2(8L+3S)/2 ... reported per output site of one parity.
    Cb = 8 * bm["d"] ** 2 * (8 if args.prec == "f64" else 4)
    cl = torch.empty(hr.hr_clover_bytes(ctx, P), dtype=torch.uint8, device="cuda")
    full_in, full_out = lat.spinor(P, full=True), lat.spinor(P, full=True)
    full_in.zero_()
    ops.append(("clover_build (per site of the FULL lattice: 4L + C)", 2 * (4 * L + Cb), lambda k: hr.hr_clover_build(cl, links, 1.0, st)))
    ops.append(("dirac (both parities: 2(8L+3S) per site pair)", 2 * (dphi_c + S), lambda k: hr.hr_dirac(args.m0, full_out, full_in, links, st)))
    ops.append(("dirac_clover (both parities: 2(8L+3S + C+3S))", 2 * (dphi_c + S + Cb + 3 * S), lambda k: hr.hr_dirac_clover(args.m0, full_out, full_in, links, cl, st)))
    # even-odd preconditioned clover operator: 2 Dphi + 2 site-local launches;
    # algorithmic bytes per even site: 2(8L+2S) + (C+2S) + (C+3S)
    Ainv = torch.empty(hr.hr_clover_bytes(ctx, P), dtype=torch.uint8, device="cuda")
    Asite = torch.empty(hr.hr_clover_bytes(ctx, P), dtype=torch.uint8, device="cuda")
    hr.hr_clover_build(Asite, links, 1.0, st)
    hr.hr_clover_finalize(ctx, P, Asite, Ainv, args.m0, st)
    t2 = lat.spinor(P)
    ops.append(("dhat_clover", 2 * dphi_c + 2 * Cb + 5 * S,
                lambda k: hr.hr_dhat_clover(sets[k % nset][2], sets[k % nset][0], sets[k % nset][1], t2, links, Asite, Ainv, st)))
    common = {"workload": cfg["name"], "dtype": args.prec, "peak_gbs": peak, "peak_source": peak_src, "sites": vh}
    for name, bps, fn in ops:
        ms = timed(fn, args.reps)
        if bps is None:   # face kernels: bytes are per launch, not per site of the volume
            gbs = face_bytes[name] / (ms * 1e-3) / 1e9
            print(json.dumps(dict(common, op=name, bytes_per_launch=face_bytes[name], face_sites=face_sites[name], ms=ms, gbs=gbs, frac=gbs / peak)))
            continue
        gbs = bps * vh / (ms * 1e-3) / 1e9
        print(json.dumps(dict(common, op=name, bytes_per_site=bps, ms=ms, gbs=gbs, frac=gbs / peak)))

    # one CG iteration, measured on a solve that cannot converge (tol = 0): time / iterations
    maxiter = 40
    ws = lat.cg_workspace(P, maxiter)
    x = lat.spinor(P)
    lat.cg_dhat(args.m0, x, sets[0][0], links, 0.0, 4, ws)
    torch.cuda.synchronize()
    n0 = hr.hr_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    it, res2, _ = lat.cg_dhat(args.m0, x, sets[0][0], links, 0.0, maxiter, ws)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / it
    bps = 4 * dphi_c + 2 * S + 8 * S
    gbs = bps * vh / (ms * 1e-3) / 1e9
    print(json.dumps(dict(common, op="cg_iteration", bytes_per_site=bps, ms=ms, gbs=gbs, frac=gbs / peak, iterations=it,
                          launches_per_iteration=(hr.hr_launch_count() - n0) / it, rel_res2=res2)))
    # BiCGstab: one iteration = 4 Dphi launches + 3 vector kernels + 1 dot; algorithmic bytes
    # 4(8L+2S) + 2S (self reads of the two fused epilogues) + 16S of vector passes
    wsb = torch.empty(hr.hr_bicgstab_workspace_bytes(ctx, P, maxiter), dtype=torch.uint8, device="cuda")
    hr.hr_bicgstab_dhat(ctx, args.m0, x, sets[0][0], links, 0.0, 4, wsb, st)
    torch.cuda.synchronize()
    n0 = hr.hr_launch_count()
    e0.record()
    it, res2, _ = hr.hr_bicgstab_dhat(ctx, args.m0, x, sets[0][0], links, 0.0, maxiter, wsb, st)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / it
    bps = 4 * dphi_c + 2 * S + 16 * S
    gbs = bps * vh / (ms * 1e-3) / 1e9
    print(json.dumps(dict(common, op="bicgstab_iteration", bytes_per_site=bps, ms=ms, gbs=gbs, frac=gbs / peak, iterations=it,
                          launches_per_iteration=(hr.hr_launch_count() - n0) / it)))
    # time to solution, same right-hand side, relative residual 1e-8 (fp64) / 1e-5 (fp32): CG on the normal equations
    # vs BiCGstab on Dhat vs the gamma5-QMR on Dhat (host-driven scalars)
    tol = 1e-8 if args.prec == "f64" else 1e-5
    for name, fn in (("cg_solve", lambda: lat.cg_dhat(args.m0, x, sets[0][0], links, tol, 2000, lat.cg_workspace(P, 2000))),
                     ("bicgstab_solve", lambda: hr.hr_bicgstab_dhat(ctx, args.m0, x, sets[0][0], links, tol, 2000,
                                                                    torch.empty(hr.hr_bicgstab_workspace_bytes(ctx, P, 2000), dtype=torch.uint8, device="cuda"), st)),
                     ("qmr_solve", lambda: hr.hr_qmr_dhat(ctx, args.m0, x, sets[0][0], links, tol, 2000,
                                                          torch.empty(hr.hr_qmr_workspace_bytes(ctx, P), dtype=torch.uint8, device="cuda"), st))):
        torch.cuda.synchronize()
        e0.record()
        it, res2, _ = fn()
        e1.record()
        torch.cuda.synchronize()
        print(json.dumps(dict(common, op=name, tol=tol, iterations=it, rel_res2=res2, ms=e0.elapsed_time(e1), bytes_per_site=0, gbs=0.0, frac=0.0)))
    if args.prec == "f64":
        # mixed precision: fp32 inner BiCGstab (to 1e-4) + fp64 true residual, same right-hand side and target
        l32 = lat.gauge(True, hr.HR_F32)
        lat.represent_links(l32, fund)
        wsm = torch.empty(hr.hr_mixed_workspace_bytes(ctx, 2000), dtype=torch.uint8, device="cuda")
        hr.hr_bicgstab_dhat_mixed(ctx, args.m0, x, sets[0][0], links, l32, tol, 1e-4, 2000, wsm, st)
        torch.cuda.synchronize()
        e0.record()
        it, outer, res2 = hr.hr_bicgstab_dhat_mixed(ctx, args.m0, x, sets[0][0], links, l32, tol, 1e-4, 2000, wsm, st)
        e1.record()
        torch.cuda.synchronize()
        print(json.dumps(dict(common, op="mixed_bicgstab_solve", tol=tol, iterations=it, outer_steps=outer, rel_res2=res2,
                              ms=e0.elapsed_time(e1), bytes_per_site=0, gbs=0.0, frac=0.0)))
    lat.close()


if __name__ == "__main__":
    main()
