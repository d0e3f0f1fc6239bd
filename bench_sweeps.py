#!/usr/bin/env python
"""bench_sweeps.py -- companion measurements of bench.py (which stays the headline): the sweeps behind the tables of
DESIGN.md and profiles/.  They import bench.py's configs, byte model and input recipe; nothing here is product code.

    python bench_sweeps.py volume  [--reps 200] [--sizes 8,12,...]      Dphi_eo and a copy against the lattice volume
    python bench_sweeps.py large_n [--reps 50] [--variants ...]         Dphi_eo against d_R at constant memory moved (Fig. 6)
    python bench_sweeps.py solver  [--config 2] [--prec f64] [--reps 50] spinor linear algebra, Dhat, solvers (Fig. 7)
    python bench_sweeps.py variants --cases '[...]' --sweeps '[...]'     kernel variants / tunings under sustained clocks
"""
from __future__ import annotations

import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

def volume(argv):
    """Volume dependence of Dphi_eo and of a streaming copy ("add 16^4, 32^4, 48^4 points
    for the curve, cf. Fig. 7's volume dependence, PAPER.md:116"; at small local lattices "the execution time
    is dominated by the kernel call overheads").
    
        python bench_sweeps.py volume [--reps 200] [--graph]
    
    SU(3) fundamental, near-identity links (config 5's recipe), L^4 lattices, fp64 and fp32.  One JSON line per point:
    time per hr_dphi_eo launch (CUDA events, back to back, alternating parity, 4 rotating buffer sets), contract and
    compulsory GB/s, and hr_spinor_copy on the same half field."""
    import torch
    import bench as B
    import lattice_inputs as li
    import paper_2405_19294_b200 as hr

    ap = argparse.ArgumentParser(prog="bench_sweeps.py volume")
    ap.add_argument("--reps", type=int, default=200)
    ap.add_argument("--sizes", default="8,12,16,24,32,48,64")
    ap.add_argument("--graph", action="store_true", help="also time 50 launches replayed from one CUDA graph (no host work between kernels)")
    args = ap.parse_args(argv)
    if not torch.cuda.is_available():
        raise SystemExit("bench_sweeps volume: no CUDA device; the product path has no CPU fallback")
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

            def timed_graph(fn, n=50):
                # the same launches captured ONCE into a CUDA graph and replayed: no host work between the kernels, i.e. the
                # time the GPU itself needs per launch (what a solver that replays a captured iteration sees)
                s = torch.cuda.Stream()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.stream(s):
                    fn_s = lambda k: fn(k, s.cuda_stream)
                    for k in range(4):
                        fn_s(k)
                    s.synchronize()
                    with torch.cuda.graph(g, stream=s):
                        for k in range(n):
                            fn_s(k)
                    g.replay()
                    s.synchronize()
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(s)
                    for _ in range(max(1, args.reps // n)):
                        g.replay()
                    e1.record(s)
                    s.synchronize()
                return e0.elapsed_time(e1) / (max(1, args.reps // n) * n)

            ms = timed(lambda k: hr.hr_dphi_eo(o[k % 4], a[k % 4], links, k & 1, st))
            msc = timed(lambda k: hr.hr_spinor_copy(lat.ctx, P, o[k % 4], a[k % 4], st))
            msg = timed_graph(lambda k, sp: hr.hr_dphi_eo(o[k % 4], a[k % 4], links, k & 1, sp)) if args.graph else None
            print(json.dumps({"workload": f"SU(3) fund {L}^4", "dtype": prec, "sites": vh, "dphi_us": ms * 1e3,
                              "dphi_graph_us": None if msg is None else msg * 1e3, "kernel": lat.variant_name(P),
                              "contract_gbs": vh * (8 * Lb + 9 * S) / (ms * 1e-3) / 1e9,
                              "compulsory_gbs": vh * (8 * Lb + 2 * S) / (ms * 1e-3) / 1e9,
                              "compulsory_frac_of_copy_peak": vh * (8 * Lb + 2 * S) / (ms * 1e-3) / 1e9 / peak,
                              "copy_us": msc * 1e3, "copy_gbs": vh * 2 * S / (msc * 1e-3) / 1e9,
                              "field_mb": (8 * Lb + 2 * S) * vh / 1e6}))
            lat.close()



# (N, rep, dims): compulsory bytes 1.6-1.9 GB in fp64 for every row
CASES = [(2, "fund", (128, 32, 32, 32)), (3, "fund", (64, 32, 32, 32)), (4, "fund", (40, 32, 32, 32)),
         (3, "sym", (48, 24, 24, 24)), (3, "adj", (48, 24, 24, 24)), (4, "sym", (56, 16, 16, 16)), (4, "adj", (48, 16, 16, 16))]
NAMES = ["site", "site_ef", "pair", "pair_ef", "site_l1", "site_pf", "colour", "bulk", "bulk2", "bulkx", "bulkx2"]


def large_n(argv):
    """Dphi_eo against the dimension d_R of the fermion representation, memory moved held about constant by shrinking the
    lattice -- the experiment of the paper's Fig. 6 ("unimproved kernel blows up; improved is stable"),
    here for every kernel flavour the library compiles for that d_R:
    
        site / site_ef   one thread per site (the paper's default kernel)
        pair / pair_ef   two threads per site (d_R <= 8)
        colour           one thread per (site, colour row): the large-d_R kernel (csrc/dphi_cp_kernel.cuh)
    
        python bench_sweeps.py large_n [--reps 50]
    
    Haar links, gaussian spinors, represented link field.  One JSON line per (representation, precision, variant): time per
    hr_dphi_eo launch (CUDA events, back to back, alternating parity, rotating buffer sets), compulsory GB/s (every byte
    once) and GFLOP/s with bench.py's per-site model."""
    import torch
    import bench as B
    import lattice_inputs as li
    import paper_2405_19294_b200 as hr

    ap = argparse.ArgumentParser(prog="bench_sweeps.py large_n")
    ap.add_argument("--reps", type=int, default=50)
    ap.add_argument("--variants", default="0,1,2,3,6")
    ap.add_argument("--cases", default="", help="comma list of d_R values to run (default: all)")
    args = ap.parse_args(argv)
    if not torch.cuda.is_available():
        raise SystemExit("bench_sweeps large_n: no CUDA device; the product path has no CPU fallback")
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



def solver(argv):
    """Measurement of the NEXT-1 rows: the paper's second benchmark, the spinor linear
    algebra of PAPER.md:108-120 / Fig. 7 ("Copy spinor field", "g5 application", "g5 mulc add assign", norms and
    inner products; SU(3) fundamental), plus hr_dhat and one CG iteration.
    
        python bench_sweeps.py solver [--config 2|3|4|5] [--prec f64|f32] [--reps 50] [--dims t,x,y,z]
    
    Prints one JSON line per operation: algorithmic bytes (S = spinor bytes per site, Vh sites: copy/g5 2S,
    g5_mulc_add_assign 3S, norm2 1S, dot 2S; Dhat 2(8L+2S)+S; CG iteration 4(8L+2S) + 2S + 8S), the time per call
    from CUDA events on the launching stream (back to back, fields larger than L2 rotate through 4 buffer sets),
    GB/s and the fraction of the measured copy peak (MEASURED_PEAKS.json).  Inputs: the seeded synthetic fields
    of bench.py's configs.  bench.py stays the headline; this script is the Fig. 7 companion."""
    import torch
    import bench as B
    import paper_2405_19294_b200 as hr

    ap = argparse.ArgumentParser(prog="bench_sweeps.py solver")
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--prec", default="f64", choices=["f64", "f32"])
    ap.add_argument("--reps", type=int, default=50)
    ap.add_argument("--m0", type=float, default=0.1)
    ap.add_argument("--dims", default="", help="t,x,y,z: the config's gauge group and representation on another lattice")
    args = ap.parse_args(argv)
    if not torch.cuda.is_available():
        raise SystemExit("bench_sweeps solver: no CUDA device; the product path has no CPU fallback")
    cfg = dict(B.CONFIGS[args.config])
    if args.dims:
        cfg["dims"] = tuple(int(x) for x in args.dims.split(","))
        cfg["name"] = "%s on %s" % (cfg["name"], "x".join(str(x) for x in cfg["dims"]))
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
    if cfg["dims"][2] % 2 == 0:
        # the faces of all four directions in ONE launch each (hr_dphi_eo_faces_pack / _apply): bytes = the sum of the per-direction ones
        fb[0] = hb
        fup, fdn = {mu: fb[mu][0] for mu in range(4)}, {mu: fb[mu][1] for mu in range(4)}
        ops.append(("faces_pack t+x+y+z (one launch)", None, lambda k: hr.hr_dphi_eo_faces_pack(15, fup, fdn, sets[k % nset][0], links, k & 1, st)))
        ops.append(("faces_apply t+x+y+z (one launch)", None,
                    lambda k: hr.hr_dphi_eo_faces_apply(15, sets[k % nset][2], fup, fdn, links, k & 1, 15, 15, st)))
        face_bytes["faces_pack t+x+y+z (one launch)"] = face_bytes["halo_pack"] + sum(face_bytes[f"face_pack {nm}"] for nm in "xyz")
        face_bytes["faces_apply t+x+y+z (one launch)"] = face_bytes["halo_apply"] + sum(face_bytes[f"face_apply {nm}"] for nm in "xyz")
        face_sites["faces_pack t+x+y+z (one launch)"] = face_sites["faces_apply t+x+y+z (one launch)"] = nface + sum(vh // cfg["dims"][mu] for mu in (1, 2, 3))
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
    # the site-diagonal matrix is fused into the Dphi epilogue where the library does so (fp64, d_R <= 4, site kernels: 2 launches
    # instead of 4); the fused path moves FEWER bytes and gets its own model: 2(8L + 3S + C) against 2(8L + 3S) + 2(C + 3S)
    hr.hr_clover_build(cl, links, 1.0, st)
    n0 = hr.hr_launch_count()
    hr.hr_dirac_clover(args.m0, full_out, full_in, links, cl, st)
    fused = hr.hr_launch_count() - n0 == 2
    ops.append(("dirac_clover, FUSED epilogue (both parities: 2(8L+3S+C))" if fused else "dirac_clover (both parities: 2(8L+3S + C+3S))",
                2 * (dphi_c + S + Cb) if fused else 2 * (dphi_c + S + Cb + 3 * S),
                lambda k: hr.hr_dirac_clover(args.m0, full_out, full_in, links, cl, st)))
    # even-odd preconditioned clover operator: 2 Dphi + 2 site-local launches;
    # algorithmic bytes per even site: 2(8L+2S) + (C+2S) + (C+3S)
    Ainv = torch.empty(hr.hr_clover_bytes(ctx, P), dtype=torch.uint8, device="cuda")
    Asite = torch.empty(hr.hr_clover_bytes(ctx, P), dtype=torch.uint8, device="cuda")
    hr.hr_clover_build(Asite, links, 1.0, st)
    hr.hr_clover_finalize(ctx, P, Asite, Ainv, args.m0, st)
    t2 = lat.spinor(P)
    ops.append(("dhat_clover, FUSED epilogues (16L + 5S + 2C)" if fused else "dhat_clover (16L + 9S + 2C)",
                2 * 8 * L + 5 * S + 2 * Cb if fused else 2 * 8 * L + 9 * S + 2 * Cb,
                lambda k: hr.hr_dhat_clover(sets[k % nset][2], sets[k % nset][0], sets[k % nset][1], t2, links, Asite, Ainv, st)))
    common = {"workload": cfg["name"], "dtype": args.prec, "peak_gbs": peak, "peak_source": peak_src, "sites": vh}
    # in-place set-up steps of the clover term: each call starts from a pristine copy (made outside the timed events)
    wk, wki = torch.empty_like(cl), torch.empty_like(cl)

    def timed_fresh(fn, reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        tot = 0.0
        for k in range(reps + 2):
            wk.copy_(cl)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            if k >= 2:
                tot += e0.elapsed_time(e1)
        return tot / reps

    hr.hr_clover_build(cl, links, 1.0, st)
    for name, bps, fn in (("clover_exp (in place: 2C per site of the full lattice)", 2 * 2 * Cb, lambda: hr.hr_clover_exp(ctx, P, wk, args.m0, st)),
                          ("clover_finalize (A in place, A^-1 out: 3C per site of the full lattice)", 2 * 3 * Cb,
                           lambda: hr.hr_clover_finalize(ctx, P, wk, wki, args.m0, st))):
        ms = timed_fresh(fn, min(args.reps, 10))
        gbs = bps * vh / (ms * 1e-3) / 1e9
        print(json.dumps(dict(common, op=name, bytes_per_site=bps, ms=ms, gbs=gbs, frac=gbs / peak)))
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





def variants(argv):
    """Dphi_eo under SUSTAINED clocks for every kernel variant / tuning asked for (the sweep behind DESIGN.md's default
    table and profiles/r2_staging.md).  A B200 running this operator back to back sits at its 1 kW power cap with the
    SM clock near 1.4-1.7 GHz; a kernel timed in a short burst runs at 1.97 GHz and reads 5-10 % faster.  Protocol per
    point: 8 launches (burst), then half a bracket of warm-up launches and a bracket of `--secs` seconds timed with CUDA
    events while NVML samples the SM clock.

        python bench_sweeps.py variants --cases '[[5,"f64","repr"],[4,"f32","fund"],[2,"f64","rows",[64,32,32,32]]]' \
               --sweeps '[{},{"variant":7},{"variant":8,"bulk_ctas":2}]' [--secs 0.5]

    case = [bench.py config (or {"N": .., "rep": ..} with dims), precision, link source repr|fund|rows, optional dims]; a sweep entry sets hr_ctx_set_tuning keys
    (variant, block, xblock, bulk_rows, bulk_stages, bulk_ctas, bulk_strip; {} = library defaults).  Inputs: one t-pair of the
    config's seeded fields repeated along t (values do not influence timing).  One JSON line per point."""
    import statistics
    import time
    import numpy as np
    import pynvml
    import torch
    import bench as B
    import lattice_inputs as li
    import paper_2405_19294_b200 as hr

    ap = argparse.ArgumentParser(prog="bench_sweeps.py variants")
    ap.add_argument("--cases", required=True)
    ap.add_argument("--sweeps", default="[{}]")
    ap.add_argument("--secs", type=float, default=0.5)
    args = ap.parse_args(argv)
    if not torch.cuda.is_available():
        raise SystemExit("bench_sweeps variants: no CUDA device; the product path has no CPU fallback")
    pynvml.nvmlInit()
    H = pynvml.nvmlDeviceGetHandleByIndex(0)
    peak, _ = B.measured_peak()
    keys = ("variant", "block", "xblock", "bulk_rows", "bulk_stages", "bulk_ctas", "bulk_strip")

    def timed(fn):
        for k in range(3):
            fn(k)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for k in range(8):
            fn(k)
        e1.record()
        torch.cuda.synchronize()
        burst = e0.elapsed_time(e1) / 8
        n = max(10, int(args.secs * 1e3 / burst))
        for k in range(max(5, n // 2)):
            fn(k)
        e0.record()
        for k in range(n):
            fn(k)
        e1.record()
        mhz = []
        while not e1.query():
            mhz.append(pynvml.nvmlDeviceGetClockInfo(H, pynvml.NVML_CLOCK_SM))
            time.sleep(0.01)
        torch.cuda.synchronize()
        return burst, e0.elapsed_time(e1) / n, (statistics.median(mhz) if mhz else None)

    for case in json.loads(args.cases):
        cid, prec, src = case[:3]
        if isinstance(cid, dict):   # {"N": 4, "rep": "fund"}: a gauge group / representation outside BASELINE.json's configs
            cfg = dict(name="SU(%d) %s" % (cid["N"], cid["rep"]), kind="haar", seeds=(1007, 2007), **cid)
        else:
            cfg = dict(B.CONFIGS[cid])
        if len(case) > 3:
            cfg["dims"] = tuple(case[3])
        P = hr.PREC_NAMES[prec]
        dims = cfg["dims"]
        vh = li.volume(dims) // 2
        U, psi = B.make_fields(dict(cfg, dims=(2,) + tuple(dims[1:])))
        U = np.concatenate([U] * (dims[0] // 2))
        psi = [np.concatenate([p] * (dims[0] // 2)) for p in psi]
        lat = hr.Lattice(dims, B.BC, cfg["N"], cfg["rep"])
        fund, links = lat.gauge(False, P), lat.gauge(True, P)
        lat.import_gauge(fund, U)
        lat.represent_links(links, fund)
        if src == "rows":
            L = lat.gauge(2, P)
            lat.compress_links(L, fund)
        else:
            L = fund if src == "fund" else links
        inp = [lat.spinor(P) for _ in range(4)]
        out = [lat.spinor(P) for _ in range(4)]
        for k in range(4):
            lat.import_spinor(inp[k], P, psi[k & 1], 1 - (k & 1))
        st = lat.stream()
        bm = B.byte_model(cfg, prec)
        w = 8 if prec == "f64" else 4
        lb = {"repr": bm["L"], "fund": bm["F"], "rows": 2 * cfg["N"] * (cfg["N"] - 1) * w}[src]
        need = vh * (8 * lb + 2 * bm["S"])
        for sw in json.loads(args.sweeps):
            try:
                for k in keys:
                    lat.set_tuning(k, sw.get(k, -1 if k == "variant" else 0))
                hr.hr_dphi_eo(out[0], inp[0], L, 0, st)
                torch.cuda.synchronize()
            except hr.HrError as exc:
                print(json.dumps({"workload": cfg["name"], "dims": list(dims), "dtype": prec, "links": src, **sw, "unavailable": str(exc)[:90]}), flush=True)
                continue
            burst, ms, mhz = timed(lambda k: hr.hr_dphi_eo(out[k % 4], inp[k % 4], L, k & 1, st))
            print(json.dumps({"workload": cfg["name"], "dims": list(dims), "dtype": prec, "links": src, **sw,
                              "burst_ms": round(burst, 4), "burst_frac": round(need / burst / 1e6 / peak, 3),
                              "sustained_ms": round(ms, 4), "sustained_frac": round(need / ms / 1e6 / peak, 3), "sm_mhz": mhz,
                              "needed_mb": round(need / 1e6, 1)}), flush=True)
        lat.close()
        del inp, out, lat
        torch.cuda.empty_cache()


SWEEPS = {"volume": volume, "large_n": large_n, "solver": solver, "variants": variants}

if __name__ == "__main__":
    if len(sys.argv) < 2 or sys.argv[1] not in SWEEPS:
        raise SystemExit(__doc__)
    SWEEPS[sys.argv[1]](sys.argv[2:])
