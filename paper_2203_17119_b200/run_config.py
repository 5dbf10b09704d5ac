"""Run one BASELINE.json configuration (c1..c5) end to end on the GPU and print one JSON report:

    python -m paper_2203_17119_b200.run_config c5 [--no-uncut]

Seeded synthetic gauge field and source (inputs.py), Dhop / Mpc^dag Mpc timings in fp32 and fp64, then the solve the
configuration names: red-black CG on Mpc^dag Mpc to cfg.tol in fp64 and in fp32-inner / fp64-outer mixed precision.
For a configuration with a Dirichlet cut (c2, c5) the same solve is repeated with the uncut operator on the same gauge
field ("Dirichlet D_Omega solve vs full-operator solve", BASELINE configs[4]; PAPER.md:34 expects the cut operator to
be the worse conditioned one).  Everything runs in libdwf_b200.so; no oracle, no CPU fallback."""
from __future__ import annotations

import argparse
import dataclasses
import json
import time

import torch

from . import api, inputs

FLOP_DHOP, FLOP_MPC = 1320, 2 * 1320 + 360


def _time(fn, reps):
    for _ in range(3):
        fn()
    s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    s.record()
    for _ in range(reps):
        fn()
    e.record()
    torch.cuda.synchronize()
    return s.elapsed_time(e) / reps


def run(cfg, U, b_np, with_sweeps=True, max_iter=50000, extras=False):
    A = api
    g = api.from_config(cfg)
    g.set_gauge(U)
    n5h = (cfg.V4 // 2) * cfg.Ls
    rep = {"dims": list(cfg.dims), "Ls": cfg.Ls, "cut": list(cfg.cut), "fused_active": bool(g.get_option("fused_active"))}
    if with_sweeps:
        for prec, name in ((A.F32, "f32"), (A.F64, "f64")):
            src = g.new_native(prec, A.FULL).normal_()
            dst = g.new_native(prec, A.FULL)
            ms = _time(lambda: g.dhop(src, A.FULL, False, prec, out=dst), 10)
            h = src.numel() // 2
            ms2 = _time(lambda: g.mdagm(src[:h], prec, out=dst[:h]), 5)
            rep[f"dhop_{name}"] = {"ms_full_volume": ms, "gflops": FLOP_DHOP * 2 * n5h / ms / 1e6}
            rep[f"mdagm_{name}"] = {"ms": ms2, "gflops": 2 * FLOP_MPC * n5h / ms2 / 1e6}
            del src, dst
    b = g.pack(b_np, A.F64, A.ODD)
    for mode, name in ((A.CG_F64, "cg_f64"), (A.CG_MIXED, "cg_mixed")):
        x, info, st = g.cg(b, cfg.tol, max_iter, mode)
        rep[name] = {"tol": cfg.tol, "status": int(st), "iters": info["iters_total"], "restarts": info["restarts"],
                     "resid_true": info["resid_true"], "seconds": info["seconds"], "launches": info["launches"]}
        del x
    if extras and any(cfg.cut) and all(c == 0 or (d // c) % 2 == 0 for d, c in zip(cfg.dims, cfg.cut)):
        # the boundary operators R^-1 (one uncut solve, eqs. 13-14) and R (two Dirichlet solves, eqs. 9-10)
        phi = g.new_native(A.F64, A.FULL).normal_()
        p = g.domain_project(phi, 2)
        rinv, i1, st1 = g.boundary_op(phi, True, cfg.tol, max_iter, A.CG_MIXED)
        rr, i2, st2 = g.boundary_op(rinv, False, cfg.tol, max_iter, A.CG_MIXED)
        rep["boundary"] = {"Rinv": {"status": int(st1), "iters": i1["iters_total"], "seconds": i1["seconds"]},
                           "R": {"status": int(st2), "iters": i2["iters_total"], "seconds": i2["seconds"]},
                           "R_Rinv_minus_P_rel": float(torch.linalg.norm(rr - p) / torch.linalg.norm(p)),
                           "boundary_fraction": float((p != 0).sum() / p.numel())}
        del phi, p, rinv, rr
    if extras:
        # SURVEY 8f NEXT-2 / NEXT-4 at full size: four shifts in one Krylov space; a 16th-order Chebyshev filter
        shifts = [0.0, 0.01, 0.1, 1.0]
        xs, info, res, st = g.multishift_cg(b, shifts, cfg.tol, max_iter)
        rep["multishift_cg"] = {"shifts": shifts, "tol": cfg.tol, "status": int(st), "iters": info["iters_total"],
                                "resid_true": res, "seconds": info["seconds"], "launches": info["launches"]}
        del xs
        for prec, name in ((A.F32, "f32"), (A.F64, "f64")):
            v = g.new_native(prec, A.ODD).normal_()
            out = g.new_native(prec, A.ODD)
            ms = _time(lambda: g.chebyshev(v, 0.0, 60.0, 16, prec, out=out), 3)
            rep[f"chebyshev16_{name}"] = {"ms": ms, "gflops": 16 * 2 * FLOP_MPC * n5h / ms / 1e6}
            del v, out
    if extras:
        rep["mrhs"] = mrhs_report(g, cfg, b)
    g.close()
    return rep


def mrhs_report(g, cfg, b, counts=(1, 2, 4, 6), hbm_gbs=None):
    """batched Dhop / Mpc^dag Mpc / CG against the number of right-hand sides.  Algorithmic bytes per
    5-D site of the Dhop: 48 B + 8 g B / (nrhs Ls): the links are loaded once per tile for all nrhs * Ls slices."""
    A = api
    n5h = (cfg.V4 // 2) * cfg.Ls
    rows = []
    for n in counts:
        try:
            g.mrhs_reserve(n)
        except api.DwfError as e:       # out of memory for this many systems
            rows.append({"nrhs": n, "skipped": str(e)})
            continue
        row = {"nrhs": n}
        for prec, name, B in ((A.F32, "f32", 4), (A.F64, "f64", 8)):
            src = g.new_mrhs(n, prec).normal_()
            dst = g.new_mrhs(n, prec)
            ms = _time(lambda: g.dhop_mrhs(src, n, A.EVEN, False, prec, out=dst), 10)
            by = n * n5h * 48 * B + (cfg.V4 // 2) * 8 * 12 * B
            by_gauge = (cfg.V4 // 2) * 8 * 12 * B
            ms2 = _time(lambda: g.mdagm_mrhs(src, n, prec, out=dst), 3)
            row[name] = {"dhop_eo_ms": ms, "dhop_ms_per_rhs": ms / n, "dhop_gflops": FLOP_DHOP * n * n5h / ms / 1e6,
                         "dhop_algorithmic_gbs": by / ms / 1e6, "gauge_share_of_bytes": by_gauge / by,
                         "bytes_per_site": by / (n * n5h), "mdagm_ms": ms2, "mdagm_ms_per_rhs": ms2 / n,
                         "mdagm_gflops": 2 * FLOP_MPC * n * n5h / ms2 / 1e6}
            del src, dst
        # n sources: the configured one and rescaled / operator-smoothed copies, so the systems differ
        fields = [b] + [g.mdagm(b, A.F64) if j % 2 else b * (0.5 ** j) for j in range(1, n)]
        bb = g.mrhs_gather(fields)
        del fields
        for mode, mname in ((A.CG_F64, "cg_f64"), (A.CG_MIXED, "cg_mixed")):
            x, infos, st = g.cg_mrhs(bb, n, cfg.tol, 50000, mode)
            row[mname] = {"status": int(st), "iters": [i["iters_total"] for i in infos], "seconds": infos[0]["seconds"],
                          "seconds_per_rhs": infos[0]["seconds"] / n, "resid_true_max": max(i["resid_true"] for i in infos)}
            del x
        del bb
        rows.append(row)
    return rows


def roofline_sweep(cfg, U, hbm_gbs):
    """SURVEY 8(d) / BASELINE configs[3]: Dhop and Mpc^dag Mpc over links in {12, 18} reals x Ls in {8, 12, 16} x {fp32, fp64},
    half-volume (EO) and full-volume Dhop.  Algorithmic bytes per 5-D site: 48 B + 8 g B / Ls (B = 4 or 8)."""
    A = api
    rows = []
    for ng in (12, 18):
        for Ls in (8, 12, 16):
            c = dataclasses.replace(cfg, Ls=Ls)
            g = api.from_config(c, compress12=int(ng == 12))
            g.set_gauge(U)
            n5h = (c.V4 // 2) * Ls
            for prec, name, B in ((A.F32, "f32", 4), (A.F64, "f64", 8)):
                src = g.new_native(prec, A.FULL).normal_()
                dst = g.new_native(prec, A.FULL)
                h = src.numel() // 2
                ms_eo = _time(lambda: g.dhop(src[:h], A.ODD, False, prec, out=dst[h:]), 20)
                ms_full = _time(lambda: g.dhop(src, A.FULL, False, prec, out=dst), 10)
                ms_mm = _time(lambda: g.mdagm(src[:h], prec, out=dst[:h]), 5)
                by = n5h * 48 * B + (c.V4 // 2) * 8 * ng * B
                rows.append({"links": ng, "Ls": Ls, "prec": name, "dhop_eo_ms": ms_eo, "dhop_full_ms": ms_full,
                             "dhop_eo_frac_hbm": by / ms_eo / 1e6 / hbm_gbs, "dhop_full_frac_hbm": 2 * by / ms_full / 1e6 / hbm_gbs,
                             "dhop_full_gflops": FLOP_DHOP * 2 * n5h / ms_full / 1e6, "mdagm_ms": ms_mm,
                             "mdagm_gflops": 2 * FLOP_MPC * n5h / ms_mm / 1e6, "fused": bool(g.get_option("fused_active"))})
                del src, dst
            g.close()
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--no-uncut", action="store_true", help="cut configurations: skip the uncut comparison solve")
    ap.add_argument("--sweep", action="store_true", help="only the Dhop / Mpc^dag Mpc roofline sweep (links x Ls x precision)")
    ap.add_argument("--hbm-gbs", type=float, default=6448.1, help="HBM roofline for --sweep (MEASURED_PEAKS.json hbm_gbs)")
    ap.add_argument("--extras", action="store_true", help="also time the multishift CG (4 shifts) and a 16th-order Chebyshev filter")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("run_config needs a CUDA device: the hot path has no CPU fallback")
    cfg = inputs.CONFIGS[args.config]
    t0 = time.perf_counter()
    U = inputs.make_gauge(cfg)
    b = inputs.source_half(cfg.dims, cfg.Ls, cfg.source_seed, parity=1)
    out = {"config": cfg.name, "params": {"M5": cfg.M5, "mf": cfg.mf, "b5": cfg.b5, "c5": cfg.c5, "gauge": cfg.gauge, "eps": cfg.eps},
           "plaquette": inputs.plaquette(U), "input_seconds": time.perf_counter() - t0}
    if args.sweep:
        out["roofline_sweep"] = roofline_sweep(cfg, U, args.hbm_gbs)
        print(json.dumps(out), flush=True)
        return
    out["as_configured"] = run(cfg, U, b, extras=args.extras)
    if any(cfg.cut) and not args.no_uncut:
        out["uncut_operator"] = run(dataclasses.replace(cfg, cut=(0, 0, 0, 0)), U, b, with_sweeps=False)
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
