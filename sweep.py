"""Latency-bandwidth sweep (BASELINE.json configs[4]) and the paper's runtime model t = T_lat + m*S/B.

Paper: bandwidth b = m*S/t with STREAM counting (Eq. 2: axpby m=3, dot m=2, mat-vec m=3);
model t(S) = T_lat + m*S/B (Eq. 3); estimators: B = mean over the largest sizes, T_lat = smallest average run
time corrected by -m*S/B and clipped at 0; minimum efficient array size ~ T_lat*B (Eq. 9).

    python sweep.py [--out DIR] [--quick] [--dg-path 0|1]            (bench.py runs `reduced` and puts its fits under "model")

Runs on cuda:0 through the C ABI (fx_time_primitive: average of back-to-back launches, CUDA events).  Writes
DIR/sweep.json and DIR/sweep.md.  Inputs: seeded uniform[-1,1) vectors (fxinputs.config4) -- synthetic stand-ins for
the vectors of the paper's benchmark program, which is not available.
"""
import argparse
import json
import math
import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

M_PASSES = {"axpby": 3, "pointwise_dot": 3, "exdot": 2, "exdot_host": 2, "exdot3": 3, "exsum": 1, "dg_apply_sym": 3, "dg_apply": 3,
            "dx_forward": 3, "dy_forward": 3, "dx_centered": 3, "dy_centered": 3}
L2_BYTES = 126e6


def fit(points, m):
    """points: [(S_bytes, t_seconds)] -> dict with the paper's estimators and a least-squares fit outside the L2 bump."""
    pts = sorted(points)
    big = [(S, t) for S, t in pts if S >= 100e6] or pts[-2:]
    bw = [m * S / t for S, t in big]
    B = sum(bw) / len(bw)
    Bstd = math.sqrt(sum((b - B) ** 2 for b in bw) / len(bw))
    small = pts[:3]
    Tlat = max(0.0, min(t - m * S / B for S, t in small))
    # least squares of t = a + S*m/Bfit over points outside the cache bump (tiny sizes and sizes with 3 vectors >= 1.5 x L2)
    ls = [(S, t) for S, t in pts if S <= 0.5e6 or 3 * S >= 1.5 * L2_BYTES]
    n = len(ls)
    sx = sum(S for S, _ in ls); sy = sum(t for _, t in ls); sxx = sum(S * S for S, _ in ls); sxy = sum(S * t for S, t in ls)
    if sum(1 for S, _ in ls if 3 * S >= 1.5 * L2_BYTES) >= 2:
        slope = (n * sxy - sx * sy) / (n * sxx - sx * sx)
        icpt = (sy - slope * sx) / n
    else:                                   # no two sizes beyond L2: a line through the cache bump means nothing
        slope, icpt = float("nan"), float("nan")
    err = max(abs((Tlat + m * S / B) / t - 1.0) for S, t in pts if not (0.5e6 < S and 3 * S < 2 * L2_BYTES))
    return {"B_GBps": B / 1e9, "B_std_GBps": Bstd / 1e9, "T_lat_us": Tlat * 1e6, "T_lat_times_B_MB": Tlat * B / 1e6,
            "lsq_B_GBps": m / slope / 1e9, "lsq_T_lat_us": icpt * 1e6, "model_max_rel_err_outside_L2_bump": err}


def reduced(fx, fi, torch, P=3, Ns=(16, 64, 256, 1024, 1536, 2048)):
    """Six sizes of config 4 at one P (18 KB ... 302 MB per vector): the fits of the five north-star primitives for bench.py"""
    pts = {}
    for N in Ns:
        c = fi.config4(P, N)
        g = fx.make_grid(**c["grid"])
        x = torch.from_numpy(c["x"]).cuda(); y = torch.from_numpy(c["y"]).cuda(); chi = torch.from_numpy(c["chi"]).cuda()
        out = torch.empty_like(x)
        S = 8.0 * g.n
        reps = int(max(10, min(1000, 0.03 / max(2e-6, 3 * S / 5e12))))
        for kind in ("axpby", "pointwise_dot", "exdot", "exdot_host", "dg_apply_sym"):
            if kind == "dg_apply_sym":
                ms = fx.time_primitive(kind, chi, x, out, reps, grid=g)
            else:
                if kind == "axpby":
                    out.copy_(y)
                ms = fx.time_primitive(kind, x, y, out, max(10, reps // (4 if kind == "exdot_host" else 1)))
            pts.setdefault(kind, []).append((S, ms * 1e-3))
        del x, y, chi, out
    res = {}
    for kind, p in pts.items():
        f = fit(p, M_PASSES[kind])
        f["m"] = M_PASSES[kind]
        f["points_MB_us"] = [[round(S / 1e6, 3), round(t * 1e6, 2)] for S, t in p]
        res[kind if kind != "dg_apply_sym" else "dg_apply_sym_P%d" % P] = f
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out"))
    ap.add_argument("--quick", action="store_true")
    ap.add_argument("--dg-path", type=int, default=0, help="fx_set_dg_path: 0 = default (CTA-tile stencil), 1 = warp-strip kernels (round 1's)")
    args = ap.parse_args()
    import numpy as np
    import torch

    import fxinputs as fi
    import paper_1807_01971_b200 as fx

    assert torch.cuda.is_available(), "sweep needs a CUDA device (no CPU fallback)"
    fx.lib()
    fx.set_dg_path(args.dg_path)
    Ns = [16, 64, 256] if args.quick else [16, 32, 64, 128, 256, 512, 1024, 2048]
    Ps = [3] if args.quick else [1, 2, 3, 4, 5]
    res = {}
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        for P in Ps:
            for N in Ns + ([4096] if (P <= 2 and not args.quick) else []):
                c = fi.config4(P, N)
                g = fx.make_grid(**c["grid"])
                n = g.n
                x = torch.from_numpy(c["x"]).cuda(); y = torch.from_numpy(c["y"]).cuda(); chi = torch.from_numpy(c["chi"]).cuda()
                out = torch.empty_like(x)
                S = 8.0 * n
                reps = int(max(10, min(2000, 0.05 / max(2e-6, 3 * S / 5e12))))
                for kind in ("axpby", "pointwise_dot", "exdot", "exdot_host", "exdot3", "exsum", "dg_apply_sym", "dg_apply",
                             "dx_forward", "dy_forward", "dx_centered", "dy_centered"):
                    if kind.startswith("dg"):
                        ms = fx.time_primitive(kind, chi, x, out, reps, grid=g)
                    elif kind.startswith("d"):
                        out.copy_(y); ms = fx.time_primitive(kind, x, y, out, reps, grid=g)
                    elif kind == "axpby":
                        out.copy_(y); ms = fx.time_primitive(kind, x, y, out, reps)
                    else:
                        ms = fx.time_primitive(kind, x, y, out, max(10, reps // (4 if kind == "exdot_host" else 1)))
                    key = kind if not kind.startswith("d") else "%s_P%d" % (kind, P)
                    res.setdefault(key, []).append({"P": P, "N": N, "n": n, "S_MB": S / 1e6, "t_us": ms * 1e3,
                                                    "GBps": M_PASSES[kind] * S / (ms * 1e-3) / 1e9})
                del x, y, chi, out
    fits = {}
    for key, pts in res.items():
        kind = key.split("_P")[0]
        fits[key] = fit([(p["S_MB"] * 1e6, p["t_us"] * 1e-6) for p in pts], M_PASSES[kind])
    os.makedirs(args.out, exist_ok=True)
    json.dump({"points": res, "fits": fits, "device": torch.cuda.get_device_name(0)}, open(os.path.join(args.out, "sweep.json"), "w"), indent=1)
    lines = ["| primitive | m | B GB/s (S >= 100 MB) | T_lat us | T_lat*B MB | least-squares B GB/s | least-squares T_lat us | model max rel. err. (outside L2 bump) |",
             "|---|---|---|---|---|---|---|---|"]
    for key, f in fits.items():
        lines.append("| %s | %d | %.0f +- %.0f | %.2f | %.3f | %.0f | %.2f | %.0f %% |" % (
            key, M_PASSES[key.split("_P")[0]], f["B_GBps"], f["B_std_GBps"], f["T_lat_us"], f["T_lat_times_B_MB"], f["lsq_B_GBps"],
            f["lsq_T_lat_us"], 100 * f["model_max_rel_err_outside_L2_bump"]))
    lines += ["", "Measured points (S = MB per vector : GB/s), sorted by size:", ""]
    for key, pts in res.items():
        lines.append("- **%s**: " % key + ", ".join("%.3g:%.0f" % (p["S_MB"], p["GBps"]) for p in sorted(pts, key=lambda q: q["S_MB"])))
    open(os.path.join(args.out, "sweep.md"), "w").write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
