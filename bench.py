#!/usr/bin/env python
"""bench.py -- one JSON line for the driver (contract: task prompt "bench.py" + tier section 4).

A "step" is one pass of the whole hot path = ONE preconditioned-CG iteration (direction update + dG apply + exact dot; the two
vector updates + preconditioner + exact dot) on BASELINE.json configs[3]: 1024 x 1024 cells, P = 3
(9.4 M fp64 unknowns, 75.5 MB per vector, working set 7 vectors = 528 MB > L2), chi / rho as configs[2].
value = algorithmic GB/s of the iteration: 11 vector passes x 8 B x n per iteration / device time.
Extra keys report the metric's other parts: exact-dot, dG-apply and axpby GB/s at >= 100 MB vectors.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--quick]
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

PASSES_FUSED = 11          # vector passes of one fused CG iteration: K1 5 (r, p_old, chi -> p, q), K2 6
METRIC = "CG-iteration algorithmic bandwidth (dG apply + exact dots + vector updates; 11 vector passes x 8 B x n per iteration)"
UNIT = "GB/s"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md 'clocks' line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx = max(mx, float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, col in (("hw_slowdown", 5), ("hw_thermal_slowdown", 6), ("sw_thermal_slowdown", 7), ("sw_power_cap", 8)):
                if len(r) > col and r[col].lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons), "samples": len(sm)}


def reduce_over_ranks(ms_local, units_local, world):
    """max time over ranks, sum of units (replicas only: DESIGN.md 8).  Uses torch.distributed when world > 1."""
    if world == 1:
        return ms_local, units_local
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    u = torch.tensor([units_local], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def time_events(fn, reps, torch):
    """CUDA-event time per call (ms) of fn over `reps` back-to-back calls on torch's current stream."""
    s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    s.record()
    for _ in range(reps):
        fn()
    e.record()
    torch.cuda.synchronize()
    return s.elapsed_time(e) / reps


def csrc_stamp():
    """sha256 (16 hex digits) of the kernel sources: profiles/traffic.json is only valid for the sources it was measured with"""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1807_01971_b200", "csrc")
    for f in sorted(os.listdir(d)):
        h.update(f.encode()); h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def cpu_info():
    model = ""
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip(); break
    except OSError:
        pass
    return {"os_cpu_count": os.cpu_count(), "cpu_model": model}


# fp64 operations per unknown of the loop kernels (ncu instruction counts): K1 = stencil 39 + direction update 3
# + exact dot 23 (incl. the halo lanes' redundant share); K2 = 3 + 23
FP64_OPS_PER_UNKNOWN = {"k1": 62.0, "k2": 26.0}


def run_fx(args):
    import numpy as np
    import torch

    import fxinputs as fi
    import paper_1807_01971_b200 as fx

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libfx has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    fx.lib()
    K, Wm = args.steps, max(args.warmup, 3)
    N = 256 if args.quick else 1024
    cfg = fi.config3(N=N)
    g = fx.make_grid(**cfg["grid"])
    n = g.n
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        chi = torch.from_numpy(cfg["chi"]).cuda(); rho = torch.from_numpy(cfg["rho"]).cuda()
        phi = torch.zeros(n, dtype=torch.float64, device="cuda")
        # ---- warm-up: W iterations through the same call (also allocates the library's work space) -------------
        fx.cg_solve(g, chi, rho, phi, 0.0, Wm)
        phi.zero_()
        fx.cg_profile(8)             # events around the whole loop and around K1, K2 of every 8th iteration (each sampled
        torch.cuda.synchronize()     # iteration costs ~9 us of serialisation; with every iteration sampled the step reads 5 % slow)
        if world > 1:
            dist.barrier()
        l0 = fx.launch_count()
        with ClockSampler(local) as clk:
            # ---- timed region: exactly K iterations; events on the library's stream around every loop kernel ---
            info = fx.cg_solve(g, chi, rho, phi, 0.0, K)
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
        prof = fx.cg_last_profile()
        launches = fx.launch_count() - l0
        fx.cg_profile(False)
        assert info.iterations == K and prof["iterations"] == K, (info.iterations, prof)
        loop_ms = prof["loop_ms"]
        ms, units = reduce_over_ranks(loop_ms, float(K) * PASSES_FUSED * 8.0 * n, world)
        value = units / (ms * 1e-3) / 1e9
        peak, peak_src = peaks()

        # ---- roofline of the dominant kernel (K1: dG apply fused with the exact dot p.Sp) ------------------------
        k_ms = {k: prof[k + "_ms"] / K for k in ("k1", "k2")}
        dom = max(k_ms, key=k_ms.get)
        bytes_per_launch = {"k1": 40.0 * n, "k2": 48.0 * n}
        achieved = bytes_per_launch[dom] / (k_ms[dom] * 1e-3) / 1e9
        names = {"k1": "k_cg_dir_apply_dot<3> (p = z + beta p, q = S p, exact dot p.q; reads r, p_old, chi, writes p, q: 40 B/unknown)",
                 "k2": "k_cg_update_tma<3> (phi,r updates + preconditioner + exact dot r.z; 48 B/unknown)"}
        roofline = {"bound": "hbm", "kernel": names[dom], "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "peak_source": peak_src, "traffic": None,
                    "frac_of_nominal_8TBs": achieved / 8000.0,
                    "per_kernel_ms": k_ms,
                    "per_kernel_GBs": {k: bytes_per_launch[k] / (k_ms[k] * 1e-3) / 1e9 for k in k_ms},
                    "kernel_share_of_step": {k: k_ms[k] / (loop_ms / K) for k in k_ms}}
        traffic_file = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(traffic_file):                                  # ncu dram bytes per launch, valid only for the sources it names
            tj = json.load(open(traffic_file))
            if tj.get("csrc_sha256_16") == csrc_stamp():
                roofline["traffic"] = tj.get(dom)
                roofline["traffic_source"] = tj.get("source")
            else:
                roofline["traffic_note"] = "profiles/traffic.json was measured with other kernel sources (%s, now %s): not reported" % (
                    tj.get("csrc_sha256_16"), csrc_stamp())
        # the second roof ("high number of 64-bit operations per memory load"): fp64 issue, measured in this run
        a8 = torch.zeros(8, dtype=torch.float64, device="cuda")
        fx.time_primitive("fp64_fma", a8, a8, a8, 2)
        t_roof = min(fx.time_primitive("fp64_fma", a8, a8, a8, 5) for _ in range(3))
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        fp64_peak = sms * fx.FP64_ROOF_FMAS_PER_SM / (t_roof * 1e-3) / 1e12          # T fp64 instructions (FMA) per second
        roofline["alu"] = {"bound": "fp64 issue", "peak_Tops": fp64_peak, "peak_source": "k_fp64_roof: %d SMs x 8 CTAs x 256 threads x 8 chains x 4096 dependent FMAs, measured in this run" % sms,
                           "kernel_ops_per_unknown": FP64_OPS_PER_UNKNOWN[dom], "kernel_ops": FP64_OPS_PER_UNKNOWN[dom] * n,
                           "achieved_Tops": FP64_OPS_PER_UNKNOWN[dom] * n / (k_ms[dom] * 1e-3) / 1e12,
                           "frac": FP64_OPS_PER_UNKNOWN[dom] * n / (k_ms[dom] * 1e-3) / 1e12 / fp64_peak,
                           "per_kernel_frac": {k: FP64_OPS_PER_UNKNOWN[k] * n / (k_ms[k] * 1e-3) / 1e12 / fp64_peak for k in k_ms}}

        # ---- the metric's other parts: primitives on >= 100 MB vectors (inputs larger than L2) --------------------
        prim = {}
        if rank == 0 and not args.no_primitives:
            nd = (1 << 22) if args.quick else (1 << 27)
            x = torch.from_numpy(fi.uniform(9001, nd)).cuda(); y = torch.from_numpy(fi.uniform(9002, nd)).cuda()
            out = torch.zeros(1, dtype=torch.float64, device="cuda")
            for _ in range(3):
                fx.exdot_async(x, y, out)
            t = time_events(lambda: fx.exdot_async(x, y, out), 20, torch)
            prim["exdot"] = {"n": nd, "MB_per_vector": 8e-6 * nd, "ms": t, "GBps": 16.0 * nd / t / 1e6, "frac_of_peak": 16.0 * nd / t / 1e6 / peak}
            for _ in range(3):
                fx.axpby(0.7, x, -0.3, y)
            t = time_events(lambda: fx.axpby(0.7, x, -0.3, y), 20, torch)
            prim["axpby"] = {"n": nd, "ms": t, "GBps": 24.0 * nd / t / 1e6, "frac_of_peak": 24.0 * nd / t / 1e6 / peak}
            for _ in range(3):
                fx.pointwise_dot(1.0, x, y, 0.0, x)
            y.copy_(torch.from_numpy(fi.uniform(9002, nd)))
            z = torch.empty_like(x)
            t = time_events(lambda: fx.pointwise_dot(1.0, x, y, 0.0, z), 20, torch)
            prim["pointwise_dot"] = {"n": nd, "ms": t, "GBps": 24.0 * nd / t / 1e6, "frac_of_peak": 24.0 * nd / t / 1e6 / peak}
            x.copy_(torch.from_numpy(fi.uniform(9001, nd))); z.copy_(torch.from_numpy(fi.uniform(9004, nd)))
            for kind, m in (("exdot3", 3), ("exsum", 1)):              # weighted dot, exact sum (device-resident result)
                fx.time_primitive(kind, x, y, z, 3)
                t = fx.time_primitive(kind, x, y, z, 20)
                prim[kind] = {"n": nd, "ms": t, "GBps": m * 8.0 * nd / t / 1e6, "frac_of_peak": m * 8.0 * nd / t / 1e6 / peak}
            xf = x.to(torch.float32); yf = z.to(torch.float32)           # binary32 inputs, exact accumulation
            for _ in range(3):
                fx.exdot_f32(xf, yf)
            t = time_events(lambda: fx.exdot_f32(xf, yf), 10, torch)
            prim["exdot_f32"] = {"n": nd, "ms": t, "GBps": 8.0 * nd / t / 1e6, "frac_of_peak": 8.0 * nd / t / 1e6 / peak,
                                 "Gelem_per_s": nd / t / 1e6, "note": "result returned to the host every call; fp64 exdot: %.0f Gelem/s" % (nd / prim["exdot"]["ms"] / 1e6)}
            del x, y, z, xf, yf
            q = torch.empty(n, dtype=torch.float64, device="cuda")
            pvec = torch.from_numpy(fi.uniform(9003, n)).cuda()
            for _ in range(3):
                fx.dg_elliptic_apply(g, chi, pvec, q, sym=True)
            t = time_events(lambda: fx.dg_elliptic_apply(g, chi, pvec, q, sym=True), 20, torch)
            for kind in ("dx_forward", "dy_forward", "dx_centered", "dy_centered"):   # the paper's "dxdy" primitive, Table 3 (m = 3)
                fx.time_primitive(kind, pvec, chi, q, 3, grid=g)
                tt = fx.time_primitive(kind, pvec, chi, q, 20, grid=g)
                prim[kind] = {"grid": "%dx%d P=3" % (N, N), "ms": tt, "GBps": 24.0 * n / tt / 1e6, "frac_of_peak": 24.0 * n / tt / 1e6 / peak}
            fx.time_primitive("arakawa", pvec, chi, q, 3, grid=g)        # the paper's second composite (Fig. 6a): 9 calls
            tt = fx.time_primitive("arakawa", pvec, chi, q, 10, grid=g)
            prim["arakawa"] = {"grid": "%dx%d P=3" % (N, N), "ms": tt, "calls": 2, "vector_passes": 9,
                               "GBps": 9 * 8.0 * n / tt / 1e6, "frac_of_peak": 9 * 8.0 * n / tt / 1e6 / peak,
                               "note": "two kernels on the tile stencil: (f, g) -> (out, h1, h2), then out += Dx h1 + Dy h2; same bits as the paper's composite of N = 9 calls, M = 34 passes (its ideal fused form: M = 4)"}
            gneu = fx.make_grid(N, N, 3, cfg["grid"]["lx"], cfg["grid"]["ly"], fx.NEU, fx.DIR_NEU)   # Neumann / mixed walls
            for _ in range(3):
                fx.dg_elliptic_apply(gneu, chi, pvec, q, sym=True)
            tn = time_events(lambda: fx.dg_elliptic_apply(gneu, chi, pvec, q, sym=True), 20, torch)
            prim["dg_apply_neumann"] = {"grid": "%dx%d P=3, bcx NEU, bcy DIR_NEU" % (N, N), "ms": tn, "GBps": 24.0 * n / tn / 1e6,
                                        "frac_of_peak": 24.0 * n / tn / 1e6 / peak}
            prim["dg_apply"] = {"grid": "%dx%d P=3" % (N, N), "n": n, "MB_per_vector": 8e-6 * n, "ms": t, "GBps": 24.0 * n / t / 1e6,
                                "frac_of_peak": 24.0 * n / t / 1e6 / peak, "note": "3 x 75.5 MB partly L2-resident between repeats"}
            del q, pvec
            # the north-star bar: dG apply at vectors >= 100 MB, every P (config 4's largest grids; P = 1 needs 4096^2 for that)
            big = {}
            for P_, N_ in ((1, 4096), (2, 2048), (3, 2048), (4, 2048), (5, 2048)) if not args.quick else ((3, 256),):
                gb = fx.make_grid(N_, N_, P_, cfg["grid"]["lx"], cfg["grid"]["ly"], fx.PER, fx.DIR)
                va = torch.rand(gb.n, dtype=torch.float64, device="cuda") + 0.5      # timing only: any finite data
                vb = torch.rand(gb.n, dtype=torch.float64, device="cuda") - 0.5
                vc = torch.empty_like(va)
                fx.time_primitive("dg_apply_sym", va, vb, vc, 3, grid=gb)
                tb = min(fx.time_primitive("dg_apply_sym", va, vb, vc, 10, grid=gb) for _ in range(2))
                big["P%d_%dx%d" % (P_, N_, N_)] = {"MB_per_vector": 8e-6 * gb.n, "ms": tb, "GBps": 24.0 * gb.n / tb / 1e6,
                                                     "frac_of_peak": 24.0 * gb.n / tb / 1e6 / peak}
                del va, vb, vc
            prim["dg_apply_100MB"] = big
            # config 1 as specified: the exact dot on every condition target and on a +-500 exponent spread, with the
            # share of elements that left the register window (the paper: the long accumulator is "rarely invoked")
            bycond = {}
            for k_ in ((20,) if args.quick else (24, 27)):
                for ci, ctarget in enumerate(fi.COND_TARGETS + ["spread500"]):
                    if ctarget == "spread500":
                        hx, hy = fi.dot_wide_spread(1 << k_)
                    else:
                        hx, hy, _ = fi.dot_family_a(k_, ci)
                    dx = torch.from_numpy(hx).cuda(); dy = torch.from_numpy(hy).cuda()
                    del hx, hy
                    for _ in range(2):
                        fx.exdot_async(dx, dy, out)
                    fx.exdot_stats(reset=True)
                    reps = 10
                    tc = time_events(lambda: fx.exdot_async(dx, dy, out), reps, torch)
                    st = fx.exdot_stats(reset=True)
                    ne = float(1 << k_) * reps
                    bycond["n2^%d_%s" % (k_, "cond%.0e" % ctarget if ctarget != "spread500" else ctarget)] = {
                        "ms": tc, "GBps": 16.0 * (1 << k_) / tc / 1e6, "frac_of_peak": 16.0 * (1 << k_) / tc / 1e6 / peak,
                        "slow_path_share": {"deposit_double_per_element": st["deposit_double"] / ne, "deposit_product_per_element": st["deposit_product"] / ne,
                                            "window_moves_per_1e6_elements": 1e6 * st["window_moves"] / ne}}
                    del dx, dy
            prim["exdot_by_condition"] = bycond
            for v in prim.values():                                  # every fraction against the nominal 8 TB/s too (north star)
                for d in (v.values() if "GBps" not in v else [v]):
                    if isinstance(d, dict) and "GBps" in d:
                        d["frac_of_nominal_8TBs"] = d["GBps"] / 8000.0

        # ---- the paper's runtime model t = T_lat + m S / B (Eq. 3; Eq. 9) on a reduced config-4 sweep -----
        model = {}
        if rank == 0 and not args.no_primitives and not args.quick:
            import sweep
            model = sweep.reduced(fx, fi, torch)

        # ---- configs[0] and configs[2] in full (small grids: latency-bound; persistent cooperative kernel) ----------------
        small = {}
        if rank == 0 and not args.no_primitives and not args.quick:
            for name, cf in (("config0_64x64_P3_tol1e-10", fi.config0()), ("config2_256x256_P3_tol1e-8", fi.config2())):
                gs = fx.make_grid(**cf["grid"])
                c_chi = torch.from_numpy(cf["chi"]).cuda(); c_rho = torch.from_numpy(cf["rho"]).cuda()
                c_phi = torch.zeros(gs.n, dtype=torch.float64, device="cuda")
                fx.cg_solve(gs, c_chi, c_rho, c_phi, cf["tol"], 20)
                c_phi.zero_()
                s_ev, e_ev = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                s_ev.record(); inf = fx.cg_solve(gs, c_chi, c_rho, c_phi, cf["tol"], cf["maxit"]); e_ev.record(); torch.cuda.synchronize()
                small[name] = {"iterations": int(inf.iterations), "status": int(inf.status), "rel_residual": inf.rel_residual,
                               "ms_total_incl_setup": s_ev.elapsed_time(e_ev), "us_per_iteration": 1e3 * s_ev.elapsed_time(e_ev) / max(1, inf.iterations)}

        # ---- e2e: the public host-buffer call; H2D of chi, rho, phi0 and D2H of phi inside the timed region -------
        hchi = torch.from_numpy(cfg["chi"]).pin_memory(); hrho = torch.from_numpy(cfg["rho"]).pin_memory()
        hphi = torch.zeros(n, dtype=torch.float64).pin_memory()
        fx.cg_solve_host(g, hchi, hrho, hphi, 0.0, 3)
        hphi.zero_()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        info2 = fx.cg_solve_host(g, hchi, hrho, hphi, 0.0, K)
        t1 = time.perf_counter()
        e_ms, e_units = reduce_over_ranks((t1 - t0) * 1e3, float(K) * PASSES_FUSED * 8.0 * n, world)
        assert info2.iterations == K
        same = bool(torch.equal(hphi, phi.cpu()))
        e2e = {"value": e_units / (e_ms * 1e-3) / 1e9, "unit": UNIT, "h2d_bytes_per_step": 3 * 8.0 * n / K, "d2h_bytes_per_step": 8.0 * n / K,
               "ms_total": e_ms, "region": "one fx_cg_solve_host call: H2D chi,rho,phi0 (pinned) + setup + K iterations + D2H phi; bytes per step = per call / K",
               "bitwise_equal_to_device_run": same}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
           "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic (seeded; fxinputs.config3: chi = 1+0.5 exp(-r^2/0.5), rho = n-N with 1e-3 uniform noise; stands in for the paper's datasets [58],[59])",
           "config": {"workload": "BASELINE.json configs[3]: dG elliptic PCG, %dx%d cells, P=3, %d fp64 unknowns, DIRxDIR, tol=0, fixed K iterations" % (N, N, n),
                      "step": "one fused PCG iteration (2 kernels)", "l2": "inputs larger than L2 (7 vectors x %.1f MB)" % (8e-6 * n),
                      "multi_gpu": "replicas only (north star: one GPU, no sharding)", "algorithmic_bytes_per_step": PASSES_FUSED * 8.0 * n},
           "clocks": clk.summary(), "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
           "cg": {"iterations": int(info.iterations), "status": int(info.status), "rel_residual": info.rel_residual},
           "primitives": prim, "small_grid_solves": small, "model": model}
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            out["cpu_baseline"] = cpu_baseline(cfg, n, quick=args.quick)
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def cpu_baseline(cfg, n, quick=False):
    """The oracle as it stands, on the host cores, bounded sample: 5 CG iterations of the same grid (t(6) - t(1))."""
    import oracle as o
    og = o.Grid(**cfg["grid"])
    its = 2 if quick else 5
    t0 = time.perf_counter(); o.cg_solve(og, cfg["chi"], cfg["rho"], cfg["phi0"], 0.0, 1); t1 = time.perf_counter()
    o.cg_solve(og, cfg["chi"], cfg["rho"], cfg["phi0"], 0.0, 1 + its); t2 = time.perf_counter()
    per_it = ((t2 - t1) - (t1 - t0)) / its
    return {"value": PASSES_FUSED * 8.0 * n / per_it / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
            "ms_per_step": per_it * 1e3, "host": cpu_info(),
            "sample": "%d CG iterations of the same %dx%d P=3 problem (time of 1+%d iterations minus time of 1), oracle/fxo.cpp single-threaded"
                      % (its, og.Nx, og.Ny, its)}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/unit; each step = one oracle CG iteration on a
    256 x 256-cell sub-sample of the workload (1/16 of the unknowns), so that K steps end within minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import fxinputs as fi
    import oracle as o
    K, Wm = args.steps, max(args.warmup, 1)
    N = 256
    cfg = fi.config3(N=N)
    og = o.Grid(**cfg["grid"])
    n = og.n
    o.cg_solve(og, cfg["chi"], cfg["rho"], cfg["phi0"], 0.0, Wm)
    t0 = time.perf_counter(); o.cg_solve(og, cfg["chi"], cfg["rho"], cfg["phi0"], 0.0, 0); t_setup = time.perf_counter() - t0
    t0 = time.perf_counter(); _, info = o.cg_solve(og, cfg["chi"], cfg["rho"], cfg["phi0"], 0.0, K); t = time.perf_counter() - t0
    ms = max(t - t_setup, 1e-9) * 1e3
    value = K * PASSES_FUSED * 8.0 * n / (ms * 1e-3) / 1e9
    sample = "each step = one oracle CG iteration on a 256x256-cell, P=3 sub-sample (1/16 of configs[3]); setup time subtracted"
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": K, "warmup": Wm,
                      "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                      "data": "synthetic (fxinputs.config3 at N=256)",
                      "config": {"workload": "BASELINE.json configs[3] (bounded sample: 256x256 cells, P=3, %d unknowns)" % n},
                      "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "host": cpu_info()},
                      "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                      "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="fx", choices=["fx", "reference"])
    ap.add_argument("--quick", action="store_true", help="256x256 grid and small vectors (smoke runs)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-primitives", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_fx(args)


if __name__ == "__main__":
    main()
