#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of arXiv:1205.0752 on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg3_production]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path over one synthetic scan: quadrature tables (a2:
gf_make_quadrature, host generation + copy), grid fill (a1: gf_make_grid_rows), evaluation of the double
integral with its reductions and stores (a3-a6: gf_eval_grid).  The workload at N=1 is BASELINE.json
configs[2], the 2048x2048-point, 512x256-node FP64 production scan the headline target is quoted on.  With N
ranks the grid keeps its box and 2048 columns and has 2048*N rows; each rank owns 2048 contiguous rows (weak
scaling; grid points are independent; no data-path collective).

value    = grid points/s of the whole job, inputs resident in HBM (the grid is produced on the device).
e2e      = the same metric through gf_eval_grid_host on pinned HOST buffers (x in, G out), copies in the
           timed region.
roofline = the evaluation kernel against the FP64 pipe (bound "alu").
cpu_baseline = the oracle as it stands, on the box's host cores, on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import gf_workloads as W

METRIC = "grid_points_per_s"
UNIT = "points/s"
# 148 SMs x 64 FP64 FMA lanes x 2 flops x 1.965 GHz (clocks.max.sm)
FP64_LANES_PER_SM = 64
N_SM = 148
# dram__bytes_read.sum + dram__bytes_write.sum of one eval kernel launch on cfg3 (profiles/, ncu --set full);
# None until a capture is committed
EVAL_KERNEL_DRAM_TRAFFIC_BYTES = 102.9e6  # profiles/r02c_eval_ncu_full.md: 67.9 MB read + 34.9 MB written (134 MB algorithmic: x in, G out)


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def workload_for(name, world):
    """The per-job workload: cfg rows x world (weak scaling), and this is all the host logic there is."""
    cfg = dict(W.CONFIGS[name])
    cfg["n_im_global"] = cfg["n_im"] * world
    return cfg


def max_over_ranks(value, world, backend_device=None):
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=backend_device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, gpu_id):
        self.rows, self.proc, self.thread = [], None, None
        self.cmd = ["nvidia-smi", "-i", str(gpu_id), "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits",
                    "-lms", "100"]

    def start(self):
        try:
            self.proc = subprocess.Popen(self.cmd, stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], None, [], set()
        for t, line in self.rows:
            if not (t0 <= t <= t1 + 0.1):
                continue
            f = [c.strip() for c in line.split(",")]
            try:
                sm.append(float(f[0]))
                smax = float(f[1])
                power.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(self.NAMES, f[3:7]):
                if v == "Active":
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "power_w_max": max(power) if power else None, "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------- oracle legs
def oracle_sample(cfg, stride):
    """Every `stride`-th index in each direction of the workload's grid (per-point cost is uniform)."""
    from oracle import gf_oracle as O
    X = O.make_grid(cfg["re"][0], cfg["re"][1], cfg["n_re"], cfg["im"][0], cfg["im"][1], cfg["n_im"],
                    spacing=cfg["spacing"], im_abs_min=cfg["im_abs_min"])
    return np.ascontiguousarray(X[::stride, ::stride]).ravel()


def oracle_step(cfg, xs):
    """One pass of the oracle over the sample: its own tables, then the triple loop (double accumulation,
    the timed variant of oracle/gf_oracle.cpp).  Returns (seconds, threads used, values)."""
    from oracle import gf_oracle as O
    t = time.perf_counter()
    contour = cfg.get("contour", "real")
    P = O.make_params(cfg["line_k"], cfg["line_pk"], cfg["cutoff2"], prefactor=W.PREFACTOR, map_scale=W.MAP_SCALE,
                      contour=contour)
    rn, rw = O.make_radial_pyramid(cfg["n_rad"], levels=1 if contour == "real" else 4, kind=W.RADIAL_RULE)
    z, wz = O.make_quadrature(cfg.get("ang", W.ANGULAR_RULE), cfg["n_ang"], measure="sqrt1mz2")
    g, used = O.eval_grid(P, rn, rw, cfg["n_rad"], z, wz, xs, accum="double")
    return time.perf_counter() - t, used, g


def cpu_baseline(cfg, stride=4):
    """The oracle's timed variant on every `stride`-th index in each direction; returns the JSON object and the
    oracle's values on that sample (for the parity_check of the GPU result bench.py has just timed)."""
    xs = oracle_sample(cfg, stride)
    dt, used, g = oracle_step(cfg, xs)
    return {"value": xs.size / dt, "unit": UNIT, "cores": used, "kind": "oracle",
            "evals_per_s": xs.size * cfg["n_rad"] * cfg["n_ang"] / dt,
            "sample": "%s: every %dth index in each direction (%d of %d points, all %dx%d nodes), %.1f s, "
                      "oracle/gf_oracle.cpp -O2, double accumulation, one thread per core"
                      % (cfg["name"], stride, xs.size, cfg["n_re"] * cfg["n_im"], cfg["n_rad"], cfg["n_ang"], dt)}, g


def parity_check(g_gpu, g_oracle, stride, what):
    """max over the sample of |G_gpu - G_oracle| / |G_oracle| (0/0 := 0, reading G17)."""
    a = np.asarray(g_gpu, dtype=np.complex128).ravel()
    b = np.asarray(g_oracle, dtype=np.complex128).ravel()
    den = np.where(b == 0, 1.0, np.abs(b))
    e = np.abs(a - b) / den
    e[(a == 0) & (b == 0)] = 0.0
    # the oracle's timed variant evaluates its terms in double: its own rounding error reaches a few 1e-12 at the
    # rare points where the contour passes a singularity of the integrand (reading G18), hence 1e-10 here;
    # the 1e-11 bar against the extended-precision variant is tests/test_gpu_parity.py's
    return {"n": int(e.size), "max_rel": float(e.max()), "tol": 1e-10, "ok": bool(e.max() <= 1e-10),
            "against": what, "sample": "every %dth index in each direction" % stride}


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    cfg = dict(W.CONFIGS[args.workload], name=args.workload, contour=args.contour)
    stride = 16
    from oracle import gf_oracle as O
    O.build()
    xs = oracle_sample(cfg, stride)
    for _ in range(args.warmup):
        oracle_step(cfg, xs)
    t = time.perf_counter()
    used = 0
    for _ in range(args.steps):
        _, used, _ = oracle_step(cfg, xs)
    dt = time.perf_counter() - t
    value = xs.size * args.steps / dt
    sample = ("each step: every %dth index in each direction of %s (%d of %d points, all %dx%d nodes); "
              "oracle/gf_oracle.cpp -O2, double accumulation, one thread per core"
              % (stride, args.workload, xs.size, cfg["n_re"] * cfg["n_im"], cfg["n_rad"], cfg["n_ang"]))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, 1, cfg["n_im"]),
            "evals_per_s": value * cfg["n_rad"] * cfg["n_ang"],
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def workload_config(cfg, world, rows_per_rank):
    def line(p):
        m2 = complex(p.get("m2", 0.0))
        return ("1/(q^2+%s)" % (("%g" % m2.real) if m2.imag == 0 else "(%g%+gi)" % (m2.real, m2.imag))) if p["kind"] == "massive" else "(q^2+%g)/(q^4+%g q^2+%g)" % (p["M2"], p["a"], p["b"])
    return {"workload": "%s: lines %s and %s, once-subtracted at p^2=0, %dx%d grid over Re[%g,%g] Im[%g,%g]%s, "
                        "%d radial Gauss-Legendre x %d angular %s nodes, cutoff %g, %s contour, complex128"
                        % (cfg["name"], line(cfg["line_k"]), line(cfg["line_pk"]), cfg["n_re"], rows_per_rank * world,
                           cfg["re"][0], cfg["re"][1], cfg["im"][0], cfg["im"][1],
                           " (log-spaced |Im|)" if cfg["spacing"] != "uniform" else "", cfg["n_rad"], cfg["n_ang"],
                           cfg.get("ang", W.ANGULAR_RULE), cfg["cutoff2"], cfg.get("contour", "real").upper()),
            "n_points": cfg["n_re"] * rows_per_rank * world, "n_rad": cfg["n_rad"], "n_ang": cfg["n_ang"],
            "contour": cfg.get("contour", "real"),
            "parallelism": "rows x%d, no collective" % world,
            "cache": "L2 flushed between steps (256 MiB write); x + G = %d MiB per rank"
                     % (cfg["n_re"] * rows_per_rank * 32 >> 20)}


# ------------------------------------------------------------------------------------- the CUDA arm
def run_ours(args):
    import torch
    import paper_1205_0752_b200 as gf
    gf.lib()  # fails loudly when the extension is missing: there is no fallback
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path runs only in the sm_100a kernels")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    cfg = workload_for(args.workload, world)
    cfg["name"] = args.workload
    cfg["contour"] = args.contour
    n_re, n_rows, n_rad, n_ang = cfg["n_re"], cfg["n_im"], cfg["n_rad"], cfg["n_ang"]
    row_first, rows_local = W.row_partition(cfg["n_im_global"], world, rank)
    assert rows_local == n_rows
    n_points_local = n_re * rows_local
    contour = args.contour
    ang_rule = cfg.get("ang", W.ANGULAR_RULE)
    P = gf.make_params(cfg["line_k"], cfg["line_pk"], cfg["cutoff2"], prefactor=W.PREFACTOR, map_scale=W.MAP_SCALE,
                       contour=contour, precision=64)
    info = gf.launch_info(P, n_rad, n_ang, n_points_local)

    x = torch.empty((rows_local, n_re), dtype=torch.complex128, device=dev)
    out = torch.empty_like(x)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    ev_k0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ev_k1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]

    def step(k=None):
        rn, rw = gf.make_radial_tables(contour, n_rad, W.RADIAL_RULE)                   # a2
        z, wz = gf.make_quadrature(ang_rule, n_ang, measure="sqrt1mz2")           # a2
        gf.make_grid_rows(cfg["re"][0], cfg["re"][1], n_re, cfg["im"][0], cfg["im"][1], cfg["n_im_global"],
                          row_first, rows_local, spacing=cfg["spacing"], im_abs_min=cfg["im_abs_min"], out=x)  # a1
        ws = gf.eval_prepare(P, rn, rw, n_rad, z, wz)                                    # a3: x-independent set-up
        if k is not None:
            ev_k0[k].record(stream)
        gf.eval_grid_prepared(P, n_rad, n_ang, ws, x, out=out)                           # a3-a6
        if k is not None:
            ev_k1[k].record(stream)
        flush.zero_()                                                                    # L2 flush

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()

    sampler = ClockSampler("GPU-" + str(torch.cuda.get_device_properties(dev).uuid).replace("GPU-", ""))
    sampler.start()
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.perf_counter()
    e0.record(stream)
    for k in range(args.steps):
        step(k)
    e1.record(stream)
    barrier()
    t1 = time.perf_counter()
    clocks = sampler.stop(t0, t1)
    ms_total = max_over_ranks(e0.elapsed_time(e1), world, dev)
    kernel_ms = float(np.mean([a.elapsed_time(b) for a, b in zip(ev_k0, ev_k1)]))
    checksum = out.view(torch.float64).abs().sum().item()
    assert np.isfinite(checksum) and checksum > 0
    out_host = out.cpu().numpy()   # the timed region's last result, for parity_check

    # ---- executed FP64 work of one launch: the kernel's own route counters (an untimed, counted launch
    #      with identical results) x the per-unit instruction counts of the SASS (gf_eval_launch_info)
    rn_c, rw_c = gf.make_radial_tables(contour, n_rad, W.RADIAL_RULE)
    z_c, wz_c = gf.make_quadrature(ang_rule, n_ang, measure="sqrt1mz2")
    out_c, counters = gf.eval_grid_counted(P, rn_c, rw_c, n_rad, z_c, wz_c, x)
    assert torch.equal(out_c.view(torch.float64), out.view(torch.float64)), "counted launch differs"
    fp64_inst, fp64_flops = gf.executed_fp64(info, counters)
    del out_c

    # ---- the FP32 comparison variant on the same scan (BASELINE.json configs[2]): untimed for `value`, own events
    fp32_variant, out32_sample = None, None
    if contour == "real":
        P32 = gf.make_params(cfg["line_k"], cfg["line_pk"], cfg["cutoff2"], prefactor=W.PREFACTOR, map_scale=W.MAP_SCALE,
                             contour="real", precision=32)
        ws32 = gf.eval_prepare(P32, rn_c, rw_c, n_rad, z_c, wz_c)
        out32 = torch.empty(x.shape, dtype=torch.complex64, device=dev)
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for i in range(3):
            if i == 2:
                f0.record(stream)
            gf.eval_grid_prepared(P32, n_rad, n_ang, ws32, x, out=out32)
        f1.record(stream)
        torch.cuda.synchronize()
        ref64 = out.to(torch.complex128)
        err32 = ((out32.to(torch.complex128) - ref64).abs() / ref64.abs().clamp_min(1e-300)).max().item()
        fp32_variant = {"kernel_ms": f0.elapsed_time(f1), "max_rel_diff_vs_fp64": err32,
                        "note": "series and NEAR loops in float, per-node set-up, EXACT lanes and the tail in FP64"}
        out32_sample = out32[::4, ::4].cpu().numpy()   # compared with the oracle on the cpu_baseline sample below
        del out32, ref64, ws32

    # ---- e2e: the host-buffer entry point, copies inside the timed region
    xh = x.cpu().pin_memory()
    outh = torch.empty(xh.shape, dtype=torch.complex128).pin_memory()
    rn_h, rw_h = gf.make_radial_tables_host(contour, n_rad, W.RADIAL_RULE)
    z_h, wz_h = gf.make_quadrature_host(ang_rule, n_ang, measure="sqrt1mz2")

    def e2e_step():
        gf.eval_grid_host(P, rn_h, rw_h, n_rad, z_h, wz_h, xh, outh)   # synchronises before returning
        flush.zero_()

    for _ in range(2):
        e2e_step()
    barrier()
    ee0, ee1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ee0.record(stream)
    for _ in range(args.steps):
        e2e_step()
    ee1.record(stream)
    barrier()
    e2e_ms = max_over_ranks(ee0.elapsed_time(ee1), world, dev)
    assert torch.equal(outh.view(torch.float64), out.cpu().view(torch.float64)), "e2e result differs from device path"
    h2d = n_points_local * 16 + 8 * (2 * rn_h.size + 2 * n_ang)
    d2h = n_points_local * 16

    # ---- the measured FP64-pipe peak at the clocks this run saw (8 independent DFMA chains per thread)
    peak_blocks, peak_threads, peak_iters = N_SM * 4, 512, 100000
    sink = torch.empty(peak_blocks * peak_threads, dtype=torch.float64, device=dev)
    best = float("inf")
    for i in range(6):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        gf.diag_fp64_peak(peak_blocks, peak_threads, peak_iters, sink)
        b.record(stream)
        torch.cuda.synchronize()
        if i:
            best = min(best, a.elapsed_time(b))
    dfma_tflops = 2.0 * 8 * peak_iters * peak_blocks * peak_threads / (best * 1e-3) / 1e12

    # ---- issue cadence of DFMA streams by operand pattern, relative to the peak stream (same shape and work)
    dfma_issue = {}
    for mode, name in ((0, "one_varying_pair"), (1, "two_varying_pairs"), (2, "three_varying_pairs"), (3, "goertzel_recurrence")):
        best_m = float("inf")
        for i in range(4):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            gf.diag_dfma_issue(mode, peak_blocks, peak_threads, peak_iters, sink)
            b.record(stream)
            torch.cuda.synchronize()
            if i:
                best_m = min(best_m, a.elapsed_time(b))
        tf = 2.0 * 8 * peak_iters * peak_blocks * peak_threads / (best_m * 1e-3) / 1e12
        dfma_issue[name] = {"tflops": tf, "cycles_per_warp_dfma_per_smsp": 2.0 * (2.0 * FP64_LANES_PER_SM * N_SM * 1.965e-3) / tf}

    if world > 1:
        torch.distributed.barrier()
    if rank != 0:
        if world > 1:
            torch.distributed.destroy_process_group()
        return 0

    sm_max = clocks["sm_max_mhz"] or 1965.0
    peak_nominal = 2.0 * FP64_LANES_PER_SM * N_SM * sm_max * 1e6 / 1e12
    achieved = fp64_flops / (kernel_ms * 1e-3) / 1e12
    n_points_job = n_points_local * world
    value = n_points_job * args.steps / (ms_total * 1e-3)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, world, rows_local),
        "evals_per_s": value * n_rad * n_ang,
        "e2e": {"value": n_points_job * args.steps / (e2e_ms * 1e-3), "unit": UNIT,
                "h2d_bytes_per_step": h2d * world, "d2h_bytes_per_step": d2h * world},
        "gpu_launches": 3 * args.steps,  # make_grid, prep_real, eval_real per step (gf_eval_grid = the last two)
        "launch": {"kernel": "eval_real_kernel<double>" if contour == "real" else "eval_contour_kernel", "grid_blocks": info["grid_blocks"],
                   "block_threads": info["block_threads"], "smem_bytes": info["smem_bytes"], "lanes_per_point": info["split"]},
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_nominal, "unit": "TFLOP/s",
                     "frac": achieved / peak_nominal, "traffic": EVAL_KERNEL_DRAM_TRAFFIC_BYTES,
                     "peak_kind": "derived: %d SMs x %d FP64 lanes x 2 x %.0f MHz (DESIGN.md)" % (N_SM, FP64_LANES_PER_SM, sm_max),
                     "peak_measured_dfma": dfma_tflops, "frac_of_measured_dfma": achieved / dfma_tflops,
                     "kernel_ms": kernel_ms, "flops_per_launch": fp64_flops,
                     "fp64_inst_per_launch": fp64_inst, "routes": counters,
                     "fp64_pipe_frac": fp64_inst / (kernel_ms * 1e-3) / (FP64_LANES_PER_SM * N_SM * sm_max * 1e6),
                     "kernel_share_of_step": kernel_ms * args.steps / ms_total},
        "dfma_issue": dfma_issue,
        "clocks": clocks,
    }
    if fp32_variant:
        line["fp32_variant"] = fp32_variant
    if world == 1 and not args.no_cpu_baseline:
        from oracle import gf_oracle as O
        O.build()
        stride = 4
        line["cpu_baseline"], g_oracle = cpu_baseline(dict(W.CONFIGS[args.workload], name=args.workload, contour=contour), stride)
        line["parity_check"] = parity_check(out_host[::stride, ::stride], g_oracle, stride,
                                            "oracle/gf_oracle.cpp, double terms (the cpu_baseline leg's own values)")
        if fp32_variant:
            p32 = parity_check(out32_sample, g_oracle, stride, "the same oracle values")
            fp32_variant["max_rel_vs_oracle"] = p32["max_rel"]
            fp32_variant["ok_1e-4"] = bool(p32["max_rel"] <= 1e-4)
    print(json.dumps(line))
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", default="cfg3_production", choices=list(W.CONFIGS))
    ap.add_argument("--contour", default="real", choices=["real", "ray_arc", "thread", "auto"],
                    help="radial contour policy (the headline and the target are REAL; the others are reported)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args(argv)
    _, _, world = dist_env()
    if world != args.gpus and world > 1:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    if args.gpus > 1 and world == 1 and args.impl == "ours":
        raise SystemExit("bench.py: launch N>1 with torch.distributed.run (one rank per GPU)")
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
