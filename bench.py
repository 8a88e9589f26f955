#!/usr/bin/env python
"""bench.py -- throughput of the arXiv 1311.3004 finite-volume step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5-16384] [--kernel fused|unfused]
    python bench.py --impl reference ...        # the CPU oracle timed on the host cores (the reference arm)

A "step" is one time step of the whole hot path (ghost rule, x-sweep, y-sweep, source step, CFL clock) over the
whole grid.  The default workload is the largest grid of BASELINE.json (C5: 16384^2 cells fp64, periodic, seeded
multi-Gaussian field, nu_W = 0.9), the one the metric's roofline target is quoted on; its state (6.4 GB) is far
larger than L2, so no flush is needed between timed steps.  Prints ONE JSON line (rank 0).

Multi-GPU: the north-star fixes one GPU and no sharding ("replicas only"): with --gpus N every rank runs
an independent replica of the workload on its own GPU, no data-path collective; value = N x cells x K / max-over-
ranks time ("weak" scaling).
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 Gcell-updates/s"          # (with --precision 32 the same quantity for the fp32 variant; `dtype` says which)
UNIT = "Gcell-updates/s"
ALG_BYTES_PER_VALUE = 6.0          # 3 fields x (1 read + 1 write) per cell-update, x 8 B (f64) or 4 B (f32)
ALG_FLOP_PER_CELL = 404.0          # the oracle's formulas, division / sqrt = 1
# derived ALU peaks (not in MEASURED_PEAKS.json): 148 SMs x lanes x FMA x 1965 MHz; 64 FP64 lanes, 128 FP32 lanes per SM
ALU_PEAK_TFLOPS = {64: 148 * 64 * 2 * 1.965e9 / 1e12, 32: 148 * 128 * 2 * 1.965e9 / 1e12}


def ncu_traffic(workload, precision):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the step kernel, from the committed `ncu --set full`
    capture of THIS kernel on THIS workload (profiles/r2_traffic.json, which names the capture) -- None when there is none:
    the figure is a property of a capture, it is not measured in the run."""
    try:
        d = json.load(open(os.path.join(ROOT, "profiles", "r2_traffic.json")))
        e = d.get(f"{workload}/f{precision}")
        return (float(e["dram_bytes_per_launch"]), e["capture"]) if e else (None, None)
    except Exception:
        return None, None


def reduce_max_ms(ms, dist, device):
    """Max over ranks of a locally measured duration (the job is as slow as its slowest replica)."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(cells_per_replica, world, steps, ms):
    """Gcell-updates/s of the whole job: every replica advances its own grid (replicas only, weak scaling)."""
    return world * cells_per_replica * steps / (ms * 1e-3) / 1e9


def make_workload(name):
    import workloads as W
    if name.startswith("C5-"):
        return W.c5_sweep(n=int(name[3:]))
    if name == "C2":
        return W.c2_pulse()
    if name == "C3":
        return W.c3_random()
    if name == "C4":
        return W.c4_hifu()
    if name == "C1":
        return W.c1_piston()
    raise SystemExit(f"unknown workload {name}")


# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs (B200_PROFILING.md)."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self, t_lo=None, t_hi=None):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except Exception:
                self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons, rows = [], [], [], set(), []
        for line in self.f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                ts = time.mktime(time.strptime(c[0].split(".")[0], "%Y/%m/%d %H:%M:%S")) + float("0." + c[0].split(".")[1])
                rows.append((ts, float(c[1]), float(c[2]), float(c[3]), c))
            except (ValueError, IndexError):
                continue
        inside = [r for r in rows if t_lo is None or (t_lo - 0.05 <= r[0] <= t_hi + 0.05)]
        for ts, a, b, p, c in (inside or rows):
            sm.append(a); mx.append(b); pw.append(p)
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            load = [s for s, p in zip(sm, pw) if p >= 0.5 * max(pw)] or sm
            out = {"sm_mhz": statistics.median(load), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                   "reasons": sorted(reasons), "samples": len(sm), "samples_in_timed_region": len(inside)}
        return out


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)", d
        except Exception:
            pass
    return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)", {}


# ---------------------------------------------------------------------------------------------------------------
# CPU legs: the oracle as it stands (oracle/, never tuned), on the host cores.  Only these two functions touch it.
ORACLE_SAMPLE_N = 2048      # one sample size for the cpu_baseline leg and the reference arm (the oracle's rate depends on it)


def _oracle_sample(w_full, n_sample=ORACLE_SAMPLE_N):
    """A bounded sample of the same workload: the workload's own generator (and seed) at n_sample^2 cells."""
    import workloads as W
    if w_full.name.startswith(("C5", "C3")):
        return W.c3_random(n=min(n_sample, w_full.nx), steps=1, nu_w=w_full.value, seed=w_full.extra["seed"],
                           name=f"{w_full.name}@{min(n_sample, w_full.nx)}^2")
    if w_full.name == "C2":
        return W.c2_pulse(n=n_sample, steps=1)
    if w_full.name == "C4":
        return W.c4_hifu(nx=n_sample, ny=n_sample // 4, steps=1, focus_cells=n_sample / 4, aperture_cells=n_sample / 12)
    return w_full


def oracle_context(w):
    from oracle.oracle import Oracle
    o = Oracle(w.nx, w.ny, w.dx, w.dy, **w.medium, threads=0)
    for side, (kind, src) in enumerate(w.bc):
        o.set_bc(side, kind, src)
    o.set_state(*[a.numpy() for a in w.init()])
    return o


def cpu_baseline(w_full, budget_s=12.0):
    """Oracle throughput on a bounded sample (about `budget_s` of CPU work) of the bench workload."""
    ws = _oracle_sample(w_full, 512)
    o = oracle_context(ws)
    o.step(1, ws.value, ws.mode)                                   # includes the pre-pass; warm-up
    t0 = time.perf_counter(); o.step(1, ws.value, ws.mode); t1 = time.perf_counter()
    rate = ws.cells / (t1 - t0)
    ws = _oracle_sample(w_full)
    steps = int(max(1, min(200, round(budget_s * rate / ws.cells))))
    o = oracle_context(ws)
    o.step(1, ws.value, ws.mode)
    t0 = time.perf_counter(); o.step(steps, ws.value, ws.mode); t1 = time.perf_counter()
    return {"value": ws.cells * steps / (t1 - t0) / 1e9, "unit": UNIT, "cores": o.threads, "kind": "oracle",
            "sample": f"{ws.name}: {ws.nx}x{ws.ny} cells x {steps} steps of the same generator and boundary rules, "
                      f"oracle/fvnl_oracle.cpp with OpenMP over rows/columns ({t1 - t0:.1f} s)"}


def run_reference(args):
    """--impl reference: the oracle, K timed steps (after W warm-up steps) on a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w_full = make_workload(args.workload)
    ws = _oracle_sample(w_full)
    o = oracle_context(ws)
    o.step(max(1, args.warmup), ws.value, ws.mode)
    t0 = time.perf_counter(); o.step(args.steps, ws.value, ws.mode); t1 = time.perf_counter()
    val = ws.cells * args.steps / (t1 - t0) / 1e9
    sample = f"{ws.name}: {ws.nx}x{ws.ny} cells per step (bounded sample of {w_full.name} {w_full.nx}x{w_full.ny})"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": (t1 - t0) * 1e3 / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w_full.name, "grid": [w_full.nx, w_full.ny], "sample": sample, "bc": "as the workload",
                   "nu_W": w_full.value},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": o.threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ---------------------------------------------------------------------------------------------------------------
def run_gpu(args):
    import torch
    import paper_1311_3004_b200 as P          # raises if libfvnl.so cannot be built / loaded: no fallback

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    w = make_workload(args.workload)
    K, Wm = args.steps, args.warmup
    s = P.Solver(w.nx, w.ny, w.dx, w.dy, **w.medium, device=dev, precision=args.precision)
    for side, (kind, src) in enumerate(w.bc):
        s.set_bc(side, kind, src)
    if args.kernel == "unfused":
        s.set_option(P.OPT_KERNEL, P.KERNEL_UNFUSED)
    if args.variant >= 0:
        s.set_option(P.OPT_VARIANT, args.variant)
    if args.rows:
        s.set_option(P.OPT_ROWS_PER_BLOCK, args.rows)
    q0 = w.init(device=dev)                    # seeded synthetic state, generated on the device (resident in HBM)
    s.set_state(*q0)
    del q0
    torch.cuda.empty_cache()
    # per-launch event pairs for the roofline; not on grids of at most 2^22 cells, where a step takes 5 ... 130 microseconds and
    # an event pair per launch (it also keeps consecutive launches from overlapping) costs up to 10 microseconds of it -- measured
    # on C2: 61 us per step with the pairs, 50 without: there the step IS the launch and the kernel time is ms / K
    per_kernel = w.cells > (1 << 22)
    s.set_option(P.OPT_KERNEL_TIMING, 1 if per_kernel else 0)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- value: state resident in HBM, K steps in one fvnl_step call, CUDA events on the solver's stream -------
    flags = s.step(Wm, w.value, w.mode)
    for k in range(4):
        s.kernel_time(k)                       # reset the per-kernel spans of the warm-up
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.7 if rank == 0 else 0.0)      # let nvidia-smi come up before the timed region
    barrier()
    l0 = s.kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_w0 = time.time()
    e0.record()
    flags |= s.step(K, w.value, w.mode)
    e1.record()
    barrier()
    t_w1 = time.time()
    launches = s.kernel_launches() - l0
    clocks = sampler.stop(t_w0, t_w1)
    ms = e0.elapsed_time(e1)
    ms = reduce_max_ms(ms, dist, dev)
    value = whole_job_value(w.cells, world, K, ms)
    step_kernel = {"fused": "k_step_ws" if args.variant in (-1, 0) else "k_step_fused"}.get(args.kernel, "k_step_ws")
    names = {P.TIMED_STEP: step_kernel, P.TIMED_XSWEEP: "k_xsweep_unfused", P.TIMED_YSWEEP: "k_ysweep_unfused",
             P.TIMED_SOURCE: "k_source_unfused"}
    spans = {names[k]: s.kernel_time(k) for k in names}
    spans = {k: v for k, v in spans.items() if v[1] > 0}
    if not per_kernel:
        if launches < K:                        # small grid: the whole call was ONE launch of the cluster kernel (fvnl_small.cuh)
            step_kernel = "k_steps_cluster"
        spans = {step_kernel: (ms, K)}          # per step: the call's device time / K (launch gaps included)
    info = s.info()

    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (device time per launch from the library's event pairs) ---------------
    peak, peak_src, peaks = measured_peaks()
    top = max(spans, key=lambda k: spans[k][0])
    top_ms = spans[top][0] / spans[top][1]
    share = spans[top][0] / ms
    traffic_src = "--traffic" if args.traffic is not None else None
    if args.traffic is None and args.kernel == "fused" and args.variant in (-1, 0):
        args.traffic, traffic_src = ncu_traffic(w.name, args.precision)
    alg_bytes = ALG_BYTES_PER_VALUE * (args.precision // 8) * w.cells
    achieved = alg_bytes / (top_ms * 1e-3) / 1e9
    roofline_hbm = {"bound": "hbm", "kernel": top, "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": args.traffic, "traffic_source": traffic_src,
                    "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes}
    rc_probe, probe_tflops = P.fvnl_probe_fp64(torch.cuda.current_stream(dev).cuda_stream)
    tf = ALG_FLOP_PER_CELL * w.cells / (top_ms * 1e-3) / 1e12
    sm_mhz = clocks.get("sm_mhz") or 1965.0
    alu_peak = ALU_PEAK_TFLOPS[args.precision]
    lanes = 64 if args.precision == 64 else 128
    roofline = {"bound": "alu", "kernel": top, "achieved": tf, "peak": alu_peak, "unit": "TFLOP/s",
                "frac": tf / alu_peak, "traffic": args.traffic, "traffic_source": traffic_src,
                "peak_source": f"derived: 148 SMs x {lanes} FP{args.precision} lanes x 2 flop x 1.965 GHz (DESIGN.md 7); "
                               f"fp{args.precision} vector pipe, not in MEASURED_PEAKS.json",
                "frac_at_observed_clock": tf / (alu_peak * sm_mhz / 1965.0),
                "fp64_probe_tflops": probe_tflops if rc_probe == 0 else None,   # DFMA-only kernel, measured in this run
                "algorithmic_flop_per_launch": ALG_FLOP_PER_CELL * w.cells, "ms_per_launch": top_ms,
                "share_of_step": share,
                "kernels": {k: {"ms_per_launch": v[0] / v[1], "launches": v[1]} for k, v in spans.items()}}

    # ---- e2e: host buffers through the C ABI, copies inside the timed region, every step ----------------------
    s.set_option(P.OPT_KERNEL_TIMING, 0)
    Ke = max(1, min(K, args.e2e_steps))
    host = s.get_state(host=True)              # pinned host memory, 3 planes
    nbytes = sum(a.numel() * a.element_size() for a in host)
    torch.cuda.synchronize(dev)
    s.set_state(*host); s.step(1, w.value, w.mode); s.get_state(out=host)      # warm-up of the path
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    for _ in range(Ke):
        s.set_state(*host)                     # H2D, 3 planes
        flags |= s.step(1, w.value, w.mode)    # pre-pass (fresh state) + one step
        s.get_state(out=host)                  # D2H, 3 planes (synchronises)
    torch.cuda.synchronize(dev)
    t1 = time.perf_counter()
    e2e = {"value": w.cells * Ke / (t1 - t0) / 1e9, "unit": UNIT, "h2d_bytes_per_step": nbytes,
           "d2h_bytes_per_step": nbytes, "steps": Ke,
           "what": "per step: fvnl_set_state(pinned host) + fvnl_step(1, nu_W) + fvnl_get_state(pinned host)"}
    # the usual way the library is driven: one copy in, K steps, one copy out
    t0 = time.perf_counter()
    s.set_state(*host); flags |= s.step(K, w.value, w.mode); s.get_state(out=host)
    torch.cuda.synchronize(dev)
    t1 = time.perf_counter()
    e2e["amortised"] = {"value": w.cells * K / (t1 - t0) / 1e9, "unit": UNIT,
                        "what": f"fvnl_set_state(host) + fvnl_step({K}) + fvnl_get_state(host), wall clock"}
    del host
    s.close()

    base = cpu_baseline(w) if not args.no_cpu else None
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": f"f{args.precision}",
        "data": "synthetic",
        "config": {"workload": w.name, "grid": [w.nx, w.ny], "cells": w.cells, "bc": [k for k, _ in w.bc],
                   "nu_W": w.value, "kernel": top if args.kernel == "fused" else "three-pass (" + top + " is the slowest of the three)",
                   "variant": args.variant, "rows_per_block": args.rows, "state_bytes": 3 * (args.precision // 8) * w.cells,
                   "precision": args.precision,
                   "l2": "state larger than L2, no flush" if 3 * (args.precision // 8) * w.cells > 4 * 126e6 else "state near/below L2 size",
                   "parallelism": "replicas only" if world > 1 else "1 GPU", "flags": int(flags),
                   "t_end_s": info["t"], "last_cfl": info["cfl"]},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "roofline_hbm": roofline_hbm,
        "cpu_baseline": base,
    }
    print(json.dumps(out))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5-16384")
    ap.add_argument("--kernel", default="fused", choices=["fused", "unfused"],
                    help="fused: the one-pass step kernel (default: k_step_ws; --variant 1: k_step_fused); unfused: three passes")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--variant", type=int, default=-1, help="launch variant of the fused kernel (tuning aid)")
    ap.add_argument("--rows", type=int, default=0, help="rows per block of the fused kernel (0 = automatic)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32],
                    help="64: the paper's precision and the metric's (default); 32: the single-precision variant (PAPER.md:464)")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    main()
