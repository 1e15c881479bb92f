#!/usr/bin/env python
"""bench.py -- batched piMPC ADMM throughput on B200 (BASELINE.json config 4), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path (a0 cache, then 200 iterations of
steps a1..a7 of Algorithm 1) over one batch of 4096 synthetic LTV MPC instances
(nx=12, nu=4, N=50, fp32).  `value` = solves/s with the stage data already
in HBM; `e2e` = the same through the C ABI with pinned HOST buffers (H2D of A, B, x0 and D2H of
x, u, du, results inside the timed region).  Multi-GPU = replicas: every rank solves its own 4096
instances, no data-path collective ("scaling": "weak").  `extras` (N=1 only) adds us/iteration for
the batch-1 configs (C1, C2, C3 sweep) and GB/s for the HBM-bound wide config (C5).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2601_14414_b200 import replicas, workloads as wl  # noqa: E402

BATCH, ITERS = 4096, 200


# -------------------------------------------------------------------------------------------------
# algorithmic work per (instance, stage, iteration) -- DESIGN.md "Roofline arithmetic"
# -------------------------------------------------------------------------------------------------
def flops_per_stage_iter(nx, nu, has_du=True):
    nb = nx + nu
    return 2 * nb * nb + 4 * (nx * nx + nx * nu) + 4 * nx * nu + 2 * nu * nu + 45 * nb + (12 * nu if has_du else 0)


def bytes_per_stage_iter(nx, nu, esz, has_du=True, packed=True):
    nb = nx + nu
    mats = nx * nx + nx * nu + (nb * (nb + 1) // 2 + nu * (nu + 1) // 2 if packed else nb * nb + nu * nu)
    vecs = 15 * nb + (6 * nu if has_du else 0)
    return (mats + vecs) * esz


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        m = json.load(open(path))
        return dict(hbm_gbs=float(m["hbm_gbs"]), sm_max_mhz=float(m.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def ncu_traffic(engine, config):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture (profiles/traffic.csv)."""
    tp = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(tp):
        return None
    for line in open(tp).read().splitlines()[1:]:
        f = line.split(",")
        if len(f) >= 4 and f[0] == str(engine) and f[1] == config:
            return int(f[3])
    return None


def alu_peak_tflops(dtype, sm_mhz, sms=148):
    """Nominal FMA peak (lanes x 2 x clock), quoted next to the MEASURED one of pimpc_measure_peaks."""
    lanes = 128 if dtype == "f32" else 64          # FP32 / FP64 FMA lanes per SM
    return sms * lanes * 2 * sm_mhz * 1e6 / 1e12


# -------------------------------------------------------------------------------------------------
# clocks sampler (B200_PROFILING.md "clocks DURING the timed region")
# -------------------------------------------------------------------------------------------------
class Clocks:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0=None, t1=None):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for t, r in self.rows if (t0 is None or t >= t0) and (t1 is None or t <= t1 + 0.15)] or \
               [r for _, r in self.rows]
        sm, mx, reasons = [], [], set()
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# -------------------------------------------------------------------------------------------------
# oracle legs (cpu_baseline and --impl reference): the ONLY places bench.py executes oracle/
# -------------------------------------------------------------------------------------------------
def oracle_solves_per_s(prob, instances, iters, threads):
    """Time the CPU oracle as it stands (single-threaded C, one call per instance) on `instances`,
    `threads` calls in flight on independent instances (ctypes releases the GIL)."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import pimpc_oracle
    pimpc_oracle.build()
    p32 = prob.rounded("f32")
    run = lambda b: pimpc_oracle.solve(**p32.instance(b), max_iters=iters, tol=0.0).c_last
    run(instances[0])
    t0 = time.perf_counter()
    with ThreadPoolExecutor(threads) as ex:
        list(ex.map(run, instances))
    dt = time.perf_counter() - t0
    return len(instances) / dt, dt


def reference_arm(args):
    rank, _, world = replicas.env_rank()
    if rank != 0:
        return 0
    cores = os.cpu_count() or 1
    sample = 256
    prob = wl.config4(batch=sample)
    vals = []
    for s in range(args.warmup + args.steps):
        v, dt = oracle_solves_per_s(prob, list(range(sample)), ITERS, cores)
        if s >= args.warmup:
            vals.append((v, dt))
    tot = sum(sample for _ in vals) / sum(dt for _, dt in vals)
    desc = f"{sample} of the {BATCH} C4 instances per step, {ITERS} iterations each, {cores} concurrent oracle calls"
    print(json.dumps({
        "impl": "reference", "metric": "batched_solves_per_s", "value": tot, "unit": "solves/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(dt for _, dt in vals) / len(vals),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args.gpus),
        "cpu_baseline": {"value": tot, "unit": "solves/s", "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": tot, "unit": "solves/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))
    return 0


def workload_config(n):
    return {"workload": "C4: 4096 independent LTV MPC instances per GPU, nx=12, nu=4, N=50, 200 ADMM iterations, "
                        "|u|<=1 |du|<=0.2 |x|<=5, rho=1 (BASELINE.json configs[3])",
            "batch_per_gpu": BATCH, "global_batch": BATCH * n, "nx": 12, "nu": 4, "N": 50, "iters": ITERS,
            "parallelism": f"replicas x{n} (instances sharded, no collective)",
            "l2": "inputs_exceed_l2 (380 MB of stage data per step vs 126 MB L2)"}


# -------------------------------------------------------------------------------------------------
def timed_loop(torch, steps, fn):
    """K steps bracketed by synchronize + CUDA events on the current stream; returns total ms."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def us_per_iteration(torch, pimpc, prob, dtype, iters, reps=7, engine="auto"):
    """(t(K) - t(0)) / K for a batch-1 config: median over reps of one solve, minus the launch floor."""
    s = pimpc.Solver(prob.nx, prob.nu, prob.N, prob.batch, dtype=dtype, engine=engine, rho=prob.rho)
    s.set_problem(prob)
    s.solve(iters); s.sync()
    def once(k):
        s.reset(); torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); s.solve(k); e1.record(); torch.cuda.synchronize()
        return e0.elapsed_time(e1)
    tk = statistics.median(once(iters) for _ in range(reps))
    t0 = statistics.median(once(0) for _ in range(reps))
    info = s.get_info()
    s.close()
    return {"us_per_iter": 1e3 * (tk - t0) / iters, "solve_ms": tk, "launch_floor_ms": t0, "iters": iters,
            "engine": info["engine"], "grid": info["grid"], "block": info["block"]}


def cstr_closed_loop(torch, pimpc, N=5000, K=1000, steps=6):
    """receding-horizon stepping at the paper's CSTR scale (N = 5000, 1000
    iterations per MPC step; its GPU code: 0.526 s median per step on an RTX 3080).  Per step: linearise on the host,
    upload the stage data, a0, shift warm start, K iterations, read u_0; the plant advances with u_0."""
    out = {}
    for dt in ("f64", "f32"):
        x = np.array(wl.CSTR["x_init"]); u = np.array([wl.CSTR["u_init"]]); t = 0.0
        s = pimpc.Solver(2, 1, N, 1, dtype=dt)
        ms, ca = [], []
        for step in range(steps):
            pp = wl.cstr_problem(x, u, t, N, iters=K)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            s.set_problem(pp)
            if step:
                s.shift(1)
            s.solve(K)
            _, ug, _, _ = s.get()
            ms.append(1e3 * (time.perf_counter() - t0))
            u = ug[0, 0, :1].astype(np.float64)
            x = wl.cstr_plant_step(x, u, t); t += wl.CSTR["Ts"]
            ca.append(float(x[0]))
        info = s.get_info()
        s.close()
        out[dt] = {"ms_per_mpc_step_median": statistics.median(ms[1:]), "ms_per_mpc_step_max": max(ms[1:]),
                   "iter_kernel_ms": info["iter_ms"], "cache_kernel_ms": info["setup_ms"], "engine": info["engine"],
                   "grid": info["grid"], "C_A_after_steps": ca[-1]}
    out["config"] = {"N": N, "iters_per_step": K, "steps_timed": steps - 1, "shape": "(2,1), the paper's own shape",
                     "paper_gpu_s_per_step": 0.526}
    return out


def extras(torch, pimpc, pk, only=None):
    """`only`: comma-separated subset of C1,C2,C3,CSTR,T1,C5 (profiling aid: `--only-extras --extras C5`)."""
    want = lambda name: only is None or name in only.split(",")
    out = {}
    if want("C1"):
        out["C1_f64"] = us_per_iteration(torch, pimpc, wl.config1(), "f64", 500)
    if want("C2"):
        for dt in ("f64", "f32"):
            out[f"C2_{dt}"] = us_per_iteration(torch, pimpc, wl.config2(), dt, 2000)
    if want("C3"):
        out.update(extras_c3(torch, pimpc))
    if want("CSTR"):
        out["CSTR_closed_loop"] = cstr_closed_loop(torch, pimpc)
    if want("T1"):
        out["paper_table1_us_per_iter_f64"] = extras_table1(torch, pimpc)
    if want("C5"):
        out.update(extras_c5(torch, pimpc, pk))
    return out


def extras_c3(torch, pimpc):
    out = {}
    sweep = {}
    for N in wl.C3_HORIZONS:
        sweep[str(N)] = us_per_iteration(torch, pimpc, wl.config3(N), "f32", 1000, reps=5)
    out["C3_f32_us_per_iter_vs_N"] = sweep
    out["C3_flatness_t10000_over_t10"] = sweep["10000"]["us_per_iter"] / max(sweep["10"]["us_per_iter"], 1e-9)
    out["C3_flatness_t10000_over_t100"] = sweep["10000"]["us_per_iter"] / max(sweep["100"]["us_per_iter"], 1e-9)
    return out


def extras_table1(torch, pimpc):
    # the paper's Table I grid (its GPU code: 530-620 us per iteration at every size)
    t1 = {}
    for nx, nu in wl.TABLE1_SHAPES:
        for N in wl.TABLE1_HORIZONS:
            r = us_per_iteration(torch, pimpc, wl.paper_random(nx, nu, N), "f64", 200, reps=3)
            t1[f"{nx},{nu},{N}"] = round(r["us_per_iter"], 2)
    return t1


def extras_c5(torch, pimpc, pk):
    out = {}
    p5 = wl.config5()
    for dt, esz in (("f32", 4), ("f64", 8)):
        s = pimpc.Solver(p5.nx, p5.nu, p5.N, p5.batch, dtype=dt, rho=p5.rho)
        s.set_problem(p5)
        s.solve(5); s.sync(); s.reset()
        s.solve(100); info = s.get_info()
        ms_it = info["iter_ms"] / 100
        balg = bytes_per_stage_iter(p5.nx, p5.nu, esz) * p5.N * p5.batch
        out[f"C5_{dt}"] = {"ms_per_iter": ms_it, "algorithmic_GBps": balg / ms_it / 1e6,
                           "frac_of_hbm_peak": balg / ms_it / 1e6 / pk["hbm_gbs"], "engine": info["engine"],
                           "solves_per_s_500it_iterations_only": p5.batch / (ms_it * 500 / 1e3),
                           "note": "iteration kernel only: excludes the a0 cache kernel and k_pack"}
        s.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--engine", default="auto")
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--only-extras", action="store_true", help="run only the C1-C3, C5 legs and print their JSON (profiling aid)")
    ap.add_argument("--extras", default=None, help="comma-separated subset of the extras: C1,C2,C3,CSTR,T1,C5")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return reference_arm(args)

    import torch
    from paper_2601_14414_b200 import pimpc          # raises if libpimpc.so is missing (no fallback)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libpimpc has no CPU fallback")
    rank, local_rank, world = replicas.init()
    torch.cuda.set_device(local_rank)
    pk = peaks()
    if args.only_extras:
        if rank == 0:
            print(json.dumps({"extras": extras(torch, pimpc, pk, args.extras)}))
        return 0

    lo, hi = replicas.weak_instance_range(BATCH, rank)
    prob = wl.config4(batch=BATCH, first_instance=lo)
    f32 = torch.float32
    A_h = torch.from_numpy(prob.A.astype(np.float32)).pin_memory()
    B_h = torch.from_numpy(prob.B.astype(np.float32)).pin_memory()
    x0_h = torch.from_numpy(prob.x0.astype(np.float32)).pin_memory()
    A_d, B_d, x0_d = A_h.cuda(), B_h.cuda(), x0_h.cuda()
    x_h = torch.empty(BATCH, prob.N, prob.nx, dtype=f32).pin_memory()
    u_h = torch.empty(BATCH, prob.N, prob.nu, dtype=f32).pin_memory()
    du_h = torch.empty(BATCH, prob.N, prob.nu, dtype=f32).pin_memory()
    res_h = torch.zeros(BATCH, pimpc.RESULT_DTYPE.itemsize, dtype=torch.uint8).pin_memory()
    onchip = pimpc.measure_peaks(torch.cuda.current_stream().cuda_stream)     # FMA-chain / smem microbenchmarks, untimed

    s = pimpc.Solver(prob.nx, prob.nu, prob.N, BATCH, dtype="f32", engine=args.engine, rho=prob.rho)
    s.set_cost(prob.Q, prob.R)
    s.set_bounds(prob.lo, prob.hi, prob.du_lo, prob.du_hi)
    iter_ms, setup_ms = [], []

    def step_resident():                       # inputs already in HBM; new stage data every step (LTV / RTI)
        s.set_stages(A_d, B_d); s.set_x0(x0_d); s.reset(); s.solve(ITERS)
        info = s.get_info()                    # waits for the solve; device times of the two kernels
        iter_ms.append(info["iter_ms"]); setup_ms.append(info["setup_ms"])

    # e2e: the calls a user makes, pinned host buffers in and out.  The batch is cut into slices of whole waves of CTAs
    # (a multiple of the SM count instances each; instances are independent), one handle and stream per slice, and the
    # loop is software-pipelined: as soon as a slice's results of step i have been read back, its inputs of step i+1 are
    # enqueued, so every step's H2D / D2H copies (all inside the timed region) overlap the other slices' solves.
    sms = s.get_info()["sm_count"]
    per = -(-BATCH // (7 * sms)) * sms
    cuts = [(a, min(a + per, BATCH)) for a in range(0, BATCH, per)]
    pair = []
    for a, b_ in cuts:
        h = pimpc.Solver(prob.nx, prob.nu, prob.N, b_ - a, dtype="f32", engine=args.engine, rho=prob.rho,
                         stream=torch.cuda.Stream().cuda_stream)
        h.set_cost(prob.Q, prob.R)
        h.set_bounds(prob.lo, prob.hi, prob.du_lo, prob.du_hi)
        pair.append((h, slice(a, b_)))

    def e2e_issue(h, sl):
        h.set_stages(A_h[sl], B_h[sl]); h.set_x0(x0_h[sl]); h.reset(); h.solve(ITERS)

    def e2e_collect(h, sl):
        h.get(x_h[sl], u_h[sl], du_h[sl], res_h[sl])

    def e2e_steps(k):
        for h, sl in pair:
            e2e_issue(h, sl)
        for step in range(k):
            for h, sl in pair:
                e2e_collect(h, sl)
                if step + 1 < k:
                    e2e_issue(h, sl)

    for _ in range(args.warmup):
        step_resident()
    iter_ms.clear(); setup_ms.clear()
    l0 = s.get_info()["total_launches"]
    clocks = Clocks(local_rank)
    if rank == 0:
        clocks.start(); time.sleep(0.3)
    replicas.barrier(local_rank)
    t0 = time.perf_counter()
    ms = timed_loop(torch, args.steps, step_resident)
    t1 = time.perf_counter()
    replicas.barrier(local_rank)
    launches = s.get_info()["total_launches"] - l0
    ck = clocks.stop(t0, t1) if rank == 0 else None
    ms = replicas.max_over_ranks(ms, local_rank)
    info = s.get_info()

    e2e_steps(max(1, args.warmup // 2))
    replicas.barrier(local_rank)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record()                               # the slices run on their own streams: events bracket full device syncs
    e2e_steps(args.steps)
    torch.cuda.synchronize()
    ev1.record(); ev1.synchronize()
    ms_e2e = ev0.elapsed_time(ev1)
    replicas.barrier(local_rank)
    ms_e2e = replicas.max_over_ranks(ms_e2e, local_rank)
    res = np.frombuffer(res_h.numpy().tobytes(), dtype=pimpc.RESULT_DTYPE)
    assert np.all(res["iters"] == ITERS) and np.all(np.isfinite(res["c"])), "bench: solver did not run"

    if rank != 0:
        return 0
    nst = BATCH * prob.N
    k_ms = statistics.mean(iter_ms)
    engine = info["engine"]
    if engine == pimpc.ENGINE_STAGED:
        alg = bytes_per_stage_iter(prob.nx, prob.nu, 4) * nst * ITERS
        roof = {"bound": "hbm", "achieved": alg / k_ms / 1e6, "peak": pk["hbm_gbs"], "unit": "GB/s",
                "kernel": "STAGED engine: 5 kernels per iteration (k_hat,k_adj,k_primal,k_dual,k_decide)", "traffic": None}
    else:
        fl = flops_per_stage_iter(prob.nx, prob.nu) * nst * ITERS
        roof = {"bound": "alu", "achieved": fl / k_ms / 1e9, "peak": max(onchip["ffma2_tflops"], onchip["ffma_tflops"]),
                "unit": "TFLOP/s", "kernel": "k_res2<float,12,4> (RESIDENT engine: one persistent launch per solve)", "traffic": None,
                "peak_nominal": alu_peak_tflops("f32", pk["sm_max_mhz"]), "measured_onchip_peaks": onchip,
                "algorithmic_GBps_if_streamed": bytes_per_stage_iter(prob.nx, prob.nu, 4) * nst * ITERS / k_ms / 1e6}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["peak_source"] = ("MEASURED_PEAKS.json hbm_gbs" if pk["source"] == "measured" else "fallback hbm_gbs") \
        if roof["bound"] == "hbm" else \
        "pimpc_measure_peaks(): FP32 FMA dependency-chain microbenchmarks (scalar FFMA and packed FFMA2; the larger one) run " \
        "on this GPU just before the timed region (the FMA pipe binds phases B and C: DESIGN.md section 6; the measured " \
        "shared-memory peak is in measured_onchip_peaks)"
    roof["kernel_ms_per_launch"] = k_ms
    roof["cache_kernel_ms"] = statistics.mean(setup_ms)
    roof["traffic"] = ncu_traffic(engine, "C4_f32")

    h2d = A_h.numel() * 4 + B_h.numel() * 4 + x0_h.numel() * 4
    d2h = (x_h.numel() + u_h.numel() + du_h.numel()) * 4 + res_h.numel()
    out = {
        "metric": "batched_solves_per_s", "value": world * BATCH * args.steps / (ms / 1e3), "unit": "solves/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(world),
        "e2e": {"value": world * BATCH * args.steps / (ms_e2e / 1e3), "unit": "solves/s", "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e / args.steps,
                "how": f"{len(pair)} handles x {per} instances (whole waves of {sms} CTAs) on their own streams, pinned host "
                       "buffers, software-pipelined: a slice's next inputs are enqueued right after its results were read"},
        "gpu_launches": int(launches), "clocks": ck, "roofline": roof,
        "engine": {1: "staged", 2: "resident", 3: "stream", 4: "coop"}.get(engine, str(engine)),
        "iterations_per_s": world * BATCH * ITERS * args.steps / (ms / 1e3),
        "us_per_iteration_batch": 1e3 * k_ms / ITERS,
    }
    if world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        n_s = 2048
        v, dt = oracle_solves_per_s(prob, list(range(n_s)), ITERS, cores)
        out["cpu_baseline"] = {"value": v, "unit": "solves/s", "cores": cores, "kind": "oracle",
                               "sample": f"first {n_s} of the {BATCH} instances, {ITERS} iterations each, once "
                                         f"({dt:.1f} s; single-threaded C oracle, {cores} instances in flight)"}
    s.close()
    for h, _ in pair:
        h.close()
    if world == 1 and not args.no_extras:
        out["extras"] = extras(torch, pimpc, pk, args.extras)
    print(json.dumps(out))
    return 0


if __name__ == "__main__":
    sys.exit(main())
