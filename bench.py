"""bench.py -- throughput of the ALM-BM hot path (BASELINE.json metric) on synthetic inputs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

One "step" = one pass of the whole hot path at one point R:
alora_eval (f + grad), alora_linesearch (quartic coefficients along D) and one alora_smatvec
(Lanczos matvec S(lambda)v).  `value` = steps/s, i.e. f+grad evaluations/s with each evaluation
accompanied by its line-search and matvec work, inputs resident in HBM.  Extra keys give the
eval-only rate, the dominant kernel's roofline, the end-to-end rate through host buffers and the
oracle timed on the host cores.  N > 1 runs N independent replicas (DESIGN.md "Multi-GPU":
replicas only), one process per GPU, value = total steps of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2505_15775_b200 import inputs  # noqa: E402

METRIC = "ALM-BM f+grad evals/sec (each step = f+grad, line-search coefficients, S(lambda)v matvec)"
UNIT = "evals/s"


def workload(idx: int, mc: str = ""):
    if idx in (1, 6) and mc:   # other grid sizes: --mc side
        return (inputs.config1 if idx == 1 else inputs.config6)(side=int(mc))
    if idx == 5 and mc:   # other rows of the paper's Table 2: --mc n,r_star
        n, rs = (int(x) for x in mc.split(","))
        return inputs.config5(n=n, r_star=rs)
    return inputs.full(idx)


def algorithmic_bytes(w, info):
    """Minimum bytes of one f+grad evaluation, SURVEY.md 8(d) / DESIGN.md "Algorithmic bytes":
    every array once (nonzeros + indices + R read + G write + y, b read + z write).
    Returns (bytes of the whole evaluation, bytes of its dominant kernel): the diagonal class is ONE
    kernel; in the general class the dominant kernel is the adjoint pass."""
    P = w.problem
    s = 4 if w.dtype == inputs.F32 else 8
    v = s
    n, m, r = P.n, P.m, w.r
    if info["cls"] == 0:
        full = info["c_nnz"]  # 2|E|
        b = 4 * (n + 1) + (full + n) * (4 + v) + 2 * n * r * s + 24 * n
        return b, b
    e_up, e_full, c_full = info["nf_A"], info["a_nnz"], info["c_nnz"]
    fwd = e_up * (8 + v) + 8 * (m + 1) + n * r * s + 8 * m
    wts = 24 * m
    adj = e_full * (8 + v) + 4 * (n + 1) + (c_full + n) * (4 + v) + 4 * (n + 1) + 8 * m + 2 * n * r * s
    return fwd + wts + adj, adj


def ncu_traffic(name: str, n: int):
    """DRAM bytes per launch of the dominant kernel from the committed ncu --set full capture
    (profiles/traffic.json, written by hand from `ncu -i ... --page raw`), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    try:
        e = json.load(open(p)).get(name, {})
        return e.get("dram_bytes_per_launch") if e.get("n") == n else None
    except (ValueError, OSError):
        return None


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def wait_first(self, keep_busy, timeout_s: float = 4.0):
        """nvidia-smi needs a few hundred ms to print its first line, longer than a short timed region: keep the GPU
        under the same load (`keep_busy` = one untimed step + sync) until the first sample is there."""
        if self.p is None:
            return
        t0 = time.perf_counter()
        while time.perf_counter() - t0 < timeout_s:
            keep_busy()
            try:
                if os.path.getsize(self.f.name) > 0:
                    return
            except OSError:
                return

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons))
        return out


def oracle_step_seconds(w, reps_budget_s: float = 20.0):
    """The oracle as it stands (single thread, fp64) on the same workload: one full step
    (f, grad, line-search coefficients, one matvec).  Returns (seconds per step, steps timed)."""
    from oracle.oracle import Oracle
    o = Oracle(w.problem)
    lam = None
    t_all, k = 0.0, 0
    while True:
        t0 = time.perf_counter()
        o.f(w.y, w.sigma, w.R)
        o.grad(w.y, w.sigma, w.R)
        o.linesearch(w.y, w.sigma, w.R, w.D)
        if lam is None:
            lam, _ = o.lam(w.y, w.sigma, w.R)
        o.smatvec(lam, w.V)
        t_all += time.perf_counter() - t0
        k += 1
        if t_all >= reps_budget_s or k >= 50:
            break
    return t_all / k, k


def aggregate_ms(ms: float, world: int, device="cuda") -> float:
    """Max over ranks of a per-rank duration (the replicas run independently; the job is as slow
    as its slowest rank)."""
    if world == 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(steps: int, world: int, ms: float) -> float:
    """Whole-job throughput: every rank processed `steps` steps."""
    return world * steps / (ms * 1e-3)


def run_reference(args, w, rank, world):
    """--impl reference: the oracle (kind: oracle, one host thread) timed on bounded work."""
    if rank != 0:
        return
    from oracle.oracle import Oracle
    o = Oracle(w.problem)
    lam, _ = o.lam(w.y, w.sigma, w.R)

    def step():
        o.f(w.y, w.sigma, w.R); o.grad(w.y, w.sigma, w.R)
        o.linesearch(w.y, w.sigma, w.R, w.D); o.smatvec(lam, w.V)

    for _ in range(min(args.warmup, 1)):
        step()
    t0 = time.perf_counter()
    k = 0
    for _ in range(args.steps):
        step(); k += 1
        if time.perf_counter() - t0 > 150.0:   # keep the whole run within a few minutes
            break
    dt = time.perf_counter() - t0
    val = k / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": k,
            "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * dt / k, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n": w.problem.n, "m": w.problem.m, "r": w.r},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle",
                             "sample": f"{k} full steps (f, grad, line-search coefficients, matvec) of {w.name}"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_solve(args, w, local, torch, binding):
    """ALM solve time (BASELINE.json metric, third part): alora_solve from a resident problem.
    Config 0 stops at KKT <= 1e-6, config 4 at relative primal infeasibility <= 1e-5."""
    P, r0 = w.problem, w.r
    t0 = time.perf_counter()
    ctx = binding.Context(P, w.dtype, device=local)
    t_create = time.perf_counter() - t0
    tdt = torch.float32 if w.dtype == inputs.F32 else torch.float64
    r_cap = args.r_cap or (64 if P.n <= 1000 else r0 + 14)
    Rbuf = torch.zeros(P.n * r_cap, dtype=tdt, device="cuda")
    Rbuf[: P.n * r0] = torch.as_tensor(w.R, dtype=tdt).cuda().reshape(-1)
    y = torch.zeros(P.m, dtype=torch.float64, device="cuda")   # Alg. 1: y0 = 0
    # config 0: KKT <= 1e-6; config 4: relative primal infeasibility <= 1e-5 (BASELINE.json); others: the paper's
    # rule, KKT (eq. 77) <= 1e-5
    kw = dict(eps=1e-6, stop_mode=0) if args.config == 0 else dict(eps=1e-5, stop_mode=1) if args.config == 4 \
        else dict(eps=1e-5, stop_mode=0)
    if args.config == 4:
        kw["it_max"] = 100   # inexact inner solves; measured 17 s against 95 s with the default 500
    if w.dtype == inputs.F32 and args.config == 5:
        kw["stall_tol"] = 1e-9   # fp32 rounding floor of f (reading 28)
    for kv in args.param:
        k, v = kv.split("=")
        kw[k] = float(v) if ("." in v or "e" in v) else int(v)
    l0 = ctx.info()["launches"]
    torch.cuda.synchronize()
    res, log, r, sg, ok = ctx.solve(binding.Params(**kw), Rbuf, r0, r_cap, y, w.sigma)
    line = {"mode": "solve", "metric": "ALM solve time", "value": res.seconds, "unit": "s", "higher_is_better": False,
            "config": {"workload": w.name, "n": P.n, "m": P.m, "r0": r0, "r_cap": r_cap, "stop": kw},
            "converged": bool(ok), "outer_iters": res.outer_iters, "n_evals": res.n_evals,
            "n_linesearch": res.n_linesearch, "n_matvec": res.n_matvec, "r_final": r, "sigma_final": sg,
            "kkt": list(res.kkt), "create_seconds": t_create, "gpu_launches": ctx.info()["launches"] - l0,
            "dtype": "f32" if w.dtype == inputs.F32 else "f64", "data": "synthetic",
            "log": [dict(t=a.t, r=a.r, sigma=a.sigma, cx=a.cx, qnorm=a.qnorm, theta1=a.theta1, inner=a.inner_iters,
                         lanczos=a.lanczos_steps, grew=a.grew, shrank=a.shrank, kkt=list(a.kkt)) for a in log]}
    print(json.dumps(line), flush=True)
    ctx.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json config index (default 1: torus MaxCut)")
    ap.add_argument("--ld", type=int, default=0, help="leading dimension of R/G/D (default r)")
    ap.add_argument("--mode", default="path", choices=["path", "solve"],
                    help="path: the hot-path step (default, the bench contract); solve: ALM solve time of the config")
    ap.add_argument("--r-cap", type=int, default=0)
    ap.add_argument("--param", action="append", default=[], help="solve mode: alora_params override, e.g. --param lbfgs_mem=3")
    ap.add_argument("--mc", default="", help="config 5: 'n,r_star' of another row of the paper's Table 2; configs 1 and 6: grid side")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    w = workload(args.config, args.mc)
    if args.impl == "reference":
        run_reference(args, w, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2505_15775_b200 import binding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    P = w.problem
    r, ld = w.r, (args.ld or w.r)
    tdt = torch.float32 if w.dtype == inputs.F32 else torch.float64
    ndt = np.float32 if w.dtype == inputs.F32 else np.float64

    def padded(a):
        out = np.zeros((P.n, ld), ndt); out[:, :r] = a
        return out

    if args.mode == "solve":
        run_solve(args, w, local, torch, binding)
        return
    ctx = binding.Context(P, w.dtype, device=local)
    info = ctx.info()
    R, D = torch.from_numpy(padded(w.R)).cuda(), torch.from_numpy(padded(w.D)).cuda()
    G = torch.empty_like(R)
    y = torch.from_numpy(w.y).cuda()
    z = torch.empty(P.m, dtype=torch.float64, device="cuda")
    lam = torch.empty(P.m, dtype=torch.float64, device="cuda")
    V = torch.from_numpy(w.V.astype(ndt)).cuda()
    W = torch.empty_like(V)
    ctx.set_dual(y, w.sigma)
    ctx.eval(R, r, ld, G, z); ctx.get_lambda(lam)

    def step():
        ctx.eval(R, r, ld, G, z, stats=False)
        ctx.linesearch(R, D, r, ld, fetch=False)
        ctx.smatvec(lam, V, 1, W, fetch=False)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:   # untimed steps of the same load until nvidia-smi has produced its first sample
        sampler.wait_first(lambda: (step(), torch.cuda.synchronize()))
    l0 = ctx.info()["launches"]
    ctx.kernel_timing(8 if args.steps >= 64 else True)   # every 8th evaluation of the timed region is bracketed by events
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    kern_ms, kern_n = ctx.kernel_timing_read()
    ctx.kernel_timing(False)
    launches = ctx.info()["launches"] - l0
    clocks = sampler.stop() if sampler else None
    ms = aggregate_ms(ms, world)
    value = whole_job_value(args.steps, world, ms)

    # eval-only rate (the metric's bare "f+grad evals/s"), same hygiene
    barrier(); e0.record()
    for _ in range(args.steps):
        ctx.eval(R, r, ld, G, z, stats=False)
    e1.record(); barrier()
    eval_only = args.steps / (e0.elapsed_time(e1) * 1e-3)
    st = ctx.get_stats(); pls = ctx.get_linesearch()

    # end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        Rh = torch.from_numpy(padded(w.R)).pin_memory()
        Gh = torch.empty_like(Rh).pin_memory()
        zh = torch.empty(P.m, dtype=torch.float64).pin_memory()
        k2 = max(3, min(args.steps, 30))
        for _ in range(3):
            ctx.eval_host(Rh.numpy(), r, ld, Gh.numpy(), zh.numpy())
        barrier(); e0.record()
        for _ in range(k2):
            ctx.eval_host(Rh.numpy(), r, ld, Gh.numpy(), zh.numpy())
        e1.record(); barrier()
        ms2 = aggregate_ms(e0.elapsed_time(e1), world)
        e2e = {"value": whole_job_value(k2, world, ms2), "unit": "evals/s (f+grad only, host R in, host G and z out)",
               "h2d_bytes_per_step": int(Rh.numel() * Rh.element_size()),
               "d2h_bytes_per_step": int(Gh.numel() * Gh.element_size() + zh.numel() * 8 + 64)}

    if rank == 0:
        peak, peak_src = peaks()
        B_eval, B = algorithmic_bytes(w, info)
        kavg_ms = kern_ms / max(1, kern_n)
        achieved = B / (kavg_ms * 1e-3) / 1e9 if kern_n else None
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32" if w.dtype == inputs.F32 else "f64",
                "data": "synthetic",
                "config": {"workload": w.name, "n": P.n, "m": P.m, "edges": w.meta.get("edges"), "r": r, "ld": ld,
                           "class": "diagonal (one fused pass)" if info["cls"] == 0 else "general (forward + adjoint)",
                           "parallelism": f"replicas x{world}", "l2": "no flush: per-step working set > 126 MB L2"
                           if B_eval > 126e6 else "no flush: working set is L2-resident (latency-bound config)"},
                "eval_only_per_s": eval_only,
                "roofline": {"bound": "hbm", "kernel": "k_rows_tiled (fused f+grad pass)" if info["cls"] == 0 else "k_rows (adjoint pass)",
                             "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                             "frac": (achieved / peak) if achieved else None, "algorithmic_bytes": B,
                             "algorithmic_bytes_whole_eval": B_eval,
                             "kernel_ms": kavg_ms, "kernel_launches_timed": kern_n, "traffic": ncu_traffic(w.name, P.n)},
                "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e,
                "check": {"f": st[0], "gnorm": float(np.sqrt(st[4])), "p": [float(x) for x in pls]}}
        if not args.no_cpu_baseline and world == 1:
            sec, k = oracle_step_seconds(w)
            line["cpu_baseline"] = {"value": 1.0 / sec, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": f"{k} full steps (f, grad, line-search coefficients, matvec) of {w.name}"}
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
