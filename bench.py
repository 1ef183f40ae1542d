"""bench.py -- throughput of the ALM-BM hot path (BASELINE.json metric) on synthetic inputs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

One "step" = one pass of the whole hot path at one point R:
alora_eval (f + grad), alora_linesearch (quartic coefficients along D, cold form) and one alora_smatvec
(Lanczos matvec S(lambda)v).  `value` = steps/s, i.e. f+grad evaluations/s with each evaluation
accompanied by its line-search and matvec work, inputs resident in HBM.  The default workload is
BASELINE.json's largest single-GPU configuration, config 4 (MaxCut, n = 2^24, r = 10, fp32): its arrays
(R 671 MB, sparse data 738 MB) are several times the 126 MB L2, so nothing is flushed between steps; for
the configurations whose working set fits in L2 (0-3, 5-7) an L2-flushed figure is reported beside the
warm one.  Extra keys: the eval-only rate, the dominant kernel's roofline (algorithmic bytes and, when a
capture of the same kernel source is committed, measured DRAM bytes), the end-to-end rate of the SAME
step through host buffers (`alora_step_host`), and the oracle timed on the host cores (one core, and one
copy per core).  N > 1 runs N independent replicas (replicas only), one process
per GPU, value = total steps of all ranks / max-over-ranks time.

`--impl reference` times the CPU oracle (oracle/) on the same metric; each of its steps is the oracle's
full step on a bounded sample of the workload (the same generator at a smaller n), scaled by the size
ratio, so that K + W steps end within a few minutes.
"""
from __future__ import annotations

import argparse
import hashlib
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
L2_BYTES = 126e6
KERNEL_SOURCES = ("rows_tiled.cuh", "kernels.cuh")     # what a traffic capture is tied to


def workload(idx: int, mc: str = ""):
    if idx in (1, 6) and mc:   # other grid sizes: --mc side
        return (inputs.config1 if idx == 1 else inputs.config6)(side=int(mc))
    if idx == 4 and mc:        # other sizes of the ring + matchings graph: --mc log2(n)
        return inputs.config4(n=1 << int(mc))
    if idx == 5 and mc:        # other rows of the paper's Table 2: --mc n,r_star
        n, rs = (int(x) for x in mc.split(","))
        return inputs.config5(n=n, r_star=rs)
    return inputs.full(idx)


def config_dict(w, world: int) -> dict:
    """The `config` object of the JSON line: identical in both arms (no run-specific keys)."""
    return {"workload": w.name, "n": int(w.problem.n), "m": int(w.problem.m), "r": int(w.r),
            "parallelism": f"replicas x{world}"}


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


def kernel_source_sha() -> str:
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        h.update(open(os.path.join(ROOT, "paper_2505_15775_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(name: str, n: int):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/traffic.json:
    dram__bytes_read.sum + dram__bytes_write.sum of one launch, with the sha of the kernel sources it was taken
    on).  None when there is no capture of this workload or the kernel sources have changed since."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        e = json.load(open(p)).get(name, {})
        if e.get("n") == n and e.get("kernel_source_sha") == kernel_source_sha():
            return e.get("dram_bytes_per_launch")
    except (ValueError, OSError):
        pass
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


# ----------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference): the only places that touch oracle/
# ----------------------------------------------------------------------------------------------
def oracle_step_fn(w):
    """One full step of the oracle as it stands (single thread, fp64): f, grad, line-search coefficients, one
    matvec with lambda of that point."""
    from oracle.oracle import Oracle
    o = Oracle(w.problem)
    lam, _ = o.lam(w.y, w.sigma, w.R)

    def step():
        o.f(w.y, w.sigma, w.R)
        o.grad(w.y, w.sigma, w.R)
        o.linesearch(w.y, w.sigma, w.R, w.D)
        o.smatvec(lam, w.V)
    return step


def oracle_step_seconds(w, budget_s: float = 15.0, max_steps: int = 50):
    """(seconds per step, steps timed) on one core."""
    step = oracle_step_fn(w)
    t_all, k = 0.0, 0
    while True:
        t0 = time.perf_counter()
        step()
        t_all += time.perf_counter() - t0
        k += 1
        if t_all >= budget_s or k >= max_steps:
            break
    return t_all / k, k


def _oracle_child(w, steps, q):
    step = oracle_step_fn(w)
    t0 = time.perf_counter()
    for _ in range(steps):
        step()
    q.put(time.perf_counter() - t0)


def oracle_all_cores(w, sec_per_step: float, budget_s: float = 15.0):
    """The oracle is single-threaded; "all cores" = one independent copy of it per core (forked after the inputs
    exist, so they are shared copy-on-write), each running the same steps concurrently.  Returns
    (steps/s of all copies together, copies) or None when memory does not allow two copies."""
    import multiprocessing as mp
    cores = os.cpu_count() or 1
    per_copy = 6 * w.R.nbytes + 16 * w.problem.m + (64 << 20)      # outputs and temporaries of one copy
    try:
        avail = int(next(ln for ln in open("/proc/meminfo") if ln.startswith("MemAvailable")).split()[1]) * 1024
    except (OSError, StopIteration):
        avail = 8 << 30
    copies = int(max(1, min(cores, avail // (2 * per_copy), 64)))
    if copies < 2:
        return None
    steps = int(max(1, min(20, budget_s / max(sec_per_step, 1e-9) / 2)))
    ctx = mp.get_context("fork")
    q = ctx.Queue()
    procs = [ctx.Process(target=_oracle_child, args=(w, steps, q)) for _ in range(copies)]
    t0 = time.perf_counter()
    for p in procs:
        p.start()
    times = [q.get() for _ in procs]
    for p in procs:
        p.join()
    wall = time.perf_counter() - t0
    return copies * steps / max(wall, max(times)), copies


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


def reference_sample(args):
    """The workload the reference arm's steps run on: the configured workload itself when the oracle does K + W
    steps of it within ~2 minutes, else the same generator at a smaller n (a power of two for config 4, a smaller
    grid for configs 1 and 6); rates are scaled by n_sample / n."""
    full_rows = {0: 800, 1: 10 ** 6, 2: 20000, 3: 10 ** 5, 4: 1 << 24, 5: 10 ** 4, 6: 10 ** 6, 7: 1 << 20}[args.config]
    us_per_row = {0: 0.8, 1: 0.35, 2: 2.1, 3: 3.0, 4: 0.55, 5: 2.7, 6: 0.43, 7: 1.7}[args.config]   # oracle, measured round 1
    budget = 100.0 / max(1, args.steps + args.warmup)          # seconds per step
    if args.mc or full_rows * us_per_row * 1e-6 <= budget:
        return workload(args.config, args.mc), 1.0, "the full workload"
    if args.config == 4:
        lg = 24
        while lg > 12 and (1 << lg) * us_per_row * 1e-6 > budget:
            lg -= 1
        ws = inputs.config4(n=1 << lg)
        return ws, (1 << lg) / full_rows, f"ring + two matchings generator (seed 1004) at n = 2^{lg}; rate scaled by 2^{lg - 24}"
    if args.config in (1, 6):
        side = 1000
        while side > 40 and side * side * us_per_row * 1e-6 > budget:
            side = int(side * 0.8)
        ws = (inputs.config1 if args.config == 1 else inputs.config6)(side=side)
        return ws, side * side / full_rows, f"same torus generator at side {side}; rate scaled by {side * side / full_rows:.4g}"
    return workload(args.config, args.mc), 1.0, "the full workload"


def run_reference(args, rank, world):
    """--impl reference: the oracle (kind: oracle, one host thread), W warm-up steps, then K timed steps."""
    if rank != 0:
        return
    ws, scale, how = reference_sample(args)
    if scale == 1.0:
        cfg = config_dict(ws, world)
    else:   # describe the FULL workload (same keys and values as the GPU arm) without building it
        full_n = {4: 1 << 24, 1: 10 ** 6, 6: 10 ** 6}[args.config]
        cfg = {"workload": ws.name, "n": full_n, "m": full_n, "r": int(ws.r), "parallelism": f"replicas x{world}"}
    step = oracle_step_fn(ws)
    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    val = args.steps / dt * scale
    sample = f"{args.steps} full oracle steps (f, grad, line-search coefficients, matvec) on {how}"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 / val, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_solve(args, w, local, torch, binding):
    """ALM solve time (BASELINE.json metric, third part): alora_solve from a resident problem, with the library's
    preset for the context dtype (alora_preset_params).  Config 0 stops at KKT <= 1e-6, config 4 at relative
    primal infeasibility <= 1e-5 (BASELINE.json), the others at the paper's rule KKT (eq. 77) <= 1e-5."""
    P, r0 = w.problem, w.r
    t0 = time.perf_counter()
    ctx = binding.Context(P, w.dtype, device=local)
    t_create = time.perf_counter() - t0
    tdt = torch.float32 if w.dtype == inputs.F32 else torch.float64
    r_cap = args.r_cap or (64 if P.n <= 1000 else r0 + 14)
    Rbuf = torch.zeros(P.n * r_cap, dtype=tdt, device="cuda")
    Rbuf[: P.n * r0] = torch.as_tensor(w.R, dtype=tdt).cuda().reshape(-1)
    y = torch.zeros(P.m, dtype=torch.float64, device="cuda")   # Alg. 1: y0 = 0
    kw = dict(eps=1e-6, stop_mode=0) if args.config == 0 else dict(eps=1e-5, stop_mode=1) if args.config == 4 \
        else dict(eps=1e-5, stop_mode=0)
    for kv in args.param:
        k, v = kv.split("=")
        kw[k] = float(v) if ("." in v or "e" in v) else int(v)
    prm = binding.Params.preset(w.dtype, **kw)
    l0 = ctx.info()["launches"]
    torch.cuda.synchronize()
    res, log, r, sg, ok = ctx.solve(prm, Rbuf, r0, r_cap, y, w.sigma)
    line = {"mode": "solve", "metric": "ALM solve time", "value": res.seconds, "unit": "s", "higher_is_better": False,
            "config": {"workload": w.name, "n": P.n, "m": P.m, "r0": r0, "r_cap": r_cap, "stop": kw,
                       "it_max": prm.it_max, "stall_tol": prm.stall_tol, "lbfgs_mem": prm.lbfgs_mem},
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
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4,
                    help="BASELINE.json config index (default 4: MaxCut n = 2^24, the largest single-GPU configuration)")
    ap.add_argument("--ld", type=int, default=0, help="leading dimension of R/G/D (default r)")
    ap.add_argument("--mode", default="path", choices=["path", "solve"],
                    help="path: the hot-path step (default, the bench contract); solve: ALM solve time of the config")
    ap.add_argument("--r-cap", type=int, default=0)
    ap.add_argument("--param", action="append", default=[], help="solve mode: alora_params override, e.g. --param lbfgs_mem=3")
    ap.add_argument("--mc", default="", help="config 5: 'n,r_star' of another row of the paper's Table 2; configs 1 and 6: grid side; config 4: log2 n")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-flush", action="store_true", help="skip the L2-flushed figures of the L2-resident configs")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    w = workload(args.config, args.mc)
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
        if ld == r:
            return np.ascontiguousarray(a, ndt)
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
    B_eval, B = algorithmic_bytes(w, info)
    resident = B_eval < 2 * L2_BYTES      # the step's arrays (partly) fit in L2: report an L2-flushed figure as well

    def step():
        ctx.eval(R, r, ld, G, z, stats=False)
        ctx.linesearch(R, D, r, ld, fetch=False)
        ctx.smatvec(lam, V, 1, W, fetch=False)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    warm = max(3, args.warmup)
    for _ in range(warm):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:   # untimed steps of the same load until nvidia-smi has produced its first sample
        sampler.wait_first(lambda: (step(), torch.cuda.synchronize()))
    l0 = ctx.info()["launches"]
    every = 8 if args.steps >= 64 else 1
    ctx.kernel_timing(every)   # every 8th evaluation of the timed region is bracketed by events
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

    # the same step with the WARM line search (what alora_solve and alora_step_host run: the line search follows an
    # evaluation of the same R and streams its gradient, reading 31) -- reported beside the cold-form `value`
    pls = ctx.get_linesearch()    # coefficients of the last cold line search of the timed region
    def step_warm():
        ctx.eval(R, r, ld, G, z, stats=False)
        ctx.linesearch(R, D, r, ld, fetch=False, warm=True)
        ctx.smatvec(lam, V, 1, W, fetch=False)
    for _ in range(3):
        step_warm()
    barrier(); e0.record()
    for _ in range(args.steps):
        step_warm()
    e1.record(); barrier()
    ms_warm = aggregate_ms(e0.elapsed_time(e1), world)
    pls_warm = ctx.get_linesearch()

    # eval-only rate (the metric's bare "f+grad evals/s"), same hygiene
    barrier(); e0.record()
    for _ in range(args.steps):
        ctx.eval(R, r, ld, G, z, stats=False)
    e1.record(); barrier()
    eval_only = args.steps / (e0.elapsed_time(e1) * 1e-3)
    st = ctx.get_stats()

    # L2-flushed figures (configs whose arrays fit in L2): a 256 MB scratch write before every step, each step timed
    # by its own event pair so that the flush is outside the timed spans
    flushed = None
    if resident and not args.no_flush:
        scratch = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        kf = min(args.steps, 50)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(kf)]
        ctx.kernel_timing(1)
        for a, b in evs:
            scratch.fill_(1)
            a.record(); step(); b.record()
        barrier()
        fk_ms, fk_n = ctx.kernel_timing_read()
        ctx.kernel_timing(False)
        fms = float(np.median([a.elapsed_time(b) for a, b in evs]))
        fms = aggregate_ms(fms, world)
        flushed = {"value": whole_job_value(1, world, fms), "unit": UNIT, "ms_per_step": fms,
                   "kernel_ms": fk_ms / max(1, fk_n), "steps": kf,
                   "how": "256 MB scratch write before every step; median of per-step CUDA-event spans"}
        del scratch

    # end to end: the SAME step through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        Rh = torch.from_numpy(padded(w.R)).pin_memory(); Dh = torch.from_numpy(padded(w.D)).pin_memory()
        Vh = torch.from_numpy(w.V.astype(ndt)).pin_memory()
        Gh = torch.empty_like(Rh).pin_memory(); Wh = torch.empty_like(Vh).pin_memory()
        zh = torch.empty(P.m, dtype=torch.float64).pin_memory()
        hargs = (Rh.numpy(), Dh.numpy(), Vh.numpy(), r, ld, Gh.numpy(), zh.numpy(), Wh.numpy())
        k2 = max(3, min(args.steps, 20))
        for _ in range(3):
            ctx.step_host(*hargs)
        barrier(); e0.record()
        for _ in range(k2):
            sth, ph, vwh = ctx.step_host(*hargs)
        e1.record(); barrier()
        ms2 = aggregate_ms(e0.elapsed_time(e1), world)
        esz = Rh.element_size()
        e2e = {"value": whole_job_value(k2, world, ms2), "unit": UNIT, "steps": k2,
               "h2d_bytes_per_step": int(2 * Rh.numel() * esz + Vh.numel() * esz),
               "d2h_bytes_per_step": int(Gh.numel() * esz + zh.numel() * 8 + Wh.numel() * esz + 8 * (16 + 16 + 16)),
               "call": "alora_step_host: R, D, V host -> G, z, W, f, p0..p4, <V,W> host"}
        assert abs(sth[0] - st[0]) <= 1e-9 * (1 + abs(st[0]))
        del Rh, Dh, Gh

    if rank == 0:
        peak, peak_src = peaks()
        kavg_ms = kern_ms / max(1, kern_n)
        achieved = B / (kavg_ms * 1e-3) / 1e9 if kern_n else None
        traffic = ncu_traffic(w.name, P.n)
        roof = {"bound": "hbm", "kernel": "k_rows_tiled (fused f+grad pass)" if info["cls"] == 0 else "k_rows (adjoint pass)",
                "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                "frac": (achieved / peak) if achieved else None, "algorithmic_bytes": B,
                "algorithmic_bytes_whole_eval": B_eval, "kernel_ms": kavg_ms, "kernel_launches_timed": kern_n,
                "traffic": traffic,
                "frac_dram": (traffic / (kavg_ms * 1e-3) / 1e9 / peak) if (traffic and kern_n) else None}
        if flushed:
            fa = B / (flushed["kernel_ms"] * 1e-3) / 1e9
            flushed.update(roofline_achieved=fa, roofline_frac=fa / peak)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": warm, "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32" if w.dtype == inputs.F32 else "f64",
                "data": "synthetic", "config": config_dict(w, world),
                "run": {"edges": w.meta.get("edges"), "ld": ld,
                        "class": "diagonal (one fused pass)" if info["cls"] == 0 else "general (forward + adjoint)",
                        "l2": ("no flush: the step's arrays (%.0f MB per evaluation) exceed the 126 MB L2 several times" % (B_eval / 1e6))
                        if not resident else "value is L2-warm (the evaluation's %.0f MB fit in L2); see `flushed`" % (B_eval / 1e6),
                        "timing": "CUDA events on the ctx stream around K steps; dominant kernel by event pairs inside alora_eval"},
                "eval_only_per_s": eval_only,
                "warm_linesearch": {"value": whole_job_value(args.steps, world, ms_warm), "unit": UNIT, "ms_per_step": ms_warm / args.steps,
                                    "what": "same step with alora_linesearch(warm=1): p1 = <G,D> from the evaluation's gradient, only the D operand gathered"},
                "roofline": roof, "flushed": flushed,
                "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e,
                "check": {"f": st[0], "gnorm": float(np.sqrt(st[4])), "p": [float(x) for x in pls], "p_warm": [float(x) for x in pls_warm]}}
        if not args.no_cpu_baseline and world == 1:
            sec, k = oracle_step_seconds(w)
            cb = {"value": 1.0 / sec, "unit": UNIT, "cores": 1, "kind": "oracle",
                  "sample": f"{k} full steps (f, grad, line-search coefficients, matvec) of {w.name}, one thread"}
            allc = oracle_all_cores(w, sec)
            if allc:
                cb["all_cores"] = {"value": allc[0], "cores": allc[1], "host_cores": os.cpu_count(),
                                   "how": "one independent copy of the single-threaded oracle per core, same step, run concurrently"}
            line["cpu_baseline"] = cb
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
