"""GPU: the fused f + grad kernel on BASELINE.json config 4 (n = 2^24, two random 40-byte neighbour rows per vertex)
against a program that only moves the traffic of that pass, measured in the same process run by
tests/probes/traffic_floor.cu (no arithmetic; per vertex 96 B streamed in, 48 B out, two random rows gathered in
the most request-efficient pattern).  DESIGN.md section 6: by algorithmic bytes the kernel sits at about 0.36 of the
streaming-copy roofline; this test pins the statement that the gap is the input's and not the kernel's -- the kernel
must stay within 15 % of the traffic-only program.  Measured: the probe's best over 3 .. 8 blocks per SM moves between
1.02 and 1.08 ms from box to box; the kernel took 1.105 - 1.118 ms while it chose between the staged tile and global
memory by a branch per neighbour, and takes 1.01 - 1.05 ms -- less than the probe, which is a program written the obvious
way, not a bound -- since it issues predicated load pairs (profiles/r2d_README.md).  The probe's numbers are printed
(-s) for profiles/."""
import json
import os
import subprocess

import pytest

from paper_2505_15775_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "probes", "traffic_floor.cu")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build_probe(out):
    subprocess.check_call([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-o", out, SRC])
    return out


def test_probe_compiles(tmp_path):
    build_probe(str(tmp_path / "probe"))


@pytest.mark.gpu
def test_config4_kernel_is_at_the_traffic_floor(tmp_path):
    import torch
    from paper_2505_15775_b200 import binding
    exe = build_probe(str(tmp_path / "probe"))
    out = subprocess.run([exe, "24", "40", "96", "48"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    floor = json.loads(out.stdout.strip().splitlines()[-1])
    w = inputs.full(4)
    P, r = w.problem, w.r
    ctx = binding.Context(P, w.dtype)
    R = torch.as_tensor(w.R, dtype=torch.float32).cuda()
    G = torch.empty_like(R)
    y = torch.as_tensor(w.y).cuda()
    z = torch.empty(P.m, dtype=torch.float64, device="cuda")
    ctx.set_dual(y, w.sigma)
    for _ in range(3):
        ctx.eval(R, r, r, G, z, stats=False)
    ctx.kernel_timing(1)
    for _ in range(20):
        ctx.eval(R, r, r, G, z, stats=False)
    ms, cnt = ctx.kernel_timing_read()
    ctx.close()
    kern = ms / cnt
    print(json.dumps({"probe": floor, "k_rows_tiled_fused_eval_ms": kern, "ratio": kern / floor["mix_ms"]}))
    assert cnt == 20 and kern <= 1.15 * floor["mix_ms"], (kern, floor)
