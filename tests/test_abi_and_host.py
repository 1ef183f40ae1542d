"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol that
include/alora.h declares, rejects bad problems without a GPU, fails loudly (no CPU fallback), and
the multi-process aggregation used by bench.py works under gloo with world_size 2."""
import ctypes
import os
import re
import subprocess
import sys
import time

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2505_15775_b200 import build
    return ctypes.CDLL(build.build())


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "alora.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(alora_[a-z_0-9]+)\s*\(", txt)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_symbols()
    assert len(names) >= 18 and "alora_eval" in names and "alora_solve" in names
    for nm in names:
        assert hasattr(lib, nm), f"{nm} declared in include/alora.h but not exported"


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "alora.h"\nint main(void){alora_params p; alora_default_params(&p); return p.k_max==300?0:1;}\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-fsyntax-only", "-I", os.path.join(ROOT, "include"), str(src)])


def test_params_struct_layout_matches_binding(lib):
    from paper_2505_15775_b200 import binding
    p = binding.Params()
    assert (p.eps, p.T_max, p.it_max, p.lbfgs_mem, p.k_max, p.gamma, p.kappa, p.tau_shrink, p.seed) == \
           (1e-5, 100, 500, 5, 300, 2.0, 0.25, 1e-8, 12345)
    from oracle import alm
    q = alm.Params()
    for f in ("eps", "stop_mode", "T_max", "tol0", "c_in", "tol_min", "it_max", "lbfgs_mem", "p_max", "k_max",
              "tau_neg", "tol_eig", "gamma", "kappa", "sigma_max", "tau_shrink", "s_max", "seed"):
        assert getattr(p, f) == getattr(q, f), f


def test_preset_matches_oracle_preset(lib):
    from paper_2505_15775_b200 import binding
    from oracle import alm
    for dt, f32 in (("f32", True), ("f64", False)):
        p, q = binding.Params.preset(dt), alm.preset_params(f32)
        for f in ("eps", "it_max", "lbfgs_mem", "stall_tol", "stall_iters", "tol0", "c_in", "tol_min", "gamma", "kappa"):
            assert getattr(p, f) == getattr(q, f), (dt, f)
    assert binding.Params.preset("f32").it_max == 100 and binding.Params.preset("f64").it_max == 500


def test_create_validates_and_has_no_cpu_fallback():
    import torch
    from paper_2505_15775_b200 import binding, inputs
    P = inputs.small(1).problem
    bad = inputs.Problem(**{**P.__dict__})
    bad.C_row = P.C_col.copy(); bad.C_col = P.C_row.copy()      # row > col somewhere
    with pytest.raises(binding.AloraError) as e:
        binding.Context(bad, "f32")
    assert e.value.status == binding.EINVAL
    bad2 = inputs.Problem(**{**P.__dict__}); bad2.b = P.b.copy(); bad2.b[3] = np.nan
    with pytest.raises(binding.AloraError) as e:
        binding.Context(bad2, "f32")
    assert e.value.status == binding.EINVAL
    if not torch.cuda.is_available():
        with pytest.raises(binding.AloraError) as e:
            binding.Context(P, "f32")
        assert e.value.status == binding.ECUDA


def test_product_path_does_not_import_oracle():
    for rel in ("paper_2505_15775_b200/binding.py", "paper_2505_15775_b200/inputs.py", "paper_2505_15775_b200/build.py"):
        src = open(os.path.join(ROOT, rel)).read()
        assert "import oracle" not in src and "from oracle" not in src, rel
    for f in os.listdir(os.path.join(ROOT, "paper_2505_15775_b200", "csrc")):
        if f.endswith((".cu", ".cuh", ".h", ".inc")):
            assert "oracle/" not in open(os.path.join(ROOT, "paper_2505_15775_b200", "csrc", f)).read(), f


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
ms = 10.0 + 5.0 * int(sys.argv[1])
out = bench.aggregate_ms(ms, 2, device="cpu")
val = bench.whole_job_value(steps=100, world=2, ms=out)
assert out == 15.0, out
assert abs(val - 2 * 100 / 15e-3) < 1e-6
dist.barrier(); dist.destroy_process_group()
print("ok")
"""


def test_replica_aggregation_gloo_world2(tmp_path):
    port = 29500 + os.getpid() % 2000
    script = tmp_path / "w.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0 and "ok" in out, err[-2000:]


def test_clock_sampler_parses_samples_and_waits_for_the_first(tmp_path, monkeypatch):
    """bench.ClockSampler with a stand-in for nvidia-smi: wait_first keeps calling the load until the
    first line is there, stop() reports the median clock and the active throttle reasons."""
    import bench
    fake = tmp_path / "nvidia-smi"
    fake.write_text("#!/bin/bash\nsleep 0.3\nfor i in 1 2 3 4 5 6 7 8 9 10; do echo '1965, 1965, Not Active, Not Active, Not Active, Active'; sleep 0.02; done\nsleep 30\n")
    fake.chmod(0o755)
    monkeypatch.setenv("PATH", str(tmp_path) + os.pathsep + os.environ["PATH"])
    s = bench.ClockSampler(0)
    calls = []
    s.wait_first(lambda: (calls.append(1), time.sleep(0.01)), timeout_s=5.0)
    assert len(calls) >= 5          # the first line took 0.3 s
    time.sleep(0.1)
    out = s.stop()
    assert out["sm_mhz"] == 1965.0 and out["sm_max_mhz"] == 1965.0 and out["reasons"] == ["sw_power_cap"]
