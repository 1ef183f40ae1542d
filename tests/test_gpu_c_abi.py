"""GPU: the C ABI driven by a plain C program (tests/c_driver/alora_c_driver.c, compiled here with gcc against
include/alora.h, linked with csrc/libalora.so and the CUDA runtime) on BASELINE.json config 0; the scalars it
prints are compared with the oracle.  Shows that the boundary needs nothing from Python or torch."""
import os
import subprocess

import numpy as np
import pytest

from paper_2505_15775_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "c_driver", "alora_c_driver.c")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def build_driver(out):
    from paper_2505_15775_b200 import build
    lib = build.build()
    subprocess.check_call(["gcc", "-std=c99", "-O1", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                           "-I", os.path.join(CUDA, "include"), SRC, "-o", out, lib,
                           "-L", os.path.join(CUDA, "lib64"), "-lcudart", "-lm",
                           "-Wl,-rpath," + os.path.dirname(lib), "-Wl,-rpath," + os.path.join(CUDA, "lib64")])
    return out


def test_c_driver_compiles(tmp_path):
    """CPU: the driver is valid C99 against the header and links with the library (no device needed)."""
    build_driver(str(tmp_path / "drv"))


@pytest.mark.gpu
def test_c_driver_matches_oracle(tmp_path, oracle_mod):
    from oracle import alm
    w = inputs.full(0)
    P, r = w.problem, w.r
    y = np.random.default_rng(3).standard_normal(P.m)
    path = tmp_path / "p.bin"
    with open(path, "wb") as f:
        np.array([P.n, P.m, P.nnzC, P.nnzA, r], np.int64).tofile(f)
        for a, dt in ((P.C_row, np.int32), (P.C_col, np.int32), (P.C_val, np.float64), (P.A_ptr, np.int64),
                      (P.A_row, np.int32), (P.A_col, np.int32), (P.A_val, np.float64), (P.b, np.float64),
                      (y, np.float64), (np.array([w.sigma]), np.float64), (w.R, np.float64), (w.D, np.float64),
                      (w.V, np.float64)):
            np.ascontiguousarray(a, dt).tofile(f)
    exe = build_driver(str(tmp_path / "drv"))
    out = subprocess.run([exe, str(path)], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    val = {ln.split()[0]: ln.split()[1:] for ln in out.stdout.splitlines() if ln.strip()}
    o = oracle_mod.Oracle(P)
    parts = o.f(y, w.sigma, w.R, parts=True)
    G = o.grad(y, w.sigma, w.R)
    den = abs(parts["cx"]) + abs(parts["yq"]) + 0.5 * w.sigma * parts["qq"]
    assert abs(float(val["f"][0]) - parts["f"]) <= 1e-10 * den
    assert abs(float(val["cx"][0]) - parts["cx"]) <= 1e-10 * den
    assert abs(np.sqrt(float(val["gg"][0])) - np.linalg.norm(G)) <= 1e-10 * np.linalg.norm(G)
    po = o.linesearch(y, w.sigma, w.R, w.D)
    for key in ("p", "pw"):
        assert np.abs(np.array([float(x) for x in val[key]]) - po).max() <= 1e-10 * np.abs(po).sum(), key
    lam, _ = o.lam(y, w.sigma, w.R)
    Wo = o.smatvec(lam, w.V)
    for key in ("vw", "vw0"):
        assert abs(float(val[key][0]) - w.V @ Wo) <= 1e-10 * np.linalg.norm(w.V) * np.linalg.norm(Wo), key
    ev = np.linalg.eigvalsh(o.smatvec(lam, np.eye(P.n)))
    assert abs(float(val["theta1"][0]) - ev[0]) < 1e-8 and val["theta1"][4] == "1"
    th3 = np.array([float(x) for x in val["theta3"][:3]])
    assert np.all(th3 >= ev[:3] - 1e-9) and abs(th3[0] - ev[0]) < 1e-8 and val["theta3"][4] == "3"
    assert int(val["warm_without_eval"][0]) == 4      # ALORA_ESTATE
    ref = alm.solve(o, w.R, np.zeros(P.m), w.sigma, alm.Params(eps=1e-6))
    assert val["solve"][1] == "1" and int(val["solve"][3]) == ref.outer_iters and int(val["solve"][5]) == ref.R.shape[1]
    assert abs(float(val["solve_cx"][0]) - o.inner_C(ref.R, ref.R)) <= 1e-6 * abs(o.inner_C(ref.R, ref.R))
    assert val["class"][0] == "0"
