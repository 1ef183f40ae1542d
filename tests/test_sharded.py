"""Row-sharded evaluation (paper_2505_15775_b200/sharded.py).

CPU: the partition and the exchange plan are checked by evaluating every shard with the ORACLE (standing in for the
kernels of a rank) -- in one process, and in two gloo processes that exchange halo rows, all-reduce z and the scalars --
against the single-rank oracle: z, every row of G and f must agree to rounding.
GPU (one device): the same with the library as the rank-local backend, the shards evaluated one after the other."""
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2505_15775_b200 import inputs, sharded

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


class OracleBackend:
    """Rank-local arithmetic by the oracle (numpy arrays): what LibraryBackend does with the CUDA library."""

    def __init__(self, shard, oracle_mod):
        self.fwd, self.adj, self.s = oracle_mod.Oracle(shard.P_fwd), oracle_mod.Oracle(shard.P_adj), shard

    def as_tensor(self, a):
        import torch
        return torch.as_tensor(np.asarray(a, float))

    def from_numpy(self, a):
        return np.asarray(a, float)

    def forward(self, R_loc):
        R_loc = np.asarray(R_loc, float)
        return self.fwd.A_op(R_loc), self.fwd.inner_C(R_loc, R_loc)

    def dual(self, z, b, y, sigma):
        z = np.asarray(z, float)
        q = z - b
        return y - sigma * q, float(y @ q), float(q @ q)

    def adjoint(self, lam, R_loc, n_own):
        R_loc = np.asarray(R_loc, float)
        G = self.adj.smatvec(np.asarray(lam, float), R_loc)[:n_own]
        return G, float(np.vdot(G, G)), float(np.vdot(G, R_loc[:n_own]))


def reference(oracle_mod, w):
    o = oracle_mod.Oracle(w.problem)
    return o.f(w.y, w.sigma, w.R), o.grad(w.y, w.sigma, w.R), o.A_op(w.R)


@pytest.mark.parametrize("idx,world", [(1, 2), (3, 2), (3, 3), (0, 4), (4, 2)])
def test_partition_and_plan_single_process(oracle_mod, idx, world):
    w = inputs.small(idx)
    P = w.problem
    sh = sharded.partition(P, world)
    assert sh[0].r0 == 0 and sh[-1].r1 == P.n and all(a.r1 == b.r0 for a, b in zip(sh, sh[1:]))
    # every stored entry is in exactly one forward shard; halo rows are remote; the plan's lists are consistent
    assert sum(s.P_fwd.nnzA for s in sh) == P.nnzA and sum(s.P_fwd.nnzC for s in sh) == P.nnzC
    for s in sh:
        assert np.all((s.halo < s.r0) | (s.halo >= s.r1)) and np.all(np.diff(s.halo) > 0)
        assert sum(len(x) for x in s.recv_slots) == len(s.halo)
        for q in range(world):
            assert len(s.send_rows[q]) == len(sh[q].recv_slots[s.rank])
            np.testing.assert_array_equal(sh[q].halo[sh[q].recv_slots[s.rank]], s.r0 + s.send_rows[q])
    out = sharded.LocalComm.eval_all(sh, [OracleBackend(s, oracle_mod) for s in sh], P.b, w.R, w.y, w.sigma)
    f, G, z = reference(oracle_mod, w)
    np.testing.assert_allclose(out["z"], z, rtol=1e-12, atol=1e-13 * (1 + np.abs(z).max()))
    np.testing.assert_allclose(out["G"], G, rtol=0, atol=1e-12 * np.abs(G).max())
    assert abs(out["f"] - f) <= 1e-12 * (1 + abs(f))
    assert abs(out["gg"] - np.vdot(G, G)) <= 1e-12 * np.vdot(G, G)


_WORKER = r"""
import sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from paper_2505_15775_b200 import inputs, sharded
from oracle import oracle
from tests.test_sharded import OracleBackend
rank = int(sys.argv[1])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=2)
oracle.build()
for idx in (1, 3):
    w = inputs.small(idx)
    P = w.problem
    s = sharded.partition(P, 2)[rank]
    ev = sharded.ShardedEvaluator(s, OracleBackend(s, oracle), sharded.TorchComm(), P.b)
    out = ev.eval(torch.as_tensor(w.R[s.r0:s.r1]), w.y, w.sigma)
    o = oracle.Oracle(P)
    f, G, z = o.f(w.y, w.sigma, w.R), o.grad(w.y, w.sigma, w.R), o.A_op(w.R)
    assert np.allclose(np.asarray(out["z"]), z, rtol=1e-12, atol=1e-13 * (1 + np.abs(z).max())), idx
    assert np.abs(np.asarray(out["G_own"]) - G[s.r0:s.r1]).max() <= 1e-12 * np.abs(G).max(), idx
    assert abs(out["f"] - f) <= 1e-12 * (1 + abs(f)), (idx, out["f"], f)
    assert abs(out["gg"] - np.vdot(G, G)) <= 1e-12 * np.vdot(G, G)
dist.barrier(); dist.destroy_process_group()
print("ok")
"""


def test_sharded_eval_gloo_world2(tmp_path):
    port = 29600 + os.getpid() % 2000
    script = tmp_path / "w.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    for p in procs:
        out, err = p.communicate(timeout=300)
        assert p.returncode == 0 and "ok" in out, err[-3000:]


@pytest.mark.gpu
@pytest.mark.parametrize("idx,world", [(1, 2), (3, 2), (3, 3)])
def test_sharded_eval_library_backend(oracle_mod, idx, world):
    """The library as the rank-local backend, shards evaluated one after the other on one GPU."""
    w = inputs.small(idx)
    P = w.problem
    tol = 2e-5 if w.dtype == inputs.F32 else 1e-10
    sh = sharded.partition(P, world)
    bes = [sharded.LibraryBackend(s, w.dtype) for s in sh]
    out = sharded.LocalComm.eval_all(sh, bes, P.b, w.R, w.y, w.sigma)
    for be in bes:
        be.close()
    f, G, z = reference(oracle_mod, w)
    o = oracle_mod.Oracle(P)
    parts = o.f(w.y, w.sigma, w.R, parts=True)
    assert np.linalg.norm(out["z"] - z) <= tol * np.linalg.norm(z)
    assert np.linalg.norm(out["G"] - G) <= tol * np.linalg.norm(G)
    assert abs(out["f"] - f) <= tol * (abs(parts["cx"]) + abs(parts["yq"]) + 0.5 * w.sigma * parts["qq"])
    assert abs(np.sqrt(out["gg"]) - np.linalg.norm(G)) <= tol * np.linalg.norm(G)
