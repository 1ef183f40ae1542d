"""Row-sharded evaluation of f, grad f and z = A(RR^T) over N ranks -- host-side plan.

STATUS: built and tested on CPU (world size 2, gloo, with the oracle standing in for the kernels of a rank) and on
one GPU (the two shards evaluated one after the other by the library); NOT measured on several GPUs -- BASELINE.json's
target is one GPU, and DESIGN.md section 8 keeps "replicas only" for bench.py.  This module holds index arithmetic,
argument marshalling and the collectives; every floating-point step runs in the library's kernels (or, in the CPU
test, in the oracle).

Plan.  Rows of R and G are partitioned into N contiguous blocks.  A rank keeps
  * its own rows plus a HALO: the remote rows its entries refer to, appended after its own rows (local index space);
  * P_fwd -- the stored entries (of every A_i and of C) whose ROW index j it owns (every stored entry (j, k), j <= k,
    belongs to exactly one rank), in local indices.  Its forward pass gives the rank's share of z and of <C,RR^T>;
    the shares add up to the full quantities (one all-reduce of the m-vector z and of one scalar);
  * P_adj -- every stored entry with an endpoint among its own rows (entries that cross the cut sit on both ranks),
    values DOUBLED, in local indices: (2C - sum_i lambda_i 2A_i) R restricted to the own rows is exactly
    grad f = 2 S(lambda) R there (doubling is exact in floating point); the halo rows of that product are discarded.
Per evaluation: (1) halo exchange of rows of R (all-to-all with fixed index lists), (2) forward pass on P_fwd,
(3) all-reduce of z, (4) lambda = y - sigma (z - b) and the dual scalars from the reduced z (replicated),
(5) adjoint pass on P_adj, (6) all-reduce of the scalars <C,RR^T>, ||G||^2, <G,R>.  MaxCut needs no step (3) in
principle (a constraint lives on one rank); the plan does not special-case it.
The line-search coefficients are not sharded here: p2 .. p4 contain products of all-reduced vectors (q1, q2), which
the C ABI does not hand out.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .inputs import Problem


@dataclass
class Shard:
    rank: int
    world: int
    r0: int                 # own rows [r0, r1) of the global problem
    r1: int
    halo: np.ndarray        # global ids of the remote rows this rank reads, ascending; local id = n_own + position
    P_fwd: Problem          # entries whose row index is own (local indices); all m constraints, the full b
    P_adj: Problem          # entries incident to own rows, values doubled (local indices)
    send_rows: list         # send_rows[q] = OWN-local ids of the rows rank q needs from this rank
    recv_slots: list        # recv_slots[q] = positions in this rank's halo block filled by rank q's rows

    @property
    def n_own(self) -> int:
        return self.r1 - self.r0

    @property
    def n_loc(self) -> int:
        return self.n_own + int(self.halo.shape[0])


def row_blocks(n: int, world: int) -> np.ndarray:
    """Boundaries of `world` contiguous row blocks of nearly equal size: rank p owns [bnd[p], bnd[p+1])."""
    return np.array([(n * p) // world for p in range(world + 1)], dtype=np.int64)


def partition(P: Problem, world: int) -> list:
    """Shards of problem P for `world` ranks (pure index arithmetic; the same on every rank)."""
    n, m = P.n, P.m
    bnd = row_blocks(n, world)
    owner = lambda idx: np.searchsorted(bnd, idx, side="right") - 1
    a_cons = np.repeat(np.arange(m, dtype=np.int64), np.diff(P.A_ptr))
    a_own_r, a_own_c = owner(P.A_row), owner(P.A_col)
    c_own_r, c_own_c = owner(P.C_row), owner(P.C_col)
    shards = []
    for p in range(world):
        r0, r1 = int(bnd[p]), int(bnd[p + 1])
        fa = a_own_r == p                                   # forward: entries whose row index is own
        fc = c_own_r == p
        ga = fa | (a_own_c == p)                            # adjoint: entries with an endpoint among the own rows
        gc = fc | (c_own_c == p)
        used = np.concatenate([P.A_row[ga], P.A_col[ga], P.C_row[gc], P.C_col[gc]]).astype(np.int64)
        halo = np.unique(used[(used < r0) | (used >= r1)])

        def loc(idx):
            idx = np.asarray(idx, np.int64)
            out = idx - r0
            rem = (idx < r0) | (idx >= r1)
            out[rem] = (r1 - r0) + np.searchsorted(halo, idx[rem])
            return out

        def sub(maskA, maskC, scale):
            ar, ac = loc(P.A_row[maskA]), loc(P.A_col[maskA])
            lo, hi = np.minimum(ar, ac), np.maximum(ar, ac)            # sym-upper in LOCAL indices
            cnt = np.bincount(a_cons[maskA], minlength=m)
            cr, cc = loc(P.C_row[maskC]), loc(P.C_col[maskC])
            return Problem(n=(r1 - r0) + int(halo.shape[0]), m=m,
                           C_row=np.minimum(cr, cc).astype(np.int32), C_col=np.maximum(cr, cc).astype(np.int32),
                           C_val=scale * P.C_val[maskC],
                           A_ptr=np.concatenate([[0], np.cumsum(cnt)]).astype(np.int64),
                           A_row=lo.astype(np.int32), A_col=hi.astype(np.int32), A_val=scale * P.A_val[maskA],
                           b=np.asarray(P.b, float).copy())
        if P.pC:
            raise NotImplementedError("a low-rank cost term couples all rows: not sharded (DESIGN.md section 8)")
        shards.append(Shard(rank=p, world=world, r0=r0, r1=r1, halo=halo, P_fwd=sub(fa, fc, 1.0), P_adj=sub(ga, gc, 2.0),
                            send_rows=[None] * world, recv_slots=[None] * world))
    for p in range(world):                                  # exchange plan: who sends which own rows to whom
        for q in range(world):
            hq = shards[q].halo
            mine = hq[(hq >= shards[p].r0) & (hq < shards[p].r1)]
            shards[p].send_rows[q] = (mine - shards[p].r0).astype(np.int64)
            shards[q].recv_slots[p] = np.searchsorted(hq, mine).astype(np.int64)
    return shards


class ShardedEvaluator:
    """f, G = grad f (own rows) and z for one rank of a row-sharded problem.

    `backend` does the rank-local arithmetic (LibraryBackend: the CUDA library; the CPU test passes an oracle-based one)
    and `comm` the three collectives (TorchComm: torch.distributed; LocalComm for a single process that holds all
    shards).  Arrays are whatever the backend works on (torch tensors / numpy arrays)."""

    def __init__(self, shard: Shard, backend, comm, b: np.ndarray):
        self.s, self.be, self.comm, self.b = shard, backend, comm, b

    def eval(self, R_own, y, sigma: float):
        s, be = self.s, self.be
        R_loc = self.comm.halo_exchange(s, R_own, be)                      # (1) own rows + halo rows
        z_part, cx_part = be.forward(R_loc)                                # (2) share of A(RR^T) and of <C,RR^T>
        z = self.comm.allreduce_sum(z_part)                                # (3)
        lam, yq, qq = be.dual(z, self.b, y, sigma)                         # (4) replicated
        G_own, gg, gr = be.adjoint(lam, R_loc, s.n_own)                    # (5) own rows of 2 S(lambda) R
        cx, gg, gr = self.comm.allreduce_scalars([cx_part, gg, gr])        # (6)
        f = cx - yq + 0.5 * sigma * qq
        return dict(f=f, cx=cx, yq=yq, qq=qq, gg=gg, gr=gr, z=z, G_own=G_own)


class TorchComm:
    """Collectives over torch.distributed (nccl on GPUs, gloo in the CPU test)."""

    def __init__(self, xp="torch"):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist

    def halo_exchange(self, s: Shard, R_own, be):
        torch, dist = self.torch, self.dist
        R_own = be.as_tensor(R_own)
        r = R_own.shape[1]
        send = torch.cat([R_own[torch.as_tensor(s.send_rows[q], device=R_own.device)] for q in range(s.world)]) \
            if s.world > 1 else R_own[:0]
        recv = torch.empty((int(s.halo.shape[0]), r), dtype=R_own.dtype, device=R_own.device)
        tmp = torch.empty_like(recv)
        if s.world > 1:
            dist.all_to_all_single(tmp, send.contiguous(), output_split_sizes=[len(x) for x in s.recv_slots],
                                   input_split_sizes=[len(x) for x in s.send_rows])
            off = 0
            for q in range(s.world):                       # rows arrive grouped by sender; put them at their halo slots
                k = len(s.recv_slots[q])
                recv[torch.as_tensor(s.recv_slots[q], device=recv.device)] = tmp[off:off + k]
                off += k
        return torch.cat([R_own, recv]).contiguous()

    def allreduce_sum(self, v):
        if self.dist.is_initialized() and self.dist.get_world_size() > 1:
            t = v if isinstance(v, self.torch.Tensor) else self.torch.from_numpy(np.ascontiguousarray(v))
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
            return t if isinstance(v, self.torch.Tensor) else t.numpy()
        return v

    def allreduce_scalars(self, vals):
        t = self.torch.tensor([float(v) for v in vals], dtype=self.torch.float64)
        if self.dist.is_initialized() and self.dist.get_world_size() > 1:
            dev = "cuda" if self.dist.get_backend() == "nccl" else "cpu"
            t = t.to(dev)
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return [float(x) for x in t.cpu()]


class LocalComm:
    """All shards in one process (one GPU, or a CPU test without process groups): the collectives become copies and
    sums over the list of per-rank values handed in by the driver loop `eval_all`."""

    @staticmethod
    def eval_all(shards, backends, b, R, y, sigma):
        import numpy as np_
        to_np = lambda a: a.detach().cpu().numpy() if hasattr(a, "detach") else np_.asarray(a)
        R = to_np(R)
        R_locs = [np_.concatenate([R[s.r0:s.r1], R[s.halo]]) for s in shards]       # halo exchange = row copies
        parts = [be.forward(be.from_numpy(Rl)) for be, Rl in zip(backends, R_locs)]
        z = sum(to_np(p[0]) for p in parts)
        cx = sum(float(p[1]) for p in parts)
        out_G, gg, gr = [], 0.0, 0.0
        for be, Rl, s in zip(backends, R_locs, shards):
            lam, yq, qq = be.dual(be.from_numpy(z), b, y, sigma)
            G_own, g2, g1 = be.adjoint(lam, be.from_numpy(Rl), s.n_own)
            out_G.append(to_np(G_own)); gg += g2; gr += g1
        return dict(f=cx - yq + 0.5 * sigma * qq, cx=cx, yq=yq, qq=qq, gg=gg, gr=gr, z=z, G=np_.concatenate(out_G))


class LibraryBackend:
    """Rank-local arithmetic by the CUDA library: two contexts (P_fwd, P_adj) on this rank's device."""

    def __init__(self, shard: Shard, dtype, device: int = 0):
        import torch
        from . import binding
        self.torch, self.s = torch, shard
        self.tdt = torch.float32 if dtype in ("f32", binding.F32) else torch.float64
        self.dev = torch.device("cuda", device)
        self.fwd = binding.Context(shard.P_fwd, dtype, device=device)
        self.adj = binding.Context(shard.P_adj, dtype, device=device)
        self.zero_y = torch.zeros(shard.P_fwd.m, dtype=torch.float64, device=self.dev)

    def as_tensor(self, a):
        return self.torch.as_tensor(a, dtype=self.tdt, device=self.dev)

    from_numpy = as_tensor

    def forward(self, R_loc):
        R_loc = self.as_tensor(R_loc)
        r = R_loc.shape[1]
        z = self.torch.empty(self.s.P_fwd.m, dtype=self.torch.float64, device=self.dev)
        self.fwd.set_dual(self.zero_y, 1.0)
        st = self.fwd.eval(R_loc, r, r, None, z)            # value-only call: z and <C_p, RR^T> of this rank's entries
        return z, float(st[1])

    def dual(self, z, b, y, sigma):
        """lambda = y - sigma (z - b) and y.q, ||q||^2 from the all-reduced z (alora_dual_terms; P_fwd carries the true b)."""
        torch = self.torch
        z = torch.as_tensor(z, dtype=torch.float64, device=self.dev)
        self._y = torch.as_tensor(y, dtype=torch.float64, device=self.dev)
        lam = torch.empty_like(z)
        self.fwd.set_dual(self._y, sigma)
        t = self.fwd.dual_terms(z, lam)
        return lam, float(t[0]), float(t[1])

    def adjoint(self, lam, R_loc, n_own):
        R_loc = self.as_tensor(R_loc)
        r = R_loc.shape[1]
        W = self.torch.empty_like(R_loc)
        self.adj.smatvec(lam, R_loc, r, W, fetch=False)     # (2C - sum lambda_i 2A_i) R: rows [0, n_own) are grad f
        gg, gr = self.adj.rowdots(W, R_loc, n_own, r, r)
        return W[:n_own], float(gg), float(gr)

    def close(self):
        self.fwd.close(); self.adj.close()
