"""the block-cyclic multi-GPU Cholesky plan of paper_2602_19683_b200/multi_gpu.py,
checked on the CPU: coverage invariants, a numpy replay of the plans of all ranks against the oracle, and a
world_size-2 gloo run with real broadcasts.  The tile arithmetic of the replay is test-only numpy/scipy (the GPU
path runs the library's kernels; tests/test_gpu_multi.py)."""
import os
import sys

import numpy as np
import pytest
import scipy.linalg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

import oracle
from paper_2602_19683_b200 import nfir


def _mg():
    torch = pytest.importorskip("torch")
    from paper_2602_19683_b200 import multi_gpu
    return multi_gpu


@pytest.mark.parametrize("M", [1, 2, 4, 7, 32])
@pytest.mark.parametrize("world", [1, 2, 3, 4, 8])
def test_plan_invariants(M, world):
    mg = _mg()
    plans = [mg.plan(M, world, r) for r in range(world)]
    for r, ops in enumerate(plans):
        bcasts = [op for op in ops if op[0] == "bcast"]
        assert [b[1] for b in bcasts] == list(range(M))                     # same collective order on every rank
        assert all(b[2] == mg.column_owner(b[1], world) for b in bcasts)
        have, applied = set(), {}
        for op in ops:
            if op[0] == "update":
                _, K, k0, k1 = op
                assert mg.column_owner(K, world) == r and k0 < k1 <= K
                assert applied.get(K, 0) == k0                              # contiguous, in order, no gap and no repeat
                assert all(P in have for P in range(k0, k1)), "uses a panel that has not arrived and been sliced"
                applied[K] = k1
            elif op[0] == "panel":
                J = op[1]
                assert mg.column_owner(J, world) == r and applied.get(J, 0) == J   # fully updated before it is factored
            elif op[0] == "slice":
                have.add(op[1])
        panels = [op[1] for op in ops if op[0] == "panel"]
        assert panels == [K for K in range(M) if mg.column_owner(K, world) == r]
    # look-ahead: between the broadcasts of J-1 and J the owner of J applies at most ONE panel (depth one) before its panel step
    if world > 1 and M > world:
        for J in range(world, M):
            ops = plans[mg.column_owner(J, world)]
            i0 = ops.index(("bcast", J - 1, mg.column_owner(J - 1, world)))
            i1 = ops.index(("panel", J))
            ups = [op for op in ops[i0:i1] if op[0] == "update"]
            assert len(ups) == 1 and ups[0][1] == J and ups[0][3] - ups[0][2] == 1


class _NumpyRank:
    """Test-only stand-in for MixedCholeskyRank: the same plan executed with numpy/scipy tile arithmetic."""

    def __init__(self, K, tile, rank, world, mg):
        self.t, self.M = tile, K.shape[0] // tile
        self.T = {(I, J): K[I * tile:(I + 1) * tile, J * tile:(J + 1) * tile].copy() for I in range(self.M) for J in range(I + 1)}
        self.ops = mg.plan(self.M, world, rank)
        self.rank = rank

    def compute(self, op):
        if op[0] == "update":
            _, K, k0, k1 = op
            for I in range(K, self.M):
                for P in range(k0, k1):
                    self.T[(I, K)] -= self.T[(I, P)] @ self.T[(K, P)].T
        elif op[0] == "panel":
            J = op[1]
            self.T[(J, J)] = np.linalg.cholesky(np.tril(self.T[(J, J)]) + np.tril(self.T[(J, J)], -1).T)
            for I in range(J + 1, self.M):
                self.T[(I, J)] = scipy.linalg.solve_triangular(self.T[(J, J)], self.T[(I, J)].T, lower=True).T
        elif op[0] == "slice":
            pass

    def pack(self, J):
        return np.stack([self.T[(I, J)] for I in range(J, self.M)])

    def unpack(self, J, buf):
        for k, I in enumerate(range(J, self.M)):
            self.T[(I, J)] = buf[k].copy()

    def dense(self):
        n = self.M * self.t
        L = np.zeros((n, n))
        for (I, J), v in self.T.items():
            L[I * self.t:(I + 1) * self.t, J * self.t:(J + 1) * self.t] = v
        return np.tril(L)


def _problem(n=256, D=4):
    X, _ = nfir.nfir_features(77, n, D)
    K = oracle.assemble(X, X, oracle.Hyper(), True)
    return K, oracle.cholesky(K)


@pytest.mark.parametrize("world", [1, 2, 3, 4, 8])
def test_numpy_replay_of_all_ranks_matches_oracle(world):
    mg = _mg()
    K, Lo = _problem()
    ranks = [_NumpyRank(K, 32, r, world, mg) for r in range(world)]
    cur = [0] * world
    for J in range(ranks[0].M):
        for r, st in enumerate(ranks):
            while st.ops[cur[r]][0] != "bcast":
                st.compute(st.ops[cur[r]]); cur[r] += 1
        root = mg.column_owner(J, world)
        buf = ranks[root].pack(J)
        for r, st in enumerate(ranks):
            if r != root:
                st.unpack(J, buf)
            cur[r] += 1
    for r, st in enumerate(ranks):
        for op in st.ops[cur[r]:]:
            st.compute(op)
        assert np.linalg.norm(st.dense() - Lo) / np.linalg.norm(Lo) <= 1e-12, r     # every rank ends with the whole factor


def _gloo_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from paper_2602_19683_b200 import multi_gpu as mg
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    K, Lo = _problem()
    st = _NumpyRank(K, 32, rank, world, mg)
    for op in st.ops:
        if op[0] == "bcast":
            J, root = op[1], op[2]
            buf = torch.from_numpy(st.pack(J)) if root == rank else torch.empty(st.M - J, 32, 32, dtype=torch.float64)
            dist.broadcast(buf, src=root)
            if root != rank:
                st.unpack(J, buf.numpy())
        else:
            st.compute(op)
    err = float(np.linalg.norm(st.dense() - Lo) / np.linalg.norm(Lo))
    # the sharding of the prediction: every test point belongs to exactly one rank, whole tile rows
    rows = [mg.shard_rows(m, t, world, rank) for (m, t) in ((128, 32), (96, 32), (4096, 1024))]
    dist.barrier()
    dist.destroy_process_group()
    np.save(f"{out}.{rank}.npy", np.array([err] + [x for ab in rows for x in ab]))


def _gloo_worker_fused(rank, world, port, out, bufs):
    """The fused transport on the CPU: every rank's tile array lives in shared memory (standing in for NVLink peer memory),
    the owner of a panel writes the finished tiles into EVERY copy (what gp_mixed_panel_bcast does block by block), and the
    "broadcast" is a barrier."""
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from paper_2602_19683_b200 import multi_gpu as mg
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    K, Lo = _problem()
    st = _NumpyRank(K, 32, rank, world, mg)
    index = {}
    for I in range(st.M):
        for J in range(I + 1):
            index[(I, J)] = I * (I + 1) // 2 + J
    views = [b.numpy() for b in bufs]                        # [ntiles, 32, 32] per rank
    for key, k in index.items():                             # this rank's tiles move into its shared array
        views[rank][k] = st.T[key]
        st.T[key] = views[rank][k]
    dist.barrier()
    for op in st.ops:
        if op[0] == "bcast":
            dist.barrier()                                   # the owner's stores are complete: nothing to copy
        elif op[0] == "panel":
            st.compute(op)                                   # (results are assigned as new arrays ...)
            J = op[1]
            for I in range(J, st.M):
                k = index[(I, J)]
                for v in views:                              # ... and stored into every copy, the own one included
                    v[k] = st.T[(I, J)]
                st.T[(I, J)] = views[rank][k]
        else:
            st.compute(op)
    err = float(np.linalg.norm(st.dense() - Lo) / np.linalg.norm(Lo))
    dist.barrier()
    dist.destroy_process_group()
    np.save(f"{out}.{rank}.npy", np.array([err]))


def test_block_cyclic_plan_with_the_fused_transport_over_shared_memory(tmp_path):
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    out = str(tmp_path / "f")
    M = 256 // 32
    bufs = [torch.zeros(M * (M + 1) // 2, 32, 32, dtype=torch.float64).share_memory_() for _ in range(2)]
    mp.spawn(_gloo_worker_fused, args=(2, 29633, out, bufs), nprocs=2, join=True)
    r = [np.load(f"{out}.{k}.npy") for k in range(2)]
    assert r[0][0] <= 1e-12 and r[1][0] <= 1e-12


def test_block_cyclic_plan_with_gloo_broadcasts(tmp_path):
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    out = str(tmp_path / "r")
    mp.spawn(_gloo_worker, args=(2, 29631, out), nprocs=2, join=True)
    r = [np.load(f"{out}.{k}.npy") for k in range(2)]
    assert r[0][0] <= 1e-12 and r[1][0] <= 1e-12
    assert list(r[0][1:]) == [0, 64, 0, 64, 0, 2048] and list(r[1][1:]) == [64, 128, 64, 96, 2048, 4096]


@pytest.mark.parametrize("m,tile,world", [(128, 32, 2), (96, 32, 2), (4096, 1024, 8), (4096, 1024, 3), (1024, 256, 4)])
def test_shard_rows_partition_the_test_points(m, tile, world):
    mg = _mg()
    edges = [mg.shard_rows(m, tile, world, r) for r in range(world)]
    assert edges[0][0] == 0 and edges[-1][1] == m
    for (a0, a1), (b0, b1) in zip(edges, edges[1:]):
        assert a1 == b0 and a0 <= a1
    assert all(a0 % tile == 0 and a1 % tile == 0 for a0, a1 in edges)
