"""Multi-GPU drivers on top of the single-GPU C ABI: one process per GPU, torch.distributed (NCCL) for the exchanges.

SURVEY.md section 8(f) row 2 / PAPER.md:203 ("extend the library to distributed multi-GPU environments"):

  * ``plan`` / ``MixedCholeskyRank``: the tiled Cholesky with its tile COLUMNS distributed block-cyclically (1-D,
    column J belongs to rank J % P).  Per step J the owner brings column J up to date, runs its FP64 panel step
    (POTRF tile task + TRSM tile tasks) and broadcasts the finished panel; every rank applies received
    panels to the columns it owns with the emulated contraction of gp_mixed_update_column (SYRK / GEMM tile tasks,
    PAPER.md:89, 136).  Look-ahead: before a rank blocks on the broadcast of panel J it applies everything it has
    received so far to the column it factors next, so per owned column there is one long contraction (efficient) and
    P - 1 short ones, and only a depth-one update plus the panel step sit between two consecutive broadcasts.
    Storage is replicated (every rank ends with the whole factor, which the prediction needs anyway: SURVEY.md 8(e));
    the trailing-update WORK is what is divided.  Two transports for the panel: an NCCL broadcast of the packed tiles
    after the panel step, or -- ``peers`` set -- the FUSED one: gp_mixed_panel_bcast stores every finished block straight
    into the other ranks' copies of the tile array over NVLink peer memory while the panel step runs, and the
    "broadcast" that follows is only a barrier (``exchange_peer_pointers`` sets the mapping up with CUDA IPC).
  * ``ShardedPredictor``: the prediction sharded by test-point tile rows: each rank
    solves V for its own test points, V^T is all-gathered once, each rank forms its block rows of Sigma.

The plan is plain data and is checked on the CPU (tests/test_multi_gpu_plan.py: coverage invariants, a numpy
replay against the oracle, a world_size-2 gloo run); the GPU path is verified on ONE GPU by running P rank states in
lock-step with device-to-device copies in place of the broadcasts (tests/test_gpu_multi.py).  UNMEASURED ON
MULTI-GPU HARDWARE: only one GPU was reachable while this was written.
"""
from __future__ import annotations

from dataclasses import dataclass

import torch

from . import binding as gp


def column_owner(J: int, world: int) -> int:
    """1-D block-cyclic ownership of tile columns."""
    return J % world


def plan(M: int, world: int, rank: int):
    """The ordered operations of `rank` for an M x M-tile factorisation on `world` ranks:
         ("update", K, k0, k1)  apply the panels [k0, k1) to the owned tile column K     (gp_mixed_update_column)
         ("panel", J)           FP64 panel step of the owned column J                    (gp_mixed_panel)
         ("bcast", J, root)     panel J (tiles (I, J), I >= J) travels from root to everyone
         ("slice", J)           digit planes of panel J                                  (gp_mixed_slice_column)
    Every rank issues the broadcasts in the same order J = 0 .. M-1."""
    owned = [K for K in range(M) if column_owner(K, world) == rank]
    applied = {K: 0 for K in owned}
    ops = []
    for J in range(M):
        root = column_owner(J, world)
        nxt = next((K for K in owned if K >= J), None)          # the column this rank factors next
        if nxt is not None and applied[nxt] < J:
            ops.append(("update", nxt, applied[nxt], J))         # catch up with everything received so far
            applied[nxt] = J
        if root == rank:
            ops.append(("panel", J))
        ops.append(("bcast", J, root))
        if J + 1 < M:
            ops.append(("slice", J))
    return ops


def panel_tile_indices(M: int, J: int):
    """Indices of the tiles (I, J), I = J .. M-1, in lower-packed storage."""
    return [I * (I + 1) // 2 + J for I in range(J, M)]


@dataclass
class MixedCholeskyRank:
    """One rank's state and the execution of its plan on its GPU.  `KL` holds the lower-packed tiles of K (all of
    them: storage is replicated) and ends as the complete factor."""
    n: int
    tile: int
    KL: torch.Tensor
    info: torch.Tensor
    rank: int
    world: int
    sched_width: int = 0
    peers: tuple = ()          # device addresses of the other ranks' KL as seen from this GPU: the fused panel broadcast

    def __post_init__(self):
        self.M = self.n // self.tile
        self.work = torch.empty(gp.gp_mixed_workspace_bytes(self.n, self.tile), dtype=torch.uint8, device=self.KL.device)
        self.tiles = self.KL.view(self.M * (self.M + 1) // 2, self.tile * self.tile)
        self.ops = plan(self.M, self.world, self.rank)
        self.reset()

    def reset(self) -> None:
        """Start a factorisation of the K that is now in `KL` (zero the counters, find the fixed-point scale)."""
        gp.gp_mixed_begin(self.KL, self.n, self.tile, self.info, self.work)

    def pack_panel(self, J: int) -> torch.Tensor:
        idx = torch.tensor(panel_tile_indices(self.M, J), device=self.KL.device)
        return self.tiles.index_select(0, idx)

    def unpack_panel(self, J: int, buf: torch.Tensor) -> None:
        idx = torch.tensor(panel_tile_indices(self.M, J), device=self.KL.device)
        self.tiles.index_copy_(0, idx, buf)

    def compute(self, op) -> None:
        kind = op[0]
        if kind == "update":
            gp.gp_mixed_update_column(self.KL, self.n, self.tile, op[1], op[2], op[3], self.work)
        elif kind == "panel":
            if self.peers:
                gp.gp_mixed_panel_bcast(self.KL, self.n, self.tile, op[1], self.sched_width, self.info, self.work, self.peers)
            else:
                gp.gp_mixed_panel(self.KL, self.n, self.tile, op[1], self.sched_width, self.info, self.work)
        elif kind == "slice":
            gp.gp_mixed_slice_column(self.KL, self.n, self.tile, op[1], self.work)
        else:
            raise ValueError(op)

    def run(self, group=None) -> None:
        """Execute the plan (one process per GPU): NCCL broadcasts of the packed panels, or, with `peers` set, the fused
        transport: the owner's panel step has already written the panel into every copy, the broadcast is a barrier."""
        import torch.distributed as dist
        for op in self.ops:
            if op[0] == "bcast" and self.peers:
                if op[2] == self.rank:
                    torch.cuda.current_stream().synchronize()        # the peer stores are complete when the panel step is
                dist.barrier(group=group)
            elif op[0] == "bcast":
                J, root = op[1], op[2]
                buf = self.pack_panel(J) if root == self.rank else torch.empty(self.M - J, self.tile * self.tile, dtype=torch.float64,
                                                                               device=self.KL.device)
                dist.broadcast(buf, src=root, group=group)
                if root != self.rank:
                    self.unpack_panel(J, buf)
            else:
                self.compute(op)


def run_lockstep(states) -> None:
    """ONE-GPU emulation of a `world`-rank run: the rank states (disjoint buffers) execute their plans step by step,
    a broadcast becomes a device-to-device copy from the root's buffer.  No kernel waits on another: every launch
    finds its inputs complete because the states advance together from one broadcast to the next."""
    cursors = [0] * len(states)
    M = states[0].M
    for J in range(M):
        for r, st in enumerate(states):
            while st.ops[cursors[r]][0] != "bcast":
                st.compute(st.ops[cursors[r]])
                cursors[r] += 1
            assert st.ops[cursors[r]][1] == J
        root = states[0].ops[cursors[0]][2]
        if states[root].peers:
            torch.cuda.current_stream().synchronize()     # fused transport: the panel step wrote every copy; this is the barrier
        else:
            buf = states[root].pack_panel(J)
            for r, st in enumerate(states):
                if r != root:
                    st.unpack_panel(J, buf.clone())
        for r in range(len(states)):
            cursors[r] += 1
    for r, st in enumerate(states):
        while cursors[r] < len(st.ops):
            st.compute(st.ops[cursors[r]])
            cursors[r] += 1


def exchange_peer_pointers(KL: torch.Tensor, group=None):
    """Addresses of the other ranks' `KL` as seen from this rank's GPU, in rank order without this rank: the `peers` of a
    MixedCholeskyRank.  Every rank shares its tensor through CUDA IPC (torch.multiprocessing's reduction of a CUDA tensor:
    cudaIpcGetMemHandle of its allocation + offset), the handles travel with all_gather_object, each rank opens the
    others' (cudaIpcOpenMemHandle) and enables peer access to their devices.  Returns (addresses, keepalive): keep
    `keepalive` referenced while the addresses are in use.  All GPUs of the node must be visible to every process.
    Verified between two processes on ONE GPU (tests/test_gpu_multi.py); across two physical GPUs (peer access over
    NVLink) it is UNVERIFIED: no such box was reachable."""
    import ctypes
    import torch.distributed as dist
    from torch.multiprocessing.reductions import reduce_tensor
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    rebuild, args = reduce_tensor(KL)
    gathered = [None] * world
    dist.all_gather_object(gathered, (rebuild, args), group=group)
    cudart = ctypes.CDLL("libcudart.so")
    views, addrs = [], []
    for r, (fn, a) in enumerate(gathered):
        if r == rank:
            continue
        t = fn(*a)                                   # a tensor on the owner's device, backed by the IPC mapping
        if t.device != KL.device:
            rc = cudart.cudaDeviceEnablePeerAccess(ctypes.c_int(t.device.index), ctypes.c_uint(0))
            if rc not in (0, 704):                   # cudaSuccess, cudaErrorPeerAccessAlreadyEnabled
                raise RuntimeError(f"cudaDeviceEnablePeerAccess({t.device.index}) failed: {rc}")
        views.append(t)
        addrs.append(int(t.data_ptr()))
    return tuple(addrs), views


# ------------------------------------------------------------------------------------------------
def shard_rows(m: int, tile: int, world: int, rank: int):
    """Contiguous range [a0, a1) of test points of `rank`: whole tile rows, the first (m / tile) % world ranks get one more."""
    Mm = m // tile
    base, extra = divmod(Mm, world)
    t0 = rank * base + min(rank, extra)
    t1 = t0 + base + (1 if rank < extra else 0)
    return t0 * tile, t1 * tile


class ShardedPredictor:
    """Prediction given L (replicated), sharded by test-point tile rows:
        rank r:  mean_r = K_{X^_r, X} alpha;   V_r^T = K_{X^_r, X} L^-T   (its own rows, no communication)
        all-gather of V^T (m x n, GP_GENERAL tiles: a rank's rows are a contiguous run of tile rows)
        rank r:  Sigma[rows_r, :] = K_{X^_r, X^} - V_r^T (V^T)^T           (full block rows: no symmetry across ranks)
    `gather` stands in for the collective: torch.distributed.all_gather_into_tensor in a real run, a concatenation in
    the one-GPU emulation."""

    def __init__(self, n: int, m: int, D: int, tile: int, h: gp.Hyper, rank: int, world: int, sched_width: int = 0, device="cuda"):
        self.n, self.m, self.D, self.tile, self.h, self.rank, self.world, self.width = n, m, D, tile, h, rank, world, sched_width
        self.a0, self.a1 = shard_rows(m, tile, world, rank)
        self.mr = self.a1 - self.a0
        dev = torch.device(device)
        self.Vt_all = torch.empty(m * n, dtype=torch.float64, device=dev)            # (m/t) x (n/t) tiles, tile-row major
        self.mean = torch.empty(max(self.mr, 1), dtype=torch.float64, device=dev)
        self.Sigma_rows = torch.empty(max(self.mr, 1), m, dtype=torch.float64, device=dev)
        _, _, fb = gp.gp_workspace_bytes(n, max(self.mr, tile), D, tile)
        self.work = torch.empty(fb, dtype=torch.uint8, device=dev)

    def local_rows(self) -> torch.Tensor:
        """This rank's slice of the V^T tile array (contiguous)."""
        return self.Vt_all[self.a0 * self.n:self.a1 * self.n]

    def solve_local(self, L: torch.Tensor, X: torch.Tensor, Xs: torch.Tensor, alpha: torch.Tensor) -> None:
        if self.mr == 0:
            return
        Xr = Xs[self.a0:self.a1].contiguous()
        gp.gp_predict_mean(X, alpha, Xr, self.h, self.mean)
        gp.gp_predict_vt(L, X, Xr, self.h, self.tile, self.width, self.local_rows(), self.work)

    def all_gather(self, group=None) -> None:
        import torch.distributed as dist
        sizes = [(shard_rows(self.m, self.tile, self.world, r)[1] - shard_rows(self.m, self.tile, self.world, r)[0]) * self.n
                 for r in range(self.world)]
        if len(set(sizes)) == 1:
            dist.all_gather_into_tensor(self.Vt_all, self.local_rows().clone(), group=group)
        else:                                       # ragged split: one broadcast per rank
            off = 0
            for r, sz in enumerate(sizes):
                if sz:
                    dist.broadcast(self.Vt_all[off:off + sz], src=r, group=group)
                off += sz

    def covariance_rows(self, Xs: torch.Tensor) -> torch.Tensor:
        if self.mr == 0:
            return self.Sigma_rows[:0]
        gp.gp_predict_cov_rows(self.Vt_all, Xs, self.n, self.a0, self.mr, self.h, self.tile, self.width, self.Sigma_rows, self.work)
        return self.Sigma_rows
