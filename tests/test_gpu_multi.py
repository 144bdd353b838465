"""SURVEY.md 8(f) row 2 and 8(e) on ONE GPU: the multi-GPU drivers of paper_2602_19683_b200/multi_gpu.py run with P rank
states in lock-step (disjoint buffers, device-to-device copies in place of the NCCL broadcasts / all-gather; no kernel waits
on another) and are compared with the oracle.  The collectives themselves are covered on the CPU with gloo
(tests/test_multi_gpu_plan.py).  Unmeasured on multi-GPU hardware."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle
from helpers import relerr
from paper_2602_19683_b200 import nfir


@pytest.fixture(scope="module")
def gp():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    from paper_2602_19683_b200 import binding
    binding.load()
    return binding


def _dense_L(gp, KL, n, tile):
    out = torch.empty(n, n, dtype=torch.float64, device="cuda")
    return gp.gp_tiles_to_dense(KL, n, n, tile, True, out).cpu().numpy()


@pytest.mark.parametrize("n,tile,world", [(1024, 128, 2), (1024, 128, 3), (1536, 256, 4), (2048, 256, 8)])
def test_block_cyclic_mixed_cholesky_in_lockstep_matches_oracle(gp, n, tile, world):
    from paper_2602_19683_b200 import multi_gpu as mg
    D = 8
    X, y = nfir.nfir_features(5 + world, n, D)
    K = oracle.assemble(X, X, oracle.Hyper(), True)
    Lo = oracle.cholesky(K)
    ntiles = (n // tile) * (n // tile + 1) // 2
    K0 = torch.empty(ntiles * tile * tile, dtype=torch.float64, device="cuda")
    dX = torch.from_numpy(X).cuda()
    gp.gp_assemble_tiles(dX, dX, gp.Hyper(), tile, gp.GP_SYM_LOWER, K0)
    states = [mg.MixedCholeskyRank(n, tile, K0.clone(), torch.zeros(1, dtype=torch.int32, device="cuda"), r, world) for r in range(world)]
    mg.run_lockstep(states)
    torch.cuda.synchronize()
    for r, st in enumerate(states):
        # a rank reports the pivots of the panels IT factored; received panels arrive factored
        assert int(st.info.item()) == 0
        L = _dense_L(gp, st.KL, n, tile)
        assert relerr(L, Lo) <= 1e-10, r                      # every rank ends with the whole factor
        np.testing.assert_allclose(L, Lo, rtol=0, atol=1e-9 * np.abs(Lo).max())
    assert torch.equal(states[0].KL, states[-1].KL) or relerr(_dense_L(gp, states[0].KL, n, tile), _dense_L(gp, states[-1].KL, n, tile)) == 0.0


@pytest.mark.parametrize("n,tile,world", [(1024, 128, 2), (1536, 256, 3), (2048, 256, 8)])
def test_block_cyclic_with_the_fused_panel_broadcast_matches_oracle_and_the_copy_transport(gp, n, tile, world):
    """gp_mixed_panel_bcast: the owner's panel step stores every finished block into the other ranks' copies of the tile
    array (here: other buffers of the same GPU standing in for NVLink peer memory), the broadcast is only a barrier.  Every
    rank must end with the oracle's factor, bit-identical in its lower part to what the copy transport gives."""
    from paper_2602_19683_b200 import multi_gpu as mg
    D = 8
    X, y = nfir.nfir_features(5 + world, n, D)
    K = oracle.assemble(X, X, oracle.Hyper(), True)
    Lo = oracle.cholesky(K)
    ntiles = (n // tile) * (n // tile + 1) // 2
    K0 = torch.empty(ntiles * tile * tile, dtype=torch.float64, device="cuda")
    dX = torch.from_numpy(X).cuda()
    gp.gp_assemble_tiles(dX, dX, gp.Hyper(), tile, gp.GP_SYM_LOWER, K0)
    bufs = [K0.clone() for _ in range(world)]
    states = [mg.MixedCholeskyRank(n, tile, bufs[r], torch.zeros(1, dtype=torch.int32, device="cuda"), r, world,
                                   peers=tuple(int(bufs[q].data_ptr()) for q in range(world) if q != r)) for r in range(world)]
    mg.run_lockstep(states)
    torch.cuda.synchronize()
    ref = [mg.MixedCholeskyRank(n, tile, K0.clone(), torch.zeros(1, dtype=torch.int32, device="cuda"), r, world) for r in range(world)]
    mg.run_lockstep(ref)
    torch.cuda.synchronize()
    L_ref = _dense_L(gp, ref[0].KL, n, tile)
    for r, st in enumerate(states):
        assert int(st.info.item()) == 0
        L = _dense_L(gp, st.KL, n, tile)
        assert relerr(L, Lo) <= 1e-10, r
        assert np.array_equal(L, L_ref), r
    with pytest.raises(gp.GpError):                            # a peer must be another buffer
        gp.gp_mixed_panel_bcast(bufs[0], n, tile, 0, 0, states[0].info, states[0].work, [int(bufs[0].data_ptr())])
    with pytest.raises(gp.GpError):
        gp.gp_mixed_panel_bcast(bufs[0], n, tile, 0, 0, states[0].info, states[0].work, [int(b.data_ptr()) for b in bufs] * 2)


@pytest.mark.parametrize("n,m,D,tile,world", [(1024, 512, 8, 128, 2), (1024, 384, 8, 128, 2), (768, 768, 5, 256, 3), (16384 // 8, 1024, 8, 256, 4)])
def test_sharded_prediction_in_lockstep_matches_oracle(gp, n, m, D, tile, world):
    from paper_2602_19683_b200 import multi_gpu as mg
    X, y = nfir.nfir_features(21, n, D)
    Xs, _ = nfir.nfir_features(22, m, D, with_targets=False)
    h = oracle.Hyper()
    p = oracle.predict(X, y, Xs, h)
    hg = gp.Hyper()
    pipe = gp.GpPipeline(n, 0, D, tile, hg)
    dX, dy, dXs = torch.from_numpy(X).cuda(), torch.from_numpy(y).cuda(), torch.from_numpy(Xs).cuda()
    pipe.assemble(dX); pipe.cholesky(); pipe.solve(dy)
    ranks = [mg.ShardedPredictor(n, m, D, tile, hg, r, world) for r in range(world)]
    for sp in ranks:
        sp.solve_local(pipe.KL, dX, dXs, pipe.alpha)
    for sp in ranks:                                          # the all-gather: every rank receives every rank's rows
        for src in ranks:
            sp.Vt_all[src.a0 * n:src.a1 * n].copy_(src.local_rows())
    mean = np.concatenate([sp.mean[:sp.mr].cpu().numpy() for sp in ranks])
    Sigma = np.concatenate([sp.covariance_rows(dXs)[:sp.mr].cpu().numpy() for sp in ranks], axis=0)
    torch.cuda.synchronize()
    assert relerr(mean, p.mean) <= 1e-9
    assert Sigma.shape == (m, m) and relerr(Sigma, p.Sigma) <= 1e-9
    np.testing.assert_allclose(Sigma, p.Sigma, rtol=0, atol=1e-9 * np.abs(p.Sigma).max())
    np.testing.assert_allclose(Sigma, Sigma.T, rtol=0, atol=1e-14)        # block rows come from different ranks: symmetric to rounding
    # V itself against the oracle (the gathered buffer, unpacked from GP_GENERAL tiles)
    Vt = torch.empty(m, n, dtype=torch.float64, device="cuda")
    gp.gp_tiles_to_dense(ranks[0].Vt_all, m, n, tile, False, Vt)
    assert relerr(Vt.cpu().numpy().T, p.V) <= 1e-9


def _ipc_worker(rank, world, port, out):
    import os
    import sys
    import torch.distributed as dist
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for q in (root, os.path.join(root, "tests")):
        if q not in sys.path:
            sys.path.insert(0, q)
    from paper_2602_19683_b200 import binding as gpb, multi_gpu as mg
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    gpb.load()
    n, tile, D = 1024, 128, 8
    X, _ = nfir.nfir_features(7, n, D)
    Lo = oracle.cholesky(oracle.assemble(X, X, oracle.Hyper(), True))
    ntiles = (n // tile) * (n // tile + 1) // 2
    KL = torch.empty(ntiles * tile * tile, dtype=torch.float64, device="cuda")
    dX = torch.from_numpy(X).cuda()
    gpb.gp_assemble_tiles(dX, dX, gpb.Hyper(), tile, gpb.GP_SYM_LOWER, KL)
    torch.cuda.synchronize()
    peers, keep = mg.exchange_peer_pointers(KL)              # CUDA IPC: the other process's tile array mapped into this one
    info = torch.zeros(1, dtype=torch.int32, device="cuda")
    st = mg.MixedCholeskyRank(n, tile, KL, info, rank, world, 0, peers)
    torch.cuda.synchronize()
    dist.barrier()
    st.run()                                                 # fused transport: panels are stored into the peer, then a barrier
    torch.cuda.synchronize()
    dist.barrier()
    dense = torch.empty(n, n, dtype=torch.float64, device="cuda")
    L = gpb.gp_tiles_to_dense(KL, n, n, tile, True, dense).cpu().numpy()
    np.save(f"{out}.{rank}.npy", np.array([relerr(L, Lo), float(info.item())]))
    dist.barrier()
    del keep
    dist.destroy_process_group()


@pytest.mark.timeout(600)
def test_fused_panel_broadcast_across_two_processes_over_cuda_ipc(gp, tmp_path):
    """The one piece of the fused transport the lock-step emulation does not reach: multi_gpu.exchange_peer_pointers (CUDA
    IPC handles through all_gather_object, cudaIpcOpenMemHandle) and MixedCholeskyRank.run() with barriers.  Two PROCESSES
    share this one GPU (host-side gloo barriers only: no kernel waits on another); each must end with the oracle's factor,
    half of whose panels arrived as stores from the other process.  Stands in for two GPUs over NVLink, which this box
    does not have."""
    import torch.multiprocessing as mp
    out = str(tmp_path / "ipc")
    try:
        mp.spawn(_ipc_worker, args=(2, 29657, out), nprocs=2, join=True)
    except Exception as e:                                   # a sandbox that forbids CUDA IPC between processes
        if "ipc" in str(e).lower():
            pytest.skip(f"CUDA IPC between processes is not available here: {str(e)[-200:]}")
        raise
    for r in range(2):
        err, info = np.load(f"{out}.{r}.npy")
        assert info == 0 and err <= 1e-10, (r, err, info)
