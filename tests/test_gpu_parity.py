"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Tolerances are north_star's: relative Frobenius error <= 1e-10 on L,
<= 1e-9 on mean and Sigma (additionally alpha <= 1e-9, K <= 1e-14; reading A11)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle
from helpers import relerr
from paper_2602_19683_b200 import nfir

TOL_K, TOL_L, TOL_ALPHA, TOL_MEAN, TOL_SIGMA = 1e-14, 1e-10, 1e-9, 1e-9, 1e-9


@pytest.fixture(scope="module")
def gp():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    from paper_2602_19683_b200 import binding
    binding.load()
    return binding


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.fixture(autouse=True)
def _auto_tuning(gp):
    """Every test starts and ends with the library's own choice of block edge and scheduling granularity."""
    gp.gp_set_block_edge(0)
    gp.gp_set_schedule_granularity(0)
    yield
    gp.gp_set_block_edge(0)
    gp.gp_set_schedule_granularity(0)


def _run_pipeline(gp, X, y, Xs, h, tile, width=0):
    n, D = X.shape
    m = Xs.shape[0]
    pipe = gp.GpPipeline(n, m, D, tile, gp.Hyper(h.lengthscale, h.vertical, h.noise, h.ell_squared), sched_width=width)
    dX, dy, dXs = _dev(X), _dev(y), _dev(Xs)
    pipe.assemble(dX)
    K = pipe.dense_L().cpu().numpy()           # lower triangle of K (strict upper zeroed)
    res = pipe.run(dX, dy, dXs)
    torch.cuda.synchronize()
    L = pipe.dense_L().cpu().numpy()
    return dict(K=K, L=L, alpha=res.alpha.cpu().numpy(), beta=res.beta.cpu().numpy(), mean=res.mean.cpu().numpy(),
                Sigma=res.Sigma.cpu().numpy(), info=int(res.info.item()))


def _check_against_oracle(out, p):
    assert out["info"] == 0
    assert relerr(out["K"], np.tril(p.K)) <= TOL_K
    assert relerr(out["L"], p.L) <= TOL_L
    assert relerr(out["beta"], p.beta) <= TOL_ALPHA
    assert relerr(out["alpha"], p.alpha) <= TOL_ALPHA
    assert relerr(out["mean"], p.mean) <= TOL_MEAN
    assert relerr(out["Sigma"], p.Sigma) <= TOL_SIGMA
    assert np.array_equal(out["Sigma"], out["Sigma"].T)          # exactly symmetric (reading A12)
    # element-wise, so that a misplaced block cannot hide in a norm
    np.testing.assert_allclose(out["L"], p.L, rtol=0, atol=1e-9 * np.abs(p.L).max())
    np.testing.assert_allclose(out["Sigma"], p.Sigma, rtol=0, atol=1e-9 * np.abs(p.Sigma).max())


@pytest.mark.parametrize("ci", [0, 1])
def test_configs_full_pipeline(gp, ci):
    cfg = nfir.CONFIGS[ci]
    X, y, Xs = nfir.make_inputs(cfg)
    h = oracle.Hyper(cfg.lengthscale, cfg.vertical, cfg.noise)
    p = oracle.predict(X, y, Xs, h)
    out = _run_pipeline(gp, X, y, Xs, h, cfg.tile)
    _check_against_oracle(out, p)


@pytest.mark.parametrize("n,m,D,tile", [
    (96, 32, 3, 32),        # block 32, 3x3 tiles, odd D
    (192, 64, 5, 64),       # block 64
    (384, 128, 8, 128),     # block 128, one block per tile
    (768, 256, 8, 256),     # block 128, 2x2 blocks per tile, 3x3 tiles
    (1536, 384, 8, 384),    # 3x3 blocks per tile, 4 tiles
    (640, 128, 16, 128),    # 5 tiles of one block, D=16
    (1024, 512, 8, 512),    # 4 blocks per tile edge
    (320, 320, 8, 160),     # tile 160 -> block 32, 5 blocks per tile edge
])
def test_shapes_spanning_tiles_and_blocks(gp, n, m, D, tile):
    """Each shape with the library's own block edge (64 or 32 at these sizes) and with the 128-block path the
    large configurations use forced on (where the tile admits it)."""
    X, y = nfir.nfir_features(n + m + D, n, D)
    Xs, _ = nfir.nfir_features(7 * n + 1, m, D, with_targets=False)
    h = oracle.Hyper()
    p = oracle.predict(X, y, Xs, h)
    for cap in (0, 128):
        gp.gp_set_block_edge(cap)
        out = _run_pipeline(gp, X, y, Xs, h, tile)
        _check_against_oracle(out, p)


@pytest.mark.parametrize("cap,g", [(128, 1), (128, 2), (128, 4), (64, 1), (64, 2), (64, 8), (32, 4), (32, 16)])
def test_block_edge_and_scheduling_granularity_do_not_change_results(gp, cap, g):
    """The block edge and the scheduling tile (g x g blocks, independent of the storage tile) only change the order
    of work: every combination matches the oracle on a 2 x 2-tile problem whose tiles hold 4 / 8 / 16 blocks per edge."""
    n, m, D, tile = 1024, 512, 8, 512
    X, y = nfir.nfir_features(91, n, D)
    Xs, _ = nfir.nfir_features(92, m, D, with_targets=False)
    h = oracle.Hyper()
    p = oracle.predict(X, y, Xs, h)
    gp.gp_set_block_edge(cap)
    gp.gp_set_schedule_granularity(g)
    assert gp.gp_block_size_for(n, tile) == cap and gp.gp_schedule_granularity(n, m, tile) == g
    out = _run_pipeline(gp, X, y, Xs, h, tile)
    _check_against_oracle(out, p)


def test_config4_hyperparameters_and_ell_switch(gp):
    X, y = nfir.nfir_features(5, 512, 16)
    Xs, _ = nfir.nfir_features(6, 256, 16, with_targets=False)
    for h in (oracle.Hyper(2.0, 1.0, 0.05, False), oracle.Hyper(2.0, 1.0, 0.05, True)):
        p = oracle.predict(X, y, Xs, h)
        out = _run_pipeline(gp, X, y, Xs, h, 256)
        _check_against_oracle(out, p)


def test_worked_examples_on_gpu_padded(gp, golden):
    """The 40-digit examples cannot be tiled (n=2,3); embed them far away from 30/29 filler points so the
    leading block of L and the predictions of the real test points are unchanged."""
    g = golden["B"]
    X3, y3, Xs2 = np.array(g["X"]), np.array(g["y"]), np.array(g["Xs"])
    n, m = 32, 32
    X = np.zeros((n, 2)); y = np.zeros(n); Xs = np.zeros((m, 2))
    X[:3], y[:3], Xs[:2] = X3, y3, Xs2
    X[3:, 0] = 1000.0 + 100.0 * np.arange(n - 3)      # kernel underflows to exactly 0 against everything
    Xs[2:, 1] = -1000.0 - 100.0 * np.arange(m - 2)
    out = _run_pipeline(gp, X, y, Xs, oracle.Hyper(), 32)
    Lg = np.array([[float(t) for t in r] for r in g["L"]])
    np.testing.assert_allclose(out["L"][:3, :3], Lg, rtol=1e-13, atol=1e-15)
    np.testing.assert_allclose(out["alpha"][:3], [float(t) for t in g["alpha"]], rtol=1e-12)
    np.testing.assert_allclose(out["mean"][:2], [float(t) for t in g["mean"]], rtol=1e-12)
    Sg = np.array([[float(t) for t in r] for r in g["Sigma"]])
    np.testing.assert_allclose(out["Sigma"][:2, :2], Sg, rtol=1e-12)


def test_tile_size_independence(gp):
    cfg = nfir.CONFIGS[1]
    X, y, Xs = nfir.make_inputs(cfg)
    h = oracle.Hyper()
    ref = _run_pipeline(gp, X, y, Xs, h, 1024)     # one tile = untiled
    for tile in (32, 128, 256, 512):
        out = _run_pipeline(gp, X, y, Xs, h, tile)
        assert relerr(out["L"], ref["L"]) <= 1e-11
        assert relerr(out["mean"], ref["mean"]) <= 1e-11
        assert relerr(out["Sigma"], ref["Sigma"]) <= 1e-11


@pytest.mark.parametrize("width", [1, 2, 7, 148])
def test_scheduler_width_does_not_change_results(gp, width):
    X, y = nfir.nfir_features(3, 768, 8)
    Xs, _ = nfir.nfir_features(4, 256, 8, with_targets=False)
    h = oracle.Hyper()
    a = _run_pipeline(gp, X, y, Xs, h, 256, width=0)
    b = _run_pipeline(gp, X, y, Xs, h, 256, width=width)
    for k in ("L", "alpha", "mean", "Sigma"):
        assert np.array_equal(a[k], b[k]), k          # same item order per block -> bitwise identical


def test_not_positive_definite_reports_column_and_terminates(gp):
    n, tile = 256, 128
    K = np.eye(n)
    K[200, 200] = -1.0
    tiles = []
    M = n // tile
    for I in range(M):
        for J in range(I + 1):
            tiles.append(K[I * tile:(I + 1) * tile, J * tile:(J + 1) * tile].ravel())
    KL = _dev(np.concatenate(tiles))
    cb, _, _ = gp.gp_workspace_bytes(n, 0, 1, tile)
    work = torch.empty(cb, dtype=torch.uint8, device="cuda")
    info = torch.zeros(1, dtype=torch.int32, device="cuda")
    gp.gp_cholesky_tiled(KL, n, tile, 0, info, work)
    torch.cuda.synchronize()
    assert int(info.item()) == 201


def test_argument_errors(gp):
    X = torch.zeros(64, 4, dtype=torch.float64, device="cuda")
    out = torch.zeros(64 * 64, dtype=torch.float64, device="cuda")
    h = gp.Hyper()
    with pytest.raises(gp.GpError) as e:
        gp.gp_assemble_tiles(X, X, h, 48, gp.GP_SYM_LOWER, out)
    assert e.value.code == gp.ERR["TILE"]
    with pytest.raises(gp.GpError) as e:
        gp.gp_assemble_tiles(X, X, gp.Hyper(lengthscale=-1.0), 32, gp.GP_SYM_LOWER, out)
    assert e.value.code == gp.ERR["HYPER"]
    with pytest.raises(gp.GpError) as e:
        gp.gp_assemble_tiles(X, X, h, 32, 5, out)
    assert e.value.code == gp.ERR["MODE"]
    info = torch.zeros(1, dtype=torch.int32, device="cuda")
    small = torch.zeros(16, dtype=torch.uint8, device="cuda")
    with pytest.raises(gp.GpError) as e:
        gp.gp_cholesky_tiled(out, 64, 32, 0, info, small)
    assert e.value.code == gp.ERR["WORKSPACE"]
    with pytest.raises(gp.GpError) as e:
        gp.gp_cholesky_tiled(out, 70, 32, 0, info, small)
    assert e.value.code == gp.ERR["TILE"]


def test_host_buffer_pipeline_matches_oracle(gp):
    """gp_pipeline_host (the end-to-end call bench.py's e2e leg times): host in, host out."""
    cfg = nfir.CONFIGS[1]
    X, y, Xs = nfir.make_inputs(cfg)
    h = oracle.Hyper(cfg.lengthscale, cfg.vertical, cfg.noise)
    p = oracle.predict(X, y, Xs, h)
    hX, hY, hXs = (torch.from_numpy(a).pin_memory() for a in (X, y, Xs))
    hMean = torch.empty(cfg.m, dtype=torch.float64).pin_memory()
    hSigma = torch.empty(cfg.m, cfg.m, dtype=torch.float64).pin_memory()
    hAlpha = torch.empty(cfg.n, dtype=torch.float64)            # pageable also works
    ws = torch.empty(gp.gp_pipeline_workspace_bytes(cfg.n, cfg.m, cfg.D, cfg.tile), dtype=torch.uint8, device="cuda")
    info = gp.gp_pipeline_host(hX, hY, hXs, gp.Hyper(h.lengthscale, h.vertical, h.noise), cfg.tile, 0, hMean, hSigma, hAlpha, ws)
    assert info == 0
    assert relerr(hAlpha.numpy(), p.alpha) <= TOL_ALPHA
    assert relerr(hMean.numpy(), p.mean) <= TOL_MEAN
    assert relerr(hSigma.numpy(), p.Sigma) <= TOL_SIGMA
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(gp.GpError) as e:
        gp.gp_pipeline_host(hX, hY, hXs, gp.Hyper(), cfg.tile, 0, hMean, hSigma, None, small)
    assert e.value.code == gp.ERR["WORKSPACE"]


def test_host_buffer_pipeline_with_the_emulated_contractions_matches_oracle(gp):
    """gp_pipeline_host_mixed: the same call with the factorisation and the covariance on the int8-emulated contraction."""
    n, m, D, tile = 1536, 512, 8, 256
    X, y = nfir.nfir_features(31, n, D)
    Xs, _ = nfir.nfir_features(32, m, D, with_targets=False)
    h = oracle.Hyper()
    p = oracle.predict(X, y, Xs, h)
    hX, hY, hXs = (torch.from_numpy(a).pin_memory() for a in (X, y, Xs))
    hMean = torch.empty(m, dtype=torch.float64).pin_memory()
    hSigma = torch.empty(m, m, dtype=torch.float64).pin_memory()
    hAlpha = torch.empty(n, dtype=torch.float64).pin_memory()
    ws = torch.empty(gp.gp_pipeline_mixed_workspace_bytes(n, m, D, tile), dtype=torch.uint8, device="cuda")
    info = gp.gp_pipeline_host(hX, hY, hXs, gp.Hyper(), tile, 0, hMean, hSigma, hAlpha, ws, mixed=True)
    assert info == 0
    assert relerr(hAlpha.numpy(), p.alpha) <= TOL_ALPHA
    assert relerr(hMean.numpy(), p.mean) <= TOL_MEAN
    assert relerr(hSigma.numpy(), p.Sigma) <= TOL_SIGMA
    small = torch.empty(gp.gp_pipeline_workspace_bytes(n, m, D, tile), dtype=torch.uint8, device="cuda")
    with pytest.raises(gp.GpError) as e:
        gp.gp_pipeline_host(hX, hY, hXs, gp.Hyper(), tile, 0, hMean, hSigma, None, small, mixed=True)
    assert e.value.code == gp.ERR["WORKSPACE"]


def test_fp64_peak_probe_launches(gp):
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    for mode in (0, 1):
        flops = gp.gp_fp64_peak_launch(mode, 10, sink)
        assert flops > 0
    torch.cuda.synchronize()
    assert float(sink.item()) == 0.0


@pytest.mark.parametrize("n,tile,D", [(1024, 256, 8), (384, 128, 4)])
def test_solve_in_place_and_repeated_on_the_same_scratch(gp, n, tile, D):
    """gp_solve publishes the pieces of beta and alpha by their VALUES (a 'not yet computed' pattern in the output vectors):
    the header allows dAlpha == dY, and the scratch of one call may be reused by the next with other right-hand sides."""
    X, y = nfir.nfir_features(61, n, D)
    _, y2 = nfir.nfir_features(62, n, D)
    h = oracle.Hyper()
    Lo = oracle.cholesky(oracle.assemble(X, X, h, True))
    pipe = gp.GpPipeline(n, 0, D, tile, gp.Hyper())
    pipe.assemble(torch.from_numpy(X).cuda())
    pipe.cholesky()
    for rhs in (y, y2, y):
        want = oracle.backward_subst(Lo, oracle.forward_subst(Lo, rhs))
        buf = torch.from_numpy(rhs.copy()).cuda()             # y in, alpha out, same buffer
        gp.gp_solve(pipe.KL, n, tile, buf, buf, None, pipe.work)
        torch.cuda.synchronize()
        assert relerr(buf.cpu().numpy(), want) <= TOL_ALPHA
        pipe.solve(torch.from_numpy(rhs).cuda())              # separate buffers: the same bits
        torch.cuda.synchronize()
        assert torch.equal(buf, pipe.alpha)


# ---------------------------------------------------------------- SURVEY.md 8(f) rows 1 and 4
@pytest.mark.parametrize("n,m,D,tile", [(128, 128, 8, 32), (1024, 1024, 8, 256), (768, 256, 5, 128), (1280, 512, 16, 256)])
def test_variance_only_and_log_marginal_likelihood(gp, n, m, D, tile):
    """gp_predict_variance (diag Sigma without W) and gp_log_marginal_likelihood against the oracle."""
    X, y = nfir.nfir_features(31, n, D)
    Xs, _ = nfir.nfir_features(32, m, D, with_targets=False)
    h = oracle.Hyper(2.0, 1.3, 0.05) if D == 16 else oracle.Hyper()
    p = oracle.predict(X, y, Xs, h, full_cov=True, variance=True)
    hg = gp.Hyper(h.lengthscale, h.vertical, h.noise, h.ell_squared)
    pipe = gp.GpPipeline(n, m, D, tile, hg)
    dX, dy, dXs = _dev(X), _dev(y), _dev(Xs)
    pipe.assemble(dX); pipe.cholesky(); pipe.solve(dy)
    var = torch.empty(m, dtype=torch.float64, device="cuda")
    gp.gp_predict_variance(pipe.KL, dX, dXs, hg, tile, 0, var, pipe.work)
    lml = torch.empty(1, dtype=torch.float64, device="cuda")
    gp.gp_log_marginal_likelihood(pipe.KL, n, tile, dy, pipe.alpha, lml)
    # the full covariance afterwards, on the same workspace: its diagonal must agree with the variance path
    gp.gp_predict_full_cov(pipe.KL, dX, dXs, hg, tile, 0, pipe.Sigma, pipe.work)
    torch.cuda.synchronize()
    assert int(pipe.info.item()) == 0
    v = var.cpu().numpy()
    assert relerr(v, p.var) <= TOL_SIGMA
    np.testing.assert_allclose(v, p.var, rtol=0, atol=1e-9 * np.abs(p.var).max())
    assert v.min() >= 0.0 and v.max() <= h.vertical
    np.testing.assert_allclose(v, np.diag(pipe.Sigma.cpu().numpy()), rtol=0, atol=1e-12)
    want = oracle.log_marginal_likelihood(p.L, y, p.alpha)
    assert abs(float(lml.item()) - want) <= 1e-10 * abs(want)


def test_variance_argument_errors(gp):
    n, m, D, tile = 128, 128, 4, 32
    X = torch.zeros(n, D, dtype=torch.float64, device="cuda")
    pipe = gp.GpPipeline(n, m, D, tile, gp.Hyper())
    var = torch.empty(m, dtype=torch.float64, device="cuda")
    with pytest.raises(gp.GpError) as e:
        gp.gp_predict_variance(pipe.KL, X, X, gp.Hyper(), 48, 0, var, pipe.work)
    assert e.value.code == gp.ERR["TILE"]
    with pytest.raises(gp.GpError) as e:
        gp.gp_predict_variance(pipe.KL, X, X, gp.Hyper(), tile, 0, var, pipe.work[:1024])
    assert e.value.code == gp.ERR["WORKSPACE"]
    with pytest.raises(gp.GpError) as e:
        gp.gp_log_marginal_likelihood(pipe.KL, n, 48, pipe.alpha, pipe.alpha, var)
    assert e.value.code == gp.ERR["TILE"]


def test_contraction_bench_launches(gp):
    """The steady-state contraction microbenchmark bench.py reports runs and counts its flop."""
    K, reps = 256, 3
    buf = (torch.rand(gp.gp_contraction_bench_bytes(K, reps) // 8 + 1, dtype=torch.float64, device="cuda") * 1e-3).view(torch.uint8)
    flop = gp.gp_contraction_bench_launch(K, reps, buf)
    torch.cuda.synchronize()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    assert flop == sms * reps * 2.0 * 128 * 128 * K
    assert torch.isfinite(buf.view(torch.float64)[: 3 * K * K]).all()


# ---------------------------------------------------------------- edge cases of the executor and the assembly
@pytest.mark.parametrize("n,m,D,tile", [
    (256, 256, 8, 256),       # a single tile: the whole factorisation is one POTRF tile task
    (2048, 2048, 4, 2048),    # 16 blocks per tile edge: 33 dependency waits per update (more than one per lane)
    (512, 128, 40, 128),      # D > 32: the assembly stages the features in two chunks
    (256, 64, 1, 64),         # D = 1
])
def test_edge_shapes(gp, n, m, D, tile):
    X, y = nfir.nfir_features(3 * n + D, n, D)
    Xs, _ = nfir.nfir_features(5 * m + D, m, D, with_targets=False)
    h = oracle.Hyper()
    p = oracle.predict(X, y, Xs, h)
    out = _run_pipeline(gp, X, y, Xs, h, tile)
    _check_against_oracle(out, p)


def test_single_worker_runs_the_whole_dag(gp):
    """sched_width = 1: one persistent CTA executes every item in list order (no deadlock, same result)."""
    n, m, D, tile = 768, 256, 8, 256
    gp.gp_set_block_edge(128)
    X, y = nfir.nfir_features(41, n, D)
    Xs, _ = nfir.nfir_features(42, m, D, with_targets=False)
    h = oracle.Hyper()
    p = oracle.predict(X, y, Xs, h)
    out = _run_pipeline(gp, X, y, Xs, h, tile, width=1)
    _check_against_oracle(out, p)


# ---------------------------------------------------------------- robustness of the inverse-based TRSM
@pytest.mark.parametrize("noise,cond_floor", [(1e-6, 1e8), (1e-8, 1e10)])
def test_ill_conditioned_factorisation(gp, noise, cond_floor):
    """L_IJ = K_IJ inv(L_JJ)^T is a product with an explicit inverse, not a substitution.  On a smooth
    D=2 problem with tiny noise (cond(K) ~ 6e8 and 6e10, reading A6 allows it) the factor must stay
    backward stable (||L L^T - K|| / ||K|| at rounding level) and its distance from the oracle must be
    of the size of the distance between two backward-stable substitution factorisations of the same K
    (the oracle and LAPACK via numpy): the explicit inverses cost no accuracy that substitution would keep."""
    n, D, tile = 1024, 2, 256
    X, y = nfir.nfir_features(77, n, D)
    h = oracle.Hyper(1.0, 1.0, noise)
    K = oracle.assemble(X, X, h, True)
    w = np.linalg.eigvalsh(K)
    assert w[-1] / w[0] >= cond_floor
    Lo = oracle.cholesky(K)
    yardstick = relerr(np.linalg.cholesky(K), Lo)            # ~1e-11 at cond 6e8, ~1e-10 at 6e10
    for cap in (64, 128):                                       # inverses of 64- and of 128-blocks
        gp.gp_set_block_edge(cap)
        pipe = gp.GpPipeline(n, 0, D, tile, gp.Hyper(1.0, 1.0, noise))
        pipe.assemble(_dev(X))
        pipe.cholesky()
        torch.cuda.synchronize()
        assert int(pipe.info.item()) == 0
        L = pipe.dense_L().cpu().numpy()
        resid = np.linalg.norm(L @ L.T - K) / np.linalg.norm(K)
        err = relerr(L, Lo)
        print(f"noise={noise:g} block={cap} cond={w[-1] / w[0]:.3g} residual={resid:.2e} |L-L_oracle|/|L_oracle|={err:.2e} "
              f"oracle-vs-LAPACK={yardstick:.2e}")
        assert resid <= 2e-14                               # measured with 128-blocks: 2e-15 at cond 6e8, 7e-15 at cond 6e10 (oracle: 7e-16)
        assert err <= 20 * yardstick
    # the solve on top of it: K alpha = y to the accuracy cond * u allows
    pipe.solve(_dev(y))
    torch.cuda.synchronize()
    alpha = pipe.alpha.cpu().numpy()
    assert np.linalg.norm(K @ alpha - y) / (np.linalg.norm(K) * np.linalg.norm(alpha)) <= 1e-14
