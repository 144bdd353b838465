"""the split-operand (Ozaki) contraction on the int8 tensor cores (tcgen05.mma kind::i8,
TMEM accumulators) against the oracle, through the C ABI.  C -= A A^T is Eq. 3's  Sigma = K** - V^T V  with
A = V^T, so oracle.posterior_cov is the expected value; a general A B^T case is checked against
the exact integer arithmetic of the planes themselves (numpy int64), which pins the digit extraction too."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle
from helpers import relerr


@pytest.fixture(scope="module")
def gp():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    from paper_2602_19683_b200 import binding
    binding.load()
    return binding


# (256, 512), (384, 1152) and (1280, 2048) take the 128 x 128 two-pass kernel, the others the 128 x 64 one (m or n not a multiple of 128)
# (1792, 256): 14 x 14 output tiles, more than the band height of the wide kernel's tile order (a band of 12 rows + one of 2)
@pytest.mark.parametrize("m,n", [(128, 32), (256, 512), (640, 1056), (384, 1152), (1280, 2048), (1792, 256)])
def test_emulated_contraction_matches_oracle_posterior_cov(gp, m, n):
    rng = np.random.default_rng(m + n)
    V = rng.uniform(-0.9, 0.9, size=(n, m))                     # |V| <= 1 as for V = L^-1 K_{X,X^} with v = 1
    Kss = rng.normal(size=(m, m))
    want = oracle.posterior_cov(V, Kss)
    A = torch.from_numpy(np.ascontiguousarray(V.T)).cuda()      # m x n, contraction index contiguous
    C = torch.from_numpy(Kss.copy()).cuda()
    planes = gp.gp_ozaki_slice(A, 2.0)
    S, b = gp.gp_ozaki_planes(), gp.gp_ozaki_digit_bits()
    assert S * b == 56 and planes.shape == (S, m, n) and int(planes.min()) >= -2 ** (b - 1) and int(planes.max()) <= 2 ** (b - 1) - 1
    gp.gp_ozaki_contract(planes, planes, 2.0, 2.0, C)
    torch.cuda.synchronize()
    got = C.cpu().numpy()
    assert relerr(got, want) <= 1e-14
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13 * np.abs(want).max())


@pytest.mark.parametrize("ma,nb,k", [(256, 192, 288), (384, 256, 640), (128, 128, 128)])
def test_planes_are_an_exact_fixed_point_expansion_and_products_are_exact(gp, ma, nb, k):
    """x / scale = sum_p d_p 2^(-b (p+1)) to 2^-57 (S planes of b-bit digits, S b = 56), and the tensor-core result equals
    the integer arithmetic of the planes recombined in FP64 (levels smallest first), bit for bit up to the last roundings
    (the 128 x 128 kernel, second and third shape, subtracts the high and the low levels in two steps)."""
    rng = np.random.default_rng(3)
    scale = 4.0
    A = rng.uniform(-1.9, 1.9, size=(ma, k)); B = rng.normal(size=(nb, k)).clip(-1.9, 1.9)
    dA, dB = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    pa, pb = gp.gp_ozaki_slice(dA, scale), gp.gp_ozaki_slice(dB, scale)
    Pa, Pb = pa.cpu().numpy().astype(np.int64), pb.cpu().numpy().astype(np.int64)
    S, b = gp.gp_ozaki_planes(), gp.gp_ozaki_digit_bits()
    w = 2.0 ** (-float(b) * np.arange(1, S + 1))
    np.testing.assert_allclose(np.tensordot(w, Pa.astype(np.float64), axes=1) * scale, A, rtol=0, atol=scale * 2.0 ** -57)
    C0 = rng.normal(size=(ma, nb))
    C = torch.from_numpy(C0.copy()).cuda()
    gp.gp_ozaki_contract(pa, pb, scale, scale, C)
    torch.cuda.synchronize()
    acc = np.zeros((ma, nb))
    for lvl in range(S - 1, -1, -1):
        s = sum(Pa[p] @ Pb[lvl - p].T for p in range(lvl + 1))          # exact int64
        acc += s.astype(np.float64) * (scale * scale * 2.0 ** (-float(b) * (lvl + 2)))
    np.testing.assert_allclose(C.cpu().numpy(), C0 - acc, rtol=0, atol=4e-16 * np.abs(C0 - acc).max())
    assert relerr(C.cpu().numpy(), C0 - A @ B.T) <= 1e-14


def test_contraction_deeper_than_one_accumulator_runs_in_segments(gp):
    """k = 20480 > 16384 (what an int32 level accumulator takes with 8-bit digits): two launches over k segments.  Operands
    near +- 0.495 scale with equal signs drive the level sums as high as they go; the expected value is exact rational
    arithmetic (a floating-point sum of 20480 terms would be the less accurate side)."""
    from fractions import Fraction
    m, k, val = 128, 20480, 0.99
    A = torch.full((m, k), val, dtype=torch.float64, device="cuda")
    A[::2] = -val
    C = torch.zeros(m, m, dtype=torch.float64, device="cuda")
    planes = gp.gp_ozaki_slice(A, 2.0)
    gp.gp_ozaki_contract(planes, planes, 2.0, 2.0, C)
    torch.cuda.synchronize()
    mag = float(Fraction(val) ** 2 * k)
    sign = np.where(np.arange(m) % 2 == 0, -1.0, 1.0)
    want = -mag * np.outer(sign, sign)
    assert relerr(C.cpu().numpy(), want) <= 1e-15


def test_slice_reports_entries_beyond_the_scale_and_bad_arguments(gp):
    X = torch.full((128, 32), 1.5, dtype=torch.float64, device="cuda")
    with pytest.raises(ValueError):
        gp.gp_ozaki_slice(X, 2.0)                                   # |x| > scale / 2
    gp.gp_ozaki_slice(X, 4.0)
    with pytest.raises(gp.GpError) as e:
        gp.gp_ozaki_slice(torch.zeros(128, 40, dtype=torch.float64, device="cuda"), 2.0)   # k % 32 != 0
    assert e.value.code == gp.ERR["SIZE"]
    p = gp.gp_ozaki_slice(torch.zeros(96, 32, dtype=torch.float64, device="cuda"), 2.0)
    with pytest.raises(gp.GpError) as e:
        gp.gp_ozaki_contract(p, p, 2.0, 2.0, torch.zeros(96, 96, dtype=torch.float64, device="cuda"))   # rows % 128 != 0
    assert e.value.code == gp.ERR["SIZE"]


# ---------------------------------------------------------------- the mixed factorisation end to end
@pytest.mark.parametrize("n,D,tile,noise", [(512, 8, 128, 0.1), (1024, 8, 256, 0.1), (2048, 8, 512, 0.1), (2048, 8, 1024, 0.1), (1536, 3, 256, 1e-3)])
def test_mixed_cholesky_matches_oracle(gp, n, D, tile, noise):
    """FP64 panels + emulated trailing updates: L against the oracle at north_star's tolerance (1e-10), and bitwise
    reproducible from run to run (integer accumulation + a fixed recombination order)."""
    from paper_2602_19683_b200 import nfir
    X, y = nfir.nfir_features(n + D, n, D)
    h = oracle.Hyper(1.0, 1.0, noise)
    K = oracle.assemble(X, X, h, True)
    Lo = oracle.cholesky(K)
    pipe = gp.GpPipeline(n, 0, D, tile, gp.Hyper(1.0, 1.0, noise))
    work = torch.empty(gp.gp_mixed_workspace_bytes(n, tile), dtype=torch.uint8, device="cuda")
    dX = torch.from_numpy(X).cuda()
    outs = []
    for _ in range(2):
        pipe.assemble(dX)
        gp.gp_cholesky_tiled_mixed(pipe.KL, n, tile, 0, pipe.info, work)
        torch.cuda.synchronize()
        assert int(pipe.info.item()) == 0
        outs.append(pipe.dense_L().cpu().numpy())
    err = relerr(outs[0], Lo)
    print(f"mixed n={n} tile={tile} noise={noise}: |L - L_oracle| / |L_oracle| = {err:.2e}")
    assert err <= 1e-10
    np.testing.assert_allclose(outs[0], Lo, rtol=0, atol=1e-9 * np.abs(Lo).max())
    assert np.array_equal(outs[0], outs[1])
    # and the rest of the pipeline runs on this factor unchanged
    pipe.solve(torch.from_numpy(y).cuda())
    torch.cuda.synchronize()
    assert relerr(pipe.alpha.cpu().numpy(), oracle.backward_subst(Lo, oracle.forward_subst(Lo, y))) <= 1e-9


def test_mixed_cholesky_reports_a_non_positive_pivot(gp):
    n, tile = 512, 128
    K = np.eye(n)
    K[300, 300] = -1.0
    tiles = [K[I * tile:(I + 1) * tile, J * tile:(J + 1) * tile].ravel() for I in range(n // tile) for J in range(I + 1)]
    KL = torch.from_numpy(np.concatenate(tiles)).cuda()
    work = torch.empty(gp.gp_mixed_workspace_bytes(n, tile), dtype=torch.uint8, device="cuda")
    info = torch.zeros(1, dtype=torch.int32, device="cuda")
    gp.gp_cholesky_tiled_mixed(KL, n, tile, 0, info, work)
    torch.cuda.synchronize()
    assert int(info.item()) == 301


# (1024, 2048, ...): Sigma has 16 x 16 output tiles: the banded tile order together with the lower-triangle selection
@pytest.mark.parametrize("n,m,D,tile", [(512, 256, 8, 128), (1024, 512, 8, 256), (2048, 1024, 5, 512), (1536, 256, 8, 256), (1024, 2048, 8, 256)])
def test_mixed_prediction_matches_oracle(gp, n, m, D, tile):
    """gp_predict_full_cov_mixed (V^T solve and W on the emulated contraction, TRSM with the diagonal tiles in FP64) on the
    factor of gp_cholesky_tiled_mixed: Sigma against the oracle at north_star's 1e-9, exactly symmetric."""
    from paper_2602_19683_b200 import nfir
    X, y = nfir.nfir_features(3 * n + m, n, D)
    Xs, _ = nfir.nfir_features(5 * n + m, m, D, with_targets=False)
    h = oracle.Hyper(1.0, 1.3, 0.1)
    p = oracle.predict(X, y, Xs, h)
    hg = gp.Hyper(1.0, 1.3, 0.1)
    pipe = gp.GpPipeline(n, m, D, tile, hg)
    dX, dXs = torch.from_numpy(X).cuda(), torch.from_numpy(Xs).cuda()
    pipe.assemble(dX)
    work = torch.empty(max(gp.gp_mixed_workspace_bytes(n, tile), gp.gp_mixed_predict_workspace_bytes(n, m, tile)), dtype=torch.uint8, device="cuda")
    gp.gp_cholesky_tiled_mixed(pipe.KL, n, tile, 0, pipe.info, work)
    gp.gp_predict_full_cov_mixed(pipe.KL, dX, dXs, hg, tile, 0, pipe.Sigma, work)
    torch.cuda.synchronize()
    assert int(pipe.info.item()) == 0
    S = pipe.Sigma.cpu().numpy()
    err = relerr(S, p.Sigma)
    print(f"mixed prediction n={n} m={m} tile={tile}: |Sigma - Sigma_oracle| / |Sigma_oracle| = {err:.2e}")
    assert err <= 1e-9
    np.testing.assert_allclose(S, p.Sigma, rtol=0, atol=1e-9 * np.abs(p.Sigma).max())
    assert np.array_equal(S, S.T)
    d = np.diag(S)
    assert d.min() >= 0.0 and d.max() <= h.vertical
    # variances only (8(f) row 1 on the emulated V^T solve): the oracle's posterior variances
    var = torch.empty(m, dtype=torch.float64, device="cuda")
    gp.gp_predict_variance_mixed(pipe.KL, dX, dXs, hg, tile, 0, var, work)
    torch.cuda.synchronize()
    want = oracle.posterior_var(p.V, h.vertical * np.ones(m))
    assert relerr(var.cpu().numpy(), want) <= 1e-9
    np.testing.assert_allclose(var.cpu().numpy(), np.diag(p.Sigma), rtol=0, atol=1e-9 * h.vertical)


# ---------------------------------------------------------------- measurement support
def test_int8_mma_issue_loop_reports_the_tensor_core_rate(gp):
    """gp_int8_mma_peak_launch: cycles per 128 x N x 32 MMA of CTA 0 (N = 64 is bound by the shared-memory operand read
    at 48, N = 128 and 256 run at the pipe's 8192 MAC per cycle: 64 and 128)."""
    cyc = torch.zeros(1, dtype=torch.int64, device="cuda")
    for n_cols, want in ((64, 48.0), (128, 64.0), (256, 128.0)):
        iters = 500
        ops = gp.gp_int8_mma_peak_launch(n_cols, iters, cyc)
        torch.cuda.synchronize()
        assert ops == 2.0 * 128 * n_cols * 32 * 16 * iters * torch.cuda.get_device_properties(0).multi_processor_count
        per = float(cyc.item()) / (16.0 * iters)
        assert want * 0.98 <= per <= want * 1.15, (n_cols, per)
    with pytest.raises(gp.GpError):
        gp.gp_int8_mma_peak_launch(96, 10, cyc)


def test_probe_launch_without_a_switch_is_the_product_kernel(gp):
    """gp_ozaki_probe_launch(0) = the 128 x 128 two-pass kernel on dense C with scales 1: same bits as gp_ozaki_contract;
    with the loads or the reductions switched off it still terminates and leaves its time stamps."""
    rng = np.random.default_rng(11)
    m, k = 384, 512
    A = torch.from_numpy(rng.uniform(-0.45, 0.45, size=(m, k))).cuda()
    planes = gp.gp_ozaki_slice(A, 1.0)
    C0 = torch.from_numpy(rng.normal(size=(m, m))).cuda()
    C1, C2 = C0.clone(), C0.clone()
    gp.gp_ozaki_contract(planes, planes, 1.0, 1.0, C1)
    gp.gp_ozaki_probe_launch(0, planes, planes, C2)
    torch.cuda.synchronize()
    assert torch.equal(C1, C2)
    assert relerr(C1.cpu().numpy(), (C0 - A @ A.T).cpu().numpy()) <= 1e-14
    for probe in (1, 2, 4):
        gp.gp_ozaki_probe_launch(probe, planes, planes, C2)
        torch.cuda.synchronize()
        t = gp.gp_ozaki_probe_stamps()
        assert len(t) == 8
    with pytest.raises(gp.GpError):
        gp.gp_ozaki_probe_launch(3, planes, planes, C2)


def test_wide_kernel_is_bit_reproducible_over_many_runs(gp):
    """Race hunt for the 128 x 128 two-pass kernel (ring slots retired by tcgen05.commit, tensor memory handed between the
    passes, staging boxes reused behind bulk-group waits): 40 runs of a multi-tile, multi-wave product must give the same
    bits (integer level sums and a fixed recombination order leave no room for run-to-run differences)."""
    rng = np.random.default_rng(5)
    m, k = 2304, 1408                      # 18 x 18 tiles (324 > 148 CTAs: two and a bit waves), 11 k-chunks
    A = torch.from_numpy(rng.uniform(-0.9, 0.9, size=(m, k))).cuda()
    planes = gp.gp_ozaki_slice(A, 2.0)
    C0 = torch.from_numpy(rng.normal(size=(m, m))).cuda()
    first = None
    for _ in range(40):
        C = C0.clone()
        gp.gp_ozaki_contract(planes, planes, 2.0, 2.0, C)
        torch.cuda.synchronize()
        if first is None:
            first = C
            assert relerr(C.cpu().numpy(), (C0 - A @ A.T).cpu().numpy()) <= 1e-14
        else:
            assert torch.equal(C, first)
