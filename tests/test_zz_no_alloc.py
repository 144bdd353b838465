"""gp_solve_noalloc: the forward/backward solves on the library's static device scratch, for callers that
cannot call cudaMalloc (CUDA graph capture, serving loops).  Its output must equal the existing gp_solve path's on two calls
in a row (the static array keeps the previous call's contents), problems beyond the fixed scratch are rejected, and the test
must pass alone in a fresh process as well as after every other test (this file is collected last on purpose)."""
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


@pytest.mark.parametrize("n,tile,D", [(2048, 256, 8), (8192, 512, 8), (96, 32, 3)])
def test_noalloc_solve_matches_the_existing_path_on_two_calls_in_a_row(gp, n, tile, D):
    X, y1 = nfir.nfir_features(41, n, D)
    _, y2 = nfir.nfir_features(42, n, D)
    pipe = gp.GpPipeline(n, 0, D, tile, gp.Hyper())
    dX = torch.from_numpy(X).cuda()
    pipe.assemble(dX)
    pipe.cholesky()
    torch.cuda.synchronize()
    assert int(pipe.info.item()) == 0
    free_before = torch.cuda.mem_get_info()[0]
    for k, y in enumerate((y1, y2, y1)):                      # the third call re-uses scratch left by a different right-hand side
        dy = torch.from_numpy(y).cuda()
        pipe.solve(dy)                                        # existing path: scratch from the caller
        torch.cuda.synchronize()
        want_alpha, want_beta = pipe.alpha.clone(), pipe.beta.clone()
        alpha = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
        beta = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
        gp.gp_solve_noalloc(pipe.KL, n, tile, dy, alpha, beta)
        torch.cuda.synchronize()
        assert relerr(alpha.cpu().numpy(), want_alpha.cpu().numpy()) <= 1e-9, k
        assert torch.equal(alpha, want_alpha), k              # same kernels, same order: in fact the same bits
        assert torch.equal(beta, want_beta), k
        alpha2 = torch.empty(n, dtype=torch.float64, device="cuda")
        gp.gp_solve_noalloc(pipe.KL, n, tile, dy, alpha2)    # beta inside the static scratch
        torch.cuda.synchronize()
        assert torch.equal(alpha2, want_alpha), k
    if n <= 2048:                                             # and against the oracle, through the dense factor
        L = pipe.dense_L().cpu().numpy()
        ref = oracle.backward_subst(L, oracle.forward_subst(L, y1))
        assert relerr(alpha.cpu().numpy(), ref) <= 1e-9
    # nothing was allocated by the calls themselves (the tensors above come from torch's cache or are freed again)
    assert torch.cuda.mem_get_info()[0] >= free_before - (64 << 20)


def test_noalloc_solve_rejects_what_does_not_fit_its_static_scratch(gp):
    dummy = torch.zeros(1024, dtype=torch.float64, device="cuda")
    with pytest.raises(gp.GpError) as e:                      # rejected before anything is touched
        gp.gp_solve_noalloc(dummy, 16384, 1024, dummy, dummy)
    assert e.value.code == gp.ERR["LIMIT"]
    assert "gp_solve_noalloc" in str(e.value) or "scratch" in str(e.value)
    gp.gp_set_block_edge(128)                                 # 128-blocks at n = 8192 would need 8 MB of inverted diagonal blocks
    try:
        with pytest.raises(gp.GpError) as e:
            gp.gp_solve_noalloc(dummy, 8192, 512, dummy, dummy)
        assert e.value.code == gp.ERR["LIMIT"]
    finally:
        gp.gp_set_block_edge(0)
    with pytest.raises(gp.GpError) as e:
        gp.gp_solve_noalloc(dummy, 100, 32, dummy, dummy)
    assert e.value.code == gp.ERR["TILE"]
