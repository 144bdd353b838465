"""The seeded NFIR-shaped generator (BASELINE.json configs; DESIGN.md input recipe)."""
import numpy as np

from paper_2602_19683_b200 import nfir


def test_configs_match_baseline_json():
    got = [(c.n, c.m, c.D, c.tile) for c in nfir.CONFIGS]
    assert got == [(128, 128, 8, 32), (1024, 1024, 8, 256), (8192, 1024, 8, 512),
                   (32768, 4096, 8, 1024), (65536, 8192, 16, 2048)]
    assert (nfir.CONFIGS[4].lengthscale, nfir.CONFIGS[4].noise) == (2.0, 0.05)
    assert all((c.lengthscale, c.vertical, c.noise) == (1.0, 1.0, 0.1) for c in nfir.CONFIGS[:4])
    assert all(c.n % c.tile == 0 and c.m % c.tile == 0 for c in nfir.CONFIGS)


def test_lag_structure_and_determinism():
    X, y = nfir.nfir_features(11, 200, 8)
    X2, y2 = nfir.nfir_features(11, 200, 8)
    assert np.array_equal(X, X2) and np.array_equal(y, y2)
    assert X.shape == (200, 8) and y.shape == (200,) and X.dtype == np.float64 and X.flags.c_contiguous
    assert np.all(np.abs(X) <= 1.0)
    # x_i = (u_i, u_{i-1}, ...): column k of row i equals column 0 of row i-k
    for k in range(1, 8):
        assert np.array_equal(X[k:, k], X[:-k, 0])
    # targets follow the recipe up to the N(0, 0.1^2) noise
    w = 0.5 ** np.arange(8)
    clean = np.sin(2.0 * X @ w) + 0.3 * X[:, 1] ** 3
    resid = y - clean
    assert 0.07 < resid.std() < 0.13 and abs(resid.mean()) < 0.03
    X3, _ = nfir.nfir_features(12, 200, 8)
    assert not np.array_equal(X, X3)


def test_make_inputs_seeds():
    cfg = nfir.CONFIGS[0]
    X, y, Xs = nfir.make_inputs(cfg)
    Xa, ya = nfir.nfir_features(1000, 128, 8)
    Xb, _ = nfir.nfir_features(2000, 128, 8, with_targets=False)
    assert np.array_equal(X, Xa) and np.array_equal(y, ya) and np.array_equal(Xs, Xb)
