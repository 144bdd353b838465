"""Pins for the CPU oracle (oracle/gp_oracle.c) against things that are NOT the oracle:
40-digit worked examples, closed forms, brute-force inversion, numpy/scipy library
routines, and the invariants north_star lists.  CPU only."""
import math

import numpy as np
import pytest
import scipy.linalg

import oracle
from oracle import Hyper
from paper_2602_19683_b200 import nfir
from helpers import gauss_jordan_inverse, relerr, se_kernel_numpy


def _f(x):
    return np.array(x, dtype=np.float64) if not isinstance(x, list) or not isinstance(x[0], list) \
        else np.array([[float(t) for t in r] for r in x])


def _fv(x):
    return np.array([float(t) for t in x])


def _fm(x):
    return np.array([[float(t) for t in r] for r in x])


# ---------------------------------------------------------------- (i) worked examples
@pytest.mark.parametrize("name", ["A", "B", "Bprime_printed_2ell", "Bprime_ell_squared"])
def test_worked_examples_40_digits(golden, name):
    g = golden[name]
    h = Hyper(g["lengthscale"], g["vertical"], g["noise"], g["ell_squared"])
    X, y, Xs = np.array(g["X"]), np.array(g["y"]), np.array(g["Xs"])
    p = oracle.predict(X, y, Xs, h)
    tol = 1e-14
    assert relerr(p.K, _fm(g["K"])) <= tol
    assert relerr(p.L, _fm(g["L"])) <= tol
    assert relerr(p.beta, _fv(g["beta"])) <= tol
    assert relerr(p.alpha, _fv(g["alpha"])) <= tol
    assert relerr(p.V, _fm(g["V"])) <= tol
    assert relerr(p.mean, _fv(g["mean"])) <= tol
    assert relerr(p.Sigma, _fm(g["Sigma"])) <= tol
    # element-wise too, so a swapped pair of entries cannot hide in a norm
    np.testing.assert_allclose(p.Sigma, _fm(g["Sigma"]), rtol=1e-13, atol=1e-15)
    np.testing.assert_allclose(p.V, _fm(g["V"]), rtol=1e-13, atol=1e-15)
    np.testing.assert_allclose(oracle.assemble(X, Xs, h, False), _fm(g["K_X_Xs"]), rtol=1e-14)


def test_printed_survey_values_example_A():
    """Literal digits printed in SURVEY.md 8(c)(i), typed in by hand (not via the json)."""
    p = oracle.predict(np.array([[0.0], [1.0]]), np.array([1.0, 2.0]), np.array([[0.5], [2.0]]), Hyper())
    np.testing.assert_allclose(p.L, [[1.0488088481701515, 0.0], [0.57830429326644473, 0.87496522467444264]], rtol=1e-14)
    np.testing.assert_allclose(p.beta, [0.95346258924559232, 1.6556183609575249], rtol=1e-14)
    np.testing.assert_allclose(p.alpha, [-0.13425787820991119, 1.8922104722202507], rtol=1e-14)
    np.testing.assert_allclose(p.mean, [1.5513877191046794, 1.1295138380566173], rtol=1e-14)
    np.testing.assert_allclose(p.Sigma, [[0.087270095454893377, -0.058988103679474658],
                                         [-0.058988103679474658, 0.61378397912183018]], rtol=1e-13)


def test_example_A_closed_forms():
    p = oracle.predict(np.array([[0.0], [1.0]]), np.array([1.0, 2.0]), np.array([[0.5], [2.0]]), Hyper())
    e = math.exp
    assert p.L[0, 0] == pytest.approx(math.sqrt(1.1), rel=1e-15)
    assert p.L[1, 0] == pytest.approx(e(-0.5) / math.sqrt(1.1), rel=1e-15)
    assert p.L[1, 1] == pytest.approx(math.sqrt(1.1 - e(-1.0) / 1.1), rel=1e-15)
    assert p.L[0, 1] == 0.0
    assert p.mean[0] == pytest.approx(3.0 * e(-0.125) / (1.1 + e(-0.5)), rel=1e-14)
    assert p.Sigma[0, 0] == pytest.approx(1.0 - 2.0 * e(-0.25) / (1.1 + e(-0.5)), rel=1e-13)


# ---------------------------------------------------------------- (ii) closed forms
@pytest.mark.parametrize("ell,v,s2,esq", [(1.0, 1.0, 0.1, False), (2.0, 1.5, 0.05, False), (2.0, 1.5, 0.05, True)])
def test_single_training_point_closed_form(ell, v, s2, esq):
    h = Hyper(ell, v, s2, esq)
    X = np.array([[0.3, -0.2, 0.9]])
    y = np.array([0.7])
    Xs = np.array([[0.1, 0.4, 0.5], [0.3, -0.2, 0.9]])
    p = oracle.predict(X, y, Xs, h)
    den = 2 * ell * ell if esq else 2 * ell
    assert p.L[0, 0] == pytest.approx(math.sqrt(v + s2), rel=1e-15)
    assert p.alpha[0] == pytest.approx(0.7 / (v + s2), rel=1e-15)
    for a in range(2):
        r2 = float(np.sum((Xs[a] - X[0]) ** 2))
        ks = v * math.exp(-r2 / den)
        assert p.mean[a] == pytest.approx(ks * 0.7 / (v + s2), rel=1e-14)
        assert p.Sigma[a, a] == pytest.approx(v - ks * ks / (v + s2), rel=1e-13)
    # test point coinciding with the training point still gets NO noise (reading A2)
    assert oracle.assemble(Xs, X, h, False)[1, 0] == pytest.approx(v, rel=1e-15)


def test_far_apart_training_points_give_scaled_identity():
    h = Hyper()
    n = 6
    X = np.zeros((n, 2))
    X[:, 0] = 100.0 * np.arange(n)          # r^2 >= 1e4: exp underflows to exactly 0
    y = np.arange(1.0, n + 1)
    Xs = X[:3] + 0.25
    p = oracle.predict(X, y, Xs, h)
    assert np.array_equal(p.K, 1.1 * np.eye(n))
    np.testing.assert_allclose(p.L, math.sqrt(1.1) * np.eye(n), rtol=1e-15)
    Kxs = se_kernel_numpy(Xs, X, 1.0, 1.0)
    Kss = se_kernel_numpy(Xs, Xs, 1.0, 1.0)
    np.testing.assert_allclose(p.Sigma, Kss - Kxs @ Kxs.T / 1.1, rtol=1e-13, atol=1e-16)
    np.testing.assert_allclose(p.mean, Kxs @ y / 1.1, rtol=1e-14)


def test_assemble_matches_broadcast_formula_rectangular():
    """Non-square, D not a power of two: catches transposed operands and index slips."""
    rng = np.random.default_rng(7)
    A, B = rng.normal(size=(13, 5)), rng.normal(size=(29, 5))
    for h in (Hyper(1.0, 1.0, 0.1), Hyper(2.0, 0.7, 0.05), Hyper(2.0, 0.7, 0.05, True)):
        K = oracle.assemble(A, B, h, add_noise_diag=False)
        assert K.shape == (13, 29)
        np.testing.assert_allclose(K, se_kernel_numpy(A, B, h.lengthscale, h.vertical, h.ell_squared), rtol=2e-15)
    Kn = oracle.assemble(A, A, Hyper(1.0, 1.0, 0.1), add_noise_diag=True)
    assert np.all(Kn.diagonal() == 1.1)            # exactly v + sigma^2
    assert np.array_equal(Kn, Kn.T)
    K0 = oracle.assemble(A, A, Hyper(1.0, 1.0, 0.1), add_noise_diag=False)
    np.testing.assert_array_equal(Kn - np.diag(Kn.diagonal()), K0 - np.diag(K0.diagonal()))


# ---------------------------------------------------------------- library routines
@pytest.mark.parametrize("n", [1, 2, 5, 37, 200])
def test_cholesky_and_substitutions_vs_numpy_scipy(n):
    rng = np.random.default_rng(n)
    G = rng.normal(size=(n, n))
    K = G @ G.T + n * np.eye(n)
    L = oracle.cholesky(K)
    np.testing.assert_allclose(L, np.linalg.cholesky(K), rtol=1e-12, atol=1e-14)
    assert np.all(np.triu(L, 1) == 0.0)
    b = rng.normal(size=n)
    np.testing.assert_allclose(oracle.forward_subst(L, b), scipy.linalg.solve_triangular(L, b, lower=True), rtol=1e-11)
    np.testing.assert_allclose(oracle.backward_subst(L, b), scipy.linalg.solve_triangular(L.T, b, lower=False), rtol=1e-11)
    B = rng.normal(size=(n, 7))
    np.testing.assert_allclose(oracle.forward_subst_cols(L, B), scipy.linalg.solve_triangular(L, B, lower=True), rtol=1e-11)
    # the multi-column backward substitution: against the library routine (a transposed-operand or wrong-direction
    # slip fails here), and bit-identical to the single-vector recurrence column by column
    Xb = oracle.backward_subst_cols(L, B)
    np.testing.assert_allclose(Xb, scipy.linalg.solve_triangular(L.T, B, lower=False), rtol=1e-11)
    for c in range(B.shape[1]):
        assert np.array_equal(Xb[:, c], oracle.backward_subst(L, np.ascontiguousarray(B[:, c])))
    # forward then backward = K^-1: K (L^-T L^-1 B) = B
    np.testing.assert_allclose(K @ oracle.backward_subst_cols(L, oracle.forward_subst_cols(L, B)), B, rtol=1e-9, atol=1e-11)
    M = rng.normal(size=(9, n))
    np.testing.assert_allclose(oracle.matvec(M, b), M @ b, rtol=1e-12, atol=1e-13)
    V = rng.normal(size=(n, 6))
    Kss = rng.normal(size=(6, 6))
    np.testing.assert_allclose(oracle.posterior_cov(V, Kss), Kss - V.T @ V, rtol=1e-12, atol=1e-12)


def test_cholesky_only_reads_lower_triangle_and_reports_bad_pivot():
    K = np.array([[4.0, 99.0], [2.0, 5.0]])         # upper entry is garbage and must be ignored
    np.testing.assert_allclose(oracle.cholesky(K), [[2.0, 0.0], [1.0, 2.0]])
    with pytest.raises(np.linalg.LinAlgError, match="column 2"):
        oracle.cholesky(np.array([[1.0, 0.0], [2.0, 1.0]]))   # 1 - 4 < 0 at column 2
    with pytest.raises(np.linalg.LinAlgError, match="column 1"):
        oracle.cholesky(np.array([[0.0, 0.0], [0.0, 1.0]]))


# ---------------------------------------------------------------- (iv) brute force
@pytest.mark.parametrize("n,m,D,seed", [(3, 2, 1, 0), (16, 9, 3, 1), (64, 40, 8, 2)])
def test_brute_force_inverse_eq2_eq3(n, m, D, seed):
    X, y = nfir.nfir_features(seed, n, D)
    Xs, _ = nfir.nfir_features(seed + 50, m, D, with_targets=False)
    for h in (Hyper(), Hyper(2.0, 1.0, 0.05), Hyper(2.0, 1.0, 0.05, True)):
        p = oracle.predict(X, y, Xs, h)
        K = se_kernel_numpy(X, X, h.lengthscale, h.vertical, h.ell_squared) + h.noise * np.eye(n)
        Kxs = se_kernel_numpy(Xs, X, h.lengthscale, h.vertical, h.ell_squared)
        Kss = se_kernel_numpy(Xs, Xs, h.lengthscale, h.vertical, h.ell_squared)
        Kinv = gauss_jordan_inverse(K)
        assert relerr(p.alpha, Kinv @ y) <= 1e-11
        assert relerr(p.mean, Kxs @ Kinv @ y) <= 1e-11                     # Eq. 2
        assert relerr(p.Sigma, Kss - Kxs @ Kinv @ Kxs.T) <= 1e-11          # Eq. 3


# ---------------------------------------------------------------- (iii) invariants on the configs
@pytest.fixture(scope="module", params=[0, 1])
def cfg_pred(request):
    cfg = nfir.CONFIGS[request.param]
    X, y, Xs = nfir.make_inputs(cfg)
    h = Hyper(cfg.lengthscale, cfg.vertical, cfg.noise)
    return cfg, X, y, Xs, h, oracle.predict(X, y, Xs, h)


def test_invariants(cfg_pred):
    cfg, X, y, Xs, h, p = cfg_pred
    K, L = p.K, p.L
    assert np.array_equal(K, K.T)
    assert np.all(K.diagonal() == h.vertical + h.noise)
    assert np.linalg.norm(L @ L.T - K) / np.linalg.norm(K) <= 1e-12
    assert np.all(L.diagonal() > 0) and np.all(np.triu(L, 1) == 0)
    assert np.linalg.norm(K @ p.alpha - y) / np.linalg.norm(y) <= 1e-10
    assert np.linalg.norm(L @ p.beta - y) / np.linalg.norm(y) <= 1e-12
    S = p.Sigma
    assert np.linalg.norm(S - S.T) / np.linalg.norm(S) <= 1e-12
    d = S.diagonal()
    assert d.min() >= 0.0 and d.max() <= h.vertical                        # variance <= prior variance
    Ssym = 0.5 * (S + S.T)
    np.linalg.cholesky(Ssym + 1e-12 * h.vertical * np.eye(cfg.m))           # PSD
    assert np.linalg.eigvalsh(Ssym).min() >= -1e-12
    # mean = V^T beta ties the backward solve to the V solve
    assert relerr(p.mean, p.V.T @ p.beta) <= 1e-11


def test_test_points_equal_training_points_identities():
    """X^ = X with noise-free test matrices (A2): mean = y - s2*alpha, Sigma = s2*(I - s2*K^-1)."""
    cfg = nfir.CONFIGS[0]
    X, y, _ = nfir.make_inputs(cfg)
    for h in (Hyper(), Hyper(2.0, 1.0, 0.05), Hyper(2.0, 1.0, 0.05, True)):
        p = oracle.predict(X, y, X, h)
        assert relerr(p.mean, y - h.noise * p.alpha) <= 1e-11
        Kinv = gauss_jordan_inverse(p.K)
        assert relerr(p.Sigma, h.noise * (np.eye(cfg.n) - h.noise * Kinv)) <= 1e-10


def test_scaling_permutation_leading_block():
    cfg = nfir.CONFIGS[0]
    X, y, Xs = nfir.make_inputs(cfg)
    h = Hyper()
    p = oracle.predict(X, y, Xs, h)
    c = 3.5
    q = oracle.predict(X, y, Xs, Hyper(h.lengthscale, c * h.vertical, c * h.noise))
    assert relerr(q.L, math.sqrt(c) * p.L) <= 1e-13
    assert relerr(q.alpha, p.alpha / c) <= 1e-11
    assert relerr(q.mean, p.mean) <= 1e-11
    assert relerr(q.Sigma, c * p.Sigma) <= 1e-11
    perm = np.random.default_rng(3).permutation(cfg.m)
    r = oracle.predict(X, y, Xs[perm], h)
    assert relerr(r.mean, p.mean[perm]) <= 1e-14
    assert relerr(r.Sigma, p.Sigma[np.ix_(perm, perm)]) <= 1e-14
    k = 50
    Lk = oracle.cholesky(p.K[:k, :k])
    assert np.array_equal(Lk, p.L[:k, :k])


def test_ell_convention_switch_coincides_at_ell_1_only():
    X, y, Xs = nfir.make_inputs(nfir.CONFIGS[0])
    a = oracle.assemble(X, X, Hyper(1.0, 1.0, 0.1, False), True)
    b = oracle.assemble(X, X, Hyper(1.0, 1.0, 0.1, True), True)
    assert np.array_equal(a, b)
    c = oracle.assemble(X, X, Hyper(2.0, 1.0, 0.1, False), True)
    d = oracle.assemble(X, X, Hyper(2.0, 1.0, 0.1, True), True)
    assert not np.allclose(c, d)
    np.testing.assert_allclose(c, oracle.assemble(X / math.sqrt(2.0), X / math.sqrt(2.0), Hyper(1.0, 1.0, 0.1), True), rtol=1e-13)
    np.testing.assert_allclose(d, oracle.assemble(X / 2.0, X / 2.0, Hyper(1.0, 1.0, 0.1), True), rtol=1e-13)


def test_oracle_thread_count_does_not_change_results():
    cfg = nfir.CONFIGS[0]
    X, y, Xs = nfir.make_inputs(cfg)
    nt = oracle.num_threads()
    p = oracle.predict(X, y, Xs, Hyper())
    oracle.set_num_threads(1)
    try:
        q = oracle.predict(X, y, Xs, Hyper())
    finally:
        oracle.set_num_threads(nt)
    for a, b in ((p.L, q.L), (p.alpha, q.alpha), (p.mean, q.mean), (p.Sigma, q.Sigma)):
        assert np.array_equal(a, b)


# ---------------------------------------------------------------- SURVEY.md 8(f) rows 1 and 4
@pytest.mark.parametrize("name", ["A", "B", "Bprime_printed_2ell", "Bprime_ell_squared"])
def test_variance_and_lml_worked_examples_40_digits(golden, name):
    """diag(Sigma) and log p(y) against the 40-digit values the golden script derives from
    the DEFINITIONS (direct inverse, determinant), not from a Cholesky factor."""
    g = golden[name]
    h = Hyper(g["lengthscale"], g["vertical"], g["noise"], g["ell_squared"])
    X, y, Xs = np.array(g["X"]), np.array(g["y"]), np.array(g["Xs"])
    p = oracle.predict(X, y, Xs, h, full_cov=False, variance=True)
    assert p.Sigma is None
    np.testing.assert_allclose(p.var, _fv(g["var"]), rtol=1e-13, atol=1e-15)
    lml = oracle.log_marginal_likelihood(p.L, y, p.alpha)
    assert abs(lml - float(g["log_marginal_likelihood"])) <= 1e-13 * abs(float(g["log_marginal_likelihood"]))


def test_lml_single_point_closed_form():
    """n = 1: log N(y; 0, v + s2) = -y^2 / (2 (v + s2)) - log(v + s2) / 2 - log(2 pi) / 2."""
    for v, s2, yv in ((1.0, 0.1, 0.7), (2.5, 0.05, -1.3)):
        h = Hyper(1.0, v, s2)
        p = oracle.fit(np.array([[0.3, -0.2]]), np.array([yv]), h)
        want = -yv * yv / (2 * (v + s2)) - 0.5 * np.log(v + s2) - 0.5 * np.log(2 * np.pi)
        assert abs(oracle.log_marginal_likelihood(p.L, np.array([yv]), p.alpha) - want) <= 1e-15 * max(1.0, abs(want))


@pytest.mark.parametrize("n,m,D,seed", [(3, 2, 1, 0), (16, 9, 3, 1), (64, 40, 8, 2)])
def test_variance_and_lml_brute_force_and_scipy(n, m, D, seed):
    from scipy.stats import multivariate_normal
    X, y = nfir.nfir_features(seed, n, D)
    Xs, _ = nfir.nfir_features(seed + 50, m, D, with_targets=False)
    for h in (Hyper(), Hyper(2.0, 1.0, 0.05), Hyper(2.0, 1.7, 0.05, True)):
        p = oracle.predict(X, y, Xs, h, full_cov=True, variance=True)
        K = se_kernel_numpy(X, X, h.lengthscale, h.vertical, h.ell_squared) + h.noise * np.eye(n)
        Kxs = se_kernel_numpy(Xs, X, h.lengthscale, h.vertical, h.ell_squared)
        Kinv = gauss_jordan_inverse(K)
        # variance: the diagonal of Eq. 3 by brute force; prior variance is v
        want = h.vertical - np.einsum("ai,ij,aj->a", Kxs, Kinv, Kxs)
        assert relerr(p.var, want) <= 1e-11
        assert np.all(p.var >= 0.0) and np.all(p.var <= h.vertical)
        np.testing.assert_allclose(p.var, np.diag(p.Sigma), rtol=1e-12, atol=1e-15)
        # log marginal likelihood: the library's multivariate normal density
        lml = oracle.log_marginal_likelihood(p.L, y, p.alpha)
        ref = multivariate_normal(mean=np.zeros(n), cov=K).logpdf(y)
        assert abs(lml - ref) <= 1e-10 * abs(ref)


def test_lml_scaling_law():
    """(v, s2, y) -> (c v, c s2, sqrt(c) y) leaves the quadratic term unchanged and adds -n/2 log c."""
    X, y = nfir.nfir_features(5, 48, 4)
    c = 3.7
    p1 = oracle.fit(X, y, Hyper(1.0, 1.0, 0.1))
    p2 = oracle.fit(X, np.sqrt(c) * y, Hyper(1.0, c * 1.0, c * 0.1))
    l1 = oracle.log_marginal_likelihood(p1.L, y, p1.alpha)
    l2 = oracle.log_marginal_likelihood(p2.L, np.sqrt(c) * y, p2.alpha)
    assert abs(l2 - (l1 - 0.5 * 48 * np.log(c))) <= 1e-11 * abs(l1)
