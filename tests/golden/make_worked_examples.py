"""Writes tests/golden/worked_examples.json: the hand-sized GP examples A, B, B' of
SURVEY.md section 8(c)(i), evaluated at 40 decimal digits with mpmath straight from the
paper's definitions -- Eq. 1, Eq. 2, Eq. 3, with
the DIRECT INVERSE K^-1 (mpmath), plus L from the textbook recurrence --
and cross-checked here between the inverse route and the Cholesky route to 1e-35.

It calls neither oracle/ nor the CUDA path: these are independent expected values.
Run:  python tests/golden/make_worked_examples.py
"""
import json
import os

from mpmath import mp, mpf, exp, sqrt, matrix, inverse, det, log, pi

mp.dps = 40


def kern(a, b, ell, v, ell_squared):
    r2 = sum((mpf(x) - mpf(y)) ** 2 for x, y in zip(a, b))
    den = 2 * mpf(ell) ** 2 if ell_squared else 2 * mpf(ell)
    return mpf(v) * exp(-r2 / den)


def example(X, y, Xs, ell, v, noise, ell_squared):
    n, m = len(X), len(Xs)
    K = matrix(n, n)
    for i in range(n):
        for j in range(n):
            K[i, j] = kern(X[i], X[j], ell, v, ell_squared) + (mpf(noise) if i == j else 0)
    Kxs = matrix(m, n)          # K_{X^,X}
    for a in range(m):
        for i in range(n):
            Kxs[a, i] = kern(Xs[a], X[i], ell, v, ell_squared)
    Kss = matrix(m, m)
    for a in range(m):
        for b in range(m):
            Kss[a, b] = kern(Xs[a], Xs[b], ell, v, ell_squared)
    yv = matrix([mpf(t) for t in y])
    # inverse route (Eq. 2, Eq. 3 literally)
    Kinv = inverse(K)
    alpha_inv = Kinv * yv
    mean_inv = Kxs * Kinv * yv
    Sigma_inv = Kss - Kxs * Kinv * Kxs.T
    # Cholesky route
    L = matrix(n, n)
    for j in range(n):
        s = K[j, j] - sum(L[j, p] ** 2 for p in range(j))
        L[j, j] = sqrt(s)
        for i in range(j + 1, n):
            L[i, j] = (K[i, j] - sum(L[i, p] * L[j, p] for p in range(j))) / L[j, j]
    beta = matrix(n, 1)
    for i in range(n):
        beta[i] = (yv[i] - sum(L[i, p] * beta[p] for p in range(i))) / L[i, i]
    alpha = matrix(n, 1)
    for i in reversed(range(n)):
        alpha[i] = (beta[i] - sum(L[p, i] * alpha[p] for p in range(i + 1, n))) / L[i, i]
    V = matrix(n, m)
    for c in range(m):
        for i in range(n):
            V[i, c] = (Kxs[c, i] - sum(L[i, p] * V[p, c] for p in range(i))) / L[i, i]
    mean = Kxs * alpha
    Sigma = Kss - V.T * V
    # log marginal likelihood of y ~ N(0, K) from the density itself (determinant and inverse), and its
    # Cholesky form
    lml_def = -(yv.T * Kinv * yv)[0] / 2 - log(det(K)) / 2 - mpf(n) / 2 * log(2 * pi)
    lml = -(yv.T * alpha)[0] / 2 - sum(log(L[i, i]) for i in range(n)) - mpf(n) / 2 * log(2 * pi)
    tol = mpf(10) ** -35
    assert abs(lml - lml_def) < tol
    assert max(abs(alpha[i] - alpha_inv[i]) for i in range(n)) < tol
    assert max(abs(mean[a] - mean_inv[a]) for a in range(m)) < tol
    assert max(abs(Sigma[a, b] - Sigma_inv[a, b]) for a in range(m) for b in range(m)) < tol

    def mat(M):
        return [[mp.nstr(M[i, j], 25) for j in range(M.cols)] for i in range(M.rows)]

    def vec(M):
        return [mp.nstr(M[i], 25) for i in range(M.rows)]

    return {"X": X, "y": y, "Xs": Xs, "lengthscale": ell, "vertical": v, "noise": noise,
            "ell_squared": bool(ell_squared), "K": mat(K), "L": mat(L), "beta": vec(beta),
            "alpha": vec(alpha), "K_X_Xs": mat(Kxs.T), "V": mat(V), "mean": vec(mean),
            "Sigma": mat(Sigma), "var": [mp.nstr(Sigma_inv[a, a], 25) for a in range(m)],
            "log_marginal_likelihood": mp.nstr(lml_def, 25)}


def main():
    XA, yA, XsA = [[0.0], [1.0]], [1.0, 2.0], [[0.5], [2.0]]
    XB, yB, XsB = [[0.0, 0.0], [1.0, 0.0], [0.0, 2.0]], [1.0, -1.0, 0.5], [[0.5, 0.5], [2.0, 2.0]]
    out = {
        "_citation": "SURVEY.md section 8(c)(i); definitions PAPER.md:63 (Eq.1), :70 (Eq.2), :76 (Eq.3), :72, :79",
        "_precision": "mpmath, 40 decimal digits, printed to 25",
        "A": example(XA, yA, XsA, 1.0, 1.0, 0.1, False),
        "B": example(XB, yB, XsB, 1.0, 1.0, 0.1, False),
        "Bprime_printed_2ell": example(XB, yB, XsB, 2.0, 1.0, 0.05, False),
        "Bprime_ell_squared": example(XB, yB, XsB, 2.0, 1.0, 0.05, True),
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "worked_examples.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    print("wrote", path)


if __name__ == "__main__":
    main()
