"""Seeded synthetic NFIR-shaped inputs and the BASELINE.json configurations.

This module holds NONE of the method's arithmetic.  It is the one piece shared by the
oracle-side tests and the CUDA-side harness: arrays are generated once here and the same
bytes are handed to both sides.  It stands in for the paper's mass-spring-damper simulator
data, which is not available; recipe from BASELINE.json `configs`
(DESIGN.md "Input recipe").
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    index: int
    n: int          # training points
    m: int          # test points (n-hat in the paper)
    D: int          # regressors (lags)
    tile: int       # tile size t (tiles per dimension M = n / t)
    lengthscale: float = 1.0
    vertical: float = 1.0
    noise: float = 0.1

    @property
    def name(self) -> str:
        return f"c{self.index}: n={self.n} m={self.m} D={self.D} tile={self.tile}"


# BASELINE.json configs 0..4. Config 2 is swept over tiles 256/512/1024; 512 is its default.
CONFIGS = (
    Config(0, 128, 128, 8, 32),
    Config(1, 1024, 1024, 8, 256),
    Config(2, 8192, 1024, 8, 512),
    Config(3, 32768, 4096, 8, 1024),
    Config(4, 65536, 8192, 16, 2048, lengthscale=2.0, vertical=1.0, noise=0.05),
)


def nfir_features(seed: int, n: int, D: int, with_targets: bool = True):
    """Force sequence u_t ~ U[-1,1], t = -(D-1)..n-1; x_i = (u_i, u_{i-1}, .., u_{i-D+1});
    y_i = sin(2 * sum_k 0.5^k u_{i-k}) + 0.3 * u_{i-1}^3 + eps_i, eps_i ~ N(0, 0.1^2).
    Draw order: all of u, then all of eps, from numpy default_rng(seed).
    Returns (X [n, D] float64 row-major, y [n] float64 or None)."""
    rng = np.random.default_rng(seed)
    u = rng.uniform(-1.0, 1.0, size=n + D - 1)
    idx = (D - 1) + np.arange(n)[:, None] - np.arange(D)[None, :]   # u index of lag k for point i
    X = np.ascontiguousarray(u[idx], dtype=np.float64)
    if not with_targets:
        return X, None
    eps = rng.normal(0.0, 0.1, size=n)
    w = 0.5 ** np.arange(D)
    lag1 = X[:, 1] if D > 1 else np.zeros(n)
    y = np.sin(2.0 * (X @ w)) + 0.3 * lag1 ** 3 + eps
    return X, np.ascontiguousarray(y, dtype=np.float64)


def make_inputs(cfg: Config, n: int | None = None, m: int | None = None):
    """(X, y, Xs) for a config; train seed 1000+c, test seed 2000+c. n/m may be overridden
    (leading-block parity, bounded CPU-baseline samples): the generator is prefix-stable in n
    for X (same u draws) but y's noise draws follow the u draws, so a prefix run is its own
    problem instance; tests that need a true prefix slice the arrays instead."""
    n = cfg.n if n is None else n
    m = cfg.m if m is None else m
    X, y = nfir_features(1000 + cfg.index, n, cfg.D, with_targets=True)
    Xs, _ = nfir_features(2000 + cfg.index, m, cfg.D, with_targets=False)
    return X, y, Xs
