"""CPU ORACLE for the planner's neural surrogate -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md P:362-407: z = (x - mu)/sigma componentwise; f_theta(x) = tanh(z W1 + b1) W2 + b2 (Eq. 24);
t_NN = exp(f_theta(x)) (Eq. 25); L(theta) = (1/N) sum_i [f_theta(x_i) - log t_i]^2 (Eq. 26).
Written out with numpy matrix products, nothing else; the gradient is NOT coded here - tests take it by central
differences of `loss`, which pins the library's analytic gradient.  Parameter layout (shared by definition with
include/mfh.h): theta = [mu (F) | sigma (F) | W1 (F x H, row-major) | b1 (H) | W2 (H) | b2].
"""
from __future__ import annotations

import numpy as np


def unpack(theta, F: int, H: int):
    th = np.asarray(theta, dtype=np.float64)
    assert th.size == 2 * F + F * H + 2 * H + 1
    o = 0
    mu = th[o:o + F]; o += F
    sigma = th[o:o + F]; o += F
    W1 = th[o:o + F * H].reshape(F, H); o += F * H
    b1 = th[o:o + H]; o += H
    W2 = th[o:o + H]; o += H
    return mu, sigma, W1, b1, W2, th[o]


def f_theta(theta, F: int, H: int, X) -> np.ndarray:
    mu, sigma, W1, b1, W2, b2 = unpack(theta, F, H)
    z = (np.asarray(X, dtype=np.float64).reshape(-1, F) - mu) / sigma
    return np.tanh(z @ W1 + b1) @ W2 + b2                      # Eq. 24


def predict(theta, F: int, H: int, X) -> np.ndarray:
    return np.exp(f_theta(theta, F, H, X))                     # Eq. 25


def loss(theta, F: int, H: int, X, t_seconds) -> float:
    r = f_theta(theta, F, H, X) - np.log(np.asarray(t_seconds, dtype=np.float64))
    return float(np.mean(r * r))                               # Eq. 26
