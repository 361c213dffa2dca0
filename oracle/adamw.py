"""ORACLE (test infrastructure): the stage-local optimizer update of Alg. 1 line 17.

AdamW with beta1 0.9, beta2 0.95, eps 1e-8, weight decay 0.1, "no decay on bias and
LayerNorm/embedding".  The paper only cites Loshchilov & Hutter; the exact form
below (decoupled decay multiplied by lr, bias correction, eps added after the
bias-corrected sqrt) is DESIGN.md reading R7; "which tensors decay" is reading R8; the
accumulated gradient G is the raw sum over the window and the update uses its mean G/k
(reading R5).
"""
from __future__ import annotations

import numpy as np

BETA1, BETA2, EPS, WEIGHT_DECAY = 0.9, 0.95, 1e-8, 0.1


def decays(name: str) -> bool:
    """Decay only the block matrices (Wqkv, Wo, W1, W2).  Biases, LN gain/bias, wte, wpe and
    the head copy of the embedding matrix do not decay (R8)."""
    return name.rsplit(".", 1)[-1] in ("wqkv", "wo", "w1", "w2")


def adamw_update(theta, m, v, G, k, t, lr, decay,
                 beta1=BETA1, beta2=BETA2, eps=EPS, weight_decay=WEIGHT_DECAY):
    """One update of one tensor, in place.  t = 1-based count of this stage's updates."""
    g = G / k
    if decay:
        theta *= (1.0 - lr * weight_decay)
    m *= beta1
    m += (1.0 - beta1) * g
    v *= beta2
    v += (1.0 - beta2) * g * g
    mhat = m / (1.0 - beta1 ** t)
    vhat = v / (1.0 - beta2 ** t)
    theta -= lr * mhat / (np.sqrt(vhat) + eps)


class StageOptimizer:
    """Per-stage state of Alg. 1: theta_i (one copy), G_i, c_i, and the local update index t."""

    def __init__(self, params: dict, k: int, **hyper):
        self.theta = {n: np.array(a, dtype=np.float64) for n, a in params.items()}
        self.m = {n: np.zeros_like(a) for n, a in self.theta.items()}
        self.v = {n: np.zeros_like(a) for n, a in self.theta.items()}
        self.G = {n: np.zeros_like(a) for n, a in self.theta.items()}
        self.k = k
        self.c = 0            # local backward counter c_i (Alg. 1 line 2)
        self.version = 0      # local update index t
        self.hyper = hyper

    def accumulate(self, grads: dict):
        """Alg. 1 line 13: G_i <- G_i + g_{m,i};  line 14-15: c_i <- c_i + 1."""
        for n, g in grads.items():
            self.G[n] += g
        self.c += 1

    def maybe_step(self, lr: float) -> bool:
        """Alg. 1 lines 16-19: if c_i = a, update theta_i with G_i, reset G_i and c_i."""
        if self.c != self.k:
            return False
        t = self.version + 1
        for n in self.theta:
            adamw_update(self.theta[n], self.m[n], self.v[n], self.G[n], self.k, t, lr, decays(n),
                         **self.hyper)
            self.G[n][...] = 0.0
        self.version = t
        self.c = 0
        return True
