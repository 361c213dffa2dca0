"""Pins for oracle/adamw.py: the closed form of the first step and torch.optim.AdamW (float64)
as a library witness for later steps.  PAPER.md:272 fixes beta1 0.9, beta2 0.95, eps 1e-8, wd 0.1."""
import numpy as np
import torch

from oracle import adamw


def test_hyperparameters_are_the_papers():
    assert (adamw.BETA1, adamw.BETA2, adamw.EPS, adamw.WEIGHT_DECAY) == (0.9, 0.95, 1e-8, 0.1)


def test_first_step_closed_form():
    """t=1: mhat = g, vhat = g^2  =>  theta1 = theta0 (1 - lr wd) - lr g / (|g| + eps)."""
    rng = np.random.default_rng(0)
    th0 = rng.standard_normal(50)
    G = rng.standard_normal(50) * 4.0
    k, lr = 4, 1e-3
    for decay in (True, False):
        th, m, v = th0.copy(), np.zeros(50), np.zeros(50)
        adamw.adamw_update(th, m, v, G, k, 1, lr, decay)
        g = G / k
        ref = th0 * ((1 - lr * 0.1) if decay else 1.0) - lr * g / (np.abs(g) + 1e-8)
        assert np.allclose(th, ref, rtol=0, atol=1e-15)


def test_matches_torch_adamw_over_several_steps():
    rng = np.random.default_rng(1)
    th0 = rng.standard_normal((7, 5))
    for decay in (True, False):
        th, m, v = th0.copy(), np.zeros_like(th0), np.zeros_like(th0)
        p = torch.tensor(th0, dtype=torch.float64, requires_grad=True)
        opt = torch.optim.AdamW([p], lr=3e-3, betas=(0.9, 0.95), eps=1e-8,
                                weight_decay=0.1 if decay else 0.0)
        for t in range(1, 8):
            G = rng.standard_normal(th0.shape)
            adamw.adamw_update(th, m, v, G, 2, t, 3e-3, decay)
            p.grad = torch.tensor(G / 2)
            opt.step()
            assert np.allclose(th, p.detach().numpy(), rtol=1e-12, atol=1e-14), (decay, t)


def test_which_tensors_decay():
    """P:272 "no decay on bias and LayerNorm/embedding"; R8."""
    yes = ["h.0.attn.wqkv", "h.3.attn.wo", "h.1.mlp.w1", "h.1.mlp.w2"]
    no = ["wte", "wpe", "head.w", "lnf.g", "lnf.b", "h.0.ln1.g", "h.0.ln2.b", "h.0.attn.bqkv",
          "h.0.attn.bo", "h.2.mlp.b1", "h.2.mlp.b2"]
    assert all(adamw.decays(n) for n in yes) and not any(adamw.decays(n) for n in no)


def test_stage_optimizer_window_semantics():
    """Alg. 1 lines 13-19: G is the raw sum, the update fires only when c == k, then G, c reset;
    a tail window (< k backwards) leaves G in place and does not update (R6)."""
    opt = adamw.StageOptimizer({"h.0.mlp.w1": np.ones((2, 2), np.float32)}, k=3)
    for i in range(2):
        opt.accumulate({"h.0.mlp.w1": np.full((2, 2), 1.0 + i)})
        assert not opt.maybe_step(1e-2) and opt.version == 0
    assert np.all(opt.G["h.0.mlp.w1"] == 3.0) and opt.c == 2
    opt.accumulate({"h.0.mlp.w1": np.full((2, 2), 3.0)})
    assert opt.maybe_step(1e-2) and opt.version == 1 and opt.c == 0
    assert np.all(opt.G["h.0.mlp.w1"] == 0.0)
    g = 6.0 / 3
    assert np.allclose(opt.theta["h.0.mlp.w1"], 1.0 * (1 - 1e-2 * 0.1) - 1e-2 * g / (g + 1e-8))
