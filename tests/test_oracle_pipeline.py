"""Pins for oracle/pipeline.py (the S-stage run): the reductions the paper fixes and a library
witness for the drift case itself.  SURVEY.md 8(c-5), BASELINE.json north_star invariants."""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

import synth
from oracle import model, pipeline
from test_oracle_layers import _torch_stage


CFG = dict(D=32, H=4, T=16, mu=2, V=64)


def _build(S, L, seed=2, perturbed=True, **kw):
    c = dict(CFG, **kw)
    specs = [model.StageSpec(s, S, L, c["D"], c["H"], c["T"], c["mu"], c["V"]) for s in range(S)]
    params = [synth.stage_params(seed, s, S, L, c["D"], c["V"], c["T"], perturbed=perturbed) for s in range(S)]
    return specs, params, c


def _tok(n, c, seed=4):
    return synth.tokens(seed, n, c["mu"], c["T"], c["V"], "zipf")


def test_single_stage_is_plain_k_step_gradient_accumulation():
    """Eq. 10 with i = N: delta == 0, and PACI on one stage is ordinary accumulation: every k
    micro-batches one AdamW step on the mean gradient.  Witness: torch autograd + torch.optim.AdamW."""
    specs, params, c = _build(1, 2)
    k, n, lr = 3, 6, 1e-2
    tok = _tok(n, c)
    r = pipeline.run_pipeline(specs, params, tok, k, lr)
    assert r["delta"] == [[0] * n] and r["version"] == [2]

    Pt = {nm: torch.tensor(np.asarray(a, np.float64), requires_grad=True) for nm, a in params[0].items()}
    from oracle.adamw import decays
    opt = torch.optim.AdamW([{"params": [Pt[nm] for nm in Pt if decays(nm)], "weight_decay": 0.1},
                             {"params": [Pt[nm] for nm in Pt if not decays(nm)], "weight_decay": 0.0}],
                            lr=lr, betas=(0.9, 0.95), eps=1e-8)
    losses = []
    for m in range(n):
        t = torch.tensor(tok[m].astype(np.int64))
        loss = _torch_stage(specs[0], Pt, t[:, :-1], t[:, 1:])
        losses.append(loss.item())
        (loss / k).backward()
        if (m + 1) % k == 0:
            opt.step()
            opt.zero_grad()
    assert np.allclose(r["losses"], losses, rtol=1e-10)
    for nm in Pt:
        assert np.allclose(r["opt"][0].theta[nm], Pt[nm].detach().numpy(), rtol=1e-8, atol=1e-11), nm


@pytest.mark.parametrize("S", [2, 3])
def test_one_window_equals_flush_bit_for_bit(S):
    """When no update falls between any forward and its backward (exactly k micro-batches),
    PACI == synchronous 1F1B-flush with m_f = k (BASELINE.json invariant)."""
    specs, params, c = _build(S, 1)
    tok = _tok(4, c)
    a = pipeline.run_pipeline(specs, params, tok, 4, 1e-2)
    b = pipeline.run_pipeline(specs, params, tok, None, 1e-2, mode="flush", m_f=4)
    assert all(d == 0 for row in a["delta"] for d in row)
    assert a["losses"] == b["losses"]
    for s in range(S):
        for nm in a["opt"][s].theta:
            assert np.array_equal(a["opt"][s].theta[nm], b["opt"][s].theta[nm])


def test_flush_is_independent_of_micro_batching():
    """"varying the number of micro-batches affects throughput but not the sequence of
    global optimizer updates".  m_f micro-batches of mu vs one micro-batch of m_f*mu."""
    S, L, m_f = 2, 1, 4
    specs, params, c = _build(S, L)
    tok = _tok(m_f, c)
    a = pipeline.run_pipeline(specs, params, tok, None, 1e-2, mode="flush", m_f=m_f)
    specs_big, _, _ = _build(S, L, mu=c["mu"] * m_f)
    big = tok.reshape(1, m_f * c["mu"], c["T"] + 1)
    b = pipeline.run_pipeline(specs_big, params, big, None, 1e-2, mode="flush", m_f=1)
    assert abs(np.mean(a["losses"]) - b["losses"][0]) < 1e-12
    for s in range(S):
        for nm in a["opt"][s].theta:
            assert np.allclose(a["opt"][s].theta[nm], b["opt"][s].theta[nm], rtol=1e-7, atol=1e-10), nm


def test_drift_case_matches_torch_backward_after_inplace_update():
    """The drift case itself (Eq. 1).  Library witness = what the paper's PyTorch patch
    enables (D.6): run torch's forward, overwrite the parameters in place, then run
    torch's backward -- autograd differentiates the saved (old) activations with the current weights."""
    spec = model.StageSpec(1, 3, 2, 32, 4, 16, 2, 64)          # interior stage
    P0 = {n: np.asarray(a, np.float64) for n, a in synth.stage_params(5, 1, 3, 2, 32, 64, 16, True).items()}
    rng = np.random.default_rng(3)
    P1 = {n: a + 0.05 * rng.standard_normal(a.shape) for n, a in P0.items()}   # "after Delta updates"
    x = rng.standard_normal((2, 16, 32))
    r = rng.standard_normal((2, 16, 32))
    out, stash = model.stage_forward(spec, P0, x)
    din, grads = model.stage_backward(spec, P1, stash, r)

    Pt = {n: torch.tensor(a, requires_grad=True) for n, a in P0.items()}
    xt = torch.tensor(x, requires_grad=True)
    ot = _torch_stage(spec, Pt, xt, None)
    with torch.no_grad():
        for n in Pt:
            Pt[n].data.copy_(torch.tensor(P1[n]))                # bypasses the version counter
    ot.backward(torch.tensor(r))
    assert np.allclose(din, xt.grad.numpy(), rtol=1e-9, atol=1e-12)
    for n in P0:
        assert np.allclose(grads[n], Pt[n].grad.numpy(), rtol=1e-9, atol=1e-12), n
    # and it is a different computation from the consistent one
    _, g_cons = model.stage_backward(spec, P0, stash, r)
    assert not np.allclose(g_cons["h.0.mlp.w1"], grads["h.0.mlp.w1"], rtol=1e-3)


def test_drift_case_linear_toy_closed_form():
    """F(h) = W h: wgrad = delta h_stash^T (no weights at all), grad h = W_current^T delta."""
    rng = np.random.default_rng(0)
    W_old, W_new = rng.standard_normal((5, 4)), rng.standard_normal((5, 4))
    h, delta = rng.standard_normal((3, 4)), rng.standard_normal((3, 5))
    y, st = model.linear_fwd(h, W_old, None)
    dh, dW, _ = model.linear_bwd(delta, st, W_new)
    assert np.allclose(y, h @ W_old.T)
    assert np.allclose(dW, sum(np.outer(delta[i], h[i]) for i in range(3)))
    assert np.allclose(dh, np.stack([W_new.T @ delta[i] for i in range(3)]))


def test_two_stage_paci_crosses_updates_and_differs_from_flush():
    """cfg-1-like run: S=2, k=4, 16 micro-batches -> stage 0 crosses one update at m=4,8,12 (SURVEY
    8(c-5)); the trajectory then differs from flush, the last stage's first window does not."""
    specs, params, c = _build(2, 1)
    tok = _tok(16, c)
    a = pipeline.run_pipeline(specs, params, tok, 4, 1e-2)
    b = pipeline.run_pipeline(specs, params, tok, None, 1e-2, mode="flush", m_f=4)
    assert a["delta"][0] == [1 if m in (4, 8, 12) else 0 for m in range(16)]
    assert a["version"] == [4, 4] and b["version"] == [4, 4]
    assert a["losses"][:4] == b["losses"][:4]
    # m=4: PACI's stage 0 forwards it BEFORE its first update (F4 precedes U1), flush after it
    assert a["losses"][4] != b["losses"][4]
    # m=5..7: both schedules forward under version 1 on both stages, and update 1 saw identical
    # gradients (first window never crosses) -> identical losses; update 2 contains m=4's drifted
    # gradient, so from m=9 on the trajectories differ.
    assert a["losses"][5:8] == b["losses"][5:8]
    assert a["losses"][9] != b["losses"][9]
    assert all(np.isfinite(a["losses"]))
