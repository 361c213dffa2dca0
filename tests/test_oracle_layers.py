"""Pins for oracle/model.py that do not come from the oracle itself:
central finite differences, closed forms / textbook invariants, and a library witness
(torch float64 ops + autograd) for the consistent-weights special case.  SURVEY.md 8(c-5)."""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

import synth
from oracle import model



def _spec(stage_index=0, n_stages=1, n_layers=1, D=16, H=4, T=8, mu=2, V=32):
    return model.StageSpec(stage_index, n_stages, n_layers, D, H, T, mu, V)


def _params(spec, seed=3, perturbed=True):
    p = synth.stage_params(seed, spec.stage_index, spec.n_stages, spec.n_layers, spec.d_model, spec.vocab,
                           spec.seq_len, perturbed=perturbed)
    # larger weights than N(0,0.02) so that every path has a gradient well above FD noise
    return {n: np.asarray(a, np.float64) * (5.0 if a.ndim == 2 else 1.0) for n, a in p.items()}


def _fd(fun, x, h=1e-5, n_probe=12, rng=None):
    """central differences of scalar fun at a few random coordinates of x (modified in place)."""
    rng = rng or np.random.default_rng(0)
    flat = x.reshape(-1)
    idx = rng.choice(flat.size, size=min(n_probe, flat.size), replace=False)
    out = []
    for i in idx:
        old = flat[i]
        flat[i] = old + h
        fp = fun()
        flat[i] = old - h
        fm = fun()
        flat[i] = old
        out.append((fp - fm) / (2 * h))
    return idx, np.array(out)


# ------------------------------------------------------------------ finite differences, whole stage

@pytest.mark.parametrize("stage_index,n_stages", [(0, 1), (0, 2), (1, 2), (1, 3)])
def test_stage_backward_matches_finite_differences(stage_index, n_stages):
    spec = _spec(stage_index, n_stages)
    P = _params(spec)
    rng = np.random.default_rng(7)
    tok = synth.tokens(5, 1, spec.micro_batch, spec.seq_len, spec.vocab, "uniform")[0]
    tgt = tok[:, 1:].astype(np.int64)
    inp = tok[:, :-1].astype(np.int64) if spec.has_embedding else rng.standard_normal(
        (spec.micro_batch, spec.seq_len, spec.d_model))
    r = rng.standard_normal((spec.micro_batch, spec.seq_len, spec.d_model))  # random cotangent

    def scalar():
        out, _ = model.stage_forward(spec, P, inp, tgt)
        return out if spec.has_head else float((out * r).sum())

    out, stash = model.stage_forward(spec, P, inp, tgt)
    din, grads = model.stage_backward(spec, P, stash, None if spec.has_head else r)
    assert set(grads) == set(P)
    for name in P:
        idx, fd = _fd(scalar, P[name], rng=rng)
        an = grads[name].reshape(-1)[idx]
        assert np.allclose(an, fd, rtol=2e-6, atol=1e-9), (name, an, fd)
    if not spec.has_embedding:
        idx, fd = _fd(scalar, inp, rng=rng)
        assert np.allclose(din.reshape(-1)[idx], fd, rtol=2e-6, atol=1e-9)
    else:
        assert din is None


# ------------------------------------------------------------------ library witness (torch autograd)

def _torch_stage(spec, P, inp, tgt):
    """The same model written with torch library ops only (F.layer_norm, F.linear,
    F.scaled_dot_product_attention, F.gelu(tanh), F.cross_entropy)."""
    D, H = spec.d_model, spec.n_heads
    if spec.has_embedding:
        x = P["wte"][inp] + P["wpe"][None, :inp.shape[1]]
    else:
        x = inp
    for l in range(spec.n_layers):
        p = f"h.{l}."
        y = F.layer_norm(x, (D,), P[p + "ln1.g"], P[p + "ln1.b"], eps=1e-5)
        qkv = F.linear(y, P[p + "attn.wqkv"], P[p + "attn.bqkv"])
        B, T, _ = qkv.shape
        q, k, v = (t.reshape(B, T, H, D // H).transpose(1, 2) for t in qkv.split(D, dim=-1))
        o = F.scaled_dot_product_attention(q, k, v, is_causal=True).transpose(1, 2).reshape(B, T, D)
        x = x + F.linear(o, P[p + "attn.wo"], P[p + "attn.bo"])
        y = F.layer_norm(x, (D,), P[p + "ln2.g"], P[p + "ln2.b"], eps=1e-5)
        x = x + F.linear(F.gelu(F.linear(y, P[p + "mlp.w1"], P[p + "mlp.b1"]), approximate="tanh"),
                         P[p + "mlp.w2"], P[p + "mlp.b2"])
    if not spec.has_head:
        return x
    z = F.linear(F.layer_norm(x, (D,), P["lnf.g"], P["lnf.b"], eps=1e-5), P[spec.head_name()])
    return F.cross_entropy(z.reshape(-1, spec.vocab), tgt.reshape(-1))


@pytest.mark.parametrize("stage_index,n_stages,n_layers", [(0, 1, 2), (1, 3, 2), (2, 3, 1)])
def test_stage_matches_torch_autograd(stage_index, n_stages, n_layers):
    spec = _spec(stage_index, n_stages, n_layers=n_layers, D=32, H=4, T=16, mu=3, V=50)
    P = _params(spec)
    rng = np.random.default_rng(11)
    tok = synth.tokens(9, 1, spec.micro_batch, spec.seq_len, spec.vocab, "zipf")[0]
    tgt = tok[:, 1:].astype(np.int64)
    inp = tok[:, :-1].astype(np.int64) if spec.has_embedding else rng.standard_normal(
        (spec.micro_batch, spec.seq_len, spec.d_model))
    r = rng.standard_normal((spec.micro_batch, spec.seq_len, spec.d_model))
    out, stash = model.stage_forward(spec, P, inp, tgt)
    din, grads = model.stage_backward(spec, P, stash, None if spec.has_head else r)

    Pt = {n: torch.tensor(a, requires_grad=True) for n, a in P.items()}
    it = torch.tensor(inp) if spec.has_embedding else torch.tensor(inp, requires_grad=True)
    ot = _torch_stage(spec, Pt, it, torch.tensor(tgt))
    if spec.has_head:
        assert abs(out - ot.item()) < 1e-12
        ot.backward()
    else:
        assert np.allclose(out, ot.detach().numpy(), rtol=1e-12, atol=1e-12)
        ot.backward(torch.tensor(r))
    for n in P:
        assert np.allclose(grads[n], Pt[n].grad.numpy(), rtol=1e-9, atol=1e-12), n
    if not spec.has_embedding:
        assert np.allclose(din, it.grad.numpy(), rtol=1e-9, atol=1e-12)


# ------------------------------------------------------------------ textbook invariants

def test_layernorm_rows_have_mean_beta_var_gamma2():
    rng = np.random.default_rng(0)
    x = rng.standard_normal((5, 7, 64)) * 3 + 1
    y, _ = model.layernorm_fwd(x, np.full(64, 2.0), np.full(64, 0.5))
    assert np.allclose(y.mean(-1), 0.5, atol=1e-12)
    assert np.allclose(y.var(-1), 4.0, rtol=1e-4)       # eps=1e-5 keeps it a hair under gamma^2
    assert np.all(y.var(-1) < 4.0)


def test_attention_causality_and_T1_and_rowsum():
    rng = np.random.default_rng(1)
    qkv = rng.standard_normal((2, 9, 3 * 24))
    o, (q, k, v, P) = model.attention_fwd(qkv, 4)
    assert np.allclose(P.sum(-1), 1.0)
    assert np.all(np.triu(P[0, 0], 1) == 0.0)
    qkv2 = qkv.copy()
    qkv2[:, 6:] += rng.standard_normal(qkv2[:, 6:].shape)   # change the future only
    o2, _ = model.attention_fwd(qkv2, 4)
    assert np.array_equal(o[:, :6], o2[:, :6])
    o1, _ = model.attention_fwd(qkv[:, :1], 4)               # T=1: softmax of one score is 1 -> o = v
    assert np.allclose(o1, qkv[:, :1, 48:])


def test_attention_head_packing_is_q_k_v_rows_with_contiguous_heads():
    """DESIGN.md R17: qkv = [q | k | v], head h = columns h*dh .. (h+1)*dh-1.  Pin: make only head 1
    of v non-zero -> only head 1's output columns are non-zero."""
    rng = np.random.default_rng(2)
    D, H, dh = 24, 4, 6
    qkv = rng.standard_normal((1, 5, 3 * D))
    qkv[..., 2 * D:] = 0.0
    qkv[..., 2 * D + dh:2 * D + 2 * dh] = 1.0
    o, _ = model.attention_fwd(qkv, H)
    assert np.allclose(o[..., dh:2 * dh], 1.0) and np.count_nonzero(o) == 5 * dh


def test_gelu_matches_library_tanh_form_and_limits():
    x = np.linspace(-6, 6, 1001)
    assert np.allclose(model.gelu_fwd(x), F.gelu(torch.tensor(x), approximate="tanh").numpy(), atol=1e-14)
    assert model.gelu_fwd(np.array(0.0)) == 0.0
    assert abs(model.gelu_fwd(np.array(10.0)) - 10.0) < 1e-12
    # within 1e-3 of the exact erf form everywhere (the tanh form is an approximation of it)
    assert np.max(np.abs(model.gelu_fwd(x) - F.gelu(torch.tensor(x)).numpy())) < 1e-3
    xt = torch.tensor(x, requires_grad=True)
    F.gelu(xt, approximate="tanh").sum().backward()
    assert np.allclose(model.gelu_bwd(np.ones_like(x), x), xt.grad.numpy(), atol=1e-13)


def test_cross_entropy_closed_forms():
    V, M = 37, 10
    z = np.zeros((1, M, V))
    tgt = np.arange(M)[None] % V
    loss, dz = model.cross_entropy_fwd_bwd(z, tgt)
    assert abs(loss - np.log(V)) < 1e-14                      # uniform logits -> ln V
    assert np.allclose(dz.sum(-1), 0.0, atol=1e-16)           # softmax - onehot sums to 0
    assert np.allclose(dz[0, 0, 0], (1.0 / V - 1.0) / M)
    z[0, :, :] = -50.0
    z[0, np.arange(M), tgt[0]] = 50.0                         # confident and right -> ~0 loss
    loss, _ = model.cross_entropy_fwd_bwd(z, tgt)
    assert loss < 1e-40 or loss == 0.0


def test_initial_loss_is_about_ln_vocab():
    """at N(0,0.02) init the loss is ln V plus about D*0.02^2/2... a small positive term."""
    spec = _spec(0, 1, n_layers=1, D=64, H=4, T=32, mu=2, V=256)
    P = {n: np.asarray(a, np.float64) for n, a in synth.stage_params(1, 0, 1, 1, 64, 256, 32).items()}
    tok = synth.tokens(1, 1, 2, 32, 256, "uniform")[0]
    loss, _ = model.stage_forward(spec, P, tok[:, :-1].astype(np.int64), tok[:, 1:].astype(np.int64))
    assert abs(loss - np.log(256)) < 0.05 and abs(np.log(256) - 5.545) < 1e-3


def test_embedding_scatter_add_brute_force():
    rng = np.random.default_rng(4)
    tok = np.array([[1, 1, 3], [3, 1, 0]])
    dx = rng.standard_normal((2, 3, 5))
    dwte, dwpe = model.embed_bwd(dx, tok, 6)
    ref = np.zeros((6, 5))
    for b in range(2):
        for t in range(3):
            ref[tok[b, t]] += dx[b, t]
    assert np.allclose(dwte, ref) and np.allclose(dwpe, dx[0] + dx[1])
    assert np.all(dwte[[2, 4, 5]] == 0)
