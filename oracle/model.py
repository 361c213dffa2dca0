"""ORACLE (test infrastructure, not the product): fp64 CPU model of one PACI pipeline stage.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this package.  It shares no code with `paper_2606_07881_b200/`.

What it computes (citations are PAPER.md line numbers, `P:n`):

* a stage function F_i (Eq. 6-7): a stack of GPT-2 pre-LN decoder blocks
  (model "GPT-2 Medium"), optionally preceded by the token+position embedding
  (first stage) and followed by final-LN + LM head + mean token cross-entropy (last
  stage; "the final layer computes the loss and the embedding layer is ... grouped with
  following transformer blocks");
* its manual backward under the stale-activation / current-weight rule of Eq. 1 and
  P:282: "the backward pass differentiates activations produced by the original forward
  pass, but evaluates the gradient with respect to the current parameter version".
  So `stage_backward` takes (a) the *stash* written by `stage_forward` -- everything that
  depends on the forward-time weights -- and (b) the *current* parameters, which are used
  ONLY where the chain rule multiplies by theta: the W in every dgrad, and the LayerNorm gain.
  Weight gradients are products of the incoming delta with stashed activations only.

The paper fixes none of the architectural constants below; they are the readings listed
in DESIGN.md ("Readings", R11-R17): tanh-GELU, LN eps 1e-5 with biased variance, QKV packed
as rows [q; k; v] with head h = rows h*dh..(h+1)*dh-1, weights stored [out, in], dropout 0.

Everything is float64 numpy.  A library matmul (`@`) serves as the contraction step; there is
no blocking, fusion or reordering beyond the formulas written here.

Two optional extensions, both off by default so that everything above is unchanged:

* `drop=(p, seed, mb_id)`: dropout ("dropout to 0.1") on the embedding output and on the output of both
  residual branches of every block (R23), mask from `oracle.dropout` (a pure function of seed,
  micro-batch id, site and element index);
* `stage_backward_checkpointed`: activation-checkpointed PACI (App. B): "discarded activations can be
  recomputed during the backward pass using the stage's current parameter version ... With checkpointing, those
  activations are instead recomputed under the current parameter version before differentiation."
"""
from __future__ import annotations

import numpy as np

from . import dropout as _dropout

LN_EPS = 1e-5                      # DESIGN.md R13
GELU_C = np.sqrt(2.0 / np.pi)      # DESIGN.md R12 (tanh form)
GELU_A = 0.044715


# ----------------------------------------------------------------------------- layers

def embed_fwd(tok, wte, wpe):
    """x[b,t,:] = wte[tok[b,t]] + wpe[t]   (first stage)."""
    B, T = tok.shape
    return wte[tok] + wpe[np.arange(T)][None, :, :]


def embed_bwd(dx, tok, vocab):
    """G_wte[tok[b,t]] += dx[b,t]; G_wpe[t] += sum_b dx[b,t]."""
    B, T, D = dx.shape
    dwte = np.zeros((vocab, D))
    np.add.at(dwte, tok.reshape(-1), dx.reshape(-1, D))
    dwpe = dx.sum(axis=0)
    return dwte, dwpe


def layernorm_fwd(x, g, b):
    """y = (x - mean) * rstd * g + b over the last axis; biased variance; stash (xhat, rstd)."""
    mean = x.mean(axis=-1, keepdims=True)
    var = ((x - mean) ** 2).mean(axis=-1, keepdims=True)
    rstd = 1.0 / np.sqrt(var + LN_EPS)
    xhat = (x - mean) * rstd
    return xhat * g + b, (xhat, rstd)


def layernorm_bwd(dy, stash, g_current):
    """Chain rule of layernorm_fwd with stashed (xhat, rstd) and the CURRENT gain (Eq. 1)."""
    xhat, rstd = stash
    dxhat = dy * g_current
    dx = rstd * (dxhat - dxhat.mean(axis=-1, keepdims=True)
                 - xhat * (dxhat * xhat).mean(axis=-1, keepdims=True))
    D = dy.shape[-1]
    dg = (dy * xhat).reshape(-1, D).sum(axis=0)
    db = dy.reshape(-1, D).sum(axis=0)
    return dx, dg, db


def linear_fwd(x, W, b):
    """y = x W^T + b, W stored [out, in]; stash x."""
    y = x @ W.T
    if b is not None:
        y = y + b
    return y, x


def linear_bwd(dy, x_stash, W_current):
    """dx = dy W_current (Eq. 1: current weights);  dW = dy^T x_stash;  db = sum_rows dy."""
    dx = dy @ W_current
    dy2 = dy.reshape(-1, dy.shape[-1])
    dW = dy2.T @ x_stash.reshape(-1, x_stash.shape[-1])
    db = dy2.sum(axis=0)
    return dx, dW, db


def _split_heads(a, H):
    B, T, D = a.shape
    return a.reshape(B, T, H, D // H).transpose(0, 2, 1, 3)  # [B,H,T,dh]


def _merge_heads(a):
    B, H, T, dh = a.shape
    return a.transpose(0, 2, 1, 3).reshape(B, T, H * dh)


def attention_fwd(qkv, H):
    """o = merge_h softmax(causal(q_h k_h^T / sqrt(dh))) v_h;  qkv[..., :D|D:2D|2D:] = q|k|v."""
    B, T, D3 = qkv.shape
    D = D3 // 3
    dh = D // H
    q, k, v = (_split_heads(qkv[..., i * D:(i + 1) * D], H) for i in range(3))
    s = (q @ k.transpose(0, 1, 3, 2)) / np.sqrt(dh)
    mask = np.tril(np.ones((T, T), dtype=bool))
    s = np.where(mask, s, -np.inf)
    s = s - s.max(axis=-1, keepdims=True)
    P = np.exp(s)
    P = P / P.sum(axis=-1, keepdims=True)
    o = _merge_heads(P @ v)
    return o, (q, k, v, P)


def attention_bwd(do, stash):
    """No parameters: pure chain rule on the stashed q, k, v, P."""
    q, k, v, P = stash
    H, dh = q.shape[1], q.shape[3]
    doh = _split_heads(do, H)
    dv = P.transpose(0, 1, 3, 2) @ doh
    dP = doh @ v.transpose(0, 1, 3, 2)
    ds = P * (dP - (dP * P).sum(axis=-1, keepdims=True))
    dq = (ds @ k) / np.sqrt(dh)
    dk = (ds.transpose(0, 1, 3, 2) @ q) / np.sqrt(dh)
    return np.concatenate([_merge_heads(dq), _merge_heads(dk), _merge_heads(dv)], axis=-1)


def gelu_fwd(p):
    """tanh-GELU: 0.5 p (1 + tanh(c (p + a p^3)))."""
    return 0.5 * p * (1.0 + np.tanh(GELU_C * (p + GELU_A * p ** 3)))


def gelu_bwd(dg, p):
    th = np.tanh(GELU_C * (p + GELU_A * p ** 3))
    dgelu = 0.5 * (1.0 + th) + 0.5 * p * (1.0 - th ** 2) * GELU_C * (1.0 + 3.0 * GELU_A * p ** 2)
    return dg * dgelu


def cross_entropy_fwd_bwd(z, tgt):
    """loss = mean_{b,t} -log softmax(z[b,t])[tgt[b,t]];  dz = (softmax - onehot) / M."""
    V = z.shape[-1]
    z2 = z.reshape(-1, V)
    t2 = tgt.reshape(-1)
    M = z2.shape[0]
    zmax = z2.max(axis=-1, keepdims=True)
    e = np.exp(z2 - zmax)
    ssum = e.sum(axis=-1, keepdims=True)
    lse = np.log(ssum) + zmax
    loss = float((lse[:, 0] - z2[np.arange(M), t2]).mean())
    dz = e / ssum
    dz[np.arange(M), t2] -= 1.0
    dz /= M
    return loss, dz.reshape(z.shape)


# ----------------------------------------------------------------------------- block

def _mask(drop, shape, site):
    """drop = (p, seed, mb_id) or None -> multiplicative mask (1/(1-p) kept, 0 dropped) or None."""
    if drop is None or drop[0] <= 0.0:
        return None
    p, seed, mb_id = drop
    return _dropout.mask(shape, p, seed, mb_id, site)


def block_fwd(x, P, pre, H, drop=None, l=0):
    """x1 = x + drop(Attn(LN1(x)));  x2 = x1 + drop(MLP(LN2(x1)))   (drop = identity unless `drop` is given)."""
    y1, st_ln1 = layernorm_fwd(x, P[pre + "ln1.g"], P[pre + "ln1.b"])
    qkv, st_qkv = linear_fwd(y1, P[pre + "attn.wqkv"], P[pre + "attn.bqkv"])
    o, st_att = attention_fwd(qkv, H)
    a, st_o = linear_fwd(o, P[pre + "attn.wo"], P[pre + "attn.bo"])
    mask_a = _mask(drop, a.shape, _dropout.site_attn(l))
    if mask_a is not None:
        a = a * mask_a
    x1 = x + a
    y2, st_ln2 = layernorm_fwd(x1, P[pre + "ln2.g"], P[pre + "ln2.b"])
    p, st_w1 = linear_fwd(y2, P[pre + "mlp.w1"], P[pre + "mlp.b1"])
    g = gelu_fwd(p)
    m, st_w2 = linear_fwd(g, P[pre + "mlp.w2"], P[pre + "mlp.b2"])
    mask_m = _mask(drop, m.shape, _dropout.site_mlp(l))
    if mask_m is not None:
        m = m * mask_m
    x2 = x1 + m
    return x2, dict(ln1=st_ln1, qkv=st_qkv, att=st_att, o=st_o, ln2=st_ln2, w1=st_w1, p=p, w2=st_w2,
                    mask_a=mask_a, mask_m=mask_m)


def block_bwd(dx2, st, Pc, pre, grads):
    """Backward of block_fwd with stash `st` and CURRENT parameters `Pc`; adds into `grads`."""
    dm = dx2 if st.get("mask_m") is None else dx2 * st["mask_m"]          # grad wrt the MLP branch output
    dg, dW2, db2 = linear_bwd(dm, st["w2"], Pc[pre + "mlp.w2"])
    dp = gelu_bwd(dg, st["p"])
    dy2, dW1, db1 = linear_bwd(dp, st["w1"], Pc[pre + "mlp.w1"])
    dln2, dg2, dbt2 = layernorm_bwd(dy2, st["ln2"], Pc[pre + "ln2.g"])
    dx1 = dx2 + dln2
    da = dx1 if st.get("mask_a") is None else dx1 * st["mask_a"]          # grad wrt the attention branch output
    do, dWo, dbo = linear_bwd(da, st["o"], Pc[pre + "attn.wo"])
    dqkv = attention_bwd(do, st["att"])
    dy1, dWqkv, dbqkv = linear_bwd(dqkv, st["qkv"], Pc[pre + "attn.wqkv"])
    dln1, dg1, dbt1 = layernorm_bwd(dy1, st["ln1"], Pc[pre + "ln1.g"])
    dx = dx1 + dln1
    for name, val in (("mlp.w2", dW2), ("mlp.b2", db2), ("mlp.w1", dW1), ("mlp.b1", db1),
                      ("ln2.g", dg2), ("ln2.b", dbt2), ("attn.wo", dWo), ("attn.bo", dbo),
                      ("attn.wqkv", dWqkv), ("attn.bqkv", dbqkv), ("ln1.g", dg1), ("ln1.b", dbt1)):
        grads[pre + name] = grads.get(pre + name, 0.0) + val
    return dx


# ----------------------------------------------------------------------------- stage

class StageSpec:
    """Static shape of one stage.  stage_index s is 0-based (paper's i = s+1), n_stages = paper's N."""

    def __init__(self, stage_index, n_stages, n_layers, d_model, n_heads, seq_len, micro_batch, vocab):
        self.stage_index, self.n_stages, self.n_layers = stage_index, n_stages, n_layers
        self.d_model, self.n_heads, self.seq_len = d_model, n_heads, seq_len
        self.micro_batch, self.vocab = micro_batch, vocab
        self.has_embedding = stage_index == 0
        self.has_head = stage_index == n_stages - 1

    def head_name(self):
        # one stage holding both ends: truly tied, one tensor (R10)
        return "wte" if self.has_embedding else "head.w"


def stage_forward(spec, P, inp, targets=None, drop=None):
    """h_{m,i} = F_i(h_{m,i-1}; theta_i)  (Eq. 7).

    inp: int tokens [mu,T] on the first stage, else h [mu,T,D].  Returns (out, stash) where out is
    h [mu,T,D], or the scalar loss on the last stage (then `targets` [mu,T] is required).
    `stash` = "activations required for backpropagation" (Alg. 1 line 7).
    mu is read off `inp`: a micro-batch may hold fewer sequences than spec.micro_batch, and the loss is
    the mean over the tokens of THIS micro-batch (R22).  drop = (p, seed, mb_id) switches dropout on.
    """
    st = {}
    if spec.has_embedding:
        st["tok"] = inp
        x = embed_fwd(inp, P["wte"], P["wpe"])
        st["mask_e"] = _mask(drop, x.shape, _dropout.SITE_EMBED)
        if st["mask_e"] is not None:
            x = x * st["mask_e"]
    else:
        x = inp
    st["blocks"] = []
    for l in range(spec.n_layers):
        x, sb = block_fwd(x, P, f"h.{l}.", spec.n_heads, drop, l)
        st["blocks"].append(sb)
    if not spec.has_head:
        return x, st
    xf, st["lnf"] = layernorm_fwd(x, P["lnf.g"], P["lnf.b"])
    z, st["head"] = linear_fwd(xf, P[spec.head_name()], None)
    loss, st["dz"] = cross_entropy_fwd_bwd(z, targets)
    return loss, st


def stage_backward(spec, Pc, stash, dout=None):
    """g_{m,i} and grad h_{m,i-1} (Alg. 1 line 12) under Eq. 1.

    Pc = the stage's CURRENT parameters.  dout = grad wrt this stage's output (None on the last
    stage, whose backward input is its own loss).  Returns (din or None, grads dict).
    """
    grads = {}
    if spec.has_head:
        dxf, dWh, _ = linear_bwd(stash["dz"], stash["head"], Pc[spec.head_name()])
        grads[spec.head_name()] = dWh
        dx, grads["lnf.g"], grads["lnf.b"] = layernorm_bwd(dxf, stash["lnf"], Pc["lnf.g"])
    else:
        dx = dout
    for l in reversed(range(spec.n_layers)):
        dx = block_bwd(dx, stash["blocks"][l], Pc, f"h.{l}.", grads)
    if spec.has_embedding:
        if stash.get("mask_e") is not None:
            dx = dx * stash["mask_e"]
        dwte, dwpe = embed_bwd(dx, stash["tok"], spec.vocab)
        grads["wte"] = grads.get("wte", 0.0) + dwte
        grads["wpe"] = dwpe
        return None, grads
    return dx, grads


def stage_backward_checkpointed(spec, Pc, stage_input, targets=None, dout=None, drop=None):
    """Activation-checkpointed PACI (App. B): nothing but the stage INPUT was kept at forward time; the
    activations "are instead recomputed under the current parameter version before differentiation".

    So: re-run F_i on the stashed input with the CURRENT parameters Pc (same dropout mask: it is a function of
    the micro-batch id), then differentiate that recomputation at Pc.  The incoming `dout` was produced by the
    ORIGINAL pipeline computation -- that is the mismatch the paper describes.  Identical to `stage_backward` of
    the stashed forward iff no update fell between forward and backward (Delta = 0).
    """
    _, stash = stage_forward(spec, Pc, stage_input, targets, drop)
    return stage_backward(spec, Pc, stash, dout)
