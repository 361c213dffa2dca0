"""Pins for the oracle's SURVEY.md 8(f) extensions -- dropout with a counter-based mask, activation-
checkpointed PACI, heterogeneous micro-batch sizes, the LR schedule -- and for the drifted
multi-stage trajectory of oracle/pipeline.py (Eq. 1 composed across stages and updates).  All `-m "not gpu"`."""
import math
import os

import numpy as np
import pytest
import torch
import torch.nn.functional as F

import synth
from oracle import dropout as odrop
from oracle import lr as olr
from oracle import model, pipeline, schedule
from oracle.adamw import decays

HERE = os.path.dirname(__file__)


def _gold():
    g = {}
    with open(os.path.join(HERE, "golden", "paper_values.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if "=" in line:
                k, v = line.rsplit("=", 1)
                g[k.strip()] = float(v)
    return g


GOLD = _gold()


# ------------------------------------------------------------------ dropout generator
def test_philox_known_answer_vectors():
    n = 0
    with open(os.path.join(HERE, "golden", "philox_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or "|" not in line:
                continue
            c, k, r = ([int(x, 16) for x in part.split()] for part in line.split("|"))
            got = odrop.philox4x32_10(*[np.array([x], dtype=np.uint64) for x in c], k[0], k[1])
            assert [int(w[0]) for w in got] == r
            n += 1
    assert n == 3


def test_dropout_mask_rate_scale_and_keys():
    p = GOLD["dropout p"]
    m = odrop.mask((64, 1000), p, seed=77, mb_id=3, site=2)
    assert set(np.unique(m)) == {0.0, 1.0 / (1.0 - p)}
    assert abs((m == 0).mean() - p) < 4 * math.sqrt(p * (1 - p) / m.size)      # keep rate
    assert abs(m.mean() - 1.0) < 4 * math.sqrt(p / (1 - p) / m.size)           # E[mask] = 1: activations unbiased
    assert np.array_equal(m, odrop.mask((64, 1000), p, 77, 3, 2))              # a pure function of its key
    for other in (odrop.mask((64, 1000), p, 78, 3, 2), odrop.mask((64, 1000), p, 77, 4, 2),
                  odrop.mask((64, 1000), p, 77, 3, 3)):
        assert 0.1 < (other != m).mean() < 0.3                                 # ~2p(1-p) = 0.18 for independent masks
    # element e uses word e % 4 of block e // 4, whatever the tensor's shape
    assert np.array_equal(m.reshape(-1)[:10], odrop.mask((10,), p, 77, 3, 2))
    assert np.all(odrop.mask((8, 8), 0.0, 1, 2, 3) == 1.0)


def _torch_stage_drop(spec, P, inp, tgt, drop):
    """torch library ops + the oracle's masks as constants: pins the chain rule through the mask."""
    D, H = spec.d_model, spec.n_heads
    p, seed, mb = drop
    mk = lambda shape, site: torch.tensor(odrop.mask(tuple(shape), p, seed, mb, site))
    if spec.has_embedding:
        x = P["wte"][inp] + P["wpe"][None, :inp.shape[1]]
        x = x * mk(x.shape, 0)
    else:
        x = inp
    for l in range(spec.n_layers):
        q_ = f"h.{l}."
        y = F.layer_norm(x, (D,), P[q_ + "ln1.g"], P[q_ + "ln1.b"], eps=1e-5)
        qkv = F.linear(y, P[q_ + "attn.wqkv"], P[q_ + "attn.bqkv"])
        B, T, _ = qkv.shape
        q, k, v = (t.reshape(B, T, H, D // H).transpose(1, 2) for t in qkv.split(D, dim=-1))
        o = F.scaled_dot_product_attention(q, k, v, is_causal=True).transpose(1, 2).reshape(B, T, D)
        a = F.linear(o, P[q_ + "attn.wo"], P[q_ + "attn.bo"])
        x = x + a * mk(a.shape, 1 + 2 * l)
        y = F.layer_norm(x, (D,), P[q_ + "ln2.g"], P[q_ + "ln2.b"], eps=1e-5)
        m = F.linear(F.gelu(F.linear(y, P[q_ + "mlp.w1"], P[q_ + "mlp.b1"]), approximate="tanh"),
                     P[q_ + "mlp.w2"], P[q_ + "mlp.b2"])
        x = x + m * mk(m.shape, 2 + 2 * l)
    if not spec.has_head:
        return x
    z = F.linear(F.layer_norm(x, (D,), P["lnf.g"], P["lnf.b"], eps=1e-5), P[spec.head_name()])
    return F.cross_entropy(z.reshape(-1, spec.vocab), tgt.reshape(-1))


@pytest.mark.parametrize("s,S", [(0, 1), (1, 3)])
def test_stage_with_dropout_matches_torch_autograd(s, S):
    spec = model.StageSpec(s, S, 2, 32, 4, 16, 2, 50)
    P = {n: np.asarray(a, np.float64) for n, a in synth.stage_params(3, s, S, 2, 32, 50, 16, True).items()}
    rng = np.random.default_rng(1)
    tok = synth.tokens(9, 1, 2, 16, 50, "zipf")[0]
    tgt = tok[:, 1:].astype(np.int64)
    inp = tok[:, :-1].astype(np.int64) if spec.has_embedding else rng.standard_normal((2, 16, 32))
    r = rng.standard_normal((2, 16, 32))
    drop = (0.25, 99, 6)
    out, stash = model.stage_forward(spec, P, inp, tgt, drop)
    din, grads = model.stage_backward(spec, P, stash, None if spec.has_head else r)
    out0, _ = model.stage_forward(spec, P, inp, tgt)
    assert not np.allclose(out, out0)                                          # the mask does something
    Pt = {n: torch.tensor(a, requires_grad=True) for n, a in P.items()}
    it = torch.tensor(inp) if spec.has_embedding else torch.tensor(inp, requires_grad=True)
    ot = _torch_stage_drop(spec, Pt, it, torch.tensor(tgt), drop)
    if spec.has_head:
        assert abs(out - ot.item()) < 1e-12
        ot.backward()
    else:
        assert np.allclose(out, ot.detach().numpy(), rtol=1e-12, atol=1e-12)
        ot.backward(torch.tensor(r))
        assert np.allclose(din, it.grad.numpy(), rtol=1e-9, atol=1e-12)
    for n in P:
        assert np.allclose(grads[n], Pt[n].grad.numpy(), rtol=1e-9, atol=1e-12), n


# ------------------------------------------------------------------ activation-checkpointed PACI
from test_oracle_layers import _torch_stage  # noqa: E402


@pytest.mark.parametrize("s,S", [(1, 3), (2, 3), (0, 2)])
def test_checkpointed_backward_is_autograd_of_the_recomputation_at_current_weights(s, S):
    """"those activations are instead recomputed under the current parameter version before
    differentiation".  Witness: torch forward + autograd entirely at the CURRENT weights P1, fed the stage input
    that was stashed and the downstream gradient of the original computation."""
    spec = model.StageSpec(s, S, 2, 32, 4, 16, 2, 64)
    P0 = {n: np.asarray(a, np.float64) for n, a in synth.stage_params(5, s, S, 2, 32, 64, 16, True).items()}
    rng = np.random.default_rng(3)
    P1 = {n: a + 0.05 * rng.standard_normal(a.shape) for n, a in P0.items()}
    tok = synth.tokens(2, 1, 2, 16, 64, "zipf")[0]
    tgt = tok[:, 1:].astype(np.int64) if spec.has_head else None
    x = tok[:, :-1].astype(np.int64) if spec.has_embedding else rng.standard_normal((2, 16, 32))
    r = None if spec.has_head else rng.standard_normal((2, 16, 32))
    din, grads = model.stage_backward_checkpointed(spec, P1, x, tgt, r)

    Pt = {n: torch.tensor(a, requires_grad=True) for n, a in P1.items()}
    xt = torch.tensor(x) if spec.has_embedding else torch.tensor(x, requires_grad=True)
    ot = _torch_stage(spec, Pt, xt, None if tgt is None else torch.tensor(tgt))
    ot.backward(None if r is None else torch.tensor(r))
    for n in P1:
        assert np.allclose(grads[n], Pt[n].grad.numpy(), rtol=1e-9, atol=1e-12), n
    if not spec.has_embedding:
        assert np.allclose(din, xt.grad.numpy(), rtol=1e-9, atol=1e-12)

    # identical to Eq. 1's stale-activation backward iff no update fell between forward and backward
    _, stash0 = model.stage_forward(spec, P0, x, tgt)
    din_same, g_same = model.stage_backward_checkpointed(spec, P0, x, tgt, r)
    din_eq1, g_eq1 = model.stage_backward(spec, P0, stash0, r)
    for n in P0:
        assert np.array_equal(g_same[n], g_eq1[n]), n
    _, g_drift = model.stage_backward(spec, P1, stash0, r)                    # Eq. 1 with Delta > 0
    name = "h.0.mlp.w1"
    assert not np.allclose(g_drift[name], grads[name], rtol=1e-3)             # the two modes differ when Delta > 0


def test_checkpointed_pipeline_equals_stashed_pipeline_iff_no_update_is_crossed():
    specs = [model.StageSpec(s, 2, 1, 32, 4, 16, 2, 64) for s in range(2)]
    params = [synth.stage_params(2, s, 2, 1, 32, 64, 16, perturbed=True) for s in range(2)]
    tok = synth.tokens(4, 8, 2, 16, 64, "zipf")
    one_window = [pipeline.run_pipeline(specs, params, tok[:4], 4, 1e-2, checkpoint=c) for c in (False, True)]
    assert all(d == 0 for row in one_window[0]["delta"] for d in row)
    for s in range(2):
        for n, th in one_window[0]["opt"][s].theta.items():
            assert np.array_equal(th, one_window[1]["opt"][s].theta[n]), n
    a, b = (pipeline.run_pipeline(specs, params, tok, 4, 1e-2, checkpoint=c) for c in (False, True))
    assert a["delta"] == b["delta"] and a["delta"][0][4] == 1                  # same schedule, same bound
    # stage 1 never crosses (Eq. 10, i = N): its own gradients agree until stage 0's drift reaches it through h
    assert a["losses"][:5] == b["losses"][:5]
    assert not np.array_equal(a["opt"][0].theta["h.0.mlp.w1"], b["opt"][0].theta["h.0.mlp.w1"])


# ------------------------------------------------------------------ drifted multi-stage trajectory
def _torch_paci_two_stages(specs, params, tok, k, lr):
    """PACI on 2 stages written with torch only: autograd graphs built at forward time, parameters overwritten IN
    PLACE (through .data, i.e. without bumping the version counter -- what the paper's PyTorch patch enables,
    P:498-513) by torch.optim.AdamW between a micro-batch's forward and its backward.  The per-stage op order is the
    classic non-flushed 1F1B order (F x (d_s + 1), then B, F alternating, then the remaining Bs; U after every k-th
    B); any interleaving of the two stages that respects the messages gives the same numbers."""
    S, n = 2, tok.shape[0]
    Pt, sh, opt, acc = [], [], [], []
    for s in range(S):
        leaves = {nm: torch.tensor(np.asarray(a, np.float64), requires_grad=True) for nm, a in params[s].items()}
        shadow = {nm: t.detach().clone().requires_grad_(True) for nm, t in leaves.items()}
        Pt.append(leaves); sh.append(shadow); acc.append({nm: torch.zeros_like(t) for nm, t in leaves.items()})
        opt.append(torch.optim.AdamW(
            [{"params": [shadow[nm] for nm in shadow if decays(nm)], "weight_decay": 0.1},
             {"params": [shadow[nm] for nm in shadow if not decays(nm)], "weight_decay": 0.0}],
            lr=lr, betas=(0.9, 0.95), eps=1e-8))
    seq = []
    for s in range(S):
        d = S - 1 - s
        ops, f, b = [], 0, 0
        for _ in range(min(d + 1, n)):
            ops.append(("F", f)); f += 1
        while b < n:
            ops.append(("B", b)); b += 1
            if b % k == 0:
                ops.append(("U", b // k))
            if f < n:
                ops.append(("F", f)); f += 1
        seq.append(ops)
    pos, fwd_msg, bwd_msg, graph, losses = [0, 0], {}, {}, [dict(), dict()], [None] * n
    cnt = [0, 0]
    while any(pos[s] < len(seq[s]) for s in range(S)):
        moved = False
        for s in range(S):
            if pos[s] == len(seq[s]):
                continue
            kind, m = seq[s][pos[s]]
            if kind == "F":
                if s == 1 and m not in fwd_msg:
                    continue
                t = torch.tensor(tok[m].astype(np.int64))
                if s == 0:
                    out = _torch_stage(specs[0], Pt[0], t[:, :-1], None)
                    graph[0][m] = out
                    fwd_msg[m] = out.detach().clone()
                else:
                    x = fwd_msg[m].clone().requires_grad_(True)
                    loss = _torch_stage(specs[1], Pt[1], x, t[:, 1:])
                    graph[1][m] = (loss, x)
                    losses[m] = loss.item()
            elif kind == "B":
                if s == 0 and m not in bwd_msg:
                    continue
                for p_ in Pt[s].values():
                    p_.grad = None
                if s == 1:
                    loss, x = graph[1].pop(m)
                    loss.backward()
                    bwd_msg[m] = x.grad.clone()
                else:
                    graph[0].pop(m).backward(bwd_msg[m])
                for nm, p_ in Pt[s].items():
                    acc[s][nm] += p_.grad
                cnt[s] += 1
            else:
                assert cnt[s] == k
                for nm in sh[s]:
                    sh[s][nm].grad = acc[s][nm] / k
                opt[s].step()
                for nm in sh[s]:
                    Pt[s][nm].data.copy_(sh[s][nm].data)         # in place, version counter untouched
                    acc[s][nm].zero_()
                cnt[s] = 0
            pos[s] += 1
            moved = True
        assert moved
    return losses, Pt, acc


@pytest.mark.parametrize("k,n", [(1, 3), (2, 5)])
def test_two_stage_drifted_trajectory_matches_torch_inplace_update_witness(k, n):
    """S = 2: stage 0's backward of micro-batch m >= k runs AFTER an update that its forward did not see
    (Delta = 1): forward under theta^(t), backward under theta^(t+1) on the stashed activations, accumulate, update,
    and the next forward under the drifted weights -- the whole glue of run_pipeline, against torch autograd with
    parameters overwritten in place between F and B.  A backward under the forward-time weights (weight stashing)
    or a recomputation would both fail this."""
    specs = [model.StageSpec(s, 2, 1, 32, 4, 16, 2, 64) for s in range(2)]
    params = [synth.stage_params(8, s, 2, 1, 32, 64, 16, perturbed=True) for s in range(2)]
    tok = synth.tokens(8, n, 2, 16, 64, "zipf")
    lr = 1e-2
    ref = pipeline.run_pipeline(specs, params, tok, k, lr)
    assert max(ref["delta"][0]) == 1 and max(ref["delta"][1]) == 0
    losses, Pt, acc = _torch_paci_two_stages(specs, params, tok, k, lr)
    assert np.allclose(ref["losses"], losses, rtol=1e-10, atol=0)
    for s in range(2):
        for nm, th in ref["opt"][s].theta.items():
            assert np.allclose(th, Pt[s][nm].detach().numpy(), rtol=1e-8, atol=1e-11), (s, nm)
            assert np.allclose(ref["opt"][s].G[nm], acc[s][nm].numpy(), rtol=1e-8, atol=1e-12), (s, nm)
    # the witness is sensitive to the drift: the consistent (flush) run gives different weights
    flush = pipeline.run_pipeline(specs, params, tok[: (n // k) * k], None, lr, mode="flush", m_f=k)
    if n % k == 0:
        assert not np.allclose(flush["opt"][0].theta["h.0.mlp.w1"], ref["opt"][0].theta["h.0.mlp.w1"], rtol=1e-6)


# ------------------------------------------------------------------ heterogeneous micro-batch sizes
def test_heterogeneous_sizes_rule_and_loss_normalisation():
    B, m = 10, 4                                    # the first B mod m micro-batches hold floor(B/m) + 1
    sizes = [B // m + (1 if i < B % m else 0) for i in range(m)]
    assert sizes == [3, 3, 2, 2] and sum(sizes) == B
    specs = [model.StageSpec(0, 1, 1, 32, 4, 16, 3, 64)]
    params = [synth.stage_params(2, 0, 1, 1, 32, 64, 16, perturbed=True)]
    tok = synth.tokens(4, m, 3, 16, 64, "zipf")
    r = pipeline.run_pipeline(specs, params, tok, m, 1e-2, n_seq=sizes)
    # each micro-batch's loss is the mean over ITS OWN tokens (R22): equal to running it alone at its own size
    for i, ns in enumerate(sizes):
        spec_i = model.StageSpec(0, 1, 1, 32, 4, 16, ns, 64)
        li, _ = model.stage_forward(spec_i, {n: np.asarray(a, np.float64) for n, a in params[0].items()},
                                    tok[i, :ns, :-1].astype(np.int64), tok[i, :ns, 1:].astype(np.int64))
        assert r["losses"][i] == li
    full = pipeline.run_pipeline(specs, params, tok, m, 1e-2)
    assert r["losses"][0] == full["losses"][0] and r["losses"][2] != full["losses"][2]


# ------------------------------------------------------------------ LR schedule
def test_lr_schedule_printed_constants_and_torch_scheduler_witness():
    peak, f = GOLD["lr peak B=256"], GOLD["lr final over peak"]
    assert abs(GOLD["lr peak B=128"] - 3 * math.sqrt(0.5) * 1e-4) < 1e-18
    N, W = 1000, 10                                                            # 1% warm-up
    assert olr.lr_at(W - 1, N, W, peak, f) == peak
    assert abs(olr.lr_at(N, N, W, peak, f) - f * peak) < 1e-18 and abs(olr.lr_at(N + 5, N, W, peak, f) - f * peak) < 1e-18
    assert abs(olr.lr_at(W + (N - W) // 2, N, W, peak, f) - peak * (f + (1 - f) / 2)) < 1e-12
    vals = [olr.lr_at(t, N, W, peak, f) for t in range(N + 1)]
    assert all(a < b for a, b in zip(vals[:W - 1], vals[1:W])) and all(a >= b for a, b in zip(vals[W:], vals[W + 1:]))
    # library witness for the cosine part: torch's CosineAnnealingLR with eta_min = f * peak
    p_ = torch.nn.Parameter(torch.zeros(1))
    opt = torch.optim.SGD([p_], lr=peak)
    sch = torch.optim.lr_scheduler.CosineAnnealingLR(opt, T_max=N - W, eta_min=f * peak)
    for t in range(W, N + 1):
        assert abs(opt.param_groups[0]["lr"] - vals[t]) < 1e-15, t
        opt.step(); sch.step()


def test_lr_by_update_is_indexed_by_each_stage_own_update_count():
    specs = [model.StageSpec(s, 2, 1, 32, 4, 16, 2, 64) for s in range(2)]
    params = [synth.stage_params(2, s, 2, 1, 32, 64, 16, perturbed=True) for s in range(2)]
    tok = synth.tokens(4, 4, 2, 16, 64, "zipf")
    a = pipeline.run_pipeline(specs, params, tok, 2, 1e-2, lr_by_update=[1e-2, 1e-2])
    b = pipeline.run_pipeline(specs, params, tok, 2, 1e-2)
    c = pipeline.run_pipeline(specs, params, tok, 2, 1e-2, lr_by_update=[1e-2, 5e-3])
    for s in range(2):
        assert np.array_equal(a["opt"][s].theta["h.0.mlp.w1"], b["opt"][s].theta["h.0.mlp.w1"])
        assert not np.array_equal(a["opt"][s].theta["h.0.mlp.w1"], c["opt"][s].theta["h.0.mlp.w1"])


def test_eta_inter_printed_value():
    g = {}
    with open(os.path.join(HERE, "golden", "paper_values.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line.startswith("eta_inter"):
                g = float(line.rsplit("=", 1)[1])
    assert abs(schedule.eta_inter(4, 9, 2) - g) < 1e-15                        # "efficiency 1/2"
    assert schedule.eta_inter(4, 9, 1) == schedule.eta_flush(4, 9)             # V = 1 reduces Eq. 4 to Eq. 3
