"""-m gpu: the SURVEY.md 8(f) rows built on the hot path -- activation-checkpointed PACI, dropout with the
shared counter-based mask, heterogeneous micro-batch sizes, the LR schedule -- and the host-side
fixes of round 2 (caller-stream ordering, id validation, counter restore, log-ring recycling), CUDA path vs oracle."""
import ctypes as C

import numpy as np
import pytest
import torch

import synth
from oracle import lr as olr
from oracle import model, pipeline as opipe
from oracle.adamw import StageOptimizer
from paper_2606_07881_b200 import binding as pb
from gpu_util import DT, TOL, dev, host, rel_l2, rounded
from test_gpu_pipeline import WTOL, _compare

pytestmark = pytest.mark.gpu


def _build(dtype, S, L, D, H, T, mu, V, k, seed=1234, **cfg):
    specs = [model.StageSpec(s, S, L, D, H, T, mu, V) for s in range(S)]
    params = [synth.stage_params(seed, s, S, L, D, V, T, perturbed=True) for s in range(S)]
    stages = []
    for s in range(S):
        st = pb.Stage(pb.make_config(s, S, L, D, H, T, mu, k, V, dtype, **cfg))
        st.load_params(params[s])
        stages.append(st)
    return specs, params, stages


SMALL = {pb.FP32: dict(D=64, H=4, T=32, V=256), pb.BF16: dict(D=128, H=2, T=128, V=512)}


# ------------------------------------------------------------------ checkpointed PACI (f-2)
@pytest.mark.parametrize("dtype", [pb.FP32, pb.BF16])
def test_checkpoint_mode_drift_case_recomputes_under_current_weights(dtype):
    """F(m0) F(m1) B(m0) U B(m1) on an interior stage with checkpoint = 1: m1's backward (Delta = 1) must differentiate
    a RECOMPUTATION of the stage under the updated weights, which differs from Eq. 1's stale-activation
    gradient; m0's (Delta = 0) equals the stashed mode."""
    c = SMALL[dtype]
    D, H, T, V, mu = c["D"], c["H"], c["T"], c["V"], 2
    spec = model.StageSpec(1, 3, 2, D, H, T, mu, V)
    params = synth.stage_params(11, 1, 3, 2, D, V, T, perturbed=True)
    st = pb.Stage(pb.make_config(1, 3, 2, D, H, T, mu, 1, V, dtype, checkpoint=1))
    st.load_params(params)
    rng = np.random.default_rng(31)
    x = [rounded(rng.standard_normal((mu, T, D)), dtype) for _ in range(2)]
    r = [rounded(rng.standard_normal((mu, T, D)) * 0.1, dtype) for _ in range(2)]
    lr = 1e-2 if dtype == pb.FP32 else 1e-3
    opt = StageOptimizer(params, 1)
    out_ref = [model.stage_forward(spec, opt.theta, x[i])[0] for i in range(2)]
    din0_ref, g0 = model.stage_backward_checkpointed(spec, opt.theta, x[0], None, r[0])
    _, stash1 = model.stage_forward(spec, opt.theta, x[1])
    opt.accumulate(g0)
    assert opt.maybe_step(lr)
    din1_ref, g1 = model.stage_backward_checkpointed(spec, opt.theta, x[1], None, r[1])
    _, g1_eq1 = model.stage_backward(spec, opt.theta, stash1, r[1])

    xd = [dev(a, dtype) for a in x]
    rd = [dev(a, dtype) for a in r]
    outs = [torch.empty(mu, T, D, device="cuda", dtype=DT[dtype]) for _ in range(2)]
    dins = [torch.empty(mu, T, D, device="cuda", dtype=DT[dtype]) for _ in range(2)]
    st.forward(0, xd[0], None, outs[0])
    st.forward(1, xd[1], None, outs[1])
    xd[1].zero_()                                  # the stage must have kept its own copy of the input
    st.backward(0, rd[0], dins[0])
    torch.cuda.synchronize()
    tol = TOL[dtype]
    for name in ("h.0.attn.wqkv", "h.1.mlp.w2", "h.0.ln1.g", "h.1.mlp.b1"):
        assert rel_l2(st.read(name, pb.GRAD_ACCUM), g0[name]) < tol, name
    assert st.maybe_step(lr) == 1
    st.backward(1, rd[1], dins[1])
    torch.cuda.synchronize()
    assert st.crossed_updates(1) == 1 and st.device_stamps(1) == (0, 1)
    for i in range(2):
        assert rel_l2(host(outs[i]), out_ref[i]) < tol
    assert rel_l2(host(dins[0]), din0_ref) < tol and rel_l2(host(dins[1]), din1_ref) < tol
    for name in ("h.0.attn.wqkv", "h.1.mlp.w1", "h.0.ln1.g", "h.1.mlp.b2", "h.0.attn.bo"):
        assert rel_l2(st.read(name, pb.GRAD_ACCUM), g1[name]) < tol, name
    if dtype == pb.FP32:   # ... and it is NOT Eq. 1's gradient: the two modes differ once an update is crossed
        assert rel_l2(st.read("h.0.ln1.g", pb.GRAD_ACCUM), g1_eq1["h.0.ln1.g"]) > 10 * tol
    st.close()


@pytest.mark.parametrize("dtype,S,k,n", [(pb.FP32, 2, 2, 6), (pb.FP32, 3, 1, 5), (pb.BF16, 2, 2, 4)])
def test_checkpoint_mode_pipeline_matches_oracle(dtype, S, k, n):
    """Whole schedule with checkpoint = 1 (embedding stage: tokens kept; head stage: targets kept, logits recomputed):
    counts exact, losses / weights within the gates, against oracle.run_pipeline(checkpoint=True)."""
    c = SMALL[dtype]
    D, H, T, V, mu, L = c["D"], c["H"], c["T"], c["V"], 2, 1
    lr = 2e-3 if dtype == pb.FP32 else 3e-4
    specs, params, stages = _build(dtype, S, L, D, H, T, mu, V, k, seed=21, checkpoint=1)
    tok = synth.tokens(21, n, mu, T, V, "zipf")
    ref = opipe.run_pipeline(specs, params, tok, k, lr, checkpoint=True)
    assert max(max(row) for row in ref["delta"]) >= 1
    out = pb.Pipeline(stages).run(torch.from_numpy(tok).cuda(), lr)
    _compare(out, ref, stages, dtype, n, 2e-5 if dtype == pb.FP32 else 5e-3, lr_bound=2 * lr)
    if dtype == pb.FP32:   # sanity: the stashed mode gives a different trajectory on the same inputs
        ref_eq1 = opipe.run_pipeline(specs, params, tok, k, lr)
        nm = "h.0.mlp.w1"
        assert rel_l2(stages[0].read(nm), ref_eq1["opt"][0].theta[nm]) > rel_l2(stages[0].read(nm), ref["opt"][0].theta[nm])


def test_checkpoint_mode_stash_slot_is_the_stage_input():
    """"each stage still keeps only a single parameter copy"; what shrinks is the stash: S - s slots of the
    stage input (+ targets) instead of S - s full activation sets, plus ONE shared full set."""
    D, H, T, mu, V, L = 1024, 16, 1024, 8, 50257, 6
    M = mu * T
    size = {}
    for ck in (0, 1):
        for s in (0, 1):
            cfg = pb.make_config(s, 4, L, D, H, T, mu, 4, V, pb.BF16, has_embedding=False, has_head=False, checkpoint=ck)
            size[ck, s] = pb.lib.paci_stage_workspace_bytes(C.byref(cfg))
    full_slot = size[0, 0] - size[0, 1]
    ck_slot = size[1, 0] - size[1, 1]
    assert ck_slot == M * D * 2                                        # one bf16 [M, D] stage input per slot
    assert size[1, 1] == size[0, 1] - 3 * full_slot + 3 * ck_slot + full_slot   # 3 slots shrink, one shared set added
    assert size[1, 0] < 0.45 * size[0, 0]                              # 8.0 GB -> 3.3 GB for the first of 4 stages x 6 blocks


# ------------------------------------------------------------------ dropout (f-3)
@pytest.mark.parametrize("dtype,s,S", [(pb.FP32, 0, 1), (pb.FP32, 1, 3), (pb.BF16, 1, 3), (pb.BF16, 0, 1)])
def test_stage_with_dropout_matches_oracle(dtype, s, S):
    c = SMALL[dtype]
    D, H, T, V, mu, L, p, seed, mb = c["D"], c["H"], c["T"], c["V"], 2, 2, 0.1, 4242, 9
    spec = model.StageSpec(s, S, L, D, H, T, mu, V)
    params = synth.stage_params(13, s, S, L, D, V, T, perturbed=True)
    st = pb.Stage(pb.make_config(s, S, L, D, H, T, mu, 1, V, dtype, dropout_p=p, dropout_seed=seed))
    st.load_params(params)
    rng = np.random.default_rng(5)
    tok = synth.tokens(5, 1, mu, T, V, "zipf")[0]
    inp_tok, tgt = tok[:, :-1].copy(), tok[:, 1:].copy()
    h = rounded(rng.standard_normal((mu, T, D)), dtype)
    dout = rounded(rng.standard_normal((mu, T, D)) * 0.1, dtype)
    P = {n: np.asarray(a, np.float64) for n, a in params.items()}
    drop = (p, seed, mb)
    ref_out, stash = model.stage_forward(spec, P, inp_tok.astype(np.int64) if spec.has_embedding else h,
                                         tgt.astype(np.int64) if spec.has_head else None, drop)
    ref_din, ref_g = model.stage_backward(spec, P, stash, None if spec.has_head else dout)
    inp = torch.from_numpy(inp_tok).cuda() if spec.has_embedding else dev(h, dtype)
    tg = torch.from_numpy(tgt).cuda() if spec.has_head else None
    out = torch.zeros(1, device="cuda") if spec.has_head else torch.empty(mu, T, D, device="cuda", dtype=DT[dtype])
    din = None if spec.has_embedding else torch.empty(mu, T, D, device="cuda", dtype=DT[dtype])
    dd = None if spec.has_head else dev(dout, dtype)
    st.forward(mb, inp, tg, out)
    st.backward(mb, dd, din)
    torch.cuda.synchronize()
    tol = TOL[dtype]
    if spec.has_head:
        assert abs(out.item() - ref_out) / abs(ref_out) < (1e-5 if dtype == pb.FP32 else 5e-3)
    else:
        assert rel_l2(host(out), ref_out) < tol
        assert rel_l2(host(din), ref_din) < tol
    for name, g in ref_g.items():
        assert rel_l2(st.read(name, pb.GRAD_ACCUM), g) < tol, (name, rel_l2(st.read(name, pb.GRAD_ACCUM), g))
    st.close()


def test_pipeline_with_dropout_checkpoint_sizes_and_lr_schedule_matches_oracle():
    """Everything of 8(f) f-2 / f-3 at once, fp32: dropout 0.1, checkpointed backward (the recomputation must
    regenerate the forward's mask), heterogeneous micro-batch sizes floor(B/m) (+1) and a warm-up + cosine learning
    rate indexed by each stage's own update count."""
    V, D, H, T, mu, S, L, k = 256, 64, 4, 32, 3, 2, 1, 2
    B, m = 16, 6
    sizes = [B // m + (1 if i < B % m else 0) for i in range(m)]          # P:274 -> [3, 3, 3, 3, 2, 2]
    assert sizes == [3, 3, 3, 3, 2, 2]
    lrs = [olr.lr_at(t, 3, 1, 2e-3) for t in range(3)]
    specs, params, stages = _build(pb.FP32, S, L, D, H, T, mu, V, k, seed=33, checkpoint=1, dropout_p=0.1,
                                   dropout_seed=777)
    tok = synth.tokens(33, m, mu, T, V, "zipf")
    ref = opipe.run_pipeline(specs, params, tok, k, None, checkpoint=True, n_seq=sizes, dropout=(0.1, 777),
                             lr_by_update=lrs)
    out = pb.Pipeline(stages).run(torch.from_numpy(tok).cuda(), 0.0, n_seq=sizes,
                                  lr_by_update=[pb.lr_schedule(t, 3, 1, 2e-3) for t in range(3)])
    _compare(out, ref, stages, pb.FP32, m, 2e-5, lr_bound=4e-3)


def test_heterogeneous_micro_batch_sizes_bf16():
    V, D, H, T, mu, S, L, k, n = 512, 128, 2, 128, 3, 2, 1, 2, 4
    sizes = [3, 2, 1, 2]
    specs, params, stages = _build(pb.BF16, S, L, D, H, T, mu, V, k, seed=41)
    tok = synth.tokens(41, n, mu, T, V, "zipf")
    ref = opipe.run_pipeline(specs, params, tok, k, 3e-4, n_seq=sizes)
    out = pb.Pipeline(stages).run(torch.from_numpy(tok).cuda(), 3e-4, n_seq=sizes)
    _compare(out, ref, stages, pb.BF16, n, 5e-3, lr_bound=6e-4)


# ------------------------------------------------------------------ host-side fixes
def test_run_is_ordered_after_the_callers_stream():
    """The token buffer is produced ASYNCHRONOUSLY on the caller's stream (a slow kernel, then a non-blocking copy
    from pinned memory); paci_pipeline_run must not read it before that work is done."""
    V, D, H, T, mu, S, L, k, n = 256, 64, 4, 32, 2, 2, 1, 2, 4
    tok = synth.tokens(7, n, mu, T, V, "uniform")
    _, _, stages = _build(pb.FP32, S, L, D, H, T, mu, V, k)
    want = pb.Pipeline(stages).run(torch.from_numpy(tok).cuda(), 1e-3)["loss"]
    _, _, stages2 = _build(pb.FP32, S, L, D, H, T, mu, V, k)
    pipe = pb.Pipeline(stages2)
    side = torch.cuda.Stream()
    pinned = torch.from_numpy(tok).pin_memory()
    buf = torch.full(tok.shape, V + 5, dtype=torch.int32, device="cuda")      # out-of-range garbage until the copy lands
    big = torch.empty(1 << 28, device="cuda")
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        for _ in range(20):
            big.normal_()                                                      # ~ms of queued work ahead of the copy
        buf.copy_(pinned, non_blocking=True)
        got = pipe.run(buf, 1e-3, stream=side)["loss"]
    assert np.allclose(got, want, rtol=1e-5)          # (atomics make runs non-bitwise; garbage tokens would be far off)


def test_out_of_range_ids_fail_the_run_without_faulting():
    V, D, H, T, mu, S, L, k, n = 256, 64, 4, 32, 2, 2, 1, 2, 2
    tok = synth.tokens(7, n, mu, T, V, "uniform")
    tok[1, 0, 5] = V + 100
    _, _, stages = _build(pb.FP32, S, L, D, H, T, mu, V, k)
    with pytest.raises(pb.PaciError) as e:
        pb.Pipeline(stages).run(torch.from_numpy(tok).cuda(), 1e-3)
    assert e.value.code == pb.EINVAL and "outside" in str(e.value)
    torch.cuda.synchronize()                                                   # the context is still healthy


def test_counters_survive_a_checkpoint_and_resume():
    """Save at version v with a half-filled window (c > 0), reload into a fresh stage with paci_stage_set_state, continue:
    the trajectory is identical to the uninterrupted one (AdamW's bias correction uses t = version + 1)."""
    D, H, T, V, mu, k = 64, 4, 32, 256, 2, 2
    params = synth.stage_params(3, 0, 1, 1, D, V, T, perturbed=True)
    tok = synth.tokens(3, 7, mu, T, V, "uniform")

    def step(st, m):
        inp = torch.from_numpy(tok[m, :, :-1].copy()).cuda()
        tgt = torch.from_numpy(tok[m, :, 1:].copy()).cuda()
        loss = torch.zeros(1, device="cuda")
        st.forward(m, inp, tgt, loss)
        st.backward(m)
        st.maybe_step(1e-2)
        torch.cuda.synchronize()
        return loss.item()

    a = pb.Stage(pb.make_config(0, 1, 1, D, H, T, mu, k, V, pb.FP32)); a.load_params(params)
    la = [step(a, m) for m in range(7)]
    b = pb.Stage(pb.make_config(0, 1, 1, D, H, T, mu, k, V, pb.FP32)); b.load_params(params)
    lb = [step(b, m) for m in range(5)]
    assert b.version == 2 and b.window_count == 1
    names = list(params)
    saved = {w: {n: b.read(n, w) for n in names} for w in (pb.PARAM, pb.GRAD_ACCUM, pb.ADAM_M, pb.ADAM_V)}
    c = pb.Stage(pb.make_config(0, 1, 1, D, H, T, mu, k, V, pb.FP32))
    for w, d in saved.items():
        for n, arr in d.items():
            c.load(n, arr, what=w)
    c.set_state(2, 1)
    assert c.version == 2 and c.window_count == 1
    lc = [step(c, m) for m in range(5, 7)]
    assert np.allclose(lb + lc, la, rtol=1e-5)         # fp32 atomics: equal up to summation order (R21)
    assert c.version == a.version == 3
    for n in names:    # (the key bias has a zero gradient: Adam turns its rounding noise into +-lr steps)
        assert rel_l2(c.read(n), a.read(n)) < (1e-4 if not n.endswith("attn.bqkv") else 5e-2), n
    # ... and a resumed stage that does NOT restore the counters takes a visibly different step (t = 1 bias correction)
    d = pb.Stage(pb.make_config(0, 1, 1, D, H, T, mu, k, V, pb.FP32))
    for w, dd in saved.items():
        for n, arr in dd.items():
            d.load(n, arr, what=w)
    d.set_state(0, 1)
    [step(d, m) for m in range(5, 7)]
    assert rel_l2(d.read("h.0.mlp.w1"), a.read("h.0.mlp.w1")) > 10 * rel_l2(c.read("h.0.mlp.w1"), a.read("h.0.mlp.w1"))
    with pytest.raises(pb.PaciError):
        c.set_state(1, k)                                                       # window count must be < k


def test_delta_log_survives_ring_recycling_with_reused_ids():
    """More than 4096 forwards with micro-batch ids 0..n-1 reused every run (what paci_pipeline_run does) and n not a
    divisor of 4096: the id -> log entry map must keep pointing at the LATEST entry of an id."""
    D, H, T, V, mu = 64, 4, 32, 256, 1
    st = pb.Stage(pb.make_config(0, 1, 0, D, H, T, mu, 1 << 20, V, pb.FP32, has_embedding=True, has_head=True))
    st.load_params(synth.stage_params(3, 0, 1, 0, D, V, T))
    inp = torch.zeros(mu, T, dtype=torch.int32, device="cuda")
    loss = torch.zeros(1, device="cuda")
    n = 7
    for it in range(4096 // n + 3):
        for m in range(n):
            st.forward(m, inp, inp, loss)
            st.backward(m)
            assert st.crossed_updates(m) == 0, (it, m)
    torch.cuda.synchronize()
    assert st.device_stamps(n - 1) == (0, 0)
    st.close()


def test_stage_worker_drives_a_real_stage_single_rank():
    """The stage-per-GPU event loop (8(f) f-1) with binding.Stage as its stage object, world size 1 (one stage holding
    both ends, no neighbour): the loop's forward / backward / update order must reproduce the oracle's S = 1 run.  The
    multi-rank transport is covered on CPU over gloo (tests/test_stage_per_gpu.py)."""
    from paper_2606_07881_b200.stage_per_gpu import StageWorker
    V, D, H, T, mu, L, k, n, lr = 256, 64, 4, 32, 2, 1, 2, 6, 2e-3
    specs, params, stages = _build(pb.FP32, 1, L, D, H, T, mu, V, k, seed=51)
    tok = synth.tokens(51, n, mu, T, V, "uniform")
    ref = opipe.run_pipeline(specs, params, tok, k, lr)
    inp = [torch.from_numpy(tok[m, :, :-1].copy()).cuda() for m in range(n)]
    tgt = [torch.from_numpy(tok[m, :, 1:].copy()).cuda() for m in range(n)]
    losses = [torch.zeros(1, device="cuda") for _ in range(n)]
    w = StageWorker(stages[0], 0, 1, lambda: torch.empty(mu, T, D, device="cuda"), None)
    rep = w.run(n, lr, inputs=lambda m: inp[m], targets=lambda m: tgt[m], losses=losses)
    torch.cuda.synchronize()
    assert rep["delta"] == ref["delta"][0] == [0] * n and rep["version"] == ref["version"][0] == n // k
    assert [e for e in rep["events"] if e[0] == "U"] == [("U", 1), ("U", 2), ("U", 3)]
    got = np.array([x.item() for x in losses])
    assert np.max(np.abs(got - np.array(ref["losses"])) / np.array(ref["losses"])) < 2e-5
    for name, th in ref["opt"][0].theta.items():
        if not name.endswith("attn.bqkv"):
            assert rel_l2(stages[0].read(name), th) < WTOL[pb.FP32], name
