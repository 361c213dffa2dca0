"""-m gpu: one stage's forward / backward / update through the C ABI vs the oracle, including the
drift case (an update between a micro-batch's forward and backward, Eq. 1) and the protocol errors."""
import numpy as np
import pytest
import torch

import synth
from oracle import model
from oracle.adamw import StageOptimizer
from paper_2606_07881_b200 import binding as pb
from gpu_util import DT, TOL, dev, host, rel_l2, rounded

pytestmark = pytest.mark.gpu


def _mk(dtype, s, S, L, D, H, T, mu, V, k, seed=11):
    spec = model.StageSpec(s, S, L, D, H, T, mu, V)
    params = synth.stage_params(seed, s, S, L, D, V, T, perturbed=True)
    st = pb.Stage(pb.make_config(s, S, L, D, H, T, mu, k, V, dtype))
    st.load_params(params)
    return spec, params, st


def _inputs(spec, dtype, seed):
    rng = np.random.default_rng(seed)
    tok = synth.tokens(seed, 1, spec.micro_batch, spec.seq_len, spec.vocab, "zipf")[0]
    inp_tok, tgt = tok[:, :-1].copy(), tok[:, 1:].copy()
    h = rounded(rng.standard_normal((spec.micro_batch, spec.seq_len, spec.d_model)), dtype)
    dout = rounded(rng.standard_normal((spec.micro_batch, spec.seq_len, spec.d_model)) * 0.1, dtype)
    return inp_tok, tgt, h, dout


def _run_gpu(st, spec, dtype, mb, inp_tok, tgt, h, dout, do_backward=True):
    M, D = spec.micro_batch * spec.seq_len, spec.d_model
    inp = torch.from_numpy(inp_tok).cuda() if spec.has_embedding else dev(h, dtype)
    tg = torch.from_numpy(tgt).cuda() if spec.has_head else None
    out = torch.zeros(1, device="cuda") if spec.has_head else torch.empty(spec.micro_batch, spec.seq_len, D,
                                                                         device="cuda", dtype=DT[dtype])
    st.forward(mb, inp, tg, out)
    keep = (inp, tg, out)
    if not do_backward:
        return out, None, keep
    din = None if spec.has_embedding else torch.empty(spec.micro_batch, spec.seq_len, D, device="cuda",
                                                      dtype=DT[dtype])
    st.backward(mb, None if spec.has_head else dev(dout, dtype), din)
    torch.cuda.synchronize()
    return out, din, keep


CASES = [  # dtype, s, S, L, D, H, T, mu, V
    (pb.FP32, 0, 2, 1, 64, 4, 32, 2, 256),     # cfg 1 stage 0
    (pb.FP32, 1, 2, 1, 64, 4, 32, 2, 256),     # cfg 1 stage 1
    (pb.FP32, 0, 1, 2, 64, 4, 32, 2, 256),     # single stage, tied head
    (pb.FP32, 1, 3, 2, 96, 3, 40, 3, 300),     # interior stage, ragged sizes
    (pb.BF16, 0, 2, 1, 128, 2, 128, 2, 1000),
    (pb.BF16, 1, 2, 1, 128, 2, 128, 2, 1000),  # ragged vocab (1000 -> padded 1024)
    (pb.BF16, 1, 3, 2, 256, 4, 128, 3, 512),   # interior, several tiles + ragged M tail (384 rows)
    (pb.BF16, 0, 1, 1, 128, 2, 128, 1, 777),   # tied head
    (pb.BF16, 1, 3, 1, 256, 4, 384, 1, 512),   # T % 128 == 0: tcgen05 attention over several key blocks
]


@pytest.mark.parametrize("dtype,s,S,L,D,H,T,mu,V", CASES)
def test_stage_forward_backward_matches_oracle(dtype, s, S, L, D, H, T, mu, V):
    spec, params, st = _mk(dtype, s, S, L, D, H, T, mu, V, k=1)
    inp_tok, tgt, h, dout = _inputs(spec, dtype, 21)
    P = {n: np.asarray(a, np.float64) for n, a in params.items()}
    ref_out, stash = model.stage_forward(spec, P, inp_tok.astype(np.int64) if spec.has_embedding else h,
                                         tgt.astype(np.int64))
    ref_din, ref_g = model.stage_backward(spec, P, stash, None if spec.has_head else dout)
    out, din, _ = _run_gpu(st, spec, dtype, 0, inp_tok, tgt, h, dout)
    tol = TOL[dtype]
    if spec.has_head:
        assert abs(out.item() - ref_out) / abs(ref_out) < (1e-5 if dtype == pb.FP32 else 5e-3)
    else:
        assert rel_l2(host(out), ref_out) < tol
    if not spec.has_embedding:
        assert rel_l2(host(din), ref_din) < tol
    for name, g in ref_g.items():
        got = st.read(name, pb.GRAD_ACCUM)
        assert rel_l2(got, g) < tol, (name, rel_l2(got, g))
    assert st.crossed_updates(0) == 0 and st.device_stamps(0) == (0, 0)
    st.close()


@pytest.mark.parametrize("dtype,D,H,T,V", [(pb.FP32, 64, 4, 32, 256), (pb.BF16, 128, 2, 128, 512)])
def test_drift_case_stale_activations_current_weights(dtype, D, H, T, V):
    """F(m0) F(m1) B(m0) U B(m1): m1's backward runs one version later than its forward (Delta = 1) and
    must use the stashed activations with the UPDATED weights (Eq. 1), not a recomputation."""
    spec, params, st = _mk(dtype, 1, 3, 2, D, H, T, 2, V, k=1)     # interior stage, d_s = 1
    a = _inputs(spec, dtype, 31)
    b = _inputs(spec, dtype, 32)
    opt = StageOptimizer(params, 1)
    _, stash0 = model.stage_forward(spec, opt.theta, a[2])
    _, stash1 = model.stage_forward(spec, opt.theta, b[2])
    _, g0 = model.stage_backward(spec, opt.theta, stash0, a[3])
    opt.accumulate(g0)
    lr = 1e-2 if dtype == pb.FP32 else 1e-3   # bf16: keep Adam's sign-flip noise (~sqrt(f)*2lr/rms) small
    assert opt.maybe_step(lr)
    ref_din, g1 = model.stage_backward(spec, opt.theta, stash1, b[3])      # current weights, old stash
    _, g1_consistent = model.stage_backward(spec, {n: np.asarray(p, np.float64) for n, p in params.items()},
                                            stash1, b[3])

    _, _, k0 = _run_gpu(st, spec, dtype, 0, *a, do_backward=False)
    _, _, k1 = _run_gpu(st, spec, dtype, 1, *b, do_backward=False)
    with pytest.raises(pb.PaciError) as e:                                  # q = 2 > d_s = 1 -> EAGAIN
        st.forward(2, k0[0], None, k0[2])
    assert e.value.code == pb.EAGAIN and st.unresolved == 2
    with pytest.raises(pb.PaciError) as e:                                  # FIFO: m1 is not the oldest
        st.backward(1, dev(b[3], dtype), torch.empty_like(k0[2]))
    assert e.value.code == pb.ESTATE
    din0 = torch.empty_like(k0[2])
    st.backward(0, dev(a[3], dtype), din0)
    with pytest.raises(pb.PaciError) as e:                                  # c == k: update pending
        st.backward(1, dev(b[3], dtype), torch.empty_like(k0[2]))
    assert e.value.code == pb.ESTATE
    assert st.maybe_step(lr) == 1 and st.version == 1 and st.maybe_step(lr) == 0
    din1 = torch.empty_like(k0[2])
    st.backward(1, dev(b[3], dtype), din1)
    torch.cuda.synchronize()
    assert st.crossed_updates(0) == 0 and st.crossed_updates(1) == 1 and st.crossed_updates(7) == -1
    assert st.device_stamps(0) == (0, 0) and st.device_stamps(1) == (0, 1)  # proven on the device
    tol = TOL[dtype]
    assert rel_l2(host(din1), ref_din) < tol
    for name in ("h.0.attn.wqkv", "h.1.mlp.w1", "h.0.ln1.g", "h.1.mlp.b2", "h.0.attn.bo"):
        got = st.read(name, pb.GRAD_ACCUM)
        assert rel_l2(got, g1[name]) < tol, name
    # ... and that it is NOT the consistent-weights gradient (the drift is visible above tolerance)
    if dtype == pb.FP32:
        got = st.read("h.0.ln1.g", pb.GRAD_ACCUM)
        assert rel_l2(got, g1_consistent["h.0.ln1.g"]) > 10 * tol
    st.close()


@pytest.mark.parametrize("dtype", [pb.FP32, pb.BF16])
def test_window_of_k_then_update_matches_oracle(dtype):
    """k micro-batches accumulate into G (raw sum), the k-th backward triggers one AdamW step on G/k."""
    D, H, T, V, k = (64, 4, 32, 256, 4) if dtype == pb.FP32 else (128, 2, 128, 512, 4)
    spec, params, st = _mk(dtype, 0, 1, 1, D, H, T, 2, V, k=k)
    opt = StageOptimizer(params, k)
    for m in range(k):
        inp_tok, tgt, h, dout = _inputs(spec, dtype, 40 + m)
        _, stash = model.stage_forward(spec, opt.theta, inp_tok.astype(np.int64), tgt.astype(np.int64))
        _, g = model.stage_backward(spec, opt.theta, stash)
        opt.accumulate(g)
        _run_gpu(st, spec, dtype, m, inp_tok, tgt, h, dout)
        if m < k - 1:
            assert st.maybe_step(1e-3) == 0 and st.window_count == m + 1
    Gsum = {n: a.copy() for n, a in opt.G.items()}
    for name in ("wte", "h.0.mlp.w2", "lnf.g"):
        assert rel_l2(st.read(name, pb.GRAD_ACCUM), Gsum[name]) < TOL[dtype], name
    theta0 = {n: np.asarray(a, np.float64) for n, a in params.items()}
    assert opt.maybe_step(1e-3) and st.maybe_step(1e-3) == 1
    assert st.version == 1 and st.window_count == 0
    for name in opt.theta:
        got = st.read(name)
        ref = opt.theta[name].reshape(-1)
        if name.endswith("attn.bqkv"):
            # The key bias has an identically ZERO gradient (softmax is invariant to a constant added to
            # every key: sum_j ds_ij = 0), so what reaches AdamW is rounding noise, which Adam normalises
            # to a step of up to +-lr.  Compare q and v parts; bound the k part by lr.
            kpart = slice(D, 2 * D)
            assert np.max(np.abs(got[kpart] - ref[kpart])) <= 1e-3 * 1.001
            got, ref = np.delete(got, np.r_[kpart]), np.delete(ref, np.r_[kpart])
        assert rel_l2(got, ref) < (1e-3 if dtype == pb.FP32 else 2e-2), name               # after one step
        assert np.count_nonzero(st.read(name, pb.GRAD_ACCUM)) == 0            # G reset
    # weight DELTA: first step ~ lr*sign(g); bf16 can flip the sign of near-zero gradients
    d_got = st.read("h.0.mlp.w1") - theta0["h.0.mlp.w1"].reshape(-1)
    d_ref = (opt.theta["h.0.mlp.w1"] - theta0["h.0.mlp.w1"]).reshape(-1)
    assert rel_l2(d_got, d_ref) < (1e-3 if dtype == pb.FP32 else 0.35)
    st.close()
