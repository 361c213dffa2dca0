"""-m gpu: empty and degenerate inputs through the C ABI.  An op given zero rows / zero elements returns PACI_OK, launches
nothing that touches memory and leaves its outputs (and the fp32 accumulators it would add into) untouched; a pipeline
run over zero micro-batches is a no-op that reports zero updates; the smallest legal shapes (one row, one micro-batch,
k = 1, one stage) agree with the oracle."""
import ctypes as C

import numpy as np
import pytest
import torch

import synth
from oracle import model
from paper_2606_07881_b200 import binding as pb
from gpu_util import DT, TOL, dev, f32, host, rel_l2, rounded

pytestmark = pytest.mark.gpu
lib = pb.lib
BOTH = [pb.FP32, pb.BF16]


def ck(rc):
    assert rc == 0, lib.paci_last_error().decode()
    torch.cuda.synchronize()


@pytest.mark.parametrize("dtype", BOTH)
def test_ops_with_zero_rows_are_no_ops(dtype):
    D, N, K, V = 128, 256, 64, 512
    sent = 7.0
    t = lambda *shape: torch.full(shape, sent, device="cuda", dtype=DT[dtype])
    g32 = lambda *shape: torch.full(shape, sent, device="cuda")
    x, y, xs, dx = t(4, D), t(4, D), t(4, D), t(4, D)
    mean, rstd, gam, bet = g32(4), g32(4), g32(D), g32(D)
    Gg, Gb, Gc = g32(D), g32(D), g32(D)
    ck(lib.paci_op_layernorm_fwd(dtype, 0, D, x.data_ptr(), None, gam.data_ptr(), bet.data_ptr(), xs.data_ptr(), y.data_ptr(),
                                 mean.data_ptr(), rstd.data_ptr(), None))
    ck(lib.paci_op_layernorm_bwd(dtype, 0, D, y.data_ptr(), x.data_ptr(), mean.data_ptr(), rstd.data_ptr(), gam.data_ptr(),
                                 None, dx.data_ptr(), Gg.data_ptr(), Gb.data_ptr(), Gc.data_ptr(), None))
    A, B, Cout, bias, Gw = t(4, K), t(N, K), t(4, N), g32(N), g32(N, K)
    for layout in (0, 1):
        ck(lib.paci_op_gemm(dtype, layout, 0, N, K, A.data_ptr(), K, B.data_ptr(), K if layout == 0 else N, bias.data_ptr(),
                            Cout.data_ptr(), N, 0, None))
    # wgrad over zero tokens: the contraction is empty, the fp32 accumulator keeps its value (beta = 1)
    ck(lib.paci_op_gemm(dtype, 2, N, K, 0, A.data_ptr(), N, A.data_ptr(), K, None, Gw.data_ptr(), K, 1, None))
    ck(lib.paci_op_gelu_fwd(dtype, 0, x.data_ptr(), y.data_ptr(), None))
    ck(lib.paci_op_gelu_bwd(dtype, 0, D, x.data_ptr(), x.data_ptr(), dx.data_ptr(), Gb.data_ptr(), None))
    ck(lib.paci_op_colsum(dtype, 0, D, x.data_ptr(), Gc.data_ptr(), None))
    ck(lib.paci_op_dropout(dtype, 0, x.data_ptr(), y.data_ptr(), 0.1, 3, 0, 0, None))
    for buf in (y, xs, dx, Cout, mean, rstd, Gg, Gb, Gc, Gw):
        assert torch.all(buf == sent), "an op over zero rows wrote to its output"


@pytest.mark.parametrize("dtype,dh,T", [(pb.FP32, 16, 32), (pb.BF16, 64, 128)])
def test_smallest_attention_one_sequence_one_head(dtype, dh, T):
    rng = np.random.default_rng(5)
    qkv, do = rng.standard_normal((1, T, 3 * dh)), rng.standard_normal((1, T, dh))
    qd, dod = dev(qkv, dtype), dev(do, dtype)
    o = torch.empty(1, T, dh, device="cuda", dtype=DT[dtype])
    lse = torch.empty(1, 1, T, device="cuda")
    ck(lib.paci_op_attention_fwd(dtype, 1, T, 1, dh, qd.data_ptr(), o.data_ptr(), lse.data_ptr(), None))
    o_ref, stash = model.attention_fwd(rounded(qkv, dtype), 1)
    assert rel_l2(host(o), o_ref) < TOL[dtype] / 4
    # row 0 attends to itself only: o[0] = v[0] exactly (softmax over one key), whatever the scores
    assert np.allclose(host(o)[0, 0], rounded(qkv, dtype)[0, 0, 2 * dh:], rtol=1e-2 if dtype == pb.BF16 else 1e-6, atol=1e-6)
    scratch = torch.empty(lib.paci_op_attention_bwd_scratch_bytes(dtype, 1, T, 1, dh), device="cuda", dtype=torch.uint8)
    dqkv = torch.empty_like(qd)
    ck(lib.paci_op_attention_bwd(dtype, 1, T, 1, dh, dod.data_ptr(), qd.data_ptr(), o.data_ptr(), lse.data_ptr(),
                                 dqkv.data_ptr(), scratch.data_ptr(), None))
    assert rel_l2(host(dqkv), model.attention_bwd(rounded(do, dtype), stash)) < TOL[dtype] / 2


def test_one_row_gemm_and_layernorm_fp32():
    rng = np.random.default_rng(9)
    A, B, bias = rng.standard_normal((1, 40)), rng.standard_normal((24, 40)), rng.standard_normal(24)
    Ad, Bd, bd = f32(A), f32(B), f32(bias)              # named: a temporary's memory would be reused before the launch
    Cout = torch.empty(1, 24, device="cuda")
    ck(lib.paci_op_gemm(pb.FP32, 0, 1, 24, 40, Ad.data_ptr(), 40, Bd.data_ptr(), 40, bd.data_ptr(), Cout.data_ptr(), 24, 0,
                        None))
    assert rel_l2(host(Cout), A @ B.T + bias) < 1e-5
    x, g, b = rng.standard_normal((1, 64)), rng.standard_normal(64), rng.standard_normal(64)
    xd, gd, betad = f32(x), f32(g), f32(b)
    y, mean, rstd = torch.empty(1, 64, device="cuda"), torch.empty(1, device="cuda"), torch.empty(1, device="cuda")
    ck(lib.paci_op_layernorm_fwd(pb.FP32, 1, 64, xd.data_ptr(), None, gd.data_ptr(), betad.data_ptr(), None, y.data_ptr(),
                                 mean.data_ptr(), rstd.data_ptr(), None))
    y_ref, _ = model.layernorm_fwd(x, g, b)
    assert rel_l2(host(y), y_ref) < 1e-5
    assert abs(float(mean[0]) - x.mean()) < 1e-5


def test_pipeline_over_zero_microbatches_is_a_no_op():
    """Alg. 1 with an empty micro-batch stream: no forward is admitted, no update happens, the weights do not move;
    the pipeline is usable afterwards."""
    from oracle import pipeline as opipe
    V, D, H, T, mu, S, L, k = 256, 64, 4, 32, 2, 2, 1, 2
    specs = [model.StageSpec(s, S, L, D, H, T, mu, V) for s in range(S)]
    params = [synth.stage_params(77, s, S, L, D, V, T, perturbed=True) for s in range(S)]
    stages = []
    for s in range(S):
        st = pb.Stage(pb.make_config(s, S, L, D, H, T, mu, k, V, pb.FP32))
        st.load_params(params[s])
        stages.append(st)
    before = [{name: st.read(name).copy() for name in params[s]} for s, st in enumerate(stages)]
    pipe = pb.Pipeline(stages)
    tok = synth.tokens(77, 4, mu, T, V, "uniform")
    dev_tok = torch.from_numpy(tok).cuda()
    out = pipe.run(dev_tok[:0].contiguous(), 1e-3)
    assert out["version"].tolist() == [0, 0]
    assert out["n_launches"] == 0
    for s, st in enumerate(stages):
        for name, w0 in before[s].items():
            assert np.array_equal(st.read(name), w0), (s, name)
    ref = opipe.run_pipeline(specs, params, tok, k, 1e-3)
    out = pipe.run(dev_tok, 1e-3)
    assert out["delta"].tolist() == ref["delta"] and out["version"].tolist() == ref["version"]
    assert np.max(np.abs(out["loss"] - np.array(ref["losses"])) / np.array(ref["losses"])) < 1e-5
