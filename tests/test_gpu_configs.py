"""-m gpu: parity on the paths bench.py takes for BASELINE.json configs[1] (GPT-2-small shape, D 768, H 12),
configs[2] (the LM-head wgrad at micro-batch 8: the range-mode split-K decomposition) and configs[4] (GPT-2-Large
shape, D 1280, H 20, micro-batch 16, single stage with the TIED head), on sampled outputs the oracle can compute one
by one, and whole stages at full width with micro-batch 1.  bf16 gates: rel-L2 <= 2e-2 (BASELINE.json north_star)."""
import numpy as np
import pytest
import torch

import synth
from oracle import model
from paper_2606_07881_b200 import binding as pb
from gpu_util import TOL, host, rel_l2, rounded
import gpu_util

pytestmark = pytest.mark.gpu
lib = pb.lib
T, V = 1024, 50257


def ck(rc):
    assert rc == 0, lib.paci_last_error().decode()


def S0():
    return torch.cuda.current_stream().cuda_stream


def _gemm_sampled(layout, Mg, Ng, Kg, accum, calls=1, n_rows=20, extra_rows=()):
    """paci_op_gemm (bf16) on random operands; returns (plan, worst rel-L2 over sampled output rows) against fp64 dot
    products of the rounded operands.  Operand rows / columns are gathered on the device, so K = 16384 x M = 50257 fits."""
    g = torch.Generator(device="cuda").manual_seed(layout * 13 + Kg + Ng)
    rng = np.random.default_rng(layout * 7 + Ng + Mg)
    a_shape = (Mg, Kg) if layout != 2 else (Kg, Mg)
    b_shape = (Ng, Kg) if layout == 0 else (Kg, Ng)
    lda = (a_shape[1] + 7) // 8 * 8                          # 16-byte row stride (M = 50257 is odd)
    A = torch.zeros(a_shape[0], lda, device="cuda", dtype=torch.bfloat16)
    A[:, :a_shape[1]] = (torch.randn(a_shape, device="cuda", generator=g) * 0.5).to(torch.bfloat16)
    B = (torch.randn(b_shape, device="cuda", generator=g) * 0.5).to(torch.bfloat16)
    bias = torch.randn(Ng, device="cuda", generator=g) if not accum else None
    C = torch.full((Mg, Ng), 2.0, device="cuda") if accum else torch.empty(Mg, Ng, device="cuda", dtype=torch.bfloat16)
    for _ in range(calls):
        ck(lib.paci_op_gemm(pb.BF16, layout, Mg, Ng, Kg, A.data_ptr(), lda, B.data_ptr(), b_shape[1],
                            bias.data_ptr() if bias is not None else None, C.data_ptr(), Ng, accum, S0()))
    plan = pb.gemm_last_plan()
    torch.cuda.synchronize()
    rows = np.unique(np.concatenate([rng.integers(0, Mg, n_rows), [0, min(255, Mg - 1), min(256, Mg - 1), Mg - 1],
                                     np.asarray(extra_rows, dtype=np.int64)]))
    ridx = torch.from_numpy(rows).cuda()
    a_rows = host(A[ridx, :Kg]) if layout != 2 else host(A[:, ridx]).T          # [n, K]
    Bm = host(B).T if layout == 0 else host(B)                                   # [K, N]
    ref = a_rows @ Bm * calls + (host(bias) if bias is not None else 2.0)
    got = host(C[ridx])
    worst = max(rel_l2(got[i], ref[i]) for i in range(len(rows)))
    return plan, worst


def test_lm_head_wgrad_takes_range_mode_and_matches():
    """Alg. 1 line 13 for G_head at the shape bench.py runs (configs[2], micro-batch 8): [50257, 1024] +=
    dz^T xf over K = 8192 tokens.  788 tiles x 128 k-blocks on 74 CTA pairs: the launcher cuts the (tile, k-block)
    space into equal contiguous ranges (range mode), flushing partial accumulators through the TMA reduce-add
    wherever a range crosses a tile.  The test ASSERTS that decomposition was taken, samples rows on both sides of
    many worker-range boundaries, pre-fills C and calls twice (beta = 1)."""
    Mg, Ng, Kg = V, 1024, 8192
    # a worker's range is units / workers = 788 * 128 / 74 k-blocks: rows around every boundary tile
    tiles_m = (Mg + 255) // 256
    per = tiles_m * 4 * 128 / 74
    edge_rows = sorted({min(Mg - 1, int((w * per // 128) % tiles_m) * 256 + off) for w in range(1, 74, 5) for off in (0, 131)})
    plan, worst = _gemm_sampled(2, Mg, Ng, Kg, 1, calls=2, n_rows=24, extra_rows=edge_rows)
    assert plan["range_mode"] == 1 and plan["tiles"] == 788 and plan["cta_group"] == 2, plan
    assert worst < 1e-4, worst


@pytest.mark.parametrize("Mg,Ng,Kg,want_range", [(V, 1280, 16384, 1), (V, 768, 8192, None)])
def test_lm_head_wgrad_other_configs(Mg, Ng, Kg, want_range):
    """The same for configs[4] (D 1280, micro-batch 16: K = 16384 tokens) and configs[1] (D 768)."""
    plan, worst = _gemm_sampled(2, Mg, Ng, Kg, 1, calls=2, n_rows=16)
    if want_range is not None:
        assert plan["range_mode"] == want_range, plan
    assert worst < 1e-4, (plan, worst)


SHAPES = []
for D_, M_ in ((768, 8192), (1280, 16384)):
    SHAPES += [(0, M_, 3 * D_, D_, 0), (0, M_, D_, D_, 0), (0, M_, 4 * D_, D_, 0), (0, M_, D_, 4 * D_, 0),      # forward
               (1, M_, D_, 3 * D_, 0), (1, M_, D_, D_, 0), (1, M_, 4 * D_, D_, 0), (1, M_, D_, 4 * D_, 0),      # dgrad
               (2, 3 * D_, D_, M_, 1), (2, D_, D_, M_, 1), (2, 4 * D_, D_, M_, 1), (2, D_, 4 * D_, M_, 1)]      # wgrad


@pytest.mark.parametrize("layout,Mg,Ng,Kg,accum", SHAPES)
def test_gemm_block_shapes_of_small_and_large_configs(layout, Mg, Ng, Kg, accum):
    """Every GEMM of one block at D = 768 (configs[1], M = 8192) and D = 1280 (configs[4], M = 16384): k-block counts
    12 and 20, N = 1280 = 5 x 256 tile tails, split-K wgrads with the beta = 1 epilogue."""
    plan, worst = _gemm_sampled(layout, Mg, Ng, Kg, accum, calls=2 if accum else 1, n_rows=12)
    assert worst < (5e-3 if not accum else 1e-4), (plan, worst)


@pytest.mark.parametrize("H,mu", [(12, 8), (20, 4)])
def test_attention_T1024_heads_of_small_and_large_configs(H, mu):
    """tcgen05 attention forward / backward at T = 1024 with H = 12 (D 768) and H = 20 (D 1280): sampled (batch, head)
    pairs against the oracle run on that head alone; lse as well."""
    D = H * 64
    rng = np.random.default_rng(H)
    qd = gpu_util.dev(rng.standard_normal((mu, T, 3 * D)) * 0.7, pb.BF16)
    dod = gpu_util.dev(rng.standard_normal((mu, T, D)) * 0.1, pb.BF16)
    o = torch.empty(mu, T, D, device="cuda", dtype=torch.bfloat16)
    lse = torch.empty(mu, H, T, device="cuda")
    ck(lib.paci_op_attention_fwd(pb.BF16, mu, T, H, 64, qd.data_ptr(), o.data_ptr(), lse.data_ptr(), S0()))
    scratch = torch.empty(lib.paci_op_attention_bwd_scratch_bytes(pb.BF16, mu, T, H, 64), device="cuda", dtype=torch.uint8)
    dqkv = torch.empty_like(qd)
    ck(lib.paci_op_attention_bwd(pb.BF16, mu, T, H, 64, dod.data_ptr(), qd.data_ptr(), o.data_ptr(), lse.data_ptr(),
                                 dqkv.data_ptr(), scratch.data_ptr(), S0()))
    torch.cuda.synchronize()
    for b, h in [(0, 0), (mu - 1, H - 1), (mu // 2, H // 2)]:
        cols = [slice(i * D + h * 64, i * D + (h + 1) * 64) for i in range(3)]
        one = np.concatenate([host(qd[b:b + 1, :, c]) for c in cols], axis=-1)          # [1, T, 192]
        o_ref, stash = model.attention_fwd(one, 1)
        sl = slice(h * 64, (h + 1) * 64)
        assert rel_l2(host(o[b, :, sl]), o_ref[0]) < TOL[pb.BF16] / 4, (b, h)
        q, k = stash[0], stash[1]
        s = np.where(np.tril(np.ones((T, T), bool)), q[0, 0] @ k[0, 0].T / 8.0, -np.inf)
        lse_ref = np.log(np.exp(s - s.max(-1, keepdims=True)).sum(-1)) + s.max(-1)
        assert rel_l2(host(lse[b, h]), lse_ref) < 1e-3
        d_ref = model.attention_bwd(host(dod[b:b + 1, :, sl]), stash)[0]
        got = np.concatenate([host(dqkv[b, :, c]) for c in cols], axis=-1)
        assert rel_l2(got, d_ref) < TOL[pb.BF16] / 2, (b, h)


def _stage_vs_oracle(D, H, s, S, L, mu=1, seed=3):
    spec = model.StageSpec(s, S, L, D, H, T, mu, V)
    params = synth.stage_params(seed, s, S, L, D, V, T, perturbed=True)
    st = pb.Stage(pb.make_config(s, S, L, D, H, T, mu, 1, V, pb.BF16))
    st.load_params(params)
    rng = np.random.default_rng(17)
    tok = synth.tokens(17, 1, mu, T, V, "zipf")[0]
    inp_tok, tgt = tok[:, :-1].copy(), tok[:, 1:].copy()
    h = rounded(rng.standard_normal((mu, T, D)), pb.BF16)
    dout = rounded(rng.standard_normal((mu, T, D)) * 0.1, pb.BF16)
    P = {n: np.asarray(a, np.float64) for n, a in params.items()}
    ref_out, stash = model.stage_forward(spec, P, inp_tok.astype(np.int64) if spec.has_embedding else h,
                                         tgt.astype(np.int64) if spec.has_head else None)
    ref_din, ref_g = model.stage_backward(spec, P, stash, None if spec.has_head else dout)
    inp = torch.from_numpy(inp_tok).cuda() if spec.has_embedding else gpu_util.dev(h, pb.BF16)
    tg = torch.from_numpy(tgt).cuda() if spec.has_head else None
    out = torch.zeros(1, device="cuda") if spec.has_head else torch.empty(mu, T, D, device="cuda", dtype=torch.bfloat16)
    din = None if spec.has_embedding else torch.empty(mu, T, D, device="cuda", dtype=torch.bfloat16)
    dd = None if spec.has_head else gpu_util.dev(dout, pb.BF16)
    st.forward(0, inp, tg, out)
    st.backward(0, dd, din)
    torch.cuda.synchronize()
    st.check_inputs()
    if spec.has_head:
        assert abs(out.item() - ref_out) / abs(ref_out) < 5e-3
    else:
        assert rel_l2(host(out), ref_out) < TOL[pb.BF16]
    if not spec.has_embedding:
        assert rel_l2(host(din), ref_din) < TOL[pb.BF16]
    for name, g in ref_g.items():
        got = st.read(name, pb.GRAD_ACCUM)
        assert rel_l2(got, g) < TOL[pb.BF16], (name, rel_l2(got, g))
    st.close()


@pytest.mark.parametrize("D,H", [(768, 12), (1280, 20)])
def test_interior_block_full_width_small_and_large(D, H):
    """One interior block at D = 768 / H = 12 and D = 1280 / H = 20, T = 1024, micro-batch 1: output, input gradient and
    every accumulated parameter gradient against the oracle."""
    _stage_vs_oracle(D, H, 1, 3, 1)


def test_head_stage_full_width_small():
    _stage_vs_oracle(768, 12, 3, 4, 0)


def test_single_stage_tied_head_bf16_full_vocab():
    """configs[4]'s structure: ONE stage holding the embedding, a block and the TIED head (R10: one tensor, the
    gradient of wte is the head wgrad PLUS the embedding scatter-add) at D = 1280, H = 20, V = 50257, T = 1024."""
    _stage_vs_oracle(1280, 20, 0, 1, 1)


@pytest.mark.parametrize("M,N_out,K_in", [(8192, 1024, 1024), (8192, 1024, 4096), (8192, 4096, 1024), (8192, 3072, 1024),
                                          (16384, 1280, 5120), (8192, 2304, 768)])
def test_backward_pair_full_size_sampled(M, N_out, K_in):
    """The one-launch dgrad + wgrad pair at the block shapes of configs[2] (and one each of configs[4], configs[1]):
    sampled rows of dx and of G_W (pre-filled, beta = 1) against fp64 dot products; the plan must be the paired one."""
    g = torch.Generator(device="cuda").manual_seed(M + N_out + K_in)
    rng = np.random.default_rng(N_out + K_in)
    dy = (torch.randn(M, N_out, device="cuda", generator=g) * 0.5).to(torch.bfloat16)
    x = (torch.randn(M, K_in, device="cuda", generator=g) * 0.5).to(torch.bfloat16)
    W = (torch.randn(N_out, K_in, device="cuda", generator=g) * 0.5).to(torch.bfloat16)
    G = torch.full((N_out, K_in), 2.0, device="cuda")
    dx = torch.empty(M, K_in, device="cuda", dtype=torch.bfloat16)
    ck(lib.paci_op_gemm_backward_pair(pb.BF16, M, N_out, K_in, dy.data_ptr(), N_out, x.data_ptr(), K_in, W.data_ptr(), K_in,
                                      G.data_ptr(), K_in, dx.data_ptr(), K_in, S0()))
    plan = pb.gemm_last_plan()
    assert plan["range_mode"] == 2 and plan["grid"] == 148, plan               # the shared, water-filled grid
    torch.cuda.synchronize()
    rows = torch.from_numpy(np.unique(np.concatenate([rng.integers(0, M, 12), [0, 255, 256, M - 1]]))).cuda()
    ref = host(dy[rows]) @ host(W)
    got = host(dx[rows])
    assert max(rel_l2(got[i], ref[i]) for i in range(len(rows))) < 5e-3
    grow = torch.from_numpy(np.unique(np.concatenate([rng.integers(0, N_out, 12), [0, 255, 256, N_out - 1]]))).cuda()
    gref = host(dy[:, grow]).T @ host(x) + 2.0
    ggot = host(G[grow])
    assert max(rel_l2(ggot[i], gref[i]) for i in range(len(grow))) < 1e-4
