"""-m gpu: every kernel through the C ABI vs the oracle's layer functions, element by element, on
seeded inputs that span several tiles and a ragged tail.  fp32 mode: rel-L2 <= 1e-5; bf16: <= 2e-2."""
import numpy as np
import pytest
import torch

import synth
from oracle import adamw as oadam
from oracle import model
from paper_2606_07881_b200 import binding as pb
from gpu_util import DT, TOL, host, rel_l2, rounded
import gpu_util

_KEEP = []


def dev(a, dtype):
    """device copy that stays alive for the whole test (a temporary whose data_ptr() was taken would be
    freed and its memory handed to the next allocation before the kernel runs)"""
    t = gpu_util.dev(a, dtype)
    _KEEP.append(t)
    return t


def f32(a):
    t = gpu_util.f32(a)
    _KEEP.append(t)
    return t


def icuda(a):
    t = torch.from_numpy(a).cuda()
    _KEEP.append(t)
    return t


@pytest.fixture(autouse=True)
def _release():
    yield
    torch.cuda.synchronize()
    _KEEP.clear()

pytestmark = pytest.mark.gpu
lib = pb.lib
S0 = None  # default stream


def ck(rc):
    assert rc == 0, lib.paci_last_error().decode()
    torch.cuda.synchronize()


BOTH = [pb.FP32, pb.BF16]


@pytest.mark.parametrize("dtype", BOTH)
@pytest.mark.parametrize("rows,D", [(37, 64), (300, 768), (129, 1024), (65, 1280)])
def test_layernorm_fwd_bwd(dtype, rows, D):
    if dtype == pb.FP32 and D > 1024:
        pytest.skip("PACI_FP32 is the small parity mode: LayerNorm rows up to 1024 floats")
    rng = np.random.default_rng(rows + D)
    x, res = rng.standard_normal((rows, D)) * 2 + 0.3, rng.standard_normal((rows, D))
    g, b = 1 + 0.1 * rng.standard_normal(D), 0.1 * rng.standard_normal(D)
    dy, dres = rng.standard_normal((rows, D)), rng.standard_normal((rows, D))
    xs_ref = rounded(rounded(x, dtype) + rounded(res, dtype), dtype)        # the stored residual stream
    y_ref, (xhat, rstd) = model.layernorm_fwd(xs_ref, g.astype(np.float32).astype(np.float64),
                                              b.astype(np.float32).astype(np.float64))
    xd, rd, gd, bd = dev(x, dtype), dev(res, dtype), f32(g), f32(b)
    xsum, y = torch.empty_like(xd), torch.empty_like(xd)
    mean, rs = torch.empty(rows, device="cuda"), torch.empty(rows, device="cuda")
    ck(lib.paci_op_layernorm_fwd(dtype, rows, D, xd.data_ptr(), rd.data_ptr(), gd.data_ptr(), bd.data_ptr(),
                                 xsum.data_ptr(), y.data_ptr(), mean.data_ptr(), rs.data_ptr(), S0))
    assert rel_l2(host(xsum), xs_ref) < 1e-7
    assert rel_l2(host(y), y_ref) < TOL[dtype] / 4
    assert rel_l2(host(rs), rstd[:, 0]) < 1e-5 and rel_l2(host(mean), xs_ref.mean(-1)) < 1e-5
    # backward with a DIFFERENT (current) gain, stashed statistics (Eq. 1)
    g2 = g + 0.05 * rng.standard_normal(D)
    dyr, dresr = rounded(dy, dtype), rounded(dres, dtype)
    dx_ref, dg_ref, db_ref = model.layernorm_bwd(dyr, (xhat, rstd), g2.astype(np.float32).astype(np.float64))
    dx_ref = dx_ref + dresr
    dx = torch.empty_like(xd)
    Gg = torch.full((D,), 0.5, device="cuda"); Gb = torch.full((D,), -0.25, device="cuda")
    Gc = torch.full((D,), 1.0, device="cuda")
    dyd, dresd, g2d = dev(dy, dtype), dev(dres, dtype), f32(g2)      # named: the buffers must outlive the launch
    ck(lib.paci_op_layernorm_bwd(dtype, rows, D, dyd.data_ptr(), xsum.data_ptr(), mean.data_ptr(),
                                 rs.data_ptr(), g2d.data_ptr(), dresd.data_ptr(), dx.data_ptr(),
                                 Gg.data_ptr(), Gb.data_ptr(), Gc.data_ptr(), S0))
    assert rel_l2(host(dx), dx_ref) < TOL[dtype] / 4
    assert rel_l2(host(Gg) - 0.5, dg_ref) < TOL[dtype] / 4          # accumulates INTO G (beta = 1)
    assert rel_l2(host(Gb) + 0.25, db_ref) < TOL[dtype] / 4
    assert rel_l2(host(Gc) - 1.0, host(dx).sum(0)) < 1e-5            # column sums of what was stored


@pytest.mark.parametrize("dtype,M,N,K", [(pb.FP32, 70, 96, 40), (pb.BF16, 300, 328, 192), (pb.BF16, 512, 1024, 256)])
def test_gemm_bias_gelu(dtype, M, N, K):
    """MLP-up with the activation in the GEMM epilogue (bf16: one tcgen05 launch, two TMA-stored tiles):
    pre-activation and gelu(pre-activation) against the oracle, ragged M / N tails included."""
    rng = np.random.default_rng(M + N)
    x, W, b = rng.standard_normal((M, K)), rng.standard_normal((N, K)) * 0.2, rng.standard_normal(N)
    xr, Wr = rounded(x, dtype), rounded(W, dtype)
    p_ref, _ = model.linear_fwd(xr, Wr, b.astype(np.float32).astype(np.float64))
    Cd = torch.empty(M, N, device="cuda", dtype=DT[dtype])
    Gd = torch.empty(M, N, device="cuda", dtype=DT[dtype])
    xd, Wd, bd = dev(x, dtype), dev(W, dtype), f32(b)
    ck(lib.paci_op_gemm_bias_gelu(dtype, M, N, K, xd.data_ptr(), K, Wd.data_ptr(), K,
                                  bd.data_ptr(), Cd.data_ptr(), Gd.data_ptr(), N, S0))
    assert rel_l2(host(Cd), p_ref) < TOL[dtype] / 4
    assert rel_l2(host(Gd), model.gelu_fwd(host(Cd))) < TOL[dtype] / 4      # gelu of what was stored
    assert rel_l2(host(Gd), model.gelu_fwd(p_ref)) < TOL[dtype] / 2


@pytest.mark.parametrize("dtype", BOTH)
def test_gelu_fwd_bwd_colsum(dtype):
    rng = np.random.default_rng(5)
    rows, cols = 203, 4 * 192
    p, dg = rng.standard_normal((rows, cols)) * 2, rng.standard_normal((rows, cols))
    pr, dgr = rounded(p, dtype), rounded(dg, dtype)
    pd = dev(p, dtype)
    out = torch.empty_like(pd)
    ck(lib.paci_op_gelu_fwd(dtype, rows * cols, pd.data_ptr(), out.data_ptr(), S0))
    assert rel_l2(host(out), model.gelu_fwd(pr)) < TOL[dtype] / 4
    dp = torch.empty_like(pd)
    G = torch.full((cols,), 2.0, device="cuda")
    ck(lib.paci_op_gelu_bwd(dtype, rows, cols, dev(dg, dtype).data_ptr(), pd.data_ptr(), dp.data_ptr(),
                            G.data_ptr(), S0))
    ref = model.gelu_bwd(dgr, pr)
    assert rel_l2(host(dp), ref) < TOL[dtype] / 4
    assert rel_l2(host(G) - 2.0, ref.sum(0)) < TOL[dtype] / 4
    G2 = torch.zeros(cols, device="cuda")
    ck(lib.paci_op_colsum(dtype, rows, cols, pd.data_ptr(), G2.data_ptr(), S0))
    assert rel_l2(host(G2), pr.sum(0)) < 1e-5
    # in place (the stage runs gelu_bwd in place)
    dgd = dev(dg, dtype)
    ck(lib.paci_op_gelu_bwd(dtype, rows, cols, dgd.data_ptr(), pd.data_ptr(), dgd.data_ptr(), None, S0))
    assert torch.equal(dgd, dp)


@pytest.mark.parametrize("dtype", BOTH)
def test_embedding_fwd_bwd_zipf(dtype):
    mu, T, D, V = 3, 40, 64, 500
    rng = np.random.default_rng(6)
    tok = synth.tokens(3, 1, mu, T, V, "zipf")[0][:, :-1].copy()
    wte, wpe = rng.standard_normal((V, D)).astype(np.float32), rng.standard_normal((T, D)).astype(np.float32)
    tokd = torch.from_numpy(tok).cuda()
    x = torch.empty(mu, T, D, device="cuda", dtype=DT[dtype])
    wted, wped = f32(wte), f32(wpe)
    ck(lib.paci_op_embed_fwd(dtype, mu, T, D, V, tokd.data_ptr(), wted.data_ptr(), wped.data_ptr(),
                             x.data_ptr(), S0))
    assert rel_l2(host(x), model.embed_fwd(tok.astype(np.int64), wte.astype(np.float64), wpe.astype(np.float64))) \
        < TOL[dtype] / 4
    dx = rng.standard_normal((mu, T, D))
    dwte, dwpe = model.embed_bwd(rounded(dx, dtype), tok.astype(np.int64), V)
    Gwte, Gwpe = torch.zeros(V, D, device="cuda"), torch.zeros(T, D, device="cuda")
    ck(lib.paci_op_embed_bwd(dtype, mu, T, D, V, tokd.data_ptr(), dev(dx, dtype).data_ptr(), Gwte.data_ptr(),
                             Gwpe.data_ptr(), S0))
    assert rel_l2(host(Gwte), dwte) < 1e-5 and rel_l2(host(Gwpe), dwpe) < 1e-5
    assert np.all(host(Gwte)[np.setdiff1d(np.arange(V), tok)] == 0)


@pytest.mark.parametrize("dtype", BOTH)
@pytest.mark.parametrize("rows,V", [(19, 256), (33, 50257), (700, 5000)])   # 700 rows: every persistent block wraps its two row buffers
def test_softmax_cross_entropy(dtype, rows, V):
    rng = np.random.default_rng(V)
    ldz = (V + 63) // 64 * 64
    z = rng.standard_normal((rows, V)) * 3
    tgt = rng.integers(0, V, rows).astype(np.int32)
    zp = np.full((rows, ldz), 7.0)      # garbage in the padding must be ignored and overwritten by 0
    zp[:, :V] = z
    zd = dev(zp, dtype)
    loss = torch.zeros(1, device="cuda")
    ck(lib.paci_op_softmax_ce(dtype, rows, V, ldz, zd.data_ptr(), icuda(tgt).data_ptr(),
                              loss.data_ptr(), S0))
    lref, dz = model.cross_entropy_fwd_bwd(rounded(z, dtype)[None], tgt.astype(np.int64)[None])
    assert abs(loss.item() - lref) / lref < 1e-5
    got = host(zd)
    assert np.all(got[:, V:] == 0)
    assert rel_l2(got[:, :V], dz[0]) < TOL[dtype] / 4


def test_adamw_flat_arena_matches_oracle_over_steps():
    rng = np.random.default_rng(8)
    n, n_decay, k = 4096 + 260, 2048, 4
    w0 = rng.standard_normal(n).astype(np.float32)
    w, m, v = f32(w0), torch.zeros(n, device="cuda"), torch.zeros(n, device="cuda")
    shadow = torch.empty(n, device="cuda", dtype=torch.bfloat16)
    ver = torch.zeros(1, device="cuda", dtype=torch.int64)
    th = w0.astype(np.float64); mo = np.zeros(n); vo = np.zeros(n)
    for t in range(1, 6):
        G = (rng.standard_normal(n) * 3).astype(np.float32)
        Gd = f32(G)
        ck(lib.paci_op_adamw(n, n_decay, w.data_ptr(), m.data_ptr(), v.data_ptr(), Gd.data_ptr(),
                             shadow.data_ptr(), k, t, 1e-2, 0.9, 0.95, 1e-8, 0.1, ver.data_ptr(), S0))
        oadam.adamw_update(th[:n_decay], mo[:n_decay], vo[:n_decay], G[:n_decay].astype(np.float64), k, t, 1e-2, True)
        oadam.adamw_update(th[n_decay:], mo[n_decay:], vo[n_decay:], G[n_decay:].astype(np.float64), k, t, 1e-2, False)
        assert torch.count_nonzero(Gd).item() == 0                      # G reset (Alg. 1 line 18)
        assert ver.item() == t                                          # device version word bumped
        assert rel_l2(host(w), th) < 1e-6 and rel_l2(host(m), mo) < 1e-6 and rel_l2(host(v), vo) < 1e-6
        assert torch.equal(shadow, w.to(torch.bfloat16))
    # weight DELTA of a step (SURVEY 8(c) note: ~lr*sign(g) on the first step)
    assert rel_l2(host(w) - w0, th - w0) < 1e-4


GEMM_SHAPES = [(64, 64, 64), (130, 72, 40), (256, 384, 128), (300, 520, 264)]


@pytest.mark.parametrize("dtype", BOTH)
@pytest.mark.parametrize("layout", [0, 1, 2])
@pytest.mark.parametrize("M,N,K", GEMM_SHAPES)
def test_gemm_layouts(dtype, layout, M, N, K):
    rng = np.random.default_rng(M * 7 + N * 3 + K + layout)
    A = rng.standard_normal((M, K)); B = rng.standard_normal((N, K)); bias = rng.standard_normal(N)
    Ar, Br = rounded(A, dtype), rounded(B, dtype)
    ref = Ar @ Br.T
    def padded(a):                                      # row stride rounded up to 8 elements (16 B in bf16),
        ld = (a.shape[1] + 7) // 8 * 8                  # with garbage in the padding: ld != extent is exercised
        buf = np.full((a.shape[0], ld), 9.0)
        buf[:, :a.shape[1]] = a
        return dev(buf, dtype), ld
    Ad, lda = padded(A if layout != 2 else A.T)         # TN: A stored [K, M]
    Bd, ldb = padded(B if layout == 0 else B.T)         # NN/TN: B stored [K, N]
    Cd = torch.empty(M, N, device="cuda", dtype=DT[dtype])
    ck(lib.paci_op_gemm(dtype, layout, M, N, K, Ad.data_ptr(), lda, Bd.data_ptr(), ldb, f32(bias).data_ptr(),
                        Cd.data_ptr(), N, 0, S0))
    assert rel_l2(host(Cd), ref + bias.astype(np.float32)) < TOL[dtype] / 4
    Cf = torch.full((M, N), 3.0, device="cuda")
    for _ in range(2):                                   # beta = 1: accumulates across calls
        ck(lib.paci_op_gemm(dtype, layout, M, N, K, Ad.data_ptr(), lda, Bd.data_ptr(), ldb, None,
                            Cf.data_ptr(), N, 1, S0))
    assert rel_l2(host(Cf) - 3.0, 2 * ref) < (1e-5 if dtype == pb.FP32 else 1e-4)


@pytest.mark.parametrize("dtype,mu,T,H,dh", [(pb.FP32, 2, 32, 4, 16), (pb.FP32, 1, 100, 3, 40),
                                              (pb.BF16, 2, 128, 3, 64), (pb.BF16, 1, 256, 2, 64),
                                              (pb.BF16, 2, 384, 2, 64), (pb.BF16, 1, 512, 1, 64)])
def test_attention_fwd_bwd(dtype, mu, T, H, dh):
    rng = np.random.default_rng(T + H)
    D = H * dh
    qkv, do = rng.standard_normal((mu, T, 3 * D)), rng.standard_normal((mu, T, D))
    if T == 512:   # large scores: the running max keeps growing, which exercises the tcgen05 kernel's lazy rescale
        qkv[..., :2 * D] *= 3.0
    qkvr, dor = rounded(qkv, dtype), rounded(do, dtype)
    o_ref, stash = model.attention_fwd(qkvr, H)
    qd = dev(qkv, dtype)
    o = torch.empty(mu, T, D, device="cuda", dtype=DT[dtype])
    lse = torch.empty(mu, H, T, device="cuda")
    ck(lib.paci_op_attention_fwd(dtype, mu, T, H, dh, qd.data_ptr(), o.data_ptr(), lse.data_ptr(), S0))
    assert rel_l2(host(o), o_ref) < TOL[dtype] / 4
    q, k = stash[0], stash[1]
    s = np.where(np.tril(np.ones((T, T), bool)), q @ k.transpose(0, 1, 3, 2) / np.sqrt(dh), -np.inf)
    lse_ref = np.log(np.exp(s - s.max(-1, keepdims=True)).sum(-1)) + s.max(-1)
    assert rel_l2(host(lse), lse_ref) < (1e-3 if dtype == pb.BF16 else 1e-5)
    dq_ref = model.attention_bwd(dor, stash)
    nb = lib.paci_op_attention_bwd_scratch_bytes(dtype, mu, T, H, dh)
    scratch = torch.empty(nb, device="cuda", dtype=torch.uint8)
    dqkv = torch.empty_like(qd)
    ck(lib.paci_op_attention_bwd(dtype, mu, T, H, dh, dev(do, dtype).data_ptr(), qd.data_ptr(), o.data_ptr(),
                                 lse.data_ptr(), dqkv.data_ptr(), scratch.data_ptr(), S0))
    assert rel_l2(host(dqkv), dq_ref) < TOL[dtype] / 2


@pytest.mark.parametrize("dtype", BOTH)
def test_dropout_mask_is_bitwise_the_oracles(dtype):
    """the CUDA kernel and oracle/dropout.py evaluate the same counter-based generator on
    the same counters, so the keep / drop decision is an integer result: it must agree EXACTLY, element by element,
    over several blocks and a ragged tail; kept values are x / (1 - p) within rounding."""
    from oracle import dropout as odrop
    rng = np.random.default_rng(2)
    n, p, seed, mb, site = 8 * 1237, 0.1, 0x1234567887654321, 70000, 5
    x = rng.standard_normal(n) + 3.0                                       # no zeros: a 0 output means "dropped"
    xd = dev(x, dtype)
    out = torch.empty_like(xd)
    ck(lib.paci_op_dropout(dtype, n, xd.data_ptr(), out.data_ptr(), p, seed, mb, site, S0))
    m = odrop.mask((n,), p, seed, mb, site)
    got = host(out)
    assert np.array_equal(got != 0, m != 0)                                # bit-exact mask
    assert rel_l2(got, rounded(x, dtype) * m) < (1e-6 if dtype == pb.FP32 else TOL[dtype] / 4)
    ck(lib.paci_op_dropout(dtype, n, xd.data_ptr(), xd.data_ptr(), p, seed, mb, site, S0))   # in place
    assert torch.equal(xd, out)
    ck(lib.paci_op_dropout(dtype, n, out.data_ptr(), xd.data_ptr(), 0.0, seed, mb, site, S0))  # p = 0: identity
    assert torch.equal(xd, out)


def test_out_of_range_token_ids_are_clamped_not_dereferenced():
    mu, T, D, V = 1, 8, 64, 50
    tok = np.array([[0, 49, 50, -1, 7, 1000000, 3, 4]], np.int32)
    wte = np.arange(V * D, dtype=np.float32).reshape(V, D) / 100
    wpe = np.zeros((T, D), np.float32)
    x = torch.empty(mu, T, D, device="cuda")
    ck(lib.paci_op_embed_fwd(pb.FP32, mu, T, D, V, icuda(tok).data_ptr(), f32(wte).data_ptr(), f32(wpe).data_ptr(),
                             x.data_ptr(), S0))
    got = host(x)[0]
    for t, want in enumerate([0, 49, 49, 0, 7, 49, 3, 4]):
        assert np.array_equal(got[t], wte[want].astype(np.float64))


@pytest.mark.parametrize("dtype", BOTH)
@pytest.mark.parametrize("M,N_out,K_in", [(130, 72, 40), (384, 256, 512), (300, 520, 264), (1024, 1024, 256)])
def test_gemm_backward_pair(dtype, M, N_out, K_in):
    """Rows a13 + a14 in ONE launch (bf16): dx = dy W with the current W (Eq. 1) and G_W += dy^T x (Alg. 1 line 13),
    the wgrad's k-blocks poured over the CTA pairs on top of the dgrad's tiles; G pre-filled and the call repeated
    (beta = 1), ragged M / N / K tails, row strides wider than the extents."""
    rng = np.random.default_rng(M + N_out + K_in)
    dy, x, W = rng.standard_normal((M, N_out)), rng.standard_normal((M, K_in)), rng.standard_normal((N_out, K_in)) * 0.3
    dyr, xr, Wr = rounded(dy, dtype), rounded(x, dtype), rounded(W, dtype)
    dx_ref, dW_ref, _ = model.linear_bwd(dyr, xr, Wr)
    def padded(a):
        ld = (a.shape[1] + 7) // 8 * 8 + 8
        buf = np.full((a.shape[0], ld), 9.0)
        buf[:, :a.shape[1]] = a
        return dev(buf, dtype), ld
    dyd, ld_dy = padded(dy); xd, ld_x = padded(x); Wd, ld_w = padded(W)
    G = torch.full((N_out, K_in), 3.0, device="cuda")
    dx = torch.empty(M, K_in, device="cuda", dtype=DT[dtype])
    for _ in range(2):
        ck(lib.paci_op_gemm_backward_pair(dtype, M, N_out, K_in, dyd.data_ptr(), ld_dy, xd.data_ptr(), ld_x, Wd.data_ptr(),
                                          ld_w, G.data_ptr(), K_in, dx.data_ptr(), K_in, S0))
    assert rel_l2(host(dx), dx_ref) < TOL[dtype] / 4
    assert rel_l2(host(G) - 3.0, 2 * dW_ref) < (1e-5 if dtype == pb.FP32 else 1e-4)


@pytest.mark.parametrize("dtype,mu,T,H,dh", [(pb.BF16, 2, 128, 3, 64), (pb.BF16, 1, 384, 4, 64), (pb.BF16, 3, 256, 5, 64),
                                              (pb.FP32, 2, 32, 4, 16)])
def test_out_proj_backward_prepares_attention_backward(dtype, mu, T, H, dh):
    """Rows a13 + a14 of the output projection with the prologue of a17 in the dgrad's epilogue (bf16 / tcgen05):
    d_o = dy Wo, G_Wo += dy^T o, and scratch <- delta = rowsum_d(d_o * o) per head, lse log2(e).  Checked against the
    oracle's linear and attention backward (the latter fed the d_o the GPU stored), and delta against its definition;
    D = H 64 spans one ragged 256-column tile (H = 3, 5) and several row tiles.  fp32: the plain pair, prepared = 0."""
    import ctypes
    rng = np.random.default_rng(7 * T + H)
    D, M = H * dh, mu * T
    qkv = rng.standard_normal((mu, T, 3 * D))
    dy, Wo = rng.standard_normal((M, D)), rng.standard_normal((D, D)) * 0.2
    qkvr, dyr, Wr = rounded(qkv, dtype), rounded(dy, dtype), rounded(Wo, dtype)
    qd = dev(qkv, dtype)
    o = torch.empty(mu, T, D, device="cuda", dtype=DT[dtype])
    lse = torch.empty(mu, H, T, device="cuda")
    ck(lib.paci_op_attention_fwd(dtype, mu, T, H, dh, qd.data_ptr(), o.data_ptr(), lse.data_ptr(), S0))
    o_host = host(o).reshape(M, D)
    do_ref, dW_ref, _ = model.linear_bwd(dyr, o_host, Wr)
    nb = lib.paci_op_attention_bwd_scratch_bytes(dtype, mu, T, H, dh)
    scratch = torch.full((nb // 4 + 1,), float("nan"), device="cuda")
    G = torch.full((D, D), 3.0, device="cuda")
    d_o = torch.empty(M, D, device="cuda", dtype=DT[dtype])
    prepared = ctypes.c_int(-1)
    ck(lib.paci_op_out_proj_backward(dtype, mu, T, H, dh, dev(dy, dtype).data_ptr(), o.data_ptr(), dev(Wo, dtype).data_ptr(),
                                     G.data_ptr(), d_o.data_ptr(), lse.data_ptr(), scratch.data_ptr(),
                                     ctypes.addressof(prepared), S0))
    assert prepared.value == (1 if dtype == pb.BF16 else 0)
    assert rel_l2(host(d_o), do_ref) < TOL[dtype] / 4
    assert rel_l2(host(G) - 3.0, dW_ref) < (1e-5 if dtype == pb.FP32 else 1e-4)
    do_host = host(d_o)                                    # what the GPU stored (bf16-rounded): backward's input
    if prepared.value:
        n = mu * H * T
        delta = host(scratch[:n]).reshape(mu, H, T)
        lse2 = host(scratch[n:2 * n]).reshape(mu, H, T)
        want = (do_host.reshape(mu, T, H, dh) * o_host.reshape(mu, T, H, dh)).sum(-1).transpose(0, 2, 1)
        assert np.abs(delta - want).max() < 1e-4 * max(1.0, np.abs(want).max())
        assert np.allclose(lse2, host(lse) * np.log2(np.e), rtol=1e-6, atol=1e-6)
    _, stash = model.attention_fwd(qkvr, H)
    dq_ref = model.attention_bwd(do_host.reshape(mu, T, D), stash)
    dqkv = torch.empty_like(qd)
    ck(lib.paci_op_attention_bwd_prepared(dtype, mu, T, H, dh, d_o.data_ptr(), qd.data_ptr(), o.data_ptr(),
                                          lse.data_ptr(), dqkv.data_ptr(), scratch.data_ptr(), S0))
    assert rel_l2(host(dqkv), dq_ref) < TOL[dtype] / 2
    dqkv2 = torch.empty_like(qd)
    ck(lib.paci_op_attention_bwd(dtype, mu, T, H, dh, d_o.data_ptr(), qd.data_ptr(), o.data_ptr(),
                                 lse.data_ptr(), dqkv2.data_ptr(), scratch.data_ptr(), S0))
    assert rel_l2(host(dqkv), host(dqkv2)) < 1e-3
