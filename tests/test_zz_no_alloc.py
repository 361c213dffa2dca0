"""paci_op_attention_bwd_static: the allocation-free attention backward (scratch in a static __device__ array of
PACI_ATTENTION_BWD_STATIC_MAX_BYTES inside the library) against the existing paci_op_attention_bwd, which takes
caller scratch -- same kernels, so the two must agree to the tolerance the op tests use (rel-L2 <= 1e-5 fp32,
<= 2e-2 bf16; in fact far closer).  Two calls in a row with DIFFERENT shapes and inputs: the second call finds the
first call's delta / lse2 / work counters in the shared array and must not be affected by them.

Named test_zz_* so that pytest collects it last: the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

from oracle import model
from paper_2606_07881_b200 import binding as pb
from gpu_util import DT, TOL, dev, host, rel_l2, rounded

lib = pb.lib


def _ck(rc):
    assert rc == 0, lib.paci_last_error().decode()
    torch.cuda.synchronize()


def _one_call(dtype, mu, T, H, dh, seed, check_no_alloc):
    rng = np.random.default_rng(seed)
    D = H * dh
    qkv, do = rng.standard_normal((mu, T, 3 * D)), rng.standard_normal((mu, T, D))
    qd, dod = dev(qkv, dtype), dev(do, dtype)
    o = torch.empty(mu, T, D, device="cuda", dtype=DT[dtype])
    lse = torch.empty(mu, H, T, device="cuda")
    _ck(lib.paci_op_attention_fwd(dtype, mu, T, H, dh, qd.data_ptr(), o.data_ptr(), lse.data_ptr(), None))
    # the existing path: caller-provided scratch
    nb = lib.paci_op_attention_bwd_scratch_bytes(dtype, mu, T, H, dh)
    assert nb <= pb.ATTENTION_BWD_STATIC_MAX_BYTES
    scratch = torch.empty(nb, device="cuda", dtype=torch.uint8)
    want = torch.empty_like(qd)
    _ck(lib.paci_op_attention_bwd(dtype, mu, T, H, dh, dod.data_ptr(), qd.data_ptr(), o.data_ptr(), lse.data_ptr(),
                                  want.data_ptr(), scratch.data_ptr(), None))
    # the new entry point: inputs and outputs only
    got = torch.full_like(qd, float("nan"))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    _ck(lib.paci_op_attention_bwd_static(dtype, mu, T, H, dh, dod.data_ptr(), qd.data_ptr(), o.data_ptr(),
                                         lse.data_ptr(), got.data_ptr(), None))
    free1 = torch.cuda.mem_get_info()[0]
    if check_no_alloc:                                    # (the first call of a process may load the module lazily)
        assert free1 == free0, f"device memory moved by {free0 - free1} bytes across the call"
    assert np.isfinite(host(got)).all()
    assert rel_l2(host(got), host(want)) < TOL[dtype] / 2
    # and both against the oracle, as tests/test_gpu_ops.py does for the existing path
    _, stash = model.attention_fwd(rounded(qkv, dtype), H)
    ref = model.attention_bwd(rounded(do, dtype), stash)
    assert rel_l2(host(got), ref) < TOL[dtype] / 2


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,first,second", [
    (pb.BF16, (2, 256, 3, 64), (1, 128, 2, 64)),          # tcgen05 kernels: delta, lse2 and two work counters in the array
    (pb.FP32, (2, 32, 4, 16), (1, 100, 3, 40)),           # FFMA parity kernels: delta in the array
])
def test_static_scratch_attention_backward_matches_existing_path_twice(dtype, first, second):
    _one_call(dtype, *first, seed=11, check_no_alloc=False)
    _one_call(dtype, *second, seed=12, check_no_alloc=True)       # finds the first call's contents in the array
    _one_call(dtype, *first, seed=13, check_no_alloc=True)        # and a larger shape after a smaller one


def test_static_scratch_rejects_shapes_beyond_the_array():
    """The size test precedes every CUDA call (runs without a GPU): mu*H*T = 8*32*4096 needs 8.4 MB > 4 MiB + 256."""
    assert lib.paci_op_attention_bwd_scratch_bytes(pb.BF16, 8, 4096, 32, 64) > pb.ATTENTION_BWD_STATIC_MAX_BYTES
    rc = lib.paci_op_attention_bwd_static(pb.BF16, 8, 4096, 32, 64, 256, 256, 256, 256, 256, None)
    assert rc == -1                                        # PACI_EINVAL
    msg = lib.paci_last_error().decode()
    assert "static array holds" in msg and "paci_op_attention_bwd" in msg
    assert lib.paci_op_attention_bwd_static(pb.BF16, 0, 128, 2, 64, 256, 256, 256, 256, 256, None) == -1
    assert lib.paci_op_attention_bwd_static(pb.BF16, 1, 128, 2, 64, None, 256, 256, 256, 256, None) == -1
