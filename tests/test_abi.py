"""CPU test: the C-ABI shared library builds, loads, and exports every symbol include/paci.h declares
(no compute calls without a GPU); host-side validation paths that do not touch the device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pb():
    from paper_2606_07881_b200 import build
    build.build(verbose=False)
    from paper_2606_07881_b200 import binding
    return binding


def _declared():
    src = open(os.path.join(ROOT, "include", "paci.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(paci_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported_and_bound(pb):
    names = _declared()
    assert len(names) >= 30
    raw = C.CDLL(pb.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), f"libpaci.so does not export {n}"
        assert n in pb.SIGNATURES, f"binding.py does not declare {n}"
    assert set(pb.SIGNATURES) == set(names)


def test_config_validation_without_gpu(pb):
    ok = pb.make_config(0, 2, 1, 64, 4, 32, 2, 4, 256, pb.FP32)
    assert pb.lib.paci_stage_workspace_bytes(C.byref(ok)) > 0
    # params of one fp32 block + embedding: 12 D^2 + 13 D + (V + T) D
    D, V, T = 64, 256, 32
    assert pb.lib.paci_stage_param_count(C.byref(ok)) == 12 * D * D + 13 * D + (V + T) * D
    bad = pb.make_config(0, 2, 1, 66, 4, 32, 2, 4, 256, pb.FP32)      # D % H != 0
    assert pb.lib.paci_stage_workspace_bytes(C.byref(bad)) == 0
    assert b"n_heads" in pb.lib.paci_last_error()
    bad = pb.make_config(0, 2, 1, 128, 4, 64, 2, 4, 256, pb.BF16)     # bf16 needs head dim 64
    assert pb.lib.paci_stage_workspace_bytes(C.byref(bad)) == 0
    bad = pb.make_config(2, 2, 1, 64, 4, 32, 2, 4, 256, pb.FP32)      # stage index out of range
    assert pb.lib.paci_stage_workspace_bytes(C.byref(bad)) == 0


def test_workspace_holds_one_parameter_copy_and_S_minus_s_stash_slots(pb):
    """one parameter copy, no extra weight memory; stage s stashes S-s micro-batches."""
    D, H, T, mu, V = 1024, 16, 1024, 8, 50257
    sizes = []
    for s in range(4):
        cfg = pb.make_config(s, 4, 6, D, H, T, mu, 4, V, pb.BF16, has_embedding=False, has_head=False)
        sizes.append(pb.lib.paci_stage_workspace_bytes(C.byref(cfg)))
        P = pb.lib.paci_stage_param_count(C.byref(cfg))
        assert P == 6 * (12 * D * D + 13 * D)
    slot = sizes[0] - sizes[1]
    assert slot > 0 and sizes[1] - sizes[2] == slot and sizes[2] - sizes[3] == slot
    M = mu * T
    per_block = 32 * D * M          # ~32 D bytes per token per block in bf16
    assert 6 * per_block <= slot <= 6 * per_block * 1.02
    fixed = sizes[3] - slot         # params (fp32 w, m, v, G + bf16 shadow = 18 B/param) + scratch
    assert fixed < 18 * P + 14 * M * D * 2 + 40 * M * D  # no second parameter copy anywhere


def test_missing_library_fails_loudly(pb):
    with pytest.raises(ImportError, match="no CPU fallback"):
        pb.load_library("/nonexistent/libpaci.so")


def test_lr_schedule_host_function_matches_oracle(pb):
    """paci_lr_schedule (1% linear warm-up, cosine to 10% of the peak) is pure host arithmetic: every step of
    a 1000-update schedule against oracle/lr.py."""
    from oracle import lr as olr
    for peak in (3e-4, 3 * 0.5 ** 0.5 * 1e-4):
        for t in list(range(0, 30)) + list(range(30, 1100, 7)):
            want = olr.lr_at(t, 1000, 10, peak)
            assert abs(pb.lr_schedule(t, 1000, 10, peak) - want) <= 1e-7 * want, t


def test_checkpoint_and_dropout_config_validation(pb):
    ok = pb.make_config(0, 2, 1, 64, 4, 32, 2, 4, 256, pb.FP32, checkpoint=1, dropout_p=0.1, dropout_seed=5)
    base = pb.make_config(0, 2, 1, 64, 4, 32, 2, 4, 256, pb.FP32)
    assert 0 < pb.lib.paci_stage_workspace_bytes(C.byref(ok))
    assert pb.lib.paci_stage_param_count(C.byref(ok)) == pb.lib.paci_stage_param_count(C.byref(base))   # one parameter copy
    for bad in (pb.make_config(0, 2, 1, 64, 4, 32, 2, 4, 256, pb.FP32, checkpoint=2),
                pb.make_config(0, 2, 1, 64, 4, 32, 2, 4, 256, pb.FP32, dropout_p=1.0),
                pb.make_config(0, 2, 1, 128, 2, 64, 2, 4, 256, pb.BF16)):     # bf16: T % 128
        assert pb.lib.paci_stage_workspace_bytes(C.byref(bad)) == 0


def test_empty_shapes_are_decided_on_the_host():
    """Empty outputs and empty contractions never reach a kernel (so this runs without a GPU): an empty output or an
    accumulate over zero tokens is PACI_OK, an OVERWRITE from an empty contraction has no value and is PACI_EINVAL."""
    from paper_2606_07881_b200 import binding as pb
    lib = pb.lib
    p = 256                                                  # never dereferenced
    for dt in (pb.FP32, pb.BF16):
        assert lib.paci_op_gemm(dt, 0, 0, 64, 64, p, 64, p, 64, None, p, 64, 0, None) == 0
        assert lib.paci_op_gemm(dt, 2, 64, 64, 0, p, 64, p, 64, None, p, 64, 1, None) == 0
        assert lib.paci_op_gemm(dt, 0, 8, 64, 0, p, 64, p, 64, None, p, 64, 0, None) == -1
        assert b"K = 0" in lib.paci_last_error()
        assert lib.paci_op_gemm_backward_pair(dt, 0, 64, 64, p, 64, p, 64, p, 64, p, 64, p, 64, None) == 0
        assert lib.paci_op_layernorm_fwd(dt, 0, 64, p, None, p, p, None, p, p, p, None) == 0
