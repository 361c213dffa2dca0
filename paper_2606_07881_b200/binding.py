"""Thin ctypes binding of libpaci.so -- argument marshalling only.

Same names as include/paci.h.  PyTorch is used for device memory and streams, nothing else: every
step of the path runs in the library's CUDA kernels.  Importing this module FAILS LOUDLY if the
shared library has not been built (`python -m paper_2606_07881_b200.build`); there is no CPU or
PyTorch fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpaci.so")

OK, EINVAL, EAGAIN, ESTATE, ECUDA = 0, -1, -2, -3, -4
FP32, BF16 = 0, 1
PARAM, GRAD_ACCUM, ADAM_M, ADAM_V = 0, 1, 2, 3
MODE_PACI, MODE_FLUSH = 0, 1


class StageConfig(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "stage_index", "n_stages", "n_layers", "d_model", "n_heads", "seq_len", "micro_batch", "k_accum",
        "vocab", "has_embedding", "has_head", "dtype")] + [(n, C.c_float) for n in (
            "beta1", "beta2", "eps", "weight_decay")] + [
        ("checkpoint", C.c_int32), ("dropout_p", C.c_float), ("dropout_seed", C.c_uint64)]


class RunReport(C.Structure):
    _fields_ = [("loss", C.POINTER(C.c_float)), ("delta", C.POINTER(C.c_int32)),
                ("version", C.POINTER(C.c_int64)), ("max_q", C.POINTER(C.c_int32)),
                ("n_slots", C.c_int64), ("n_launches", C.c_int64), ("elapsed_ms", C.c_float)]


class ProfEntry(C.Structure):
    _fields_ = [("launches", C.c_int64), ("sampled", C.c_int64)] + [(n, C.c_double) for n in (
        "flops", "bytes", "sampled_flops", "sampled_bytes", "sampled_ms")]


PROF_NCAT = 15
ATTENTION_BWD_STATIC_MAX_BYTES = 4 * 1024 * 1024 + 256   # PACI_ATTENTION_BWD_STATIC_MAX_BYTES (include/paci.h)

# name -> (restype, argtypes); every symbol include/paci.h declares
_vp, _i, _i64, _sz, _f = C.c_void_p, C.c_int, C.c_int64, C.c_size_t, C.c_float
SIGNATURES = {
    "paci_stage_workspace_bytes": (_sz, [C.POINTER(StageConfig)]),
    "paci_stage_param_count": (_sz, [C.POINTER(StageConfig)]),
    "paci_stage_create": (_i, [C.POINTER(StageConfig), _vp, _sz, _vp, C.POINTER(_vp)]),
    "paci_stage_destroy": (_i, [_vp]),
    "paci_stage_tensor_numel": (_sz, [_vp, C.c_char_p]),
    "paci_stage_load": (_i, [_vp, _i, C.c_char_p, _vp, _sz, _vp]),
    "paci_stage_read": (_i, [_vp, _i, C.c_char_p, _vp, _sz, _vp]),
    "paci_forward": (_i, [_vp, _i64, _vp, _vp, _vp, _vp]),
    "paci_forward_var": (_i, [_vp, _i64, C.c_int32, _vp, _vp, _vp, _vp]),
    "paci_backward": (_i, [_vp, _i64, _vp, _vp, _vp]),
    "paci_maybe_step": (_i, [_vp, _f, _vp]),
    "paci_lr_schedule": (_f, [_i64, _i64, _i64, _f, _f]),
    "paci_stage_set_state": (_i, [_vp, _i64, C.c_int32, _vp]),
    "paci_stage_check": (_i, [_vp, _vp]),
    "paci_version": (_i64, [_vp]),
    "paci_unresolved": (C.c_int32, [_vp]),
    "paci_window_count": (C.c_int32, [_vp]),
    "paci_crossed_updates": (C.c_int32, [_vp, _i64]),
    "paci_stage_device_stamps": (_i, [_vp, _i64, C.POINTER(_i64), C.POINTER(_i64), _vp]),
    "paci_last_error": (C.c_char_p, []),
    "paci_pipeline_workspace_bytes": (_sz, [C.POINTER(_vp), C.c_int32]),
    "paci_pipeline_create": (_i, [C.POINTER(_vp), C.c_int32, _vp, _sz, C.POINTER(_vp)]),
    "paci_pipeline_destroy": (_i, [_vp]),
    "paci_pipeline_run": (_i, [_vp, _vp, C.c_int32, _i64, C.c_int32, _f, _vp, C.POINTER(RunReport)]),
    "paci_pipeline_run_var": (_i, [_vp, _vp, C.c_int32, _i64, _vp, C.c_int32, _f, _vp, _i64, _vp,
                                   C.POINTER(RunReport)]),
    "paci_partition": (_i, [C.c_int32, C.c_int32, _vp, _vp, _vp, C.c_double, _vp, C.POINTER(C.c_double),
                            C.POINTER(C.c_double)]),
    "paci_op_gemm": (_i, [_i, _i, _i, _i, _i, _vp, _i, _vp, _i, _vp, _vp, _i, _i, _vp]),
    "paci_op_gemm_backward_pair": (_i, [_i, _i, _i, _i, _vp, _i, _vp, _i, _vp, _i, _vp, _i, _vp, _i, _vp]),
    "paci_op_gemm_bias_gelu": (_i, [_i, _i, _i, _i, _vp, _i, _vp, _i, _vp, _vp, _vp, _i, _vp]),
    "paci_op_layernorm_fwd": (_i, [_i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "paci_op_layernorm_bwd": (_i, [_i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "paci_op_gelu_fwd": (_i, [_i, _sz, _vp, _vp, _vp]),
    "paci_op_gelu_bwd": (_i, [_i, _i, _i, _vp, _vp, _vp, _vp, _vp]),
    "paci_op_colsum": (_i, [_i, _i, _i, _vp, _vp, _vp]),
    "paci_op_attention_fwd": (_i, [_i, _i, _i, _i, _i, _vp, _vp, _vp, _vp]),
    "paci_op_attention_bwd": (_i, [_i, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "paci_op_attention_bwd_scratch_bytes": (_sz, [_i, _i, _i, _i, _i]),
    "paci_op_out_proj_backward": (_i, [_i, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "paci_op_attention_bwd_prepared": (_i, [_i, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "paci_op_attention_bwd_static": (_i, [_i, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp]),
    "paci_op_embed_fwd": (_i, [_i, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp]),
    "paci_op_embed_bwd": (_i, [_i, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp]),
    "paci_op_dropout": (_i, [_i, _sz, _vp, _vp, _f, C.c_uint64, _i64, C.c_int32, _vp]),
    "paci_op_softmax_ce": (_i, [_i, _i, _i, _i, _vp, _vp, _vp, _vp]),
    "paci_op_adamw": (_i, [_sz, _sz, _vp, _vp, _vp, _vp, _vp, _i, _i64, _f, _f, _f, _f, _f, _vp, _vp]),
    "paci_profile_begin": (_i, [C.c_int32]),
    "paci_profile_end": (_i, [C.POINTER(ProfEntry)]),
    "paci_profile_category_name": (C.c_char_p, [C.c_int32]),
    "paci_launch_count": (_i64, []),
    "paci_gemm_last_plan": (None, [C.POINTER(C.c_int32)]),
}


def load_library(path: str = LIB_PATH) -> C.CDLL:
    if not os.path.exists(path):
        raise ImportError(
            f"{path} not found: the CUDA extension is not built. Run `python -m paper_2606_07881_b200.build` "
            "(needs nvcc with sm_100a). There is no CPU fallback.")
    lib = C.CDLL(path)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)      # AttributeError if the library does not export it
        fn.restype, fn.argtypes = res, args
    return lib


lib = load_library()


class PaciError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: code {code}: {lib.paci_last_error().decode()}")


def check(rc, where):
    if rc < 0:
        raise PaciError(rc, where)
    return rc


def _ptr(t):
    """device / host pointer of a torch tensor, numpy array, int or None"""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _stream(stream=None):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream


def make_config(stage_index, n_stages, n_layers, d_model, n_heads, seq_len, micro_batch, k_accum, vocab,
                dtype, has_embedding=None, has_head=None, beta1=0.9, beta2=0.95, eps=1e-8, weight_decay=0.1,
                checkpoint=0, dropout_p=0.0, dropout_seed=0):
    """AdamW defaults are the paper's."""
    return StageConfig(stage_index, n_stages, n_layers, d_model, n_heads, seq_len, micro_batch, k_accum, vocab,
                       int(stage_index == 0 if has_embedding is None else has_embedding),
                       int(stage_index == n_stages - 1 if has_head is None else has_head),
                       dtype, beta1, beta2, eps, weight_decay, int(checkpoint), float(dropout_p), int(dropout_seed))


def gemm_last_plan() -> dict:
    out = (C.c_int32 * 6)()
    lib.paci_gemm_last_plan(out)
    return dict(zip(("cta_group", "block_n", "splits", "range_mode", "grid", "tiles"), list(out)))


def partition(t, s, a, n_stages, budget) -> dict:
    """App. D.5: cut points of the memory-constrained min-max partition."""
    t, s, a = (np.ascontiguousarray(v, dtype=np.float64) for v in (t, s, a))
    cuts = np.zeros(n_stages + 1, np.int32)
    mt, mo = C.c_double(), C.c_double()
    rc = check(lib.paci_partition(len(t), n_stages, t.ctypes.data, s.ctypes.data, a.ctypes.data, float(budget),
                                  cuts.ctypes.data, C.byref(mt), C.byref(mo)), "paci_partition")
    return dict(cuts=cuts.tolist(), max_time=mt.value, max_overshoot=mo.value, fallback=bool(rc))


def lr_schedule(step, total_steps, warmup_steps, peak, final_frac=0.1) -> float:
    return float(lib.paci_lr_schedule(step, total_steps, warmup_steps, peak, final_frac))


class Stage:
    """Owns the device workspace (a torch uint8 tensor) and the paci_stage handle."""

    def __init__(self, cfg: StageConfig, device="cuda:0"):
        import torch
        self.cfg = cfg
        self.device = torch.device(device)
        nbytes = lib.paci_stage_workspace_bytes(C.byref(cfg))
        if nbytes == 0:
            raise PaciError(EINVAL, "paci_stage_workspace_bytes")
        self.workspace_bytes = nbytes
        self.ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.ws.data_ptr() + 255) // 256 * 256
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            check(lib.paci_stage_create(C.byref(cfg), base, nbytes, _stream(), C.byref(h)), "paci_stage_create")
        self.handle = h
        self.act_dtype = torch.bfloat16 if cfg.dtype == BF16 else torch.float32

    def close(self, _destroy=lib.paci_stage_destroy):      # bound at definition: module globals are gone at shutdown
        if getattr(self, "handle", None):
            _destroy(self.handle)
            self.handle = None

    __del__ = close

    def _dev(self):
        import torch
        return torch.cuda.device(self.device)

    def numel(self, name):
        return lib.paci_stage_tensor_numel(self.handle, name.encode())

    def load(self, name, array, what=PARAM):
        a = np.ascontiguousarray(array, dtype=np.float32)
        with self._dev():
            check(lib.paci_stage_load(self.handle, what, name.encode(), a.ctypes.data, a.size, _stream()),
                  f"paci_stage_load({name})")

    def load_params(self, params: dict):
        for n, a in params.items():
            self.load(n, a)

    def read(self, name, what=PARAM, shape=None):
        n = self.numel(name)
        if n == 0:
            raise KeyError(name)
        out = np.empty(n, dtype=np.float32)
        with self._dev():
            check(lib.paci_stage_read(self.handle, what, name.encode(), out.ctypes.data, n, _stream()),
                  f"paci_stage_read({name})")
        return out.reshape(shape) if shape is not None else out

    def forward(self, mb_id, inp, targets=None, out=None, stream=None, raise_on_again=True, n_seq=None):
        with self._dev():
            if n_seq is None:
                rc = lib.paci_forward(self.handle, mb_id, _ptr(inp), _ptr(targets), _ptr(out), _stream(stream))
            else:
                rc = lib.paci_forward_var(self.handle, mb_id, n_seq, _ptr(inp), _ptr(targets), _ptr(out),
                                          _stream(stream))
        if rc == EAGAIN and not raise_on_again:
            return rc
        return check(rc, "paci_forward")

    def backward(self, mb_id, dout=None, din=None, stream=None):
        with self._dev():
            return check(lib.paci_backward(self.handle, mb_id, _ptr(dout), _ptr(din), _stream(stream)),
                         "paci_backward")

    def maybe_step(self, lr, stream=None):
        with self._dev():
            return check(lib.paci_maybe_step(self.handle, lr, _stream(stream)), "paci_maybe_step")

    def set_state(self, version, window_count):
        with self._dev():
            check(lib.paci_stage_set_state(self.handle, version, window_count, _stream()), "paci_stage_set_state")

    def check_inputs(self):
        with self._dev():
            check(lib.paci_stage_check(self.handle, _stream()), "paci_stage_check")

    @property
    def version(self):
        return lib.paci_version(self.handle)

    @property
    def unresolved(self):
        return lib.paci_unresolved(self.handle)

    @property
    def window_count(self):
        return lib.paci_window_count(self.handle)

    def crossed_updates(self, mb_id):
        return lib.paci_crossed_updates(self.handle, mb_id)

    def device_stamps(self, mb_id):
        vF, vB = C.c_int64(), C.c_int64()
        with self._dev():
            check(lib.paci_stage_device_stamps(self.handle, mb_id, C.byref(vF), C.byref(vB), _stream()),
                  "paci_stage_device_stamps")
        return vF.value, vB.value


class Pipeline:
    """S stages on one GPU driven by paci_pipeline_run."""

    def __init__(self, stages):
        import torch
        self.stages = list(stages)
        S = len(self.stages)
        arr = (C.c_void_p * S)(*[s.handle for s in self.stages])
        self._arr = arr
        nbytes = lib.paci_pipeline_workspace_bytes(arr, S)
        if nbytes == 0:
            raise PaciError(EINVAL, "paci_pipeline_workspace_bytes")
        self.device = self.stages[0].device
        self.ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.ws.data_ptr() + 255) // 256 * 256
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            check(lib.paci_pipeline_create(arr, S, base, nbytes, C.byref(h)), "paci_pipeline_create")
        self.handle = h

    def close(self, _destroy=lib.paci_pipeline_destroy):   # bound at definition: module globals are gone at shutdown
        if getattr(self, "handle", None):
            _destroy(self.handle)
            self.handle = None

    __del__ = close

    def run(self, tokens, lr, mode=MODE_PACI, want_loss=True, want_delta=True, n_seq=None, lr_by_update=None,
            stream=None):
        """tokens: int32 [n, mu, T+1]; a torch CUDA tensor (resident) or a numpy / torch CPU array (host).
        n_seq: optional int32 [n] heterogeneous micro-batch sizes; lr_by_update: optional float32
        array, the learning rate of each stage's u-th update during this run (PAPER.md:272 schedule).
        The run is ordered after the work already enqueued on `stream` (default: torch's current stream)."""
        import torch
        S = len(self.stages)
        n = int(tokens.shape[0])
        on_host = isinstance(tokens, np.ndarray) or (hasattr(tokens, "is_cuda") and not tokens.is_cuda)
        if isinstance(tokens, np.ndarray):
            assert tokens.dtype == np.int32 and tokens.flags.c_contiguous
        else:
            assert tokens.dtype == torch.int32 and tokens.is_contiguous()
        loss = np.zeros(n, np.float32)
        delta = np.full((S, n), -1, np.int32)
        version = np.zeros(S, np.int64)
        max_q = np.zeros(S, np.int32)
        rep = RunReport(loss.ctypes.data_as(C.POINTER(C.c_float)) if want_loss else None,
                        delta.ctypes.data_as(C.POINTER(C.c_int32)) if want_delta else None,
                        version.ctypes.data_as(C.POINTER(C.c_int64)), max_q.ctypes.data_as(C.POINTER(C.c_int32)),
                        0, 0, 0.0)
        sizes = None if n_seq is None else np.ascontiguousarray(n_seq, dtype=np.int32)
        lrs = None if lr_by_update is None else np.ascontiguousarray(lr_by_update, dtype=np.float32)
        with torch.cuda.device(self.device):
            if sizes is None and lrs is None:
                rc = lib.paci_pipeline_run(self.handle, _ptr(tokens), int(on_host), n, mode, lr, _stream(stream),
                                           C.byref(rep))
            else:
                rc = lib.paci_pipeline_run_var(self.handle, _ptr(tokens), int(on_host), n, _ptr(sizes), mode, lr,
                                               _ptr(lrs), 0 if lrs is None else lrs.size, _stream(stream),
                                               C.byref(rep))
        check(rc, "paci_pipeline_run")
        return dict(loss=loss, delta=delta, version=version, max_q=max_q, n_slots=rep.n_slots,
                    n_launches=rep.n_launches, elapsed_ms=rep.elapsed_ms)


def profile_begin(sample_stride: int):
    check(lib.paci_profile_begin(sample_stride), "paci_profile_begin")


def profile_end() -> dict:
    """category name -> dict(launches, sampled, flops, bytes, sampled_flops, sampled_bytes, sampled_ms)"""
    arr = (ProfEntry * PROF_NCAT)()
    check(lib.paci_profile_end(arr), "paci_profile_end")
    return {lib.paci_profile_category_name(i).decode(): {f: getattr(arr[i], f) for f, _ in ProfEntry._fields_}
            for i in range(PROF_NCAT)}
