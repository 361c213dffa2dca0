"""Helpers for the `-m gpu` parity tests (CUDA path vs oracle on the same seeded inputs)."""
import numpy as np
import torch

from paper_2606_07881_b200 import binding as pb

DT = {pb.FP32: torch.float32, pb.BF16: torch.bfloat16}
# parity gates of BASELINE.json north_star: rel-L2 <= 1e-5 (fp32 mode), <= 2e-2 (bf16 mode)
TOL = {pb.FP32: 1e-5, pb.BF16: 2e-2}


def dev(a, dtype):
    """numpy (any float) -> CUDA tensor of the activation dtype"""
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda().to(DT[dtype]).contiguous()


def f32(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def host(t):
    return t.detach().float().cpu().numpy().astype(np.float64)


def rel_l2(got, ref):
    got = np.asarray(got, np.float64).reshape(-1)
    ref = np.asarray(ref, np.float64).reshape(-1)
    den = np.linalg.norm(ref)
    return float(np.linalg.norm(got - ref) / den) if den > 0 else float(np.linalg.norm(got))


def rounded(a, dtype):
    """what the GPU sees after the input is stored in its activation dtype (bf16 mode rounds inputs)"""
    return host(dev(a, dtype))


def sync_ok():
    torch.cuda.synchronize()
