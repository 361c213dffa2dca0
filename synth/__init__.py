"""Seeded synthetic inputs shared by the oracle tests and the CUDA tests/bench.

This module holds NONE of the method's arithmetic: it only draws token ids and
initial weights.  Neither `oracle/` nor `paper_2606_07881_b200/` imports it; the
tests and `bench.py` call it and hand the same arrays to both sides.

Stand-in for the paper's data (App. B "Models and data"): the paper
trains on OpenWebText tokenised with the GPT-2 tokenizer into 1024-token blocks.
That dataset is not available here; BASELINE.json replaces it by i.i.d. synthetic
token ids of the same shape -- uniform for the tiny config, Zipf(s=1.1) over the
vocabulary for the GPT-2-shaped configs.

PRNG: numpy's Philox (a 64-bit counter-based generator), keyed by
(seed, stream-id), so every tensor gets its own independent, reproducible stream.
"""
from __future__ import annotations

import zlib

import numpy as np

INIT_STD = 0.02  # BASELINE.json configs: "weights N(0,0.02)"


def _rng(seed: int, stream: str) -> np.random.Generator:
    key = (int(seed) & 0xFFFFFFFFFFFFFFFF, zlib.crc32(stream.encode()))
    return np.random.Generator(np.random.Philox(key=np.array(key, dtype=np.uint64)))


def zipf_cdf(vocab: int, s: float = 1.1) -> np.ndarray:
    """fp64 cumulative table of P(rank r) ~ r^-s, r = 1..vocab (id = r-1)."""
    w = np.arange(1, vocab + 1, dtype=np.float64) ** (-s)
    c = np.cumsum(w)
    return c / c[-1]


def tokens(seed: int, n_microbatches: int, micro_batch: int, seq_len: int, vocab: int,
           dist: str = "zipf", s: float = 1.1) -> np.ndarray:
    """int32 ids [n_microbatches, micro_batch, seq_len + 1]; column t+1 is the target of t."""
    rng = _rng(seed, f"tokens/{dist}")
    shape = (n_microbatches, micro_batch, seq_len + 1)
    if dist == "uniform":
        return rng.integers(0, vocab, size=shape, dtype=np.int64).astype(np.int32)
    if dist == "zipf":
        u = rng.random(size=shape)
        ids = np.searchsorted(zipf_cdf(vocab, s), u, side="left")
        return np.minimum(ids, vocab - 1).astype(np.int32)
    raise ValueError(dist)


def param_names(n_layers: int, has_embedding: bool, has_head: bool):
    """Stage-local tensor names, in the order of SURVEY.md 8(b)."""
    names = []
    if has_embedding:
        names += ["wte", "wpe"]
    for l in range(n_layers):
        p = f"h.{l}."
        names += [p + "ln1.g", p + "ln1.b", p + "attn.wqkv", p + "attn.bqkv", p + "attn.wo", p + "attn.bo",
                  p + "ln2.g", p + "ln2.b", p + "mlp.w1", p + "mlp.b1", p + "mlp.w2", p + "mlp.b2"]
    if has_head:
        names += ["lnf.g", "lnf.b"]
        if not has_embedding:
            names += ["head.w"]  # stage-local copy of the embedding matrix (reading R10)
    return names


def param_shape(name: str, d_model: int, vocab: int, seq_len: int):
    D = d_model
    leaf = name.split(".", 2)[-1] if name.startswith("h.") else name
    return {
        "wte": (vocab, D), "wpe": (seq_len, D), "head.w": (vocab, D),
        "ln1.g": (D,), "ln1.b": (D,), "ln2.g": (D,), "ln2.b": (D,), "lnf.g": (D,), "lnf.b": (D,),
        "attn.wqkv": (3 * D, D), "attn.bqkv": (3 * D,), "attn.wo": (D, D), "attn.bo": (D,),
        "mlp.w1": (4 * D, D), "mlp.b1": (4 * D,), "mlp.w2": (D, 4 * D), "mlp.b2": (D,),
    }[leaf]


def stage_params(seed: int, stage_index: int, n_stages: int, n_layers: int, d_model: int, vocab: int,
                 seq_len: int, perturbed: bool = False, first_block: int | None = None) -> dict:
    """fp32 initial parameters of one stage (dict name -> float32 array).

    Matrices, wte, wpe ~ N(0, 0.02); biases 0; LN gain 1, LN bias 0.
    `perturbed=True` (tests only): biases and LN bias ~ N(0,0.02), LN gain ~ 1+N(0,0.02), so
    that the bias/affine gradient paths are exercised before the first update.
    The head copy on the last stage is drawn from the SAME stream as stage 0's wte
    ("tied at init", reading R10).
    """
    has_emb = stage_index == 0
    has_head = stage_index == n_stages - 1
    out = {}
    for name in param_names(n_layers, has_emb, has_head):
        shape = param_shape(name, d_model, vocab, seq_len)
        if name in ("wte", "head.w"):
            stream = "param/wte"  # same values on both stages
        elif name in ("wpe", "lnf.g", "lnf.b"):
            stream = f"param/{name}"
        else:  # transformer block l of this stage = global block stage_index*n_layers + l
            l = int(name.split(".")[1])
            base = stage_index * n_layers if first_block is None else first_block   # unequal splits name their first block
            stream = f"param/h.{base + l}." + name.split(".", 2)[2]
        rng = _rng(seed, stream)
        leaf = name.rsplit(".", 1)[-1]
        if len(shape) == 2:
            a = rng.standard_normal(shape) * INIT_STD
        elif leaf == "g":
            a = 1.0 + (rng.standard_normal(shape) * INIT_STD if perturbed else 0.0) * np.ones(shape)
        else:
            a = rng.standard_normal(shape) * INIT_STD if perturbed else np.zeros(shape)
        out[name] = np.ascontiguousarray(a, dtype=np.float32)
    return out
