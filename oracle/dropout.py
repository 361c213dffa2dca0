"""ORACLE (test infrastructure): dropout with a counter-based mask ("dropout to 0.1").

The paper gives the rate only.  Where dropout sits is DESIGN.md reading R23 (GPT-2's residual / embedding
dropout: on the embedding output and on the output of both residual branches of every block; no dropout on the
attention probabilities).  The random numbers are not free inputs here: forward and backward of one micro-batch
run at different times (and, in checkpointed PACI, the forward runs twice), so the mask is a pure function of
(seed, micro-batch id, site, element index), evaluated by BOTH sides from the published generator

    Philox4x32-10  (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as 1, 2, 3", SC'11):
    10 rounds of  (c0, c1, c2, c3) <- (hi(M1*c2) ^ c1 ^ k0,  lo(M1*c2),  hi(M0*c0) ^ c3 ^ k1,  lo(M0*c0)),
    with the key bumped by (W0, W1) between rounds;  M0 = 0xD2511F53, M1 = 0xCD9E8D57, W0 = 0x9E3779B9,
    W1 = 0xBB67AE85.

Element e (row-major index inside the micro-batch's tensor) is kept iff word e % 4 of
Philox(counter = (e//4 low 32 bits, e//4 high 32 bits, mb_id mod 2^32, site), key = (seed low, seed high))
is >= floor(p * 2^32); kept values are multiplied by 1/(1-p).

Pins (tests/test_oracle_dropout.py): the generator's known-answer vectors; keep rate; E[mask] = 1.
"""
from __future__ import annotations

import numpy as np

M0, M1 = 0xD2511F53, 0xCD9E8D57
W0, W1 = 0x9E3779B9, 0xBB67AE85
MASK32 = 0xFFFFFFFF


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Vectorised over numpy uint64 arrays holding 32-bit values.  Returns the four output words."""
    c0, c1, c2, c3 = (np.asarray(c, dtype=np.uint64) & np.uint64(MASK32) for c in (c0, c1, c2, c3))
    k0, k1 = int(k0) & MASK32, int(k1) & MASK32
    for _ in range(10):
        p0 = np.uint64(M0) * c0            # < 2^64: both factors are < 2^32
        p1 = np.uint64(M1) * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & np.uint64(MASK32)
        hi1, lo1 = p1 >> np.uint64(32), p1 & np.uint64(MASK32)
        c0, c1, c2, c3 = hi1 ^ c1 ^ np.uint64(k0), lo1, hi0 ^ c3 ^ np.uint64(k1), lo0
        k0, k1 = (k0 + W0) & MASK32, (k1 + W1) & MASK32
    return c0, c1, c2, c3


def threshold(p: float) -> int:
    return min(int(np.floor(p * 4294967296.0)), MASK32)


def mask(shape, p: float, seed: int, mb_id: int, site: int) -> np.ndarray:
    """fp64 array of `shape`: 1/(1-p) where the element is kept, 0 where it is dropped."""
    n = int(np.prod(shape))
    nblk = (n + 3) // 4
    blk = np.arange(nblk, dtype=np.uint64)
    words = philox4x32_10(blk & np.uint64(MASK32), blk >> np.uint64(32), np.uint64(mb_id & MASK32), np.uint64(site),
                          seed & MASK32, (seed >> 32) & MASK32)
    r = np.stack(words, axis=1).reshape(-1)[:n]            # word j of block b -> element 4 b + j
    keep = r >= np.uint64(threshold(p))
    return (keep.astype(np.float64) / (1.0 - p)).reshape(shape)


SITE_EMBED = 0


def site_attn(l: int) -> int:
    return 1 + 2 * l


def site_mlp(l: int) -> int:
    return 2 + 2 * l
