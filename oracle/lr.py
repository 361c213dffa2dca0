"""ORACLE (test infrastructure): the learning-rate schedule of App. B.

"We use a linear warmup [26] over 1% of training steps followed by cosine decay [16] to 10% of the peak value."
The paper gives no formula; reading R16: with t the 0-based index of the update the rate is used for,

    t <  W : peak * (t + 1) / W                                   (reaches the peak at the last warm-up step)
    t >= W : peak * (f + (1 - f) * (1 + cos(pi * (t - W) / (N - W))) / 2),  and peak * f for t >= N,

W = warm-up steps, N = total steps, f = 0.1.  In PACI every stage indexes the schedule by its OWN local update
count ("local update index"): there is no global step to read.
"""
from __future__ import annotations

import math


def lr_at(step: int, total_steps: int, warmup_steps: int, peak: float, final_frac: float = 0.1) -> float:
    if warmup_steps > 0 and step < warmup_steps:
        return peak * (step + 1) / warmup_steps
    if step >= total_steps or total_steps <= warmup_steps:
        return peak * final_frac
    prog = (step - warmup_steps) / (total_steps - warmup_steps)
    return peak * (final_frac + (1.0 - final_frac) * 0.5 * (1.0 + math.cos(math.pi * prog)))
