"""ORACLE (test infrastructure): the S-stage PACI / 1F1B-flush pipeline, executed in fp64.

Runs the ops of `oracle.schedule.simulate` in order with the real stage arithmetic of
`oracle.model` and the per-stage optimizer of `oracle.adamw`: forward under the parameters the
stage holds at that moment, stash, backward under the parameters it holds when the backward
runs (Eq. 1), G += g, update every k-th local backward (Alg. 1).
"""
from __future__ import annotations

import numpy as np

from . import model, schedule
from .adamw import StageOptimizer


def run_pipeline(specs, params, tokens, k, lr, mode="paci", m_f=None, sim_kwargs=None, hyper=None,
                 checkpoint=False, n_seq=None, dropout=None, lr_by_update=None):
    """specs: list of model.StageSpec (one per stage); params: list of dict name->array;
    tokens: int [n_mb, mu, T+1] (targets are tokens shifted by one).

    Optional:
      checkpoint    activation-checkpointed PACI: a stage keeps only its input and recomputes its forward
                    under the CURRENT parameters at backward time (model.stage_backward_checkpointed);
      n_seq         int [n_mb]: micro-batch m holds only the first n_seq[m] sequences of tokens[m] (heterogeneous
                    micro-batch sizes);
      dropout       (p, seed): dropout with the counter-based mask of oracle.dropout, keyed by the micro-batch id;
      lr_by_update  list: learning rate of a stage's u-th update (each stage indexes it by its own update count).

    Returns dict(losses[n_mb], delta[s][m], version[s], opt[s] (StageOptimizer: theta, m, v, G),
                 sim (the schedule record)).
    """
    S = len(specs)
    n_mb = tokens.shape[0]
    sim = schedule.simulate(S, n_mb, k, mode=mode, m_f=m_f, **(sim_kwargs or {}))
    k_eff = m_f if mode == "flush" else k
    opt = [StageOptimizer(params[s], k_eff, **(hyper or {})) for s in range(S)]
    stash = [dict() for _ in range(S)]
    h = [dict() for _ in range(S)]       # forward messages into stage s
    dh = [dict() for _ in range(S)]      # backward messages into stage s
    losses = [None] * n_mb
    delta = [[None] * n_mb for _ in range(S)]
    vF = [[None] * n_mb for _ in range(S)]
    for (_, _, s, kind, m) in sim["ops"]:
        spec = specs[s]
        ns = tokens.shape[1] if n_seq is None else int(n_seq[m])
        drop = None if dropout is None else (dropout[0], dropout[1], m)
        if kind == "F":
            inp = tokens[m, :ns, :-1].astype(np.int64) if s == 0 else h[s].pop(m)
            tgt = tokens[m, :ns, 1:].astype(np.int64) if spec.has_head else None
            vF[s][m] = opt[s].version
            out, st = model.stage_forward(spec, opt[s].theta, inp, tgt, drop)
            stash[s][m] = (inp, tgt) if checkpoint else st          # checkpoint: the stage input is all that is kept
            if spec.has_head:
                losses[m] = out
            else:
                h[s + 1][m] = out
        elif kind == "B":
            dout = None if spec.has_head else dh[s].pop(m)
            delta[s][m] = opt[s].version - vF[s][m]
            if checkpoint:
                inp, tgt = stash[s].pop(m)
                din, grads = model.stage_backward_checkpointed(spec, opt[s].theta, inp, tgt, dout, drop)
            else:
                din, grads = model.stage_backward(spec, opt[s].theta, stash[s].pop(m), dout)
            opt[s].accumulate(grads)
            if s > 0:
                dh[s - 1][m] = din
        else:  # "U"
            lr_now = lr if lr_by_update is None else lr_by_update[opt[s].version]
            stepped = opt[s].maybe_step(lr_now)
            assert stepped and opt[s].version == m
    assert delta == sim["delta"]
    return dict(losses=losses, delta=delta, version=[o.version for o in opt], opt=opt, sim=sim)
