#!/usr/bin/env python
"""bench.py -- the PACI stage-step benchmark (contract in DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config medium] [--impl reference]

One STEP = one global batch (n_micro micro-batches) pushed through the S emulated stages of the
asynchronous 1F1B pipeline on one GPU by `paci_pipeline_run`: every row of SURVEY.md 8(a) runs --
embedding, the block stacks forward and backward, LM head + cross-entropy, wgrad accumulation into
fp32 in the GEMM epilogue, one fused AdamW per stage every k micro-batches, version / crossed-update
bookkeeping.  Metric (BASELINE.json): tokens/s per PACI stage step = stage steps x tokens per
micro-batch / time, i.e. S * n_micro * mu * T / t_step (mean over the S stages of the pipeline; the
whole-pipeline tokens/s is the same number / S and is printed as `pipeline_tokens_per_s`).

Prints ONE JSON line on rank 0.  N > 1 (torchrun): N independent replicas, no data-path collective
("replicas only"); barrier + max-over-ranks timing.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

# BASELINE.json `configs`, in order.  n_micro = micro-batches per step (one global batch).
CONFIGS = {
    "tiny":    dict(idx=0, V=256,   D=64,   H=4,  T=32,   S=2, L=1, mu=2,  k=4, n_micro=16, dtype="fp32",
                    dist="uniform", lr=1e-3),
    "small":   dict(idx=1, V=50257, D=768,  H=12, T=1024, S=4, L=3, mu=8,  k=4, n_micro=16, dtype="bf16",
                    dist="zipf", lr=3e-4),
    "medium":  dict(idx=2, V=50257, D=1024, H=16, T=1024, S=4, L=6, mu=8,  k=4, n_micro=16, dtype="bf16",
                    dist="zipf", lr=3e-4),
    "medium8": dict(idx=3, V=50257, D=1024, H=16, T=1024, S=8, L=3, mu=8,  k=4, n_micro=32, dtype="bf16",
                    dist="zipf", lr=3e-4),
    "large":   dict(idx=4, V=50257, D=1280, H=20, T=1024, S=1, L=9, mu=16, k=8, n_micro=16, dtype="bf16",
                    dist="zipf", lr=3e-4),
}
METRIC = "tokens/s per PACI stage step (GPT-2 Medium, bf16)"
UNIT = "tokens/s"
SEED = 1   # timing seed; parity uses 1234


def workload_name(name, c):
    return (f"configs[{c['idx']}] {name}: V={c['V']} D={c['D']} H={c['H']} T={c['T']} "
            f"{c['S']} emulated stages x {c['L']} pre-LN blocks, micro-batch {c['mu']}, k={c['k']}, "
            f"{c['n_micro']} micro-batches per step, {c['dtype']} compute / fp32 master+m+v+G, "
            f"{c['dist']} tokens, N(0,0.02) weights")


# ------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 9:
                continue
            try:
                sm.append(float(parts[1])); mx.append(float(parts[2])); pw.append(float(parts[3]))
            except ValueError:
                continue
            for n, v in zip(names, parts[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = sorted(s for s, p in zip(sm, pw) if p > 0.5 * max(pw)) or sorted(sm)
        return {"sm_mhz": busy[len(busy) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------ peaks
def measured_peaks():
    """MEASURED_PEAKS.json (driver-written) or the profiling guide's stated fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm=d["hbm_gbs"], tf_burst=d["bf16_tflops"],
                    tf_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]), source="measured")
    return dict(hbm=6650.0, tf_burst=1590.0, tf_sustained=1400.0, source="fallback")


def ncu_traffic(kernel_key):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full summary, or None."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            parts = [x.strip() for x in line.split(",")]
            if parts and parts[0] == kernel_key and len(parts) >= 3:
                try:
                    return float(parts[1]) + float(parts[2])
                except ValueError:
                    return None
    return None


# ------------------------------------------------------------------------------------ CPU oracle leg
def oracle_sample(c, steps, warmup):
    """Times the fp64 oracle AS IT STANDS on the host cores, on a bounded sample of the workload: one
    PACI stage step (F, B with G += g, and the AdamW update divided by k as in the workload) of ONE
    stage at full width and depth (L blocks, D, H, T, V), with micro-batch 1.  The stage is the
    interior stage s=1 when S >= 3 (the stage kind SURVEY.md 8(d) defines the metric on), else stage 0.
    Returns (tokens/s per stage step, info)."""
    import synth
    from oracle import model
    from oracle.adamw import StageOptimizer
    S, L, D, H, T, V, k = c["S"], c["L"], c["D"], c["H"], c["T"], c["V"], c["k"]
    mu = 1
    s = 1 if S >= 3 else 0
    spec = model.StageSpec(s, S, L, D, H, T, mu, V)
    opt = StageOptimizer(synth.stage_params(SEED, s, S, L, D, V, T), 1)
    tok = synth.tokens(SEED, steps + warmup, mu, T, V, c["dist"])
    rng = np.random.default_rng(SEED)
    per_step = []
    for it in range(steps + warmup):
        inp = tok[it, :, :-1].astype(np.int64) if spec.has_embedding else rng.standard_normal((mu, T, D))
        tgt = tok[it, :, 1:].astype(np.int64) if spec.has_head else None
        dout = None if spec.has_head else rng.standard_normal((mu, T, D)) * 1e-3
        t0 = time.perf_counter()
        _, stash = model.stage_forward(spec, opt.theta, inp, tgt)
        _, grads = model.stage_backward(spec, opt.theta, stash, dout)
        opt.accumulate(grads)
        t_fb = time.perf_counter() - t0
        t0 = time.perf_counter()
        assert opt.maybe_step(c["lr"])
        t_u = time.perf_counter() - t0
        per_step.append(t_fb + t_u / k)
    timed = per_step[warmup:]
    t = sum(timed) / len(timed)
    host = len(os.sched_getaffinity(0))
    try:
        from threadpoolctl import threadpool_info
        threads = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    except Exception:
        threads = host
    kind = "interior" if 0 < s < S - 1 else ("first" if S > 1 else "only")
    info = dict(cores=min(threads, host), host_cores=host, s_per_step=t,
                sample=(f"fp64 numpy oracle: one stage step of the {kind} stage s={s} at full width and depth "
                        f"({L} blocks, D={D}, H={H}, T={T}), micro-batch 1 instead of {c['mu']} ({mu * T} tokens): "
                        f"F + B (G += g) + AdamW time/{k}; {len(timed)} timed step(s); BLAS threads {threads} "
                        f"of {host} host cores"))
    return mu * T / t, info


def oracle_one_thread(c):
    """SURVEY.md 8(d) also asks for a 1-thread figure: the same oracle, ONE block of the interior stage at full
    width (micro-batch 1), F + B only, timed with the BLAS pool limited to one thread and again with all threads."""
    import synth
    from oracle import model
    from threadpoolctl import threadpool_limits
    S, D, H, T, V = c["S"], c["D"], c["H"], c["T"], c["V"]
    s = 1 if S >= 3 else 0
    spec = model.StageSpec(s, max(S, 3) if s == 1 else S, 1, D, H, T, 1, V)
    if spec.has_embedding or spec.has_head:
        return None
    theta = {n: np.asarray(a, np.float64) for n, a in synth.stage_params(SEED, s, spec.n_stages, 1, D, V, T).items()}
    rng = np.random.default_rng(SEED)
    inp, dout = rng.standard_normal((1, T, D)), rng.standard_normal((1, T, D)) * 1e-3

    def once():
        t0 = time.perf_counter()
        _, stash = model.stage_forward(spec, theta, inp, None)
        model.stage_backward(spec, theta, stash, dout)
        return time.perf_counter() - t0
    once()
    t_all = once()
    with threadpool_limits(limits=1):
        t_one = once()
    return {"value": T / t_one, "unit": UNIT, "cores": 1, "all_cores_value": T / t_all,
            "sample": f"one block of the interior stage (D={D}, H={H}, T={T}), micro-batch 1, F + B, fp64 numpy oracle"}


def run_reference(args, c, name):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    val, info = oracle_sample(c, args.steps, args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": info["s_per_step"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(name, c)},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": info["cores"], "kind": "oracle",
                             "sample": info["sample"]},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------ CUDA leg
def build_pipeline(pb, c, device, layers=None, checkpoint=0):
    """layers: blocks per stage (default: the equal split of BASELINE.json, c['L'] each)."""
    import synth
    dt = pb.BF16 if c["dtype"] == "bf16" else pb.FP32
    layers = list(layers) if layers is not None else [c["L"]] * c["S"]
    stages, first = [], 0
    for s in range(c["S"]):
        st = pb.Stage(pb.make_config(s, c["S"], layers[s], c["D"], c["H"], c["T"], c["mu"], c["k"], c["V"], dt,
                                     checkpoint=checkpoint), device=device)
        st.load_params(synth.stage_params(SEED, s, c["S"], layers[s], c["D"], c["V"], c["T"], first_block=first))
        first += layers[s]
        stages.append(st)
    return stages, pb.Pipeline(stages)


def free_pipeline(torch, stages, pipe):
    pipe.close()
    for st in stages:
        st.close()
    stages.clear()
    torch.cuda.empty_cache()


def timed_steps(pipe, tok_dev, lr, first, steps, S, tokens_per_step):
    """Device time of `steps` pipeline steps on resident tokens -> (tokens/s per stage step, ms per step)."""
    ms = 0.0
    for i in range(steps):
        ms += pipe.run(tok_dev[first + i], lr, want_delta=False)["elapsed_ms"]
    return S * tokens_per_step * steps / (ms * 1e-3), ms / steps


def partition_profile(pb, c, per_stage):
    """Per-layer profile for App. D.5 from THIS build's own measurements: the layers are the L*S
    transformer blocks (the embedding grouped with the first) plus the final layer that computes the
    loss.  t_l = forward time (the paper's proxy), s_l = bytes of parameters + gradient accumulator + optimizer state
    (+ bf16 shadow), a_l = bytes stashed for backward per micro-batch (from paci_stage_workspace_bytes)."""
    import ctypes as C
    S, L, D, H, T, mu, V, k = c["S"], c["L"], c["D"], c["H"], c["T"], c["mu"], c["V"], c["k"]
    dt = pb.BF16 if c["dtype"] == "bf16" else pb.FP32

    def ws(s_idx, n_layers, emb, head):
        cfg = pb.make_config(s_idx, 2, n_layers, D, H, T, mu, k, V, dt, has_embedding=emb, has_head=head)
        return pb.lib.paci_stage_workspace_bytes(C.byref(cfg))

    def nparams(n_layers, emb, head):
        cfg = pb.make_config(0, 2, n_layers, D, H, T, mu, k, V, dt, has_embedding=emb, has_head=head)
        return pb.lib.paci_stage_param_count(C.byref(cfg))
    a_block = (ws(0, 2, False, False) - ws(1, 2, False, False)) - (ws(0, 1, False, False) - ws(1, 1, False, False))
    a_head = ws(0, 0, False, True) - ws(1, 0, False, True)
    bpp = 18.0 if dt == pb.BF16 else 16.0
    s_block = bpp * (nparams(2, False, False) - nparams(1, False, False))
    s_head = bpp * nparams(0, False, True)
    s_emb = bpp * (nparams(1, True, False) - nparams(1, False, False))
    t_block = per_stage[1 if S >= 3 else 0]["t_fwd_ms"] / L
    t_emb = max(per_stage[0]["t_fwd_ms"] - L * t_block, 0.0) if S > 1 else 0.0
    t_head = max(per_stage[S - 1]["t_fwd_ms"] - L * t_block, 0.0)
    n_blocks = L * S
    t = [t_block] * n_blocks + [t_head]
    s_ = [s_block] * n_blocks + [s_head]
    a = [float(a_block)] * n_blocks + [float(a_head)]
    t[0] += t_emb
    s_[0] += s_emb
    return t, s_, a


def run_partition(pb, torch, c, stages, pipe, per_stage, tok_dev, lr, device, steps=2):
    """--partition auto: App. D.5 (Eq. 12-15) fed by this build's own per-layer profile; the S stages
    then hold unequal numbers of blocks.  One GPU serialises the emulated stages, so the gain shows where the paper
    puts it: the slowest stage bounds a pipeline's steady-state throughput (PAPER.md:460 'bottle-necked by the slowest
    stage')."""
    S, L, mu, T, k = c["S"], c["L"], c["mu"], c["T"], c["k"]
    t, s_, a = partition_profile(pb, c, per_stage)
    budget = 180e9 / S                     # the S emulated stages share one 180 GB B200
    part = pb.partition(t, s_, a, S, budget)
    cuts = part["cuts"]
    layers = [cuts[j + 1] - cuts[j] for j in range(S)]
    layers[-1] -= 1                        # the last group's final layer is the head, not a block
    free_pipeline(torch, stages, pipe)
    stages2, pipe2 = build_pipeline(pb, c, device, layers=layers)
    pipe2.run(tok_dev[0], lr, want_delta=False)
    value, ms = timed_steps(pipe2, tok_dev, lr, 1, steps, S, c["n_micro"] * mu * T)
    st2 = per_stage_times(pb, torch, dict(c), stages2, reps=2)
    free_pipeline(torch, stages2, pipe2)
    slow = lambda ps: max(p["t_fwd_ms"] + p["t_bwd_ms"] + p["t_step_ms"] / k for p in ps)
    return {"profile": {"t_block_ms": t[1], "t_first_ms": t[0], "t_head_ms": t[-1], "s_block_bytes": s_[1],
                        "a_block_bytes": a[1], "a_head_bytes": a[-1], "budget_bytes": budget},
            "cuts": cuts, "blocks_per_stage": layers, "fallback": part["fallback"],
            "predicted_max_stage_fwd_ms": part["max_time"],
            "equal_split": {"blocks_per_stage": [L] * S, "slowest_stage_ms": slow(per_stage),
                            "pipeline_tokens_per_s_bound": mu * T / (slow(per_stage) * 1e-3)},
            "partitioned": {"slowest_stage_ms": slow(st2), "pipeline_tokens_per_s_bound": mu * T / (slow(st2) * 1e-3),
                            "tokens_per_s_per_stage_step_one_gpu": value, "ms_per_step_one_gpu": ms,
                            "per_stage": st2}}


def per_stage_times(pb, torch, c, stages, reps=3):
    """t_F, t_B, t_step of every stage kind through paci_forward / paci_backward / paci_maybe_step
    (SURVEY.md 8(d) "Procedure"): tokens/s per stage step = M / (t_F + t_B + t_step / k)."""
    S, mu, T, D, V, k = c["S"], c["mu"], c["T"], c["D"], c["V"], c["k"]
    act = torch.bfloat16 if c["dtype"] == "bf16" else torch.float32
    g = torch.Generator(device="cuda").manual_seed(SEED)
    out = []
    mb = 1 << 20
    for s, st in enumerate(stages):
        emb, head = s == 0, s == S - 1
        inp = (torch.randint(0, V, (mu, T), device="cuda", dtype=torch.int32, generator=g) if emb
               else torch.randn(mu, T, D, device="cuda", generator=g).to(act))
        tgt = torch.randint(0, V, (mu, T), device="cuda", dtype=torch.int32, generator=g) if head else None
        o = torch.zeros(1, device="cuda") if head else torch.empty(mu, T, D, device="cuda", dtype=act)
        dout = None if head else (torch.randn(mu, T, D, device="cuda", generator=g) * 1e-3).to(act)
        din = None if emb else torch.empty(mu, T, D, device="cuda", dtype=act)
        tf, tb, tu = [], [], []
        for r in range(reps + 1):
            for j in range(k):
                e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
                e[0].record(); st.forward(mb, inp, tgt, o); e[1].record()
                st.backward(mb, dout, din); e[2].record()
                stepped = st.maybe_step(c["lr"]); e[3].record()
                mb += 1
                torch.cuda.synchronize()
                if r > 0:
                    tf.append(e[0].elapsed_time(e[1])); tb.append(e[1].elapsed_time(e[2]))
                    if stepped:
                        tu.append(e[2].elapsed_time(e[3]))
        f, b, u = float(np.median(tf)), float(np.median(tb)), float(np.median(tu))
        out.append({"stage": s, "t_fwd_ms": round(f, 4), "t_bwd_ms": round(b, 4), "t_step_ms": round(u, 4),
                    "tokens_per_s": mu * T / ((f + b + u / k) * 1e-3)})
    return out


def run_ours(args, c, name):
    import torch
    from paper_2606_07881_b200 import replicas
    rank, world, local = replicas.init_from_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    device = f"cuda:{local}"
    from paper_2606_07881_b200 import binding as pb
    import synth

    S, mu, T, n_micro, k = c["S"], c["mu"], c["T"], c["n_micro"], c["k"]
    tokens_per_step = n_micro * mu * T
    stages, pipe = build_pipeline(pb, c, device)
    ws_total = sum(st.workspace_bytes for st in stages)
    n_batches = args.warmup + 2 * args.steps
    tok_host = synth.tokens(SEED + rank, n_batches * n_micro, mu, T, c["V"], c["dist"])
    tok_host = tok_host.reshape(n_batches, n_micro, mu, T + 1)
    tok_dev = torch.from_numpy(tok_host).to(device)
    tok_pinned = torch.from_numpy(tok_host).pin_memory()
    lr = c["lr"]

    for w in range(args.warmup):                                     # untimed warm-up steps
        pipe.run(tok_dev[w], lr, want_delta=False)

    # ---- timed region 1: inputs resident in HBM (this is `value`; no profiling inside)
    clocks = ClockSampler(local)
    replicas.barrier(); torch.cuda.synchronize()
    clocks.start()
    dev_ms, launches = 0.0, 0
    delta_max, losses = 0, []
    t0 = time.perf_counter()
    for i in range(args.steps):
        out = pipe.run(tok_dev[args.warmup + i], lr)
        dev_ms += out["elapsed_ms"]; launches += out["n_launches"]
        delta_max = max(delta_max, int(out["delta"].max())); losses.append(float(out["loss"].mean()))
    torch.cuda.synchronize()
    wall_ms = (time.perf_counter() - t0) * 1e3
    replicas.barrier()
    value, max_ms = replicas.whole_job_throughput(dev_ms, S * tokens_per_step * args.steps)
    ms_per_step = max_ms / args.steps

    # ---- timed region 1b: the SAME K steps again with the in-library sampler on (every n-th kernel bracketed by
    # CUDA events and made to run alone, which costs the step a few percent: hence not inside region 1)
    pb.profile_begin(args.sample_stride)
    prof_ms = 0.0
    for i in range(args.steps):
        prof_ms += pipe.run(tok_dev[args.warmup + i], lr, want_delta=False)["elapsed_ms"]
    torch.cuda.synchronize()
    prof = pb.profile_end()
    clk = clocks.stop()
    replicas.barrier()

    # ---- timed region 2: end to end through the C ABI with HOST token buffers (pinned), loss read back
    replicas.barrier(); torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(args.steps):
        out = pipe.run(tok_pinned[args.warmup + args.steps + i], lr, want_delta=False)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    replicas.barrier()
    e2e_value, _ = replicas.whole_job_throughput(e2e_ms, S * tokens_per_step * args.steps)

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel (the tcgen05 GEMM) from the sampled in-library events
    peaks = measured_peaks()
    cats = {}
    for n, e in prof.items():
        if e["launches"] == 0:
            continue
        d = {"launches": e["launches"], "sampled": e["sampled"], "sampled_ms": round(e["sampled_ms"], 3)}
        if e["sampled_ms"] > 0:
            if e["flops"] > 0:
                d["tflops"] = round(e["sampled_flops"] / e["sampled_ms"] * 1e-9, 1)
                d["frac"] = round(d["tflops"] / peaks["tf_sustained"], 3)
            else:
                d["gbs"] = round(e["sampled_bytes"] / e["sampled_ms"] * 1e-6, 1)
                d["frac"] = round(d["gbs"] / peaks["hbm"], 3)
            # this category's estimated share of the step: mean sampled duration x launches
            d["est_ms_per_step"] = round(e["sampled_ms"] / e["sampled"] * e["launches"] / args.steps, 3)
        cats[n] = d
    g = [prof[n] for n in ("gemm_fwd", "gemm_dgrad", "gemm_wgrad", "gemm_bwd_pair")]
    g_ms = sum(e["sampled_ms"] for e in g)
    g_flops = sum(e["sampled_flops"] for e in g)
    g_n = sum(e["sampled"] for e in g)
    achieved = g_flops / g_ms * 1e-9 if g_ms > 0 else 0.0
    roofline = {"bound": "tensor", "kernel": "gemm_tc_kernel (tcgen05 bf16, all GEMM launches of the step)",
                "achieved": round(achieved, 1), "peak": peaks["tf_sustained"], "unit": "TFLOP/s",
                "frac": round(achieved / peaks["tf_sustained"], 4),
                "peak_source": f"{peaks['source']} sustained bf16 (kernel timed inside a long step)",
                "traffic": ncu_traffic("gemm_tc_kernel"),
                "flops_per_launch": g_flops / g_n if g_n else None,
                "ms_per_launch": g_ms / g_n if g_n else None,
                "sampled_launches": g_n, "sample_stride": args.sample_stride}

    stage_times = per_stage_times(pb, torch, c, stages) if not args.no_stage_times else None
    extras = {}
    if args.partition == "auto" and stage_times is not None and S > 1:
        extras["partition"] = run_partition(pb, torch, c, stages, pipe, stage_times, tok_dev, lr, device)
    else:
        free_pipeline(torch, stages, pipe)
    if not args.no_extras:
        # activation-checkpointed PACI on the same workload: the stash shrinks to the stage input and
        # every backward first recomputes its stage's forward under the current weights
        st_ck, pipe_ck = build_pipeline(pb, c, device, checkpoint=1)
        pipe_ck.run(tok_dev[0], lr, want_delta=False)
        v_ck, ms_ck = timed_steps(pipe_ck, tok_dev, lr, 1, min(2, args.steps), S, tokens_per_step)
        ws_ck = sum(st.workspace_bytes for st in st_ck)
        free_pipeline(torch, st_ck, pipe_ck)
        extras["checkpointed_paci"] = {"value": v_ck, "unit": UNIT, "ms_per_step": ms_ck, "stage_workspace_bytes": ws_ck,
                                       "note": "checkpoint=1: backward = recompute under current weights + differentiate"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": c["dtype"], "data": "synthetic",
            "config": {"workload": workload_name(name, c), "n_stages": S, "tokens_per_step": tokens_per_step,
                       "stage_steps_per_step": S * n_micro, "stage_workspace_bytes": ws_total,
                       "l2": "inputs larger than L2 (each step streams > 20 GB of weights and stashed activations)",
                       "parallelism": "replicas only" if world > 1 else "1 GPU, S emulated stages on per-stage streams",
                       "gemm_backend": "tcgen05"},
            "pipeline_tokens_per_s": value / S, "wall_ms_per_step": wall_ms / args.steps,
            "sampled_region_ms_per_step": prof_ms / args.steps,
            "clocks": clk,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": n_micro * mu * (T + 1) * 4,
                    "d2h_bytes_per_step": n_micro * 4, "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": launches,
            "roofline": roofline, "kernels": cats,
            "max_crossed_updates": delta_max, "mean_loss_per_step": losses}
    if stage_times is not None:
        line["per_stage"] = stage_times
    if extras:
        line["extras"] = extras
    if world == 1 and not args.no_cpu_baseline:
        val, info = oracle_sample(c, 3, 1)                # 3 timed oracle steps after 1 warm-up step (~25 s of host time)
        line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": info["cores"], "kind": "oracle",
                                "sample": info["sample"]}
        try:
            one = oracle_one_thread(c)
            if one is not None:
                line["cpu_baseline"]["one_thread"] = one
        except Exception as e:                       # the 1-thread figure is an extra, never a reason to lose the line
            line["cpu_baseline"]["one_thread"] = {"unavailable": repr(e)[:200]}
    print(json.dumps(line))
    return 0



# ------------------------------------------------------------------------------------ k sweep (configs[3])
def run_k_sweep(args, c, name):
    """BASELINE.json configs[3]: the same model split into S emulated stages, k in {1,2,4,8}: PACI and
    1F1B-flush (groups of m_f = k micro-batches, Table 4's matched comparison) on the same GPU.
    Per k: crossed-update counts Delta_{m,s} (max per stage against the bound ceil((S-1-s)/k), Eq. 10
    P:398), versions, device time of the run, and the EMULATED pipeline step time: one GPU serialises the
    stages, so bubbles cannot show in wall time; the virtual makespan is the schedule's logical slot count
    (every stage does at most one F or B per slot, `n_slots` of paci_pipeline_run) x the measured mean
    op time (t_F + t_B) / 2 of an interior stage.  flush / PACI is then compared with Eq. 3."""
    import math
    import torch
    from paper_2606_07881_b200 import binding as pb
    import synth
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(0)
    S, mu, T, n = c["S"], c["mu"], c["T"], c["n_micro"]
    tok = torch.from_numpy(synth.tokens(SEED, n, mu, T, c["V"], c["dist"])).cuda()
    rows = []
    for k in (1, 2, 4, 8):
        ck = dict(c, k=k)
        row = {"k": k, "bound_max": math.ceil((S - 1) / k)}
        for mode, tag in ((pb.MODE_PACI, "paci"), (pb.MODE_FLUSH, "flush")):
            stages, pipe = build_pipeline(pb, ck, "cuda:0")
            pipe.run(tok, ck["lr"], mode=mode, want_delta=False)              # warm-up run
            out = pipe.run(tok, ck["lr"], mode=mode)
            d = out["delta"]
            row[tag] = {"ms": out["elapsed_ms"], "n_slots": int(out["n_slots"]),
                        "max_delta_per_stage": [int(x) for x in d.max(axis=1)],
                        "versions": [int(v) for v in out["version"]],
                        "tokens_per_s_per_stage_step": S * n * mu * T / (out["elapsed_ms"] * 1e-3)}
            if tag == "paci":
                row["bound_per_stage"] = [math.ceil((S - 1 - s) / k) for s in range(S)]
                row["bound_holds"] = all(a <= b for a, b in zip(row[tag]["max_delta_per_stage"], row["bound_per_stage"]))
                st = per_stage_times(pb, torch, ck, stages, reps=2)[1]          # an interior stage
                row["t_op_ms"] = (st["t_fwd_ms"] + st["t_bwd_ms"]) / 2
            pipe.close()
            for s_ in stages:
                s_.close()
            del stages, pipe
            torch.cuda.empty_cache()
        t_op = row["t_op_ms"]
        row["virtual_ms"] = {"paci": row["paci"]["n_slots"] * t_op, "flush": row["flush"]["n_slots"] * t_op}
        # steady state: PACI needs 2k slots per k micro-batches, a flush group (k + S - 1) * 2
        row["eta_flush_eq3"] = k / (k + S - 1)
        row["eta_measured_slots"] = 2 * n / row["flush"]["n_slots"] if row["flush"]["n_slots"] else None   # PACI steady state: 2 slots per micro-batch
        rows.append(row)
    line = {"metric": "k sweep: crossed updates and emulated step time, PACI vs 1F1B-flush", "n_gpus": 1,
            "config": {"workload": workload_name(name, c), "n_microbatches": n}, "data": "synthetic",
            "dtype": c["dtype"], "sweep": rows}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------ energy per op
class PowerSampler:
    """mean board power / SM clock while one op runs back to back (nvidia-smi -lms 50)."""

    def __init__(self, gpu_index):
        self.gpu = gpu_index

    def __enter__(self):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", "--query-gpu=power.draw,clocks.sm",
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None
        return self

    def __exit__(self, *exc):
        w, mhz = [], []
        if self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.p.kill()
            self.f.flush()
            self.f.seek(0)
            for line in self.f.read().splitlines():
                parts = [x.strip() for x in line.split(",")]
                try:
                    w.append(float(parts[0])); mhz.append(float(parts[1]))
                except (ValueError, IndexError):
                    continue
        self.f.close()
        os.unlink(self.f.name)
        n = len(w) // 3                                    # drop the ramp: keep the last two thirds
        w, mhz = w[n:], mhz[n:]
        self.watts = sum(w) / len(w) if w else None
        self.mhz = sum(mhz) / len(mhz) if mhz else None
        return False


def run_energy(args, c, name):
    """`--energy`: every kernel of one block at the config's shapes, run alone and back to back for ~2.5 s each under
    the board's power cap: mean W, SM clock, us per call and mJ per call (= W x us), with cuBLAS (torch) on the same
    GEMM shapes beside ours.  The step is power-capped, so mJ per call is what a kernel costs it."""
    import ctypes
    import torch
    from paper_2606_07881_b200 import binding as pb
    lib = pb.lib
    torch.cuda.set_device(0)
    bf = torch.bfloat16
    D, H, T, mu = c["D"], c["H"], c["T"], c["mu"]
    M = mu * T
    S0 = lambda: torch.cuda.current_stream().cuda_stream
    rows = []

    def run(label, fn, flops=None, secs=2.5):
        for _ in range(20):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n, t0 = 0, time.time()
        with PowerSampler(0) as ps:
            e0.record()
            while time.time() - t0 < secs:
                for _ in range(200):
                    fn()
                n += 200
                torch.cuda.synchronize()
            e1.record()
            torch.cuda.synchronize()
        us = e0.elapsed_time(e1) * 1e3 / n
        r = {"op": label, "watts": ps.watts, "sm_mhz": ps.mhz, "us_per_call": round(us, 2),
             "mj_per_call": round(ps.watts * us * 1e-3, 2) if ps.watts else None}
        if flops:
            r["tflops"] = round(flops / us * 1e-6, 1)
        rows.append(r)
        time.sleep(0.5)

    def rnd(*shape, scale=1.0):
        return (torch.randn(*shape, device="cuda") * scale).to(bf)

    keep = []                                              # tensors whose data_ptr() the closures captured

    def ours_fwd(N, K, gelu=False):
        A, B, bias = rnd(M, K), rnd(N, K, scale=0.02), torch.randn(N, device="cuda")
        Cc, G = torch.empty(M, N, device="cuda", dtype=bf), torch.empty(M, N, device="cuda", dtype=bf)
        keep.extend([A, B, bias, Cc, G])
        if gelu:
            return lambda: lib.paci_op_gemm_bias_gelu(pb.BF16, M, N, K, A.data_ptr(), K, B.data_ptr(), K, bias.data_ptr(),
                                                      Cc.data_ptr(), G.data_ptr(), N, S0())
        return lambda: lib.paci_op_gemm(pb.BF16, 0, M, N, K, A.data_ptr(), K, B.data_ptr(), K, bias.data_ptr(),
                                        Cc.data_ptr(), N, 0, S0())

    def cublas_fwd(N, K):
        A, B, bias = rnd(M, K), rnd(N, K, scale=0.02), rnd(N)
        keep.extend([A, B, bias])
        return lambda: torch.nn.functional.linear(A, B, bias)

    def ours_pair(N_out, K_in):
        dy, x, W = rnd(M, N_out), rnd(M, K_in), rnd(N_out, K_in, scale=0.02)
        G, dx = torch.zeros(N_out, K_in, device="cuda"), torch.empty(M, K_in, device="cuda", dtype=bf)
        keep.extend([dy, x, W, G, dx])
        return lambda: lib.paci_op_gemm_backward_pair(pb.BF16, M, N_out, K_in, dy.data_ptr(), N_out, x.data_ptr(), K_in,
                                                      W.data_ptr(), K_in, G.data_ptr(), K_in, dx.data_ptr(), K_in, S0())

    def cublas_pair(N_out, K_in):                          # the same two products, both with bf16 outputs
        dy, x, W = rnd(M, N_out), rnd(M, K_in), rnd(N_out, K_in, scale=0.02)
        keep.extend([dy, x, W])

        def f():
            torch.matmul(dy, W)
            torch.matmul(dy.t(), x)
        return f

    for label, N, K, gelu in (("QKV forward", 3 * D, D, False), ("out-proj forward", D, D, False),
                              ("MLP-up forward + GELU epilogue", 4 * D, D, True), ("MLP-down forward", D, 4 * D, False)):
        run(f"gemm_tc {label} {M}x{N}x{K}", ours_fwd(N, K, gelu), 2.0 * M * N * K)
        run(f"cuBLAS  F.linear {M}x{N}x{K}" + (" (no GELU)" if gelu else ""), cublas_fwd(N, K), 2.0 * M * N * K)
    for label, N_out, K_in in (("Wqkv", 3 * D, D), ("W1", 4 * D, D), ("W2", D, 4 * D), ("Wo", D, D)):
        run(f"gemm_tc backward pair {label} (dgrad + fp32 wgrad accumulate)", ours_pair(N_out, K_in), 4.0 * M * N_out * K_in)
        run(f"cuBLAS  dgrad + wgrad {label} (two matmuls, bf16 out)", cublas_pair(N_out, K_in), 4.0 * M * N_out * K_in)
    qkv, do = rnd(mu, T, 3 * D), rnd(mu, T, D)
    o, lse, dqkv = torch.empty(mu, T, D, device="cuda", dtype=bf), torch.empty(mu, H, T, device="cuda"), torch.empty_like(qkv)
    scratch = torch.empty(lib.paci_op_attention_bwd_scratch_bytes(pb.BF16, mu, T, H, D // H), device="cuda", dtype=torch.uint8)
    fl = 2.0 * mu * H * T * T * (D // H)
    run("attention forward", lambda: lib.paci_op_attention_fwd(pb.BF16, mu, T, H, D // H, qkv.data_ptr(), o.data_ptr(),
                                                               lse.data_ptr(), S0()), fl)
    run("attention backward", lambda: lib.paci_op_attention_bwd(pb.BF16, mu, T, H, D // H, do.data_ptr(), qkv.data_ptr(),
                                                                o.data_ptr(), lse.data_ptr(), dqkv.data_ptr(),
                                                                scratch.data_ptr(), S0()), 2 * fl)
    x, res, g, b = rnd(M, D), rnd(M, D), torch.randn(D, device="cuda"), torch.randn(D, device="cuda")
    xs, y, dx = torch.empty_like(x), torch.empty_like(x), torch.empty_like(x)
    mean, rstd = torch.empty(M, device="cuda"), torch.empty(M, device="cuda")
    Gg, Gb, Gc = (torch.zeros(D, device="cuda") for _ in range(3))
    run("LayerNorm forward (+ residual)", lambda: lib.paci_op_layernorm_fwd(
        pb.BF16, M, D, x.data_ptr(), res.data_ptr(), g.data_ptr(), b.data_ptr(), xs.data_ptr(), y.data_ptr(),
        mean.data_ptr(), rstd.data_ptr(), S0()))
    run("LayerNorm backward (+ residual, column sums)", lambda: lib.paci_op_layernorm_bwd(
        pb.BF16, M, D, y.data_ptr(), xs.data_ptr(), mean.data_ptr(), rstd.data_ptr(), g.data_ptr(), res.data_ptr(),
        dx.data_ptr(), Gg.data_ptr(), Gb.data_ptr(), Gc.data_ptr(), S0()))
    dg, pp = rnd(M, 4 * D), rnd(M, 4 * D)
    dp, Gb4 = torch.empty_like(pp), torch.zeros(4 * D, device="cuda")
    run("GELU backward + b1 column sums", lambda: lib.paci_op_gelu_bwd(pb.BF16, M, 4 * D, dg.data_ptr(), pp.data_ptr(),
                                                                       dp.data_ptr(), Gb4.data_ptr(), S0()))
    per_block = sum(r["mj_per_call"] or 0.0 for r in rows if not r["op"].startswith("cuBLAS"))
    per_block += sum((r["mj_per_call"] or 0.0) for r in rows if r["op"].startswith("LayerNorm"))   # two of each per block
    print(json.dumps({"metric": "energy per kernel call under the board's power cap", "n_gpus": 1,
                      "config": {"workload": workload_name(name, c)}, "data": "synthetic (N(0,1) activations)",
                      "dtype": "bf16", "mj_per_block_fwd_bwd": round(per_block, 1), "ops": rows}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="medium", choices=sorted(CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--sample-stride", type=int, default=29,
                    help="time every n-th library op with CUDA events; a sampled op runs alone on the GPU")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-stage-times", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the checkpointed-PACI extra measurement")
    ap.add_argument("--partition", default="equal", choices=["equal", "auto"],
                    help="auto: also run App. D.5's partitioner on this build's own per-layer profile and report "
                         "the partitioned pipeline as an EXTRA (the headline stays on BASELINE.json's equal split)")
    ap.add_argument("--k-sweep", action="store_true", help="BASELINE.json configs[3]: k in {1,2,4,8}, PACI vs flush")
    ap.add_argument("--energy", action="store_true",
                    help="W, SM clock, us and mJ per call of every block kernel run alone under the power cap, cuBLAS beside")
    args = ap.parse_args()
    c = CONFIGS[args.config]
    if args.impl == "reference":
        return run_reference(args, c, args.config)
    if args.energy:
        return run_energy(args, c, args.config)
    if args.k_sweep:
        return run_k_sweep(args, CONFIGS["medium8"] if args.config == "medium" else c, "medium8" if args.config == "medium" else args.config)
    return run_ours(args, c, args.config)


if __name__ == "__main__":
    sys.exit(main())
