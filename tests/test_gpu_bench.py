"""-m gpu: bench.py end to end as the driver calls it (one JSON line with the contract's keys), and the 8-stage
configuration (BASELINE.json configs[3]) through `bench.py --config medium8`: the only reproducer of the LayerNorm
ring-phase hang of round 1 (8 stage streams at full width), kept as a regression test.  Barrier waits trap after 4 s,
so a protocol error fails the subprocess instead of hanging the GPU."""
import json
import math
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench(*args, timeout=900):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                       timeout=timeout, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]
    return json.loads(lines[0])


def test_bench_line_contract_on_the_tiny_config():
    d = _bench("--config", "tiny", "--steps", "2", "--warmup", "3")
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert key in d, key
    assert d["value"] > 0 and d["gpu_launches"] > 0 and d["data"] == "synthetic" and d["vs_baseline"] is None
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    assert set(d["roofline"]) >= {"bound", "achieved", "peak", "unit", "frac", "traffic"}
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["extras"]["checkpointed_paci"]["value"] > 0
    assert d["extras"]["checkpointed_paci"]["stage_workspace_bytes"] < d["config"]["stage_workspace_bytes"]


def test_bench_medium8_two_steps():
    d = _bench("--config", "medium8", "--steps", "2", "--warmup", "1", "--no-cpu-baseline", "--no-stage-times",
               "--no-extras")
    assert d["config"]["n_stages"] == 8 and d["value"] > 0
    assert d["max_crossed_updates"] <= math.ceil(7 / 4)                     # Eq. 2: N = 8, a = 4
    assert all(math.isfinite(x) for x in d["mean_loss_per_step"])
