"""bench.py's rank handling on real devices: `--gpus N` without torchrun spawns N ranks that
share out the cfg4a batch with no data-path collective.  The 2-rank case needs 2 GPUs and is skipped below that; the
1-rank case runs everywhere a GPU is."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*args):
    env = dict(os.environ)
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        env.pop(k, None)
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, env=env,
                         timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


def test_single_rank_line_has_the_contract_keys():
    d = run_bench("--workload", "cfg1", "--steps", "3", "--warmup", "3", "--no-per-config", "--no-cpu-baseline")
    assert d["n_gpus"] == 1 and d["scaling"] == "weak" and d["gpu_launches"] > 0 and d["dtype"] == "f64"
    assert d["roofline"]["bound"] in ("l2", "hbm") and d["roofline"]["peak"] > 9000.0       # the library's own L2 probe
    assert d["e2e"]["api"] == "sn_poisson_solve_host" and d["e2e"]["h2d_bytes_per_step"] > 0
    assert d["clocks"]["sm_mhz"] and d["config"]["workload"].startswith("cfg1")


def test_two_ranks_share_the_batch():
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs 2 GPUs")
    d = run_bench("--gpus", "2", "--steps", "1", "--warmup", "3", "--no-cpu-baseline")
    assert d["n_gpus"] == 2 and d["scaling"] == "strong"
    assert d["config"]["workload"].startswith("cfg4a") and d["config"]["batch_per_gpu"] == 32
