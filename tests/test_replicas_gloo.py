"""`bench.py --gpus N` plumbing on CPU: world_size 2, backend gloo.  The path does not shard
(DESIGN.md "replicas only"): ranks exchange nothing but the barrier and the max-over-ranks of
their device time, and the job throughput is sum(units) / max(time)."""
import os
import socket
import subprocess
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent

WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["SWS_ROOT"])
from paper_1403_5044_b200 import replicas
assert replicas.init("gloo")
rank = int(os.environ["RANK"])
replicas.barrier()
local_ms = 100.0 if rank == 0 else 250.0          # rank 1 is the slow replica
mx = replicas.max_over_ranks(local_ms)
sm = replicas.sum_over_ranks(18.0)
tp = replicas.job_throughput(18.0, local_ms)
assert mx == 250.0, mx
assert sm == 36.0, sm
assert abs(tp - 36.0 / 0.25) < 1e-9, tp
replicas.barrier()
replicas.finalize()
print(f"rank {rank} ok")
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_gloo(tmp_path):
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), SWS_ROOT=str(ROOT))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for rank, p in enumerate(procs):
        out, _ = p.communicate(timeout=180)
        assert p.returncode == 0, out
        assert f"rank {rank} ok" in out


def test_single_process_is_a_noop():
    code = ("import sys; sys.path.insert(0, %r)\n"
            "from paper_1403_5044_b200 import replicas\n"
            "assert not replicas.init('gloo')\n"
            "assert replicas.max_over_ranks(3.5) == 3.5 and replicas.job_throughput(10, 500.0) == 20.0\n"
            % str(ROOT))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    subprocess.run([sys.executable, "-c", code], check=True, env=env)


def test_reference_arm_prints_contract_line():
    """bench.py --impl reference: the oracle on the host cores, one JSON line with the base keys."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--ref-rows", "64", "--config", "cfg3_181x61"],
                         check=True, capture_output=True, text=True, env=env, cwd=ROOT).stdout
    line = json.loads(out.strip().splitlines()[-1])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
              "higher_is_better", "scaling", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in line, k
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["config"]["workload"] == "cfg3_181x61"
