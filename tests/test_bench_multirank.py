"""bench.py with more than one rank (CPU, gloo, world_size 2): the path does not shard (replicas
only), so all there is to the N > 1 case is the barrier, the max over ranks of the timed region, the sum of the replicas'
cell-steps, and rank 0 alone printing the JSON line."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(script_args, port):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port)] + script_args
    env = dict(os.environ, OMP_NUM_THREADS="1")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)


def _json_lines(text):
    return [json.loads(l) for l in text.splitlines() if l.startswith("{")]


def test_time_is_max_over_ranks_and_value_is_the_sum_of_replicas():
    r = _torchrun([os.path.join(ROOT, "tests", "multirank_worker.py")], 29641)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1                                  # rank 0 alone prints
    assert lines[0]["world"] == 2
    assert lines[0]["ms"] == 20.0                           # the slower rank's time
    assert abs(lines[0]["value"] - 2 * 1000 * 5 / 20e-3 / 1e9) < 1e-15


def test_reference_arm_runs_on_rank_0_only():
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "3", "--warmup", "1",
                   "--workload", "cfg1"], 29642)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
