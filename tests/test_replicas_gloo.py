"""N > 1 path of bench.py on the CPU (`gloo`, world_size 2): DESIGN.md section 8 -- the path does not shard inside one
run (BASELINE.json: one GPU, no collectives), so `bench.py --gpus N` runs N independent replicas; what is distributed is
only the host logic tested here: per-rank seeds, the max-over-ranks time, the whole-job value, and rank 0 alone printing
the reference arm's line."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(script_args, timeout=600):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port())] + script_args
    env = dict(os.environ, OMP_NUM_THREADS="2")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def _json_lines(out):
    return [json.loads(ln) for ln in out.splitlines() if ln.startswith("{")]


def test_replica_logic_world_size_2_gloo():
    r = _torchrun([os.path.join("tests", "gloo_worker.py")])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1                                            # rank 0 alone prints
    d = lines[0]
    assert d["world"] == 2 and d["seeds_differ"] and d["seed0"] is None
    assert d["ms"] == 20.0                                            # max over ranks of (10, 20)
    assert d["value"] == d["units"] * 5 * 2 / 20e-3                   # both replicas' units over the slowest rank's time


def test_reference_arm_under_torchrun_prints_one_line():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
