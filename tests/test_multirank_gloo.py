"""N > 1 host logic of bench.py on CPU: two `gloo` ranks, no GPU.

The path shards by (batch, head) with no data-path collective; what the ranks exchange is only the timing
(max over ranks) and the unit count (sum over ranks).  This test runs that exchange with world_size 2."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import bench
rank, world, local, inited = bench.dist_setup(2)
assert inited and world == 2 and rank == int(os.environ["RANK"])
bench.barrier(inited)
# rank r "took" 10 + 5 r ms for 100 (r + 1) units: whole job = max time, summed units
t, u = bench.aggregate(10.0 + 5.0 * rank, 100.0 * (rank + 1), inited, "cpu")
bench.barrier(inited)
import torch.distributed as dist
dist.destroy_process_group()
print(json.dumps({{"rank": rank, "t": t, "u": u}}))
"""


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_aggregate_is_max_time_and_summed_units_over_two_gloo_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180) for p in procs]
    for p, (out, err) in zip(procs, outs):
        assert p.returncode == 0, err[-2000:]
    import json
    res = [json.loads(out.strip().splitlines()[-1]) for out, _ in outs]
    for r in res:
        assert r["t"] == 15.0 and r["u"] == 300.0


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="1", CUDA_VISIBLE_DEVICES="")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--workload", "tiny_tf_fp32"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert p.returncode == 0, p.stderr[-2000:]
    assert p.stdout.strip() == ""        # ranks other than 0 exit 0 without work or output


def test_reference_arm_prints_one_json_line_on_rank_zero():
    import json
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    env.pop("RANK", None); env.pop("WORLD_SIZE", None)
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--workload", "tiny_tf_fp32"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert p.returncode == 0, p.stderr[-2000:]
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
