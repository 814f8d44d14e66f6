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


# ---------------------------------------------------------------------------------------------- Ulysses
ULYSSES_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r}); sys.path.insert(0, os.path.join({root!r}, "tests"))
import numpy as np, torch, torch.distributed as dist
import oracle
from paper_2606_25473_b200 import ulysses
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size={world})
rank, P = dist.get_rank(), dist.get_world_size()
B, H, d, L, F = 2, 4, 16, 6, 2                      # teacher forcing: N = 2 F L = 24 tokens, sharded over P ranks
N = 2 * F * L
g = torch.Generator().manual_seed(7)                # every rank draws the same global tensors, then keeps its shard
full = [torch.randn((B, H, N, d), generator=g, dtype=torch.float32) for _ in range(6)]
n = N // P
shard = [x[:, :, rank * n:(rank + 1) * n].contiguous() for x in full]
om = oracle.teacher_forcing_mask(L, F)
calls = []
def local_op(q, k, v, tq, tk, tv):                  # the test's stand-in for the CUDA call: the oracle on this rank's heads
    assert q.shape == (B, H // P, N, d)
    calls.append(1)
    o, to, lse = oracle.attn_jvp(om, *[t.numpy() for t in (q, k, v, tq, tk, tv)], 1.0 / np.sqrt(d))
    return torch.from_numpy(o).float(), torch.from_numpy(to).float(), torch.from_numpy(lse).float()
# round trip of the two exchanges alone
hs = ulysses.seq_to_head_shard(shard)
for t in range(6):
    assert torch.equal(hs[t], full[t][:, rank * (H // P):(rank + 1) * (H // P)])      # all tokens of my heads, in order
back = ulysses.head_to_seq_shard(hs)
for t in range(6):
    assert torch.equal(back[t], shard[t])
o, to, lse = ulysses.ulysses_attn_jvp(local_op, *shard)
ro, rto, rlse = oracle.attn_jvp(om, *[t.numpy() for t in full], 1.0 / np.sqrt(d))     # the undistributed result
err_o = float(np.abs(o.numpy() - ro[:, :, rank * n:(rank + 1) * n]).max())
err_to = float(np.abs(to.numpy() - rto[:, :, rank * n:(rank + 1) * n]).max())
err_lse = float(np.abs(lse.numpy() - rlse[:, rank * (H // P):(rank + 1) * (H // P)]).max())
dist.barrier()
dist.destroy_process_group()
print(json.dumps({{"rank": rank, "err_o": err_o, "err_to": err_to, "err_lse": err_lse, "calls": len(calls),
                  "shape": list(o.shape)}}))
"""


def _run_ranks(tmp_path, source, world):
    import json
    script = tmp_path / "worker.py"
    script.write_text(source)
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="2")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (out, err) in zip(procs, outs):
        assert p.returncode == 0, err[-3000:]
    return [json.loads(out.strip().splitlines()[-1]) for out, _ in outs]


def test_ulysses_all_to_all_round_trip_and_distributed_result_equals_the_undistributed_one(tmp_path):
    """Two gloo ranks, sequence-sharded inputs: one packed all-to-all in (six tensors), the local op on H/P heads with
    the full sequence and the unchanged mask, one packed all-to-all out."""
    for world in (2, 4):
        res = _run_ranks(tmp_path, ULYSSES_WORKER.format(root=ROOT, world=world), world)
        assert sorted(r["rank"] for r in res) == list(range(world))
        for r in res:
            assert r["calls"] == 1 and r["shape"] == [2, 4, 24 // world, 16]
            assert r["err_o"] < 1e-6 and r["err_to"] < 1e-6 and r["err_lse"] < 1e-6
