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
G = {groups}
B, H, d, L, F = 2, 8, 16, 6, 2                      # teacher forcing: N = 2 F L = 24 tokens, sharded over P ranks
N = 2 * F * L
g = torch.Generator().manual_seed(7)                # every rank draws the same global tensors, then keeps its shard
full = [torch.randn((B, H, N, d), generator=g, dtype=torch.float32) for _ in range(7)]      # q k v tq tk tv dO
n, h, hg = N // P, H // P, H // (P * G)
shard = [x[:, :, rank * n:(rank + 1) * n].contiguous() for x in full]
om = oracle.teacher_forcing_mask(L, F)
calls = []
def local_op(grp, q, k, v, tq, tk, tv):             # the test's stand-in for the CUDA call: the oracle on one head group
    assert q.shape == (B, hg, N, d)
    calls.append(grp)
    o, to, lse = oracle.attn_jvp(om, *[t.numpy() for t in (q, k, v, tq, tk, tv)], 1.0 / np.sqrt(d))
    return torch.from_numpy(o).float(), torch.from_numpy(to).float(), torch.from_numpy(lse).float()
def local_bwd(grp, q, k, v, o, lse, dout):
    res = [oracle.attn_bwd_head(om, q[b, x].numpy(), k[b, x].numpy(), v[b, x].numpy(), dout[b, x].numpy(), 1.0 / np.sqrt(d))
           for b in range(B) for x in range(hg)]
    return tuple(torch.from_numpy(np.stack([r[i] for r in res]).reshape(B, hg, N, d)).float() for i in range(3))
# the index arithmetic alone: pack -> all-to-all -> unpack gives all tokens of my heads of group grp, in order
for grp in range(G):
    recv, work = ulysses._exchange(ulysses.pack_seq_shard(shard[:6], P, grp, G), None, True)
    work.wait()
    hs = ulysses.unpack_head_shard(recv)
    for t in range(6):
        assert torch.equal(hs[t], full[t][:, rank * h + grp * hg:rank * h + (grp + 1) * hg])
    back, work = ulysses._exchange(ulysses.pack_head_shard(hs, P), None, True)
    work.wait()
    outs = [torch.zeros_like(x) for x in shard[:6]]
    ulysses.unpack_seq_shard(back, outs, grp, G)
    for t in range(6):
        sel = torch.zeros(H, dtype=torch.bool)
        for j in range(P):
            sel[j * h + grp * hg:j * h + (grp + 1) * hg] = True
        assert torch.equal(outs[t][:, sel], shard[t][:, sel]) and torch.count_nonzero(outs[t][:, ~sel]) == 0
# the zero-copy chunk lists: every [n, d] block lands where the kernel reads it, and comes back where the caller reads it
for grp in range(G):
    heads = [torch.full((B, hg, N, d), float("nan")) for _ in range(6)]
    ulysses._exchange_p2p(ulysses.p2p_chunks_in(shard[:6], heads, P, rank, grp, G), rank, None).wait()
    for t in range(6):
        assert torch.equal(heads[t], full[t][:, rank * h + grp * hg:rank * h + (grp + 1) * hg])
    outs = [torch.zeros_like(x) for x in shard[:6]]
    ulysses._exchange_p2p(ulysses.p2p_chunks_out(heads, outs, P, rank, grp, G), rank, None).wait()
    for t in range(6):
        sel = torch.zeros(H, dtype=torch.bool)
        for j in range(P):
            sel[j * h + grp * hg:j * h + (grp + 1) * hg] = True
        assert torch.equal(outs[t][:, sel], shard[t][:, sel]) and torch.count_nonzero(outs[t][:, ~sel]) == 0
# both exchange modes give the same bits
o2, to2, saved2 = ulysses.ulysses_attn_jvp(local_op, *shard[:6], head_groups=G, mode="packed")
dq2, dk2, dv2 = ulysses.ulysses_attn_bwd(local_bwd, saved2, shard[6], head_groups=G, mode="packed")
calls.clear()
o, to, saved = ulysses.ulysses_attn_jvp(local_op, *shard[:6], head_groups=G)
dq, dk, dv = ulysses.ulysses_attn_bwd(local_bwd, saved, shard[6], head_groups=G)
for a, b in zip((o, to, dq, dk, dv), (o2, to2, dq2, dk2, dv2)):
    assert torch.equal(a, b)
sl = slice(rank * n, (rank + 1) * n)
ro, rto, rlse = oracle.attn_jvp(om, *[t.numpy() for t in full[:6]], 1.0 / np.sqrt(d))     # the undistributed result
err = dict(o=float(np.abs(o.numpy() - ro[:, :, sl]).max()), to=float(np.abs(to.numpy() - rto[:, :, sl]).max()))
lse = torch.cat([s[4] for s in saved], dim=1)        # head-sharded: [B, H/P, N] of my heads
err["lse"] = float(np.abs(lse.numpy() - rlse[:, rank * h:(rank + 1) * h]).max())
for name, got, i in (("dq", dq, 0), ("dk", dk, 1), ("dv", dv, 2)):
    ref = np.stack([[oracle.attn_bwd_head(om, *[full[t][b, x].numpy() for t in (0, 1, 2, 6)], 1.0 / np.sqrt(d))[i]
                     for x in range(H)] for b in range(B)])
    err[name] = float(np.abs(got.numpy() - ref[:, :, sl]).max())
dist.barrier()
dist.destroy_process_group()
print(json.dumps({{"rank": rank, "err": err, "calls": calls, "shape": list(o.shape)}}))
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
    """gloo ranks, sequence-sharded inputs: per head group one packed all-to-all in (six tensors), the local op on the
    group's heads with the full sequence and the unchanged mask, one packed all-to-all out; then
    the backward direction (dO in; dQ, dK, dV out) on the head-sharded q, k, v, o, lse the forward left on the rank."""
    for world, groups in ((2, 1), (2, 2), (4, 2)):
        res = _run_ranks(tmp_path, ULYSSES_WORKER.format(root=ROOT, world=world, groups=groups), world)
        assert sorted(r["rank"] for r in res) == list(range(world))
        for r in res:
            assert r["calls"] == list(range(groups)) and r["shape"] == [2, 8, 24 // world, 16]
            assert max(r["err"].values()) < 1e-5, r["err"]


def test_bench_ulysses_arm_dry_run_on_two_gloo_ranks():
    """`torch.distributed.run --nproc-per-node 2 bench.py --gpus 2 --ulysses` without CUDA: the exchange pipeline of the
    Ulysses arm (two head groups, async all-to-alls) on gloo with a no-op local op; rank 0 prints one JSON line."""
    import json
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="2")
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        env.pop(k, None)
    p = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
                        "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--ulysses",
                        "--steps", "2", "--warmup", "1", "--workload", "tiny_tf_fp32", "--head-groups", "1"],
                       env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-3000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["mode"] == "ulysses" and line["dry_run"] and line["n_gpus"] == 2 and line["scaling"] == "strong"
    assert line["backend"] == "gloo" and line["collectives_per_step"] == 2 and line["value"] is None
    assert line["a2a_bytes_in_per_rank"] == 6 * 1 * 2 * 48 * 64 * 4 // 2
