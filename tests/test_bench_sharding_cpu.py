"""The N > 1 path of bench.py on CPU: two gloo ranks shard the sites of an edge (no data-path collective) and agree on
the max-over-ranks time; the reference arm runs on rank 0 only."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    idx = bench.shard_atoms(rank, 3, 8)
    t = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")
    # the partial maps of the shards add up to the map of the union (sites are independent: eq. 14) -- checked with a
    # stand-in per-site contribution, since the contraction itself needs the GPU
    contrib = torch.zeros(8, dtype=torch.float64)
    contrib[idx] = torch.arange(8, dtype=torch.float64)[idx] + 1.0
    dist.all_reduce(contrib)
    q.put((rank, idx.tolist(), t, contrib.tolist()))
    dist.destroy_process_group()


def test_two_ranks_shard_sites_and_take_the_max_time():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got[0][1] == [0, 1, 2] and got[1][1] == [3, 4, 5]                 # disjoint contiguous blocks
    assert got[0][2] == got[1][2] == 15.0                                    # max over ranks on both
    assert got[0][3] == got[1][3] == [1.0, 2.0, 3.0, 4.0, 5.0, 6.0, 0.0, 0.0]


def test_shard_clamps_at_the_end_of_the_edge():
    import bench
    assert bench.shard_atoms(2, 3, 8).tolist() == [6, 7]
    assert bench.shard_atoms(3, 3, 8).tolist() == []
    assert bench.max_over_ranks(3.5, 1) == 3.5


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` (the oracle timed on the host cores) at quarter scale: one JSON line with the keys
    the driver reads; ranks other than 0 print nothing."""
    import json
    import subprocess
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--scale", "4", "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "amplitudes/s" and d["value"] > 0 and d["higher_is_better"] is True
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    r1 = subprocess.run(cmd, capture_output=True, text=True, env=dict(env, RANK="1", WORLD_SIZE="2"), timeout=600)
    assert r1.returncode == 0 and not [l for l in r1.stdout.splitlines() if l.startswith("{")]


def test_sample_sites_spreads_a_step_over_planes_and_ranks():
    """bench.sample_sites: --atoms sites spread evenly over the first --planes ionisation planes; ranks take disjoint blocks
    inside every plane ("atoms spread over planes")."""
    import bench
    from bip_inputs.specimen import make_workload
    e = make_workload("cfg1", scale=2, nz=8).edges[0]
    planes = np.unique(e.slice)
    a = bench.sample_sites(e, 0, 4, 2)
    b = bench.sample_sites(e, 1, 4, 2)
    assert len(a) == len(b) == 4 and not set(a.tolist()) & set(b.tolist())
    assert sorted(set(e.slice[a].tolist())) == planes[:2].tolist() == sorted(set(e.slice[b].tolist()))
    assert np.bincount(e.slice[a])[planes[:2]].tolist() == [2, 2]


def test_gpus_flag_must_match_the_launch():
    """`--gpus N` under a launcher that started a different number of ranks fails loudly instead of running 1 GPU."""
    import subprocess
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "8"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0 and "does not match WORLD_SIZE" in (r.stderr + r.stdout)
