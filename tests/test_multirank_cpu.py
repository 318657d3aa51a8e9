"""N > 1 host logic on CPU: world_size-2 gloo runs of the reduction used by bench.py, and the
reference arm under torchrun (rank 0 alone prints one JSON line, the other rank exits 0)."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CFG5_PAIRS = [580, 653, 2006, 1938, 3152, 3218, 3644, 3660]      # coupled pairs of the eight J^pi of config 5 (oracle tables)


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    from paper_1404_5253_b200 import shard
    import wpcd_inputs as wi

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert shard.rank_world() == (rank, rank, world)
    # each rank: its own lattice, a fake step time and unit count
    p = wi.WORKLOADS["cfg1"].grid(seed_offset=shard.lattice_seed_offset(rank))
    ms, units = 1.0 + rank, 1000.0 * (rank + 1)
    ms_max, units_sum = shard.reduce_step(dist, "cpu", ms, units)
    mine = shard.assign_round_robin(list(range(5)), rank, world)
    # the J^pi matrices of config 5 dealt by cost (coupled channel pairs), as bench.py does for the nd workloads
    jpis = wi.WORKLOADS["cfg5"].jpis
    dealt = shard.assign_balanced(jpis, CFG5_PAIRS, rank, world)
    np.save(os.path.join(out_dir, f"grid{rank}.npy"), p)
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"ms_max": ms_max, "units_sum": units_sum, "mine": mine, "value": shard.throughput(ms_max, units_sum), "dealt": dealt}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_gloo_world2_reduction(tmp_path):
    import torch.multiprocessing as mp

    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0, r1 = (json.load(open(tmp_path / f"r{k}.json")) for k in (0, 1))
    assert r0["ms_max"] == r1["ms_max"] == 2.0            # the slowest rank
    assert r0["units_sum"] == r1["units_sum"] == 3000.0   # all ranks' units
    assert r0["value"] == 3000.0 / 2e-3
    assert sorted(r0["mine"] + r1["mine"]) == [0, 1, 2, 3, 4] and r0["mine"] == [0, 2, 4]
    # the union of the ranks' matrices is the workload, nothing twice, loads within 1 % of each other
    import wpcd_inputs as wi
    jpis = [list(j) for j in wi.WORKLOADS["cfg5"].jpis]
    assert sorted(r0["dealt"] + r1["dealt"]) == sorted(jpis) and not [j for j in r0["dealt"] if j in r1["dealt"]]
    load = [sum(CFG5_PAIRS[jpis.index(j)] for j in r["dealt"]) for r in (r0, r1)]
    assert abs(load[0] - load[1]) <= 0.01 * sum(load)
    g0, g1 = np.load(tmp_path / "grid0.npy"), np.load(tmp_path / "grid1.npy")
    assert g0.shape == g1.shape and g0[0] == g1[0] == 0.0 and g0[-1] == g1[-1] and not np.array_equal(g0, g1)


def test_reference_arm_under_torchrun_world2():
    port = 31500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "cfg1",
           "--steps", "1", "--warmup", "0"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                 # rank 0 alone prints
    rec = json.loads(lines[0])
    assert rec["impl"] == "reference" and rec["n_gpus"] == 2 and rec["value"] > 0
    assert rec["cpu_baseline"]["kind"] == "oracle" and rec["e2e"]["h2d_bytes_per_step"] == 0


def test_assign_balanced_partitions_any_world():
    """Every rank computes the same deal; the union is the job list for any world size, more ranks than jobs leave ranks idle."""
    sys.path.insert(0, ROOT)
    from paper_1404_5253_b200 import shard

    items = list(range(8))
    for world in (1, 2, 3, 4, 8, 11):
        parts = [shard.assign_balanced(items, CFG5_PAIRS, r, world) for r in range(world)]
        assert sorted(sum(parts, [])) == items
        loads = [sum(CFG5_PAIRS[k] for k in p) for p in parts]
        assert max(loads) <= max(max(CFG5_PAIRS), 1.1 * sum(CFG5_PAIRS) / world)
        assert parts[0] and 7 in parts[0]                    # the largest matrix goes to rank 0 (it prints the line)
