"""The N > 1 path of bench.py is "replicas only": no data-path collective, the only
cross-rank traffic is the MAX reduction of the per-rank step time.  World size 2 over gloo on CPU."""
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert bench.dist_env() == (rank, rank, world)
    mine = 1.5 + rank                      # rank 1 is the slow replica
    total = bench.max_over_ranks(mine, world, "cpu")
    dist.barrier()
    q.put((rank, total, bench.aggregate_updates_per_s(total, world)))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [2.5, 2.5]            # both ranks see the slowest replica's time
    assert [r[2] for r in res] == [800.0, 800.0]        # 2 replicas -> 2 updates per 2.5 ms step: throughput, not latency


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.25, 1) == 3.25 and bench.aggregate_updates_per_s(4.0, 1) == 250.0
    assert bench.dist_env()[2] >= 1


def test_reference_arm_runs_without_a_gpu_and_prints_the_contract_line():
    """bench.py --impl reference: the CPU oracle on a bounded sample; rank > 0 exits silently."""
    import json
    import subprocess
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "3", "--scale", "0.04",
           "--steps", "1", "--warmup", "0", "--reference-budget-s", "2"]
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "config",
              "cpu_baseline", "e2e"):
        assert k in line, k
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    out1 = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=dict(env, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1"))
    assert out1.returncode == 0 and out1.stdout.strip() == ""


def test_slab_ranges_partition_the_mipmap():
    """bench.py --partition slab: the ranks' voxel ranges are disjoint, aligned, balanced and cover everything."""
    sys.path.insert(0, ROOT)
    import bench
    for n in (1438087680, 4096, 4097, 5, 299648):
        for world in (1, 2, 3, 4, 8):
            r = [bench.slab_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            for (a0, a1), (b0, b1) in zip(r, r[1:]):
                assert a1 == b0 and a0 <= a1
            sizes = [b - a for a, b in r]
            assert all(a % 4096 == 0 for a, _ in r)
            assert max(sizes) - min(sizes) <= 4096 or n < 4096 * world


def test_committed_traffic_table_is_readable_by_bench():
    """roofline.traffic comes from profiles/roofline_traffic.csv (ncu dram bytes per launch of the dominant kernel)."""
    sys.path.insert(0, ROOT)
    import bench
    t = bench.ncu_traffic("cfg3_neocortex_shaped", "k_colorize")
    assert t is not None and 0.9 * 8 * 1438087061 < t < 1.1 * 8 * 1438087061          # about the algorithmic 8 B / voxel
    assert bench.ncu_traffic("cfg5_dag_stress", "k_colorize_tile") > 24 * 512 ** 3   # random gathers: far above it
    assert bench.ncu_traffic("cfg5_dag_stress", "k_level") > 60 * 2 ** 26
    assert bench.ncu_traffic("no_such_workload", "k_colorize") is None
