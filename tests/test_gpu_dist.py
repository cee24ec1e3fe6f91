"""The N > 1 path of bench.py on hardware (replicas + voxel-slab partition, no data-path collective).

The GPU box has ONE device, so two ranks share cuda:0 and talk over gloo (`--dist-backend gloo`): the ranks' kernels never
wait on one another -- the only cross-rank traffic is the barrier and the MAX reduction of the step time -- so this is
the real N = 2 code path (rendezvous, slab slicing on the device, mg_tf_update_host on a slab, rank-0 JSON line), not a
stand-in for two GPUs; its timings are not scaling numbers.  Each rank dumps the host copy of its colourised slab; the
stitched mipmap is compared with the oracle element by element."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SCALE = 0.1
TOL = 1e-5


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _launch(tmp_path, partition):
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    dump = str(tmp_path / f"dump_{partition}")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3", "--warmup", "3",
           "--scale", str(SCALE), "--partition", partition, "--dist-backend", "gloo", "--dump-dir", dump,
           "--no-cpu-baseline", "--no-render", "--no-query", "--no-packed", "--no-attr"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [l for l in out.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]                       # rank 0 alone prints
    return json.loads(lines[0]), [np.load(os.path.join(dump, f"rank{r}.npz")) for r in range(2)]


def _oracle_mipmap(tf_update):
    """RGBA8 of every voxel of the concatenated mipmap by the oracle, from the host-side assembly of the same config."""
    from paper_2009_02702_b200 import workload
    w = workload.make(3, SCALE, load=False)
    hg = w.host_graph
    ref_nodes = oracle.graph_eval(hg["child_a"], hg["child_b"], hg["weight"], hg["n_leaves"], w.tf(tf_update).astype(np.float64))
    flat = np.zeros(w.n_voxels_padded, dtype=np.uint32)              # padding voxels hold node 0 (workload.py)
    for s0, lv in zip(w.level_start, w.host_idx):
        flat[s0:s0 + lv.size] = lv.reshape(-1)
    return w, ref_nodes, oracle.lookup(flat, ref_nodes)


def _rgba8_close(got, ref_c):
    code = oracle.to_rgba8(ref_c).astype(np.int64)
    diff = got.astype(np.int64) - code
    scaled = np.clip(ref_c, 0.0, 1.0) * 255.0
    near = np.abs(scaled - np.floor(scaled) - 0.5) <= 255 * TOL + 1e-4
    return bool(((diff == 0) | ((np.abs(diff) == 1) & near)).all())


def test_slab_partition_world2_stitches_to_the_oracle_mipmap(tmp_path):
    line, dumps = _launch(tmp_path, "slab")
    assert line["n_gpus"] == 2 and line["scaling"] == "strong" and "slab" in line["config"]["parallelism"]
    assert line["value"] == line["ms_per_step"] > 0 and line["e2e"]["value"] > 0
    n_pad = int(dumps[0]["n_voxels_padded"])
    lo0, hi0, lo1, hi1 = (int(dumps[r][k]) for r in range(2) for k in ("v_lo", "v_hi"))
    assert lo0 == 0 and hi0 == lo1 and hi1 == n_pad and lo1 % 4096 == 0 and abs((hi0 - lo0) - (hi1 - lo1)) <= 4096
    assert line["e2e"]["d2h_bytes_per_step"] == 4 * (hi0 - lo0)       # rank 0's slab only
    w, ref_nodes, ref_c = _oracle_mipmap(int(dumps[0]["tf_update"]))
    assert w.n_voxels_padded == n_pad
    stitched = np.concatenate([dumps[0]["out"], dumps[1]["out"]]).reshape(-1, 4)
    assert stitched.shape[0] == n_pad
    assert _rgba8_close(stitched, ref_c)
    for d in dumps:                                                  # graph + propagation replicated on both ranks
        assert np.abs(d["nodes"] - ref_nodes).max() <= TOL
    assert np.array_equal(dumps[0]["nodes"], dumps[1]["nodes"])


def test_replicas_world2_each_rank_holds_the_whole_oracle_mipmap(tmp_path):
    line, dumps = _launch(tmp_path, "replicas")
    assert line["n_gpus"] == 2 and line["scaling"] == "weak" and "replicas" in line["config"]["parallelism"]
    assert line["value"] == line["ms_per_step"] > 0                  # latency of one update: not divided by N
    assert abs(line["updates_per_s"] - 2e3 / line["ms_per_step"]) < 1e-6 * line["updates_per_s"]
    w, ref_nodes, ref_c = _oracle_mipmap(int(dumps[0]["tf_update"]))
    for d in dumps:
        assert int(d["v_lo"]) == 0 and int(d["v_hi"]) == w.n_voxels_padded
        assert _rgba8_close(d["out"].reshape(-1, 4), ref_c)
        assert np.abs(d["nodes"] - ref_nodes).max() <= TOL
