#!/usr/bin/env python
"""bench.py -- TF-update latency of the Mixture Graph hot path on B200 (contract: see DESIGN.md §Measurement).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--format rgba8|rgba16f]
  python bench.py --impl reference ...      # the CPU fp64 oracle, as it stands, on the host cores

One "step" = one full transfer-function update = every §8(a) device row:
  a4 leaf assignment + a5 level-synchronous propagation (mg_propagate, TF already in HBM)
  a6 colourise of EVERY mip level (mg_colorize over the concatenated node-index mipmap).
`value` = milliseconds per TF update with all inputs resident in HBM (CUDA events on the launch
stream, barrier + synchronize on both sides, max over ranks).  `e2e` = the same update through
mg_tf_update_host: TF from pinned HOST memory, colourised mipmap copied back to pinned HOST memory,
both copies inside the timed region.  Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tf_update_latency_ms"
UNIT = "ms"
FALLBACK_HBM_GBS = 6650.0            # /opt/skills/guides/B200_PROFILING.md fallback ("of fallback")
NOMINAL_HBM_GBS = 8000.0             # BASELINE.json north_star "~8 TB/s"
BYTES_PER_VOXEL = {"rgba8": 8, "rgba16f": 12}       # 4 B index + 4 B (8 B) output
BYTES_PER_NODE_L2 = 28               # 12 B a/b/w stream + 16 B colour store (gathers hit L2), §8(d)
BYTES_PER_NODE_DRAM = 60             # + two 16-B gathers when the fp32 palette exceeds L2 (config 5), §8(d)
BYTES_GATHER_BEYOND_L2 = {"rgba8": 4, "rgba16f": 8}    # per-voxel palette gather, counted only when the palette exceeds L2 (config 5):
                                                        # the entry the kernel really reads (RGBA8 / 4 x fp16 palette), not the 16-B
BYTES_GATHER_SURVEY = 16                                # fp32 entry SURVEY.md §8(d) counts (kept beside it as *_survey)
L2_BYTES = 126e6


def parse_args():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=300)
    p.add_argument("--warmup", type=int, default=10)
    p.add_argument("--impl", choices=["b200", "reference"], default="b200")
    p.add_argument("--config", type=int, default=3, help="BASELINE.json config 1-5 (default 3: 2048x2048x300)")
    p.add_argument("--scale", type=float, default=1.0, help="geometric down-scale of the config (debugging only)")
    p.add_argument("--format", choices=["rgba8", "rgba16f"], default="rgba8")
    p.add_argument("--e2e-steps", type=int, default=0, help="0 = min(steps, 8)")
    p.add_argument("--no-cpu-baseline", action="store_true")
    p.add_argument("--no-e2e", action="store_true")
    p.add_argument("--no-attr", action="store_true", help="skip the extra NEXT-1 measurement (multi-attribute propagation)")
    p.add_argument("--host-mipmap", action="store_true",
                   help="configs 1-4: build the whole histogram mipmap on the host (default: the two finest levels are classified "
                        "on the device, NEXT-4 front end; same graph and node indices either way)")
    p.add_argument("--device-levels", action="store_true",
                   help="configs 1-4: build the levels >= 1 of the histogram mipmap on the device too (mg_mipmap_levels_build: merge + "
                        "hash-cons per level; the host continues above the last level whose mixtures a warp can merge); same graph "
                        "and node indices, shorter setup")
    p.add_argument("--partition", choices=["replicas", "slab"], default="replicas",
                   help="N > 1: independent replicas of the whole update (default, weak scaling) or ONE update whose colourise is "
                        "split into N contiguous voxel slabs with the graph replicated (strong scaling, SURVEY.md 8(e)); no collective either way")
    p.add_argument("--dist-backend", choices=["nccl", "gloo"], default="nccl",
                   help="N > 1: process-group backend for the barrier and the max-over-ranks timing reduction (the only cross-rank "
                        "traffic).  gloo lets several ranks share one GPU (rank r uses device r mod device_count): how the N > 1 "
                        "code path is exercised on a one-GPU box (tests/test_gpu_dist.py); its timings are not scaling numbers")
    p.add_argument("--dump-dir", default=None,
                   help="every rank writes rank<r>.npz there: its voxel range and the host copy of its colourised mipmap slab as "
                        "the last mg_tf_update_host of the e2e leg left it (tests compare the stitched slabs with the oracle)")
    p.add_argument("--relabel", action="store_true", help="(the default on config 5; kept for old command lines)")
    p.add_argument("--no-relabel", action="store_true",
                   help="config 5: load the DAG in the caller's numbering instead of with MG_RELABEL (every level sorted by its "
                        "children: the higher child becomes a sequential sweep, 2.02 -> 1.72 ms)")
    p.add_argument("--no-query", action="store_true", help="skip the extra NEXT-4 measurement (mixture LUT + range queries)")
    p.add_argument("--render-empty-background", action="store_true",
                   help="render section: make the first leaf (config 4: background ID 0) exactly transparent, the case "
                        "empty-space skipping is for (L271)")
    p.add_argument("--render-alpha-zero-frac", type=float, default=None,
                   help="render section: fraction of segments made exactly transparent (default: the config's own)")
    p.add_argument("--no-render", action="store_true", help="skip the extra NEXT-2 measurement (ray-marcher over the paletted mipmap)")
    p.add_argument("--no-packed", action="store_true", help="skip the extra NEXT-3 measurement (bit-packed node IDs)")
    p.add_argument("--cpu-sample-voxels", type=int, default=1 << 31, help="oracle sample size (>= the mipmap = whole workload)")
    p.add_argument("--reference-budget-s", type=float, default=90.0)
    return p.parse_args()


# ------------------------------------------------------------------------------------------------
# clocks: sample SM clock + throttle reasons DURING the timed region (NVML in a thread)
# ------------------------------------------------------------------------------------------------

class ClockSampler:
    def __init__(self, device_index: int, period_s: float = 0.02):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self._idx, self._period = device_index, period_s
        self.error = None

    def _visible_index(self) -> int:
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            ids = [v.strip() for v in vis.split(",") if v.strip()]
            if self._idx < len(ids) and ids[self._idx].isdigit():
                return int(ids[self._idx])
        return self._idx

    def _run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self._visible_index())
            self.max_mhz = int(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            names = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                     "hw_power_brake_slowdown": 0x80, "sw_power_cap": 0x4, "sync_boost": 0x10,
                     "applications_clocks_setting": 0x2}
            while not self._stop.is_set():
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
                time.sleep(self._period)
        except Exception as exc:                      # noqa: BLE001 -- reported in the JSON, never fatal
            self.error = repr(exc)

    def __enter__(self):
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._thr.join(timeout=5)

    def summary(self) -> dict:
        out = {"sm_mhz": (float(np.median(self.samples)) if self.samples else None), "sm_max_mhz": self.max_mhz,
               "reasons": sorted(self.reasons), "samples": len(self.samples)}
        if self.error:
            out["error"] = self.error
        return out


# ------------------------------------------------------------------------------------------------
# the oracle as a timed CPU baseline (cpu_baseline leg and --impl reference): test infrastructure,
# executed here only, as it stands (oracle/__init__.py: graph_eval_levels + colourise_rgba8)
# ------------------------------------------------------------------------------------------------

def _sample_plan(w, n_sample: int):
    """Leading voxels of every mip level, in proportion to the level's size (>= 1 voxel each)."""
    frac = min(1.0, n_sample / max(1, w.n_voxels))
    return [max(1, int(np.ceil(v * frac))) if v else 0 for v in w.level_voxels]


def oracle_step(w, tf64, plan, chunk: int = 1 << 25, n_threads: int = 0):
    """One TF update by the oracle on a sample: (propagate seconds, colourise seconds, threads); n_threads = 0: all cores."""
    import oracle
    g = w.host_graph
    levels = [w.host_level(l) for l in range(len(plan))]           # (a download when level 0 only lives on the device)
    t0 = time.perf_counter()
    c, used = oracle.graph_eval_levels(g["child_a"], g["child_b"], g["weight"], g["n_leaves"], tf64, n_threads=n_threads)
    t1 = time.perf_counter()
    for lvl, n in zip(levels, plan):
        flat = lvl.reshape(-1)
        for o in range(0, n, chunk):
            oracle.colourise_rgba8(flat[o:min(n, o + chunk)], c, n_threads=n_threads)
    t2 = time.perf_counter()
    return t1 - t0, t2 - t1, int(used)


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(w, n_sample: int) -> dict:
    plan = _sample_plan(w, n_sample)
    tf64 = w.tf(0).astype(np.float64)
    tp, tc, used = oracle_step(w, tf64, plan)
    n_s = sum(plan)
    ms = 1e3 * (tp + tc * (w.n_voxels / n_s))
    # the same oracle on ONE thread (SURVEY.md 8(d) "Oracle timing (i)"; the paper's CPU figures, are multi-core):
    # full propagation, colourise on an eighth of the sample, scaled
    plan1 = _sample_plan(w, max(1, n_s // 8))
    tp1, tc1, used1 = oracle_step(w, tf64, plan1, n_threads=1)
    n_s1 = sum(plan1)
    ms1 = 1e3 * (tp1 + tc1 * (w.n_voxels / n_s1))
    return {"value": ms, "unit": UNIT, "cores": used, "kind": "oracle", "cpu_model": cpu_model(), "host_cores": os.cpu_count(),
            "sample": f"full fp64 level-synchronous propagation of all {w.stats['n_nodes']} nodes ({1e3 * tp:.1f} ms) + "
                      f"fp64 lookup/RGBA8 conversion of the leading {n_s} of {w.n_voxels} voxels (same share of every "
                      f"mip level, {1e3 * tc:.1f} ms), colourise time scaled to the whole mipmap",
            "propagate_ms": 1e3 * tp, "colorize_sample_ms": 1e3 * tc, "sample_voxels": n_s,
            "threads_1_ms": ms1, "threads_1_propagate_ms": 1e3 * tp1, "threads_1_cores": used1,
            "threads_1_sample": f"one thread: full propagation ({1e3 * tp1:.1f} ms) + the leading {n_s1} voxels "
                                f"({1e3 * tc1:.1f} ms), colourise time scaled to the whole mipmap"}


def workload_config(w, args, n_gpus: int) -> dict:
    s = w.stats
    cfg = {"workload": w.name, "baseline_config": args.config, "mip_voxels": w.n_voxels, "mip_levels": len(w.level_voxels),
           "nodes": s["n_nodes"], "leaves": s["n_leaves"], "topo_depth": s["depth"], "output": args.format,
           "parallelism": "single GPU" if n_gpus == 1 else
                          (f"{n_gpus}-way voxel-slab partition of colourise, graph and propagation replicated (no collective)"
                           if getattr(args, "partition", "replicas") == "slab" else f"{n_gpus} independent replicas (no collective)"),
           "l2": "inputs larger than L2 (node-index stream %.2f GB per step, L2 126 MB); no explicit flush" % (4e-9 * w.n_voxels)}
    if "quant_bits" in s:
        cfg["quant_bits"] = s["quant_bits"]
    cfg["tf_sequence"] = "%s, %d distinct updates cycled in order" % (w.cfg.get("tf_sequence", "random"),
                                                                       max(1, min(args.steps + args.warmup, w.n_updates)))
    if args.scale != 1.0:
        cfg["scale"] = args.scale
    return cfg


# ------------------------------------------------------------------------------------------------
# distributed plumbing: one process per GPU, replicas only -- the only
# cross-rank traffic is the timing reduction (max over ranks)
# ------------------------------------------------------------------------------------------------

def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def max_over_ranks(value: float, world: int, device="cpu") -> float:
    """MAX over all ranks of a per-rank duration (the only cross-rank traffic of a replica run)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def slab_range(n_voxels_padded: int, rank: int, world: int, align: int = 4096):
    """Voxel range [lo, hi) of rank's slab: the concatenated mipmap cut into `world` contiguous pieces whose
    boundaries are multiples of `align` voxels (one colourise CTA; keeps every 16-byte vector aligned).  The
    pieces are disjoint, cover [0, n_voxels_padded) and differ by at most `align` voxels."""
    blocks = -(-int(n_voxels_padded) // align)
    lo = (blocks * rank // world) * align
    hi = (blocks * (rank + 1) // world) * align
    return min(lo, n_voxels_padded), min(hi, n_voxels_padded)


def aggregate_updates_per_s(ms_per_step: float, world: int) -> float:
    """Whole-job THROUGHPUT of a replica run: `world` independent replicas finish `world` updates per step time.
    (The latency metric itself does not improve with replicas: every update still takes ms_per_step.)"""
    return max(1, world) / (ms_per_step * 1e-3)


def peak_hbm_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    except Exception:                                   # noqa: BLE001
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(workload: str, kernel: str):
    """dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/), or None."""
    path = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    try:
        with open(path) as f:
            for line in f:
                p = [x.strip() for x in line.split(",")]
                if len(p) >= 4 and p[0] == workload and p[1] == kernel:
                    return float(p[2]) + float(p[3])
    except OSError:
        pass
    return None


def run_b200(args) -> dict:
    import torch
    import torch.distributed as dist

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the hot path has no CPU fallback)")
    device_index = local_rank % torch.cuda.device_count()           # (> 1 rank per GPU only with --dist-backend gloo)
    torch.cuda.set_device(device_index)
    red_dev = "cuda"
    if world > 1:
        if args.dist_backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", device_index))
        else:
            dist.init_process_group("gloo")
            red_dev = "cpu"
    from paper_2009_02702_b200 import mg, workload

    w = workload.make(args.config, args.scale, relabel=(args.config == 5 and not args.no_relabel),
                      device_mipmap=("levels" if args.device_levels else True) if (not args.host_mipmap and args.config != 5) else False)
    g = w.graph
    info = g.info
    n_nodes, n_internal = int(info.n_nodes), int(info.n_internal)
    fmt = mg.MG_RGBA8 if args.format == "rgba8" else mg.MG_RGBA16F
    out_bytes = 4 if args.format == "rgba8" else 8
    nodes = torch.empty((n_nodes, 4), dtype=torch.float32, device="cuda")
    out = torch.empty(w.n_voxels_padded * out_bytes, dtype=torch.uint8, device="cuda")
    n_tf = max(1, min(args.steps + args.warmup, w.n_updates))             # the config's own update sequence (100 TFs), in order
    tfs = [torch.from_numpy(w.tf(u)).cuda() for u in range(n_tf)]          # resident in HBM before the timed region
    stream = torch.cuda.current_stream()
    st = stream.cuda_stream
    slab = args.partition == "slab" and world > 1
    v_lo, v_hi = slab_range(w.n_voxels_padded, rank, world) if slab else (0, w.n_voxels_padded)
    idx_part, out_part, n_part = w.d_idx[v_lo:v_hi], out[v_lo * out_bytes:v_hi * out_bytes], v_hi - v_lo

    def step(k: int):
        g.propagate(tfs[k % n_tf], nodes, st)
        g.colorize(idx_part, n_part, nodes, out_part, fmt=fmt, stream=st, from_last_propagate=True)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for k in range(args.warmup):
        step(k)
    barrier()
    K = args.steps
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = mg.kernel_launch_count()
    with ClockSampler(device_index) as clocks:
        barrier()
        t_begin.record(stream)
        for k in range(K):
            e = ev[k]
            e[0].record(stream)
            g.propagate(tfs[(args.warmup + k) % n_tf], nodes, st)
            e[1].record(stream)
            g.colorize(idx_part, n_part, nodes, out_part, fmt=fmt, stream=st, from_last_propagate=True)
            e[2].record(stream)
        t_end.record(stream)
        barrier()
    launches = mg.kernel_launch_count() - launches0
    total_ms = t_begin.elapsed_time(t_end)
    prop_ms = np.array([e[0].elapsed_time(e[1]) for e in ev])
    col_ms = np.array([e[1].elapsed_time(e[2]) for e in ev])
    total_ms = max_over_ranks(total_ms, world, red_dev)
    ms_per_step = total_ms / K

    # ---- the same colourise WITHOUT the reuse flag: mg_colorize's default first derives the palette from node_rgba
    derive = None
    if rank == 0:
        kd = min(K, 20)
        evd = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(kd)]
        g.propagate(tfs[0], nodes, st)
        for _ in range(2):
            g.colorize(idx_part, n_part, nodes, out_part, fmt=fmt, stream=st)
        for k in range(kd):
            evd[k][0].record(stream)
            g.colorize(idx_part, n_part, nodes, out_part, fmt=fmt, stream=st)
            evd[k][1].record(stream)
        torch.cuda.synchronize()
        derive = float(np.mean([e[0].elapsed_time(e[1]) for e in evd]))

    # ---- SURVEY.md section 8(d)'s metric as the paper timed it: "GPU timings include the data upload of one float4 color per
    # source" -- mg_propagate_host from PINNED host TFs (H2D of n_leaves float4 + propagation), alone
    # and followed by the colourise of all levels; CUDA events on the launch stream, the config's TF sequence in order
    upload = None
    if rank == 0:
        ku = min(K, 100)
        tf_pin = [torch.from_numpy(w.tf(u)).pin_memory() for u in range(min(n_tf, ku))]
        for k in range(3):
            g.propagate_host(tf_pin[k % len(tf_pin)], nodes, st)
        torch.cuda.synchronize()
        evu = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(ku)]
        for k in range(ku):
            evu[k][0].record(stream)
            g.propagate_host(tf_pin[k % len(tf_pin)], nodes, st)
            evu[k][1].record(stream)
        torch.cuda.synchronize()
        ph = np.array([e[0].elapsed_time(e[1]) for e in evu])
        for k in range(ku):
            evu[k][0].record(stream)
            g.propagate_host(tf_pin[k % len(tf_pin)], nodes, st)
            g.colorize(idx_part, n_part, nodes, out_part, fmt=fmt, stream=st, from_last_propagate=True)
            evu[k][1].record(stream)
        torch.cuda.synchronize()
        uh = np.array([e[0].elapsed_time(e[1]) for e in evu])
        upload = {"propagate_host_ms": float(ph.mean()), "propagate_host_ms_median": float(np.median(ph)),
                  "update_incl_tf_upload_ms": float(uh.mean()), "update_incl_tf_upload_ms_median": float(np.median(uh)),
                  "tf_upload_bytes": int(w.n_leaves * 16), "steps": ku,
                  "what": "mg_propagate_host (pinned host TF -> H2D -> all levels): the quantity the paper times (L371-L373), and the "
                          "same followed by mg_colorize of every mip level"}
        del tf_pin

    # ---- NEXT-3 variant: the same update with the node IDs bit-packed at r(l) bits per voxel (Table 1)
    packed = None
    if not args.no_packed and rank == 0:
        w.pack()
        lv = w.packed_levels
        for k in range(3):
            g.propagate(tfs[k % n_tf], nodes, st)
            g.colorize_packed(w.d_packed, lv, nodes, out, fmt=fmt, stream=st, from_last_propagate=True)
        torch.cuda.synchronize()
        kp = min(K, 100)
        evp = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(kp)]
        for k in range(kp):
            evp[k][0].record(stream)
            g.propagate(tfs[k % n_tf], nodes, st)
            evp[k][1].record(stream)
            g.colorize_packed(w.d_packed, lv, nodes, out, fmt=fmt, stream=st, from_last_propagate=True)
            evp[k][2].record(stream)
        torch.cuda.synchronize()
        pc = float(np.mean([e[1].elapsed_time(e[2]) for e in evp]))
        pt = float(np.mean([e[0].elapsed_time(e[2]) for e in evp]))
        in_bytes = sum(l["bits"] * l["n_voxels"] for l in lv) / 8.0
        algo = in_bytes + out_bytes * w.n_voxels
        packed = {"tf_update_ms": pt, "colorize_ms": pc, "bits_per_voxel": 8.0 * in_bytes / w.n_voxels,
                  "bits_per_level": [l["bits"] for l in lv], "algorithmic_bytes_per_launch": algo,
                  "achieved_gbs": algo / (pc * 1e-3) / 1e9, "steps": kp, "kernel": "k_colorize_packed",
                  "what": "NEXT-3: node IDs stored as (id - i_min(l)) at r(l) bits per voxel (PAPER.md Table 1, Eq. 15-16)"}
        w.d_packed = None

    # ---- NEXT-1 variant: the same graph pass for other attributes (opacity alone; 4 TFs batched as 16 channels)
    attr = None
    if not args.no_attr and rank == 0:
        attr = {"what": "NEXT-1 mg_propagate_attr: C channels per node in ONE pass over the graph arrays (PAPER.md L269, L271, L277)",
                "steps": min(K, 100)}
        for C_, label in ((1, "opacity_only_c1_ms"), (16, "four_tfs_batched_c16_ms")):
            leaf = torch.rand((int(info.n_leaves), C_), dtype=torch.float32, device="cuda")
            xa = torch.empty((n_nodes, C_), dtype=torch.float32, device="cuda")
            for _ in range(3):
                g.propagate_attr(leaf, xa, C_, st)
            torch.cuda.synchronize()
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record(stream)
            for _ in range(attr["steps"]):
                g.propagate_attr(leaf, xa, C_, st)
            a1.record(stream)
            torch.cuda.synchronize()
            attr[label] = a0.elapsed_time(a1) / attr["steps"]
            del leaf, xa

    # ---- NEXT-2: ray-march the paletted mipmap (1600 x 1200, 0.5-voxel steps: L414), with and without ESS (L271)
    render = None
    if not args.no_render and rank == 0 and len(w.mip_dims) > 1:
        from paper_2009_02702_b200 import synth
        view = synth.render_view(w.cfg)
        rtf = synth.render_tf(w.tf(0) if args.render_alpha_zero_frac is None else
                              synth.random_tf(w.n_leaves, w.cfg.get("seed", 0), alpha_zero_frac=args.render_alpha_zero_frac))
        if args.render_empty_background:
            rtf[0, 3] = 0.0
        g.propagate(torch.from_numpy(rtf).cuda(), nodes, st)
        img = torch.empty((view["height"], view["width"], 4), dtype=torch.float32, device="cuda")
        desc = w.mip_desc()
        render = {"what": "NEXT-2 mg_render: pinhole ray-marcher over the node-index mipmap + fp32 palette, per-sample LOD, "
                          "manual trilinear + inter-level blend, opacity correction, hierarchical empty-space skipping "
                          "(PAPER.md L267-L271, L414)", "width": view["width"], "height": view["height"],
                  "step_voxels": view["step_voxels"], "tf": f"config TF, opacities x {synth.RENDER_ALPHA_SCALE}" + (", first leaf transparent" if args.render_empty_background else ""),
                  "frames": 10}
        # the empty-space mask of mg_ess_mask_build (rebuilt per TF update: timed on its own) turns R6's climb into one load
        mask = None
        if 3 <= len(w.mip_dims) <= 18:
            mask = torch.empty(w.level_voxels[2], dtype=torch.int16, device="cuda")
            for _ in range(2):
                g.ess_mask_build(w.d_idx, desc, nodes, view["ess_threshold"], mask, st)
            m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            m0.record(stream)
            for _ in range(10):
                g.ess_mask_build(w.d_idx, desc, nodes, view["ess_threshold"], mask, st)
            m1.record(stream)
            torch.cuda.synchronize()
            render["ess_mask_build_ms"] = m0.elapsed_time(m1) / 10
            render["ess_mask_mbytes"] = 2e-6 * w.level_voxels[2]
        for label, thr, fl, use_mask in (("ess", view["ess_threshold"], view["flags"], True), ("no_ess", -1.0, view["flags"], False),
                                         ("ess_climb", view["ess_threshold"], view["flags"], False),
                                         ("ess_generic_mipmap", view["ess_threshold"], 0, True), ("no_ess_generic_mipmap", -1.0, 0, False)):
            v = mg.view_struct(dict(view, ess_threshold=thr, flags=fl))
            mk = mask if use_mask else None
            stats = torch.zeros(4, dtype=torch.int64, device="cuda")
            for _ in range(2):
                g.render(w.d_idx, desc, nodes, v, img, None, st, ess_mask_device=mk)
            torch.cuda.synchronize()
            r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            r0.record(stream)
            for _ in range(render["frames"]):
                g.render(w.d_idx, desc, nodes, v, img, None, st, ess_mask_device=mk)
            r1.record(stream)
            g.render(w.d_idx, desc, nodes, v, img, stats, st, ess_mask_device=mk)
            torch.cuda.synchronize()
            ms = r0.elapsed_time(r1) / render["frames"]
            ev_, sk_, un_, _ = (int(x) for x in stats.cpu().numpy())
            render[label] = {"ms_per_frame": ms, "fps": 1e3 / ms, "samples_composited": ev_, "samples_skipped": sk_,
                             "samples_one_leaf_shortcut": un_, "samples_per_s": (ev_ + sk_) / (ms * 1e-3),
                             "ess_mask": bool(use_mask and mask is not None)}
        render["ess_speedup"] = render["no_ess"]["ms_per_frame"] / render["ess"]["ms_per_frame"]
        # ESS only pays where most samples can be skipped: report the fraction it skipped in this view next to the ratio, and
        # which of the two kernels a caller should run here (the faster one; both produce the same image)
        e_ = render["ess"]
        render["ess_skippable_fraction"] = e_["samples_skipped"] / max(1, e_["samples_skipped"] + e_["samples_composited"])
        render["ess_pays_in_this_view"] = bool(render["ess_speedup"] > 1.0)
        render["best_ms_per_frame"] = min(render["ess"]["ms_per_frame"], render["no_ess"]["ms_per_frame"])
        del mask
        render["histogram_mipmap_flag_speedup"] = render["no_ess_generic_mipmap"]["ms_per_frame"] / render["no_ess"]["ms_per_frame"]
        render["coverage"] = float((img[..., 3] > 0).float().mean().item())
        del img

    # ---- NEXT-4: mixture lookup table + range queries (Table 4: random cubes of 16^3 .. 256^3 voxels, FA vs naive)
    query = None
    if not args.no_query and rank == 0 and len(w.mip_dims) > 1 and w.host_graph is not None and "weight_sigma" in w.host_graph:
        from paper_2009_02702_b200 import synth
        g.mixture_lut(w.host_graph["weight_sigma"]).close()          # warm-up build (module load, allocator state)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        lut = g.mixture_lut(w.host_graph["weight_sigma"])
        torch.cuda.synchronize()
        t_build = time.perf_counter() - t0
        nl = int(info.n_leaves)
        nq = 64
        query = {"what": "NEXT-4: device mixture LUT (mu, dmu per node, Eq. 18) and batched range queries, footprint assembly "
                         "vs naive (PAPER.md sections 3.5-3.6, Table 4)", "lut_build_ms": 1e3 * t_build,
                 "lut_entries": int(lut.info.nnz), "lut_mbytes": lut.info.device_bytes / 1e6, "queries_per_batch": nq,
                 "paper_context": "Table 4 (10-core CPU, ms per query FA / naive): 16^3 0.11-0.15 / 0.40-0.44; 64^3 1.3-2.1 / 12.9-29.5; "
                                  "256^3 25-394 / 1200-70500", "sizes": {}}
        desc = w.mip_desc()
        e_buf = torch.empty((nq, nl), dtype=torch.float64, device="cuda")
        d_buf = torch.empty((nq, nl), dtype=torch.float64, device="cuda")
        f_buf = torch.empty((nq,), dtype=torch.int64, device="cuda")
        c = w.cfg
        for side in (16, 32, 64, 128, 256):
            boxes = np.array(synth.query_boxes(c["dims"], side, nq, seed=c.get("seed", 0)), dtype=np.uint64)
            row = {}
            for label, mode, reps in (("fa", mg.MG_QUERY_FA, 10), ("naive", mg.MG_QUERY_NAIVE, 3)):
                lut.range_query(w.d_idx, desc, boxes, e_buf, d_buf, f_buf, mode=mode, stream=st)
                torch.cuda.synchronize()
                q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                q0.record(stream)
                for _ in range(reps):
                    lut.range_query(w.d_idx, desc, boxes, e_buf, d_buf, f_buf, mode=mode, stream=st)
                q1.record(stream)
                torch.cuda.synchronize()
                row[label + "_ms_per_query"] = q0.elapsed_time(q1) / reps / nq
                row[label + "_fetches"] = float(f_buf.double().mean().item())
            row["fetches_saved"] = 1.0 - row["fa_fetches"] / row["naive_fetches"]
            row["speedup"] = row["naive_ms_per_query"] / row["fa_ms_per_query"]
            query["sizes"][str(side)] = row
        lut.close()
        del e_buf, d_buf, f_buf

    # ---- e2e: host TF in, host mipmap out, through the public C-ABI call (rank-local, then max)
    e2e = None
    if not args.no_e2e:
        ke = args.e2e_steps or min(K, 8)
        tf_pinned = [torch.from_numpy(w.tf(u)).pin_memory() for u in range(min(n_tf, ke))]
        out_host = torch.empty(max(n_part, 1) * out_bytes, dtype=torch.uint8).pin_memory()
        for k in range(2):
            g.tf_update_host(tf_pinned[k % len(tf_pinned)], nodes, idx_part, n_part, out_part, out_host, fmt=fmt, stream=st)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for k in range(ke):
            g.tf_update_host(tf_pinned[k % len(tf_pinned)], nodes, idx_part, n_part, out_part, out_host, fmt=fmt, stream=st)
        e1.record(stream)
        barrier()
        e2e_ms = e0.elapsed_time(e1)
        e2e_ms = max_over_ranks(e2e_ms, world, red_dev)
        if args.dump_dir:
            os.makedirs(args.dump_dir, exist_ok=True)
            np.savez(os.path.join(args.dump_dir, f"rank{rank}.npz"), v_lo=v_lo, v_hi=v_hi, out=out_host.numpy().copy(),
                     nodes=nodes.cpu().numpy(), tf_update=(ke - 1) % len(tf_pinned), n_voxels_padded=w.n_voxels_padded)
        e2e = {"value": e2e_ms / ke, "unit": UNIT,
               "h2d_bytes_per_step": int(w.n_leaves * 16), "d2h_bytes_per_step": int(n_part * out_bytes), "steps": ke,
               "d2h_gbs": n_part * out_bytes / (e2e_ms / ke * 1e-3) / 1e9,
               "what": "mg_tf_update_host: pinned-host TF -> H2D -> propagate -> colourise all levels -> D2H of the whole "
                       "mipmap into pinned host memory (PCIe-bound: d2h_gbs = the output bytes over the whole step time)"}
        del out_host

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return {}

    peak, peak_src = peak_hbm_gbs()
    bpv = BYTES_PER_VOXEL[args.format]
    beyond_l2 = 16.0 * n_nodes > L2_BYTES                 # the fp32 palette (16 B per node) does not fit L2: config 5 only
    bpv_survey = bpv + BYTES_GATHER_SURVEY
    if beyond_l2:
        bpv += BYTES_GATHER_BEYOND_L2[args.format]
    col_avg = float(col_ms.mean())
    prop_avg = float(prop_ms.mean())
    algo_bytes = float(bpv) * w.n_voxels * (n_part / max(1, w.n_voxels_padded))      # rank 0's share (all of it unless --partition slab)
    achieved = algo_bytes / (col_avg * 1e-3) / 1e9
    kernel = "k_colorize"
    col_launches = (launches / K) - int(info.n_launches_propagate)                    # > 1: one sweep per palette tile
    roofline = {"bound": "hbm", "kernel": kernel, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": ncu_traffic(w.name, kernel), "algorithmic_bytes_per_launch": algo_bytes,
                "algorithmic_bytes_per_voxel": bpv, "avg_launch_ms": col_avg, "peak_source": peak_src,
                "timing": "CUDA events on the launch stream around every mg_colorize of the timed region"}
    if col_launches > 1:
        roofline["kernel"] = kernel = "k_colorize_tile"
        roofline["traffic"] = ncu_traffic(w.name, kernel)
        roofline["launches_per_step"] = col_launches
    if beyond_l2:
        roofline["algorithmic_bytes_per_voxel_survey"] = bpv_survey
        roofline["achieved_at_survey_bytes"] = achieved * bpv_survey / bpv
        roofline["note"] = ("palette beyond the L2: one sweep per palette tile (<= 88 MB); achieved = the algorithmic bytes of the whole "
                            "colourise / the time of all its sweeps; traffic = DRAM bytes of all sweeps")
    prop_roofline = None
    if beyond_l2:
        # config 5: propagation is truly bandwidth-bound too -- report both; `roofline` is the one that takes longer
        pa = float(BYTES_PER_NODE_DRAM) * n_internal
        prop_roofline = {"bound": "hbm", "kernel": "k_level", "achieved": pa / (prop_avg * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                         "frac": pa / (prop_avg * 1e-3) / 1e9 / peak, "traffic": ncu_traffic(w.name, "k_level"),
                         "algorithmic_bytes_per_launch": pa, "algorithmic_bytes_per_node": BYTES_PER_NODE_DRAM,
                         "avg_launch_ms": prop_avg, "launches_per_step": int(info.n_launches_propagate),
                         "note": "all levels of one mg_propagate together (one launch per level)"}
        if prop_avg > col_avg:
            roofline, prop_roofline = prop_roofline, roofline
    res = {
        # latency of ONE update: replicas do not shorten it (each rank runs a whole update; max over ranks), a slab
        # partition does (strong scaling).  The whole-job throughput of a replica run is `updates_per_s`.
        "metric": METRIC, "value": ms_per_step, "unit": UNIT, "n_gpus": world,
        "updates_per_s": aggregate_updates_per_s(ms_per_step, 1 if slab else world),
        "steps": K, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "strong" if slab else "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": workload_config(w, args, world),
        "propagate_ms": prop_avg, "colorize_ms": col_avg, "propagate_ms_min": float(prop_ms.min()), "colorize_ms_min": float(col_ms.min()),
        "propagate_ms_median": float(np.median(prop_ms)), "colorize_ms_median": float(np.median(col_ms)),
        "update_ms_median": float(np.median(prop_ms + col_ms)), "update_ms_min": float((prop_ms + col_ms).min()),
        "nodes_per_s": n_internal / (prop_avg * 1e-3), "voxels_per_s": w.n_voxels * (n_part / max(1, w.n_voxels_padded)) / (col_avg * 1e-3),
        "hbm_gbs_step": (algo_bytes + BYTES_PER_NODE_L2 * n_internal) / (ms_per_step * 1e-3) / 1e9,
        "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
        "roofline": roofline,
        "gpu_launches": int(launches), "clocks": clocks.summary(),
        "paper_context": "RTX Titan palette update (propagation only, incl. TF upload): 3.5 / 11.3 / 12.1 ms for 1.03 / 5.20 / 1.93 M "
                         "nodes (PAPER.md L373); the paper never materialises the RGBA mipmap (L221)",
        "setup_s": dict({k: round(v, 3) for k, v in w.stats.items() if k.endswith("_s")},
                        **({"device_levels_done": w.stats["device_levels_done"]} if "device_levels_done" in w.stats else {})),
    }
    if derive is not None:
        res["colorize_deriving_palette_ms"] = derive      # mg_colorize's default (no MG_PALETTE_FROM_LAST_PROPAGATE): + k_convert_palette
    if upload is not None:
        res["propagate_host_ms"] = upload["propagate_host_ms"]             # section 8(d): what the paper timed (L371-L373)
        res["update_incl_tf_upload_ms"] = upload["update_incl_tf_upload_ms"]
        res["tf_upload"] = upload
    if prop_roofline is not None:
        res["roofline_second_kernel"] = prop_roofline
    if packed is not None:
        packed["frac"] = packed["achieved_gbs"] / peak
        res["packed"] = packed
    if attr is not None:
        res["attr"] = attr
    if render is not None:
        res["render"] = render
    if query is not None:
        res["query"] = query
    if e2e is not None:
        res["e2e"] = e2e
    if world == 1 and not args.no_cpu_baseline and w.host_idx is not None:
        res["cpu_baseline"] = cpu_baseline(w, args.cpu_sample_voxels)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return res


# ------------------------------------------------------------------------------------------------
# --impl reference: there is no reference implementation (the paper ships no code), so this arm
# times the CPU fp64 oracle, as it stands, on the host cores; each step a bounded sample
# ------------------------------------------------------------------------------------------------

def run_reference(args) -> dict:
    rank, local_rank, world = dist_env()
    if rank != 0:
        return {}
    import torch
    if torch.cuda.is_available():
        torch.cuda.set_device(local_rank)
    from paper_2009_02702_b200 import workload
    # the oracle's inputs (graph + node-index mipmap) come from the same seeded assembly as the GPU arm
    w = workload.make(args.config, args.scale, device_synth=torch.cuda.is_available(), load=False)
    tf64 = [w.tf(u).astype(np.float64) for u in range(4)]
    # calibrate the per-step sample so that steps + warmup fit the budget
    probe = _sample_plan(w, 1 << 22)
    tp, tc, used = oracle_step(w, tf64[0], probe)
    per_voxel = tc / sum(probe)
    n_total = args.steps + args.warmup
    budget_per_step = max(0.05, args.reference_budget_s / max(1, n_total) - tp)
    n_sample = int(min(w.n_voxels, max(1 << 16, budget_per_step / per_voxel)))
    plan = _sample_plan(w, n_sample)
    n_s = sum(plan)
    for k in range(args.warmup):
        oracle_step(w, tf64[k % 4], plan)
    t0 = time.perf_counter()
    tps, tcs = [], []
    for k in range(args.steps):
        a, b, used = oracle_step(w, tf64[(args.warmup + k) % 4], plan)
        tps.append(a)
        tcs.append(b)
    wall = time.perf_counter() - t0
    tp, tc = float(np.mean(tps)), float(np.mean(tcs))
    ms = 1e3 * (tp + tc * (w.n_voxels / n_s))
    sample = (f"per step: full fp64 propagation of {w.stats['n_nodes']} nodes + lookup/RGBA8 of the leading {n_s} of "
              f"{w.n_voxels} voxels (same share of every mip level); colourise time scaled to the whole mipmap")
    cfg = workload_config(w, args, 1)
    cfg["output"] = "rgba8"
    return {"impl": "reference", "metric": METRIC, "value": ms, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(1, args.steps), "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
            "cpu_baseline": {"value": ms, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample, "cpu_model": cpu_model(),
                             "host_cores": os.cpu_count()},
            "e2e": {"value": ms, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "propagate_ms": 1e3 * tp, "colorize_sample_ms": 1e3 * tc,
            "note": "no reference implementation exists for this paper; this arm is the repo's CPU fp64 oracle (test "
                    "infrastructure), a deliberately plain program: the ratio against it is not the headline"}


def main():
    args = parse_args()
    res = run_reference(args) if args.impl == "reference" else run_b200(args)
    if res:
        print(json.dumps(res), flush=True)


if __name__ == "__main__":
    main()
