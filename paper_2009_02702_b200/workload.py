"""Assemble one of the BASELINE.json configs end to end on the current CUDA device.

Plumbing only (none of the method's arithmetic): volume generator (synth / synth_gpu) -> host
builder (libmg_builder.so: a0-a2) -> mg_load_graph (a3) -> the per-voxel node indices of every
mip level uploaded into ONE device buffer.  Used by bench.py, by the full-size parity tests and
by __graft_entry__; nothing here imports ``oracle/``.

Device layout of the mipmap (indices and outputs alike): the mip levels are concatenated finest
first; level l starts at voxel ``level_start[l]``, a multiple of 64 voxels (256 B for the uint32
indices and the RGBA8 output, 512 B for fp16), so that every level is a self-contained, vector-
aligned sub-buffer a renderer can bind on its own, and ONE mg_colorize call over
``n_voxels_padded`` voxels covers all levels.  Padding voxels hold node index 0.
"""
from __future__ import annotations

import time

import numpy as np

from . import builder, synth


class _LazyMg:
    """``mg`` (the ctypes binding of libmg.so) is loaded on first use: a workload assembled with ``load=False`` for the
    reference arm of bench.py (generator + host builder + oracle) then never maps the CUDA library."""

    def __getattr__(self, name):
        from . import mg as _mg
        return getattr(_mg, name)


mg = _LazyMg()

LEVEL_ALIGN = 64          # voxels


class Workload:
    """A loaded graph plus its device-resident node-index mipmap."""

    def __init__(self, name: str):
        self.name = name
        self.graph: mg.Graph | None = None
        self.host_graph: dict | None = None       # child_a, child_b, weight, level_offsets, n_leaves (builder numbering = library numbering)
        self.mip_dims: list = []                  # [(X_l, Y_l, Z_l)]
        self.level_start: list = []               # first voxel of level l in the concatenated buffers
        self.level_voxels: list = []              # voxels of level l
        self.n_voxels = 0                         # real voxels (sum of level_voxels)
        self.n_voxels_padded = 0                  # extent of the concatenated buffers
        self.d_idx = None                         # torch int32 [n_voxels_padded] (uint32 values)
        self.host_idx = None                      # list of numpy uint32 views per level (builder-owned) or arrays
        self.build_result = None                  # keeps the builder-owned arrays alive
        self.stats: dict = {}
        self.n_leaves = 0
        self.cfg: dict = {}
        self.seg = None                           # uint32 [Z, Y, X] segmentation (only with keep_seg)
        self.d_packed = None                      # torch uint8: bit-packed streams of all levels (after pack())
        self.packed_levels = None                 # list of dicts (n_voxels, out_offset, byte_offset, bits, i_min)
        self.packed_bytes = 0
        self.perm = None                          # uint32 [n_nodes]: library index of the caller's node (only after MG_RELABEL)

    @property
    def n_updates(self) -> int:
        """Length of the config's TF-update sequence (BASELINE.json: 100 consecutive updates)."""
        return int(self.cfg.get("n_updates", 100))

    def tf(self, update: int = 0) -> np.ndarray:
        """fp32 [n_leaves, 4]: update number ``update`` of this config's TF sequence (synth recipe).  "random": an
        independent TF per update; "single_segment" (config 4): update u is update u - 1 with ONE random segment re-drawn."""
        c = self.cfg
        seed = c.get("seed", 0)
        if c.get("tf_sequence", "random") != "single_segment":
            return synth.random_tf(self.n_leaves, seed, update=update, alpha_zero_frac=c.get("alpha_zero_frac", 0.0))
        chain = self.__dict__.setdefault("_tf_chain", [synth.random_tf(self.n_leaves, seed, update=0,
                                                                       alpha_zero_frac=c.get("alpha_zero_frac", 0.0))])
        while len(chain) <= update:
            chain.append(synth.single_segment_update(chain[-1], seed, len(chain)))
        return chain[update].copy()

    def host_level(self, l: int) -> np.ndarray:
        """Node indices of mip level ``l`` on the host, flat uint32 (downloaded when the host never had them)."""
        if self.host_idx is not None and self.host_idx[l] is not None:
            return self.host_idx[l].reshape(-1)
        s = self.level_start[l]
        return self.d_idx[s:s + self.level_voxels[l]].cpu().numpy().view(np.uint32)

    def mip_desc(self) -> "mg.MgMipmapDesc":
        """The mg_mipmap_desc of the concatenated device mipmap (input of mg_render)."""
        return mg.mipmap_desc(self.level_start, self.mip_dims)

    def pack(self) -> None:
        """NEXT-3: derive the bit-packed form of the device mipmap (Table 1 (8), (9), (A)): per level
        i_min(l), r(l) (Eq. 15-16) and one packed stream; fills d_packed / packed_levels."""
        import torch
        st = torch.cuda.current_stream().cuda_stream
        levels, pos = [], 0
        for s0, nv in zip(self.level_start, self.level_voxels):
            lo, hi = mg.index_range(self.d_idx[s0:s0 + nv], nv, st)
            bits = mg.bits_per_voxel(lo, hi)
            levels.append(dict(n_voxels=nv, out_offset=s0, byte_offset=pos, bits=bits, i_min=lo))
            pos += mg.packed_stream_bytes(nv, bits)
        self.d_packed = torch.empty(pos, dtype=torch.uint8, device="cuda")
        for l, (s0, nv) in zip(levels, zip(self.level_start, self.level_voxels)):
            mg.pack_indices(self.d_idx[s0:s0 + nv], nv, l["i_min"], l["bits"], self.d_packed[l["byte_offset"]:], st)
        torch.cuda.synchronize()
        self.packed_levels = levels
        self.packed_bytes = pos

    def close(self) -> None:
        self.d_packed = None
        if self.graph is not None:
            self.graph.close()
            self.graph = None
        self.d_idx = None
        self.host_idx = None
        if self.build_result is not None:
            self.build_result.close()
            self.build_result = None


def _layout(level_voxels):
    start, pos = [], 0
    for n in level_voxels:
        start.append(pos)
        pos += -(-n // LEVEL_ALIGN) * LEVEL_ALIGN
    return start, pos


def _upload_levels(w: Workload, levels) -> None:
    import torch
    w.level_voxels = [int(a.size) for a in levels]
    w.level_start, w.n_voxels_padded = _layout(w.level_voxels)
    w.n_voxels = sum(w.level_voxels)
    d = torch.zeros(max(w.n_voxels_padded, 1), dtype=torch.int32, device="cuda")
    chunk = 1 << 27                                # 512 MB pieces through pageable memory
    for s, a in zip(w.level_start, levels):
        flat = a.reshape(-1).view(np.int32)
        for o in range(0, flat.size, chunk):
            e = min(flat.size, o + chunk)
            d[s + o:s + e].copy_(torch.from_numpy(flat[o:e]))
    w.d_idx = d
    w.host_idx = levels


def from_volume(seg: np.ndarray, name: str = "volume", cfg: dict | None = None, keep_host: bool = True,
                load: bool = True, **builder_params) -> Workload:
    """Builder + load + upload for a uint32 [Z, Y, X] segment-ID volume.  ``load=False`` stops after the
    builder (host arrays only: what bench.py's reference arm needs; no device is touched)."""
    w = Workload(name)
    w.cfg = dict(cfg or {})
    t0 = time.perf_counter()
    r = builder.build(seg, **builder_params)
    t1 = time.perf_counter()
    g = r.graph()
    w.host_graph = g
    w.n_leaves = g["n_leaves"]
    w.mip_dims = r.mip_dims
    if load:
        w.graph = mg.Graph(g["child_a"], g["child_b"], g["weight"], g["n_leaves"], level_offsets=g["level_offsets"],
                           leaf_segment_id=g["leaf_segment_id"])
    t2 = time.perf_counter()
    levels = [r.node_idx(l, copy=False) for l in range(r.info.n_mip_levels)]
    if load:
        _upload_levels(w, levels)
    else:
        w.level_voxels = [int(a.size) for a in levels]
        w.level_start, w.n_voxels_padded = _layout(w.level_voxels)
        w.n_voxels = sum(w.level_voxels)
        w.host_idx = levels
    t3 = time.perf_counter()
    i = r.info
    w.stats = dict(builder_s=t1 - t0, load_graph_s=t2 - t1, upload_idx_s=t3 - t2, n_nodes=int(i.n_nodes),
                   n_leaves=int(i.n_leaves), depth=int(i.depth), quant_bits=int(i.quant_bits),
                   n_distinct_mixtures=int(i.n_distinct_mixtures), nnz_per_voxel=i.nnz_total / max(1, i.n_voxels_total),
                   n_mip_levels=int(i.n_mip_levels), builder_mipmap_s=i.seconds_mipmap,
                   builder_factorise_s=i.seconds_factorise, builder_finalise_s=i.seconds_finalise,
                   phi2_exact=int(i.phi2_exact), n_stage1=int(i.n_stage1), n_stage2=int(i.n_stage2), n_big=int(i.n_big),
                   level_sizes=np.diff(g["level_offsets"].astype(np.int64)).tolist())
    if keep_host:
        w.build_result = r
    else:
        w.host_idx = None
        r.close()
    return w


def from_volume_device_levels(seg_dev, name: str = "volume", cfg: dict | None = None, store_capacity=(0, 0),
                              **builder_params) -> Workload:
    """``from_volume_device`` with the levels >= 1 of the histogram mipmap built on the device too
    (mg_mipmap_levels_build: merge + hash-cons per level, as far up as the mixtures stay small), the host builder
    continuing above the last finished level (mgb_build_from_levels) and the device-built levels turned into node
    indices in place (mg_mipmap_remap_handles).  Same graph and node indices as ``from_volume``; ``host_idx[l]`` is None
    for the levels below the last device-built one.  ``store_capacity`` = (mixtures, entries) of the device store
    (mg_mipmap_levels_build_ex; 0 = the library's sizing): a level that does not fit is continued on the host."""
    import torch
    w = Workload(name)
    w.cfg = dict(cfg or {})
    Z, Y, X = (int(d) for d in seg_dev.shape)
    dims = builder.mip_chain((X, Y, Z))                 # the library's statement of L80, not a Python restatement
    w.mip_dims = dims
    w.level_voxels = [a * b * c for a, b, c in dims]
    w.level_start, w.n_voxels_padded = _layout(w.level_voxels)
    w.n_voxels = sum(w.level_voxels)
    st = torch.cuda.current_stream().cuda_stream
    t0 = time.perf_counter()
    w.d_idx = torch.zeros(w.n_voxels_padded, dtype=torch.int32, device="cuda")
    n0 = w.level_voxels[0]
    ids = mg.mipmap_leaf_index(seg_dev, n0, w.d_idx[:n0], stream=st)
    table = mg.MixtureTable(w.d_idx, dims[0], ids.size, w.d_idx, w.level_start, stream=st, cap_mixtures=store_capacity[0],
                            cap_entries=store_capacity[1]) if len(dims) > 1 else None
    Ld = int(table.info.levels_done) if table is not None else 0
    if Ld == 0:                                    # nothing for the device to do (1 x 1 x 1, or huge mixtures at level 1)
        if table is not None:
            table.close()
        w.d_idx = None
        return from_volume_device(seg_dev, name=name, cfg=cfg, **builder_params)
    mix = table.export()
    s_d, n_d = w.level_start[Ld], w.level_voxels[Ld]
    handles = w.d_idx[s_d:s_d + n_d].cpu().numpy().view(np.uint32)
    nnz_levels, n_dev_mix = int(table.info.nnz_levels), int(table.info.n_mixtures)
    table.close()
    t1 = time.perf_counter()
    r, nodes = builder.build_from_levels(dims[0], ids, Ld, handles, mix, nnz_levels, **builder_params)
    t2 = time.perf_counter()
    g = r.graph()
    w.host_graph = g
    w.n_leaves = g["n_leaves"]
    assert r.mip_dims == dims
    w.graph = mg.Graph(g["child_a"], g["child_b"], g["weight"], g["n_leaves"], level_offsets=g["level_offsets"],
                       leaf_segment_id=g["leaf_segment_id"])
    t3 = time.perf_counter()
    d_nodes = torch.from_numpy(nodes.view(np.int32)).cuda() if nodes.size else torch.zeros(1, dtype=torch.int32, device="cuda")
    s1 = w.level_start[1]
    mg.mipmap_remap_handles(w.d_idx[s1:], s_d + n_d - s1, d_nodes, nodes.size, st)       # levels 1 .. Ld are contiguous but for padding zeros
    w.host_idx = [None] * Ld + [r.node_idx(l, copy=False) for l in range(Ld, r.info.n_mip_levels)]
    for l in range(Ld + 1, len(dims)):
        a = w.host_idx[l]
        w.d_idx[w.level_start[l]:w.level_start[l] + a.size].copy_(torch.from_numpy(a.reshape(-1).view(np.int32)))
    torch.cuda.synchronize()
    t4 = time.perf_counter()
    i = r.info
    w.stats = dict(front_end_s=t1 - t0, builder_s=t2 - t1, load_graph_s=t3 - t2, upload_idx_s=t4 - t3, n_nodes=int(i.n_nodes),
                   n_leaves=int(i.n_leaves), depth=int(i.depth), quant_bits=int(i.quant_bits),
                   n_distinct_mixtures=int(i.n_distinct_mixtures), nnz_per_voxel=i.nnz_total / max(1, i.n_voxels_total),
                   n_mip_levels=int(i.n_mip_levels), builder_mipmap_s=i.seconds_mipmap,
                   builder_factorise_s=i.seconds_factorise, builder_finalise_s=i.seconds_finalise,
                   device_mipmap=True, device_levels_done=Ld, n_device_mixtures=n_dev_mix,
                   level_sizes=np.diff(g["level_offsets"].astype(np.int64)).tolist())
    w.build_result = r
    return w


def from_volume_device(seg_dev, name: str = "volume", cfg: dict | None = None, **builder_params) -> Workload:
    """The same assembly as ``from_volume`` for a segment-ID volume that is ALREADY ON THE DEVICE (torch int32
    [Z, Y, X], uint32 values): the two finest mip levels are classified by the device front end
    (mg_mipmap_leaf_index / mg_mipmap_front_level1, writing level 0's node indices straight into the mipmap
    buffer), the host builder continues from the list of non-pure level-1 parents (mgb_build_from_level1), and
    only the levels >= 1 are uploaded.  Same graph and same node indices as ``from_volume`` on the same volume;
    ``host_idx[0]`` is None (level 0 never exists on the host; ``host_level(0)`` downloads it)."""
    import torch
    w = Workload(name)
    w.cfg = dict(cfg or {})
    Z, Y, X = (int(d) for d in seg_dev.shape)
    dims = builder.mip_chain((X, Y, Z))                 # the library's statement of L80, not a Python restatement
    w.mip_dims = dims
    w.level_voxels = [a * b * c for a, b, c in dims]
    w.level_start, w.n_voxels_padded = _layout(w.level_voxels)
    w.n_voxels = sum(w.level_voxels)
    st = torch.cuda.current_stream().cuda_stream
    t0 = time.perf_counter()
    w.d_idx = torch.zeros(w.n_voxels_padded, dtype=torch.int32, device="cuda")
    n0 = w.level_voxels[0]
    ids = mg.mipmap_leaf_index(seg_dev, n0, w.d_idx[:n0], stream=st)
    level1 = mixed_voxel = mixed_children = np.zeros(0, np.uint32)
    if len(dims) > 1:
        n1, s1 = w.level_voxels[1], w.level_start[1]
        cap = max(1024, n1 // 16)
        while True:
            mv = torch.empty(cap, dtype=torch.int32, device="cuda")
            mc = torch.empty((cap, 8), dtype=torch.int32, device="cuda")
            n_mixed = mg.mipmap_front_level1(w.d_idx[:n0], dims[0], w.d_idx[s1:s1 + n1], mv, mc, cap, stream=st)
            if n_mixed <= cap:
                break
            cap = n_mixed
        level1 = w.d_idx[s1:s1 + n1].cpu().numpy().view(np.uint32)
        mixed_voxel = mv[:n_mixed].cpu().numpy().view(np.uint32)
        mixed_children = mc[:n_mixed].cpu().numpy().view(np.uint32)
        del mv, mc
    t1 = time.perf_counter()
    r = builder.build_from_level1(dims[0], ids, level1, mixed_voxel, mixed_children, **builder_params)
    t2 = time.perf_counter()
    g = r.graph()
    w.host_graph = g
    w.n_leaves = g["n_leaves"]
    assert r.mip_dims == dims
    w.graph = mg.Graph(g["child_a"], g["child_b"], g["weight"], g["n_leaves"], level_offsets=g["level_offsets"],
                       leaf_segment_id=g["leaf_segment_id"])
    t3 = time.perf_counter()
    w.host_idx = [None] + [r.node_idx(l, copy=False) for l in range(1, r.info.n_mip_levels)]
    for s, a in zip(w.level_start[1:], w.host_idx[1:]):
        w.d_idx[s:s + a.size].copy_(torch.from_numpy(a.reshape(-1).view(np.int32)))
    torch.cuda.synchronize()
    t4 = time.perf_counter()
    i = r.info
    w.stats = dict(front_end_s=t1 - t0, builder_s=t2 - t1, load_graph_s=t3 - t2, upload_idx_s=t4 - t3, n_nodes=int(i.n_nodes),
                   n_leaves=int(i.n_leaves), depth=int(i.depth), quant_bits=int(i.quant_bits),
                   n_distinct_mixtures=int(i.n_distinct_mixtures), nnz_per_voxel=i.nnz_total / max(1, i.n_voxels_total),
                   n_mip_levels=int(i.n_mip_levels), builder_mipmap_s=i.seconds_mipmap,
                   builder_factorise_s=i.seconds_factorise, builder_finalise_s=i.seconds_finalise,
                   n_level1_mixed=int(mixed_voxel.size), device_mipmap=True,
                   level_sizes=np.diff(g["level_offsets"].astype(np.int64)).tolist())
    w.build_result = r
    return w


def from_dag(child_a, child_b, weight, level_offsets, n_leaves: int, node_idx: np.ndarray, name: str = "dag",
             cfg: dict | None = None, relabel: bool = False, load: bool = True) -> Workload:
    """A ready-made level-contiguous DAG plus ONE node-index volume (config 5).  ``relabel`` loads it with
    MG_RELABEL (the library sorts every level by its children for gather locality) and renumbers the
    device index volume accordingly; ``Workload.perm`` then maps the caller's node numbers to the library's."""
    w = Workload(name)
    w.cfg = dict(cfg or {})
    w.n_leaves = int(n_leaves)
    t0 = time.perf_counter()
    if load:
        w.graph = mg.Graph(child_a, child_b, weight, n_leaves, level_offsets=level_offsets,
                           flags=mg.MG_RELABEL if relabel else 0)
    t1 = time.perf_counter()
    w.host_graph = dict(child_a=child_a, child_b=child_b, weight=weight, level_offsets=np.asarray(level_offsets),
                        n_leaves=int(n_leaves))
    w.mip_dims = [(int(node_idx.size), 1, 1)]
    if load:
        _upload_levels(w, [node_idx.reshape(-1)])
    else:
        w.level_voxels, w.level_start = [int(node_idx.size)], [0]
        w.n_voxels = w.n_voxels_padded = int(node_idx.size)
        w.host_idx = [node_idx.reshape(-1)]
    if relabel and load:
        import torch
        w.perm = w.graph.node_permutation()
        w.graph.relabel_indices(w.d_idx, w.n_voxels_padded, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    t2 = time.perf_counter()
    off = np.asarray(level_offsets, dtype=np.int64)
    w.stats = dict(load_graph_s=t1 - t0, upload_idx_s=t2 - t1, n_nodes=int(child_a.size), n_leaves=int(n_leaves),
                   depth=int(off.size - 2), level_sizes=np.diff(off).tolist())
    return w


def make(cfg_id: int, scale: float = 1.0, device_synth: bool = True, keep_seg: bool = False,
         relabel: bool = False, load: bool = True, device_mipmap: bool | str = False, **builder_params) -> Workload:
    """BASELINE.json config ``cfg_id`` (1-5); ``scale`` < 1 gives a geometrically similar smaller
    instance (tests).  Volumes are generated on the GPU (bit-identical to synth.py) unless
    ``device_synth`` is False.  ``keep_seg`` keeps the generated volume in ``Workload.seg``."""
    if cfg_id == 5:
        c = dict(synth.CONFIGS[5])
        n_nodes = max(1 << 10, int(round(c["n_nodes"] * scale)))
        n_leaves = max(16, int(round(c["n_leaves"] * scale)))
        n_vox = max(1 << 10, int(round(c["volume_voxels"] * scale)))
        t0 = time.perf_counter()
        a, b, wt, off = synth.random_dag(n_nodes, c["n_levels"], n_leaves, c["seed"])
        idx = synth.random_node_idx(n_vox, n_nodes, c["seed"])
        t1 = time.perf_counter()
        w = from_dag(a, b, wt, off, n_leaves, idx, name=c["name"] + (f"_x{scale:g}" if scale != 1.0 else ""), cfg=c,
                     relabel=relabel, load=load)
        w.stats["synth_s"] = t1 - t0
        return w
    c = synth.scaled_config(cfg_id, scale)
    if "quant_bits" in c:
        builder_params.setdefault("quant_bits", c["quant_bits"])
    t0 = time.perf_counter()
    if device_mipmap:
        import torch
        from . import synth_gpu
        seg_dev = synth_gpu.make_volume(c)
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        assemble = from_volume_device_levels if device_mipmap == "levels" else from_volume_device
        w = assemble(seg_dev, name=c["name"], cfg=c, **builder_params)
        if keep_seg:
            w.seg = seg_dev.cpu().numpy().view(np.uint32)
        del seg_dev
        torch.cuda.empty_cache()
        w.stats["synth_s"] = t1 - t0
        return w
    if device_synth:
        import torch
        from . import synth_gpu
        seg = synth_gpu.make_volume(c).cpu().numpy().view(np.uint32)
        torch.cuda.empty_cache()
    else:
        seg = synth.make_volume(c)
    t1 = time.perf_counter()
    w = from_volume(seg, name=c["name"], cfg=c, load=load, **builder_params)
    if keep_seg:
        w.seg = seg                                # the generator's volume (tests: input of the oracle)
    del seg
    w.stats["synth_s"] = t1 - t0
    return w
