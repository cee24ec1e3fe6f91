"""Full-size parity: BASELINE.json's configs in the launch configuration bench.py times.

The whole workload is assembled exactly as bench.py does (workload.make with the device front end of the
histogram mipmap: GPU volume generator -> mg_mipmap_leaf_index / mg_mipmap_front_level1 -> host builder ->
mg_load_graph -> ONE concatenated node-index mipmap, ONE mg_colorize call over all levels).  The oracle cannot colourise 1.4 G voxels element by element in seconds, so:
  * node colours: EVERY node against the same-graph oracle (O-4), leaves bit-exact, max-abs <= 1e-5;
  * level 0 (87 % of the voxels): EVERY voxel -- its colour must be the RGBA8 code of TF[S(v)] (I5, L223),
    with S from the input generator (not from the builder) and the 4 x n_leaves codes from the oracle;
  * every other level: EVERY voxel against the oracle's lookup/conversion on the same graph (host-built node
    indices), and padding voxels against node 0;
  * quantised-graph colour vs the DIRECT definition C_dir = sum_s H[s] TF[s] on the generator's volume: EVERY voxel of
    EVERY level >= 1 (oracle.direct_colour_level, O-3c), max-abs <= 2e-3 (north_star), and every voxel whose index is a
    leaf must have C_dir == TF[leaf] to 1e-12 (a mixed voxel taken for pure fails);
  * the graph's symbolic mixtures mu against the histograms H (O-3 brute force): max ||mu - H||_1 (I11) and the bound
    I12 on every voxel of every level whose dense histogram table fits 2 GB (levels >= 5 or 6: where the mixtures have
    hundreds of components and the quantisation error peaks, Table 2) and on >= 1000 mixed voxels of each finer
    level.  The per-level maxima go to $MG_PARITY_REPORT_DIR/direct_parity_cfg<N>.json when that is set (DESIGN.md
    section 9 quotes them).
"""
import json
import os

import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-5
TOL_DIRECT = 2e-3


@pytest.fixture(scope="module")
def libs():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2009_02702_b200 import mg, workload
    torch.cuda.set_device(0)
    return mg, workload


def _leaf_index_chunked(S):
    """Sorted distinct IDs and per-voxel leaf number of a big volume (same result as oracle.leaf_index,
    slab by slab to bound memory)."""
    mx = int(S.max())
    cnt = np.zeros(mx + 1, dtype=np.int64)
    for z in range(S.shape[0]):
        cnt += np.bincount(S[z].reshape(-1), minlength=mx + 1)
    ids = np.flatnonzero(cnt).astype(np.uint32)
    lut = np.zeros(mx + 1, dtype=np.uint32)
    lut[ids] = np.arange(ids.size, dtype=np.uint32)
    out = np.empty(S.shape, dtype=np.uint32)
    for z in range(S.shape[0]):
        out[z] = lut[S[z]]
    return ids, out


def _rgba8_close(got, ref_c):
    """got uint8 [n,4] vs oracle colours fp64 [n,4]: equal codes, or +-1 next to a rounding boundary."""
    code = oracle.to_rgba8(ref_c).astype(np.int64)
    diff = got.astype(np.int64) - code
    if not diff.any():
        return True
    scaled = np.clip(ref_c, 0.0, 1.0) * 255.0
    near = np.abs(scaled - np.floor(scaled) - 0.5) <= 255 * TOL + 1e-4
    return bool(((diff == 0) | ((np.abs(diff) == 1) & near)).all())


def _run_update(mg, w, tf, fmt):
    g = w.graph
    nodes = torch.full((g.info.n_nodes, 4), float("nan"), dtype=torch.float32, device="cuda")
    bpv = 4 if fmt == mg.MG_RGBA8 else 8
    out = torch.full((w.n_voxels_padded * bpv,), 0xAB, dtype=torch.uint8, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    g.propagate(torch.from_numpy(tf).cuda(), nodes, st)
    g.colorize(w.d_idx, w.n_voxels_padded, nodes, out, fmt=fmt, stream=st, from_last_propagate=True)   # as bench.py does
    torch.cuda.synchronize()
    return nodes, out


def _check_nodes(w, nodes, tf):
    hg = w.host_graph
    ref = oracle.graph_eval(hg["child_a"], hg["child_b"], hg["weight"], hg["n_leaves"], tf.astype(np.float64))
    got = nodes.cpu().numpy()
    nl = hg["n_leaves"]
    assert np.array_equal(got[:nl].view(np.uint32), tf.view(np.uint32)), "leaves not bit-exact"
    err = float(np.abs(got - ref).max())
    assert err <= TOL, err
    return ref


def _sample_positions(n, k, seed, stream):
    k = min(k, n)
    pos = (synth.u64(seed, stream, np.arange(k, dtype=np.uint64)) % np.uint64(n)).astype(np.int64)
    edge = np.concatenate([np.arange(min(n, 70)), np.arange(max(0, n - 70), n)])
    return np.unique(np.concatenate([pos, edge]))


def _check_mipmap_every_voxel(w, out, tf, ref_nodes, seg_index, sample_seed):
    """The colourised RGBA8 mipmap `out` (all levels, padded layout) of one update, EVERY voxel: level 0 must be the code of
    TF[S(v)] (I5, L223; S from the generator, the codes from the oracle), every other level the oracle's lookup +
    conversion on the same graph with the node indices the host builder produced; padding voxels are node 0."""
    out4 = out.view(-1, 4)
    code_tf = torch.from_numpy(oracle.to_rgba8(tf.astype(np.float64)).view(np.uint32).reshape(-1).astype(np.int64)).cuda()
    n0 = w.level_voxels[0]
    flat = seg_index.reshape(-1)
    out32 = out.view(torch.int32)
    bad = 0
    step = 1 << 27
    for o in range(0, n0, step):
        e = min(n0, o + step)
        s = torch.from_numpy(flat[o:e].astype(np.int64)).cuda()
        exp = code_tf[s]
        got = out32[o:e].to(torch.int64) & 0xFFFFFFFF
        bad += int((got != exp).sum().item())
    assert bad == 0, f"{bad} level-0 voxels differ from code(TF[S(v)])"
    for l, (s0, nv) in enumerate(zip(w.level_start, w.level_voxels)):
        if l == 0:                                                       # additionally on samples through the oracle's lookup
            pos = _sample_positions(nv, 200000, sample_seed, l)
            got = out4[torch.from_numpy(pos + s0).cuda()].cpu().numpy()
            assert _rgba8_close(got, oracle.lookup(seg_index.reshape(-1)[pos], ref_nodes)), "level 0"
        else:
            idx_l = w.host_idx[l].reshape(-1)
            chunk = 1 << 23
            for o in range(0, nv, chunk):
                e = min(nv, o + chunk)
                got = out4[s0 + o:s0 + e].cpu().numpy()
                assert _rgba8_close(got, oracle.lookup(idx_l[o:e], ref_nodes)), f"level {l}, voxels {o}..{e}"
        pad_end = w.level_start[l + 1] if l + 1 < len(w.level_start) else w.n_voxels_padded
        if pad_end > s0 + nv:                                            # padding voxels: node 0
            padv = out4[s0 + nv:pad_end].cpu().numpy()
            assert _rgba8_close(padv, np.broadcast_to(ref_nodes[0], padv.shape).copy())


def _check_update_sequence(mg, w, seg_index, cfg_id, n_updates=100):
    """The config's OWN update sequence as BASELINE.json names it -- config 2: "100 consecutive random TF updates", config
    4: "per-update TF changes one random segment" (the paper performs full updates only, L221, "whenever the user changes
    the color transfer function", L373) -- enqueued back to back with no host synchronisation in between.  node_rgba is
    snapshotted after every update (stream-ordered copies) and EVERY node of EVERY update is compared with the same-graph
    oracle (leaves bit-exact, 1e-5); the colourised mipmap of the first, the middle and the last update is checked on
    every voxel."""
    g = w.graph
    n_nodes = int(g.info.n_nodes)
    assert w.n_updates >= n_updates
    tfs = [w.tf(u) for u in range(n_updates)]
    changed = [int((tfs[u] != tfs[u - 1]).any(axis=1).sum()) for u in range(1, n_updates)]
    if w.cfg.get("tf_sequence") == "single_segment":
        assert max(changed) == 1 and sum(changed) >= n_updates - 5          # one segment per update (a re-draw may repeat a value)
    else:
        assert min(changed) > 0.9 * w.n_leaves                              # independent TFs
    st = torch.cuda.current_stream().cuda_stream
    d_tfs = [torch.from_numpy(t).cuda() for t in tfs]
    nodes = torch.full((n_nodes, 4), float("nan"), dtype=torch.float32, device="cuda")
    snaps = torch.empty((n_updates, n_nodes, 4), dtype=torch.float32, device="cuda")
    out = torch.full((w.n_voxels_padded * 4,), 0xAB, dtype=torch.uint8, device="cuda")
    keep = {u: torch.empty_like(out) for u in (0, n_updates // 2, n_updates - 1)}
    torch.cuda.synchronize()
    for u in range(n_updates):
        g.propagate(d_tfs[u], nodes, st)
        g.colorize(w.d_idx, w.n_voxels_padded, nodes, out, fmt=mg.MG_RGBA8, stream=st, from_last_propagate=True)
        snaps[u].copy_(nodes, non_blocking=True)
        if u in keep:
            keep[u].copy_(out, non_blocking=True)
    torch.cuda.synchronize()
    hg = w.host_graph
    nl = hg["n_leaves"]
    worst = 0.0
    for u in range(n_updates):
        ref = oracle.graph_eval(hg["child_a"], hg["child_b"], hg["weight"], nl, tfs[u].astype(np.float64))
        got = snaps[u].cpu().numpy()
        assert np.array_equal(got[:nl].view(np.uint32), tfs[u].view(np.uint32)), f"update {u}: leaves not bit-exact"
        err = float(np.abs(got - ref).max())
        assert err <= TOL, (u, err)
        worst = max(worst, err)
        if u in keep:
            _check_mipmap_every_voxel(w, keep[u], tfs[u], ref, seg_index, 500 + u)
    print(f"cfg {cfg_id}: {n_updates} consecutive updates ({w.cfg.get('tf_sequence', 'random')}), every node of every update: "
          f"max |err| = {worst:.2e}; mipmaps of updates {sorted(keep)} checked on every voxel")


@pytest.mark.parametrize("cfg_id", [3, 2, 4])
def test_volume_config_full_size(libs, cfg_id):
    mg, workload = libs
    w = workload.make(cfg_id, keep_seg=True, device_mipmap=True)              # the assembly bench.py uses by default
    try:
        c = synth.CONFIGS[cfg_id]
        X, Y, Z = c["dims"]
        assert w.host_idx[0] is None                                             # level 0 never existed on the host
        assert w.mip_dims == oracle.mip_dims((X, Y, Z))                     # O-1 at full size (Table 2 totals)
        assert w.n_voxels == sum(x * y * z for x, y, z in w.mip_dims)
        tf = w.tf(1)
        nodes, out = _run_update(mg, w, tf, mg.MG_RGBA8)
        ref_nodes = _check_nodes(w, nodes, tf)
        out4 = out.view(-1, 4)

        ids, seg_index = _leaf_index_chunked(w.seg)
        assert np.array_equal(ids, w.host_graph["leaf_segment_id"])
        _check_mipmap_every_voxel(w, out, tf, ref_nodes, seg_index, 77 + cfg_id)

        # ---- quantised graph vs the DIRECT histogram (north_star's second tolerance; I11 / I12)
        _check_direct_histogram(w, cfg_id, tf, nodes.cpu().numpy().astype(np.float64), seg_index, ids.size)
        _check_render_full_size(mg, w, tf, seg_index)
        if cfg_id in (2, 4):                                                 # the configs BASELINE.json names by their update sequence
            del nodes, out
            _check_update_sequence(mg, w, seg_index, cfg_id)
    finally:
        w.close()


def _check_direct_histogram(w, cfg_id, tf, nodes_host, seg_index, nl, dense_bytes=2 << 30, n_sample=1000, tol=TOL_DIRECT,
                            first_level=1, tag=""):
    """GPU node colours (fp32, quantised graph) against C_dir = sum_s H_s TF[s] with H by brute force from the
    generator's volume (O-3), and the graph's symbolic mixtures mu (O-5) against H."""
    hg = w.host_graph
    tf64 = tf.astype(np.float64)
    mu = oracle.symbolic_eval_sparse(hg["child_a"], hg["child_b"], hg["weight"], nl)
    span = float(tf64.max() - tf64.min())
    report = {"config": cfg_id, "quant_bits": int(w.stats["quant_bits"]), "n_nodes": int(w.stats["n_nodes"]),
              "depth": int(w.stats["depth"]), "tolerance": TOL_DIRECT, "levels": []}
    worst_c = worst_l1 = 0.0
    for l in range(first_level, len(w.mip_dims)):
        xl, yl, zl = w.mip_dims[l]
        idx_l = w.host_idx[l].reshape(-1)
        nv = idx_l.size
        if nv * nl * 8 <= dense_bytes:                                     # every voxel of the level
            H = oracle.brute_force_level(seg_index, nl, l).reshape(nv, nl)
            vox = np.arange(nv)
        else:                                                              # >= n_sample mixed voxels (a pure voxel is a leaf: exact)
            mixed = np.flatnonzero(idx_l >= nl)
            if mixed.size == 0:
                continue
            if mixed.size <= 2 * n_sample:
                vox = mixed
            else:                                                          # draws with replacement: a third more than needed
                k = n_sample + n_sample // 3
                vox = np.unique(mixed[(synth.u64(5, 300 + l, np.arange(k, dtype=np.uint64)) % np.uint64(mixed.size)).astype(np.int64)])
                assert vox.size >= n_sample
            H = np.stack([oracle.brute_force_histogram(seg_index, nl, l, int(v % xl), int((v // xl) % yl), int(v // (xl * yl)))
                          for v in vox])
        assert np.abs(H.sum(axis=1) - 1.0).max() < 1e-12
        node = idx_l[vox].astype(np.int64)
        err_c = np.abs(nodes_host[node] - H @ tf64).max(axis=1)
        l1 = np.abs(mu[node].toarray() - H).sum(axis=1)
        assert (err_c <= 0.5 * l1 * span + 2e-6).all(), f"I12 violated on level {l}"
        report["levels"].append({"level": l, "voxels": int(nv), "checked": int(vox.size), "every_voxel": bool(vox.size == nv),
                                 "max_abs_colour": float(err_c.max()), "max_l1_mixture": float(l1.max())})
        worst_c, worst_l1 = max(worst_c, float(err_c.max())), max(worst_l1, float(l1.max()))
    # ---- EVERY voxel of EVERY level >= first_level against the direct definition C_dir = sum_s H[s] TF[s] (O-3c: accumulated
    # from the generator's volume, coarse z-slab by z-slab; no histogram table).  A voxel the builder calls pure (its index
    # is a leaf) must BE pure: C_dir equals TF[leaf] to rounding -- a mixed voxel mis-classified as pure fails here.
    worst_all = 0.0
    done = {r["level"]: r for r in report["levels"]}
    for l in range(first_level, len(w.mip_dims)):
        xl, yl, zl = w.mip_dims[l]
        idx_l = w.host_idx[l].reshape(-1)
        per_k = xl * yl
        dk = max(1, (1 << 24) // per_k)
        lvl_max, n_pure, pure_max = 0.0, 0, 0.0
        for k0 in range(0, zl, dk):
            k1 = min(zl, k0 + dk)
            c_dir = oracle.direct_colour_level(seg_index, tf64, l, k0, k1).reshape(-1, 4)
            node = idx_l[k0 * per_k:k1 * per_k].astype(np.int64)
            lvl_max = max(lvl_max, float(np.abs(nodes_host[node] - c_dir).max()))
            pure = node < nl
            if pure.any():
                n_pure += int(pure.sum())
                pure_max = max(pure_max, float(np.abs(c_dir[pure] - tf64[node[pure]]).max()))
        assert pure_max <= 1e-12, f"level {l}: a voxel indexed as a leaf is not pure (|C_dir - TF[leaf]| = {pure_max:.3e})"
        assert lvl_max <= tol, f"level {l}: max |C_graph - C_dir| over all {idx_l.size} voxels = {lvl_max:.3e}"
        r = done.get(l)
        if r is None:
            r = {"level": l, "voxels": int(idx_l.size), "checked": 0, "every_voxel": False, "max_abs_colour": 0.0, "max_l1_mixture": 0.0}
            report["levels"].append(r)
        r.update(colour_checked_on="all", max_abs_colour_all_voxels=lvl_max, pure_voxels=n_pure, max_abs_pure_vs_tf=pure_max)
        worst_all = max(worst_all, lvl_max)
    report["levels"].sort(key=lambda r: r["level"])
    report["max_abs_colour_all_voxels"] = worst_all
    worst_c = max(worst_c, worst_all)
    report["max_abs_colour"], report["max_l1_mixture"] = worst_c, worst_l1
    print(f"cfg {cfg_id} (b = {report['quant_bits']}, {report['n_nodes']} nodes, depth {report['depth']}): max |C_graph - C_dir| = "
          f"{worst_c:.3e}, max ||mu - H||_1 = {worst_l1:.3e}; per level: " +
          ", ".join(f"l{r['level']}:{r['max_abs_colour']:.1e}/{r['max_l1_mixture']:.1e}({r['checked']})" for r in report["levels"]) +
          f"; colour on ALL voxels of every level: max {worst_all:.3e}")
    out_dir = os.environ.get("MG_PARITY_REPORT_DIR")
    if out_dir:
        os.makedirs(out_dir, exist_ok=True)
        with open(os.path.join(out_dir, f"direct_parity_cfg{cfg_id}{tag}.json"), "w") as f:
            json.dump(report, f, indent=1)
    assert worst_c <= tol, worst_c
    return report


def test_config4_at_the_papers_bitrate_is_reported(libs):
    """Config 4 at the paper's b = 9 (L305), which its synthetic stand-in does NOT carry inside north_star's 2e-3
    (SURVEY.md Q7 expected as much: Table 2's max error 0.005 in l1 allows 2.5e-3 in colour): the same check as above
    on every voxel of the levels >= 5 (where the error peaks), asserted only against I12 and 3e-3, and written to
    the report as direct_parity_cfg4_b9.json.  The config itself is built at b = 10, the smallest bitrate that meets
    the tolerance (synth.CONFIGS[4])."""
    mg, workload = libs
    w = workload.make(4, keep_seg=True, quant_bits=9)
    try:
        assert w.stats["quant_bits"] == 9
        tf = w.tf(1)
        g = w.graph
        nodes = torch.empty((g.info.n_nodes, 4), dtype=torch.float32, device="cuda")
        g.propagate(torch.from_numpy(tf).cuda(), nodes)
        torch.cuda.synchronize()
        _check_nodes(w, nodes, tf)
        ids, seg_index = _leaf_index_chunked(w.seg)
        r = _check_direct_histogram(w, 4, tf, nodes.cpu().numpy().astype(np.float64), seg_index, ids.size, tol=3e-3,
                                    first_level=5, tag="_b9")
        assert r["max_abs_colour"] > 0.5 * TOL_DIRECT                   # (it is the tolerance's order of magnitude)
    finally:
        w.close()


def _check_render_full_size(mg, w, tf, seg_index):
    """NEXT-2 in bench.py's launch configuration (synth.render_view: 1600 x 1200, 0.5-voxel steps, ESS 1e-8,
    spacing 1:1:7): sampled pixels + the image corners against the oracle's per-ray march on the same
    pyramid (tolerance: tests/test_gpu_render.py), and the ESS-off image must equal the ESS-on image."""
    g = w.graph
    rtf = synth.render_tf(tf)
    nodes = torch.empty((g.info.n_nodes, 4), dtype=torch.float32, device="cuda")
    g.propagate(torch.from_numpy(rtf).cuda(), nodes)
    view = synth.render_view(w.cfg)
    W, H = view["width"], view["height"]
    img = torch.full((H, W, 4), float("nan"), dtype=torch.float32, device="cuda")
    img_off = torch.full((H, W, 4), float("nan"), dtype=torch.float32, device="cuda")
    img_plain = torch.full((H, W, 4), float("nan"), dtype=torch.float32, device="cuda")
    stats = torch.zeros(12, dtype=torch.int64, device="cuda")
    desc = w.mip_desc()
    assert view["flags"] == mg.MG_VIEW_HISTOGRAM_MIPMAP            # what bench.py times
    g.render(w.d_idx, desc, nodes, view, img, stats[0:4])
    g.render(w.d_idx, desc, nodes, dict(view, ess_threshold=-1.0), img_off, stats[4:8])
    g.render(w.d_idx, desc, nodes, dict(view, flags=0), img_plain, stats[8:12])
    # mg_render_ex with the empty-space mask (what bench.py times as "ess"): same image, same counters as the climb
    mask = torch.empty(w.level_voxels[2], dtype=torch.int16, device="cuda")
    g.ess_mask_build(w.d_idx, desc, nodes, view["ess_threshold"], mask)
    img_mask = torch.full((H, W, 4), float("nan"), dtype=torch.float32, device="cuda")
    stats_mask = torch.zeros(4, dtype=torch.int64, device="cuda")
    g.render(w.d_idx, desc, nodes, view, img_mask, stats_mask, ess_mask_device=mask)
    torch.cuda.synchronize()
    assert torch.equal(img, img_mask) and torch.equal(stats[0:4], stats_mask)
    del mask, img_mask
    got, got_off = img.cpu().numpy().astype(np.float64), img_off.cpu().numpy().astype(np.float64)
    st = stats.cpu().numpy().reshape(3, 4)
    assert np.isfinite(got).all() and got[..., 3].max() > 0.5
    assert st[1, 1] == 0 and st[0, 0] <= st[1, 0] and st[2, 2] == 0
    if w.cfg.get("alpha_zero_frac", 0.0) > 0:                      # configs without a transparent segment have nothing to skip
        assert st[0, 1] > 0 and st[0, 0] < st[1, 0]
    if w.cfg.get("zscale", 1) > 1:                                  # lambda > 0 somewhere: the coarse-first shortcut fires
        assert st[0, 2] > 0
    assert st[0, :2].sum() == st[1, :2].sum() == st[2, :2].sum()
    assert np.abs(got - got_off).max() <= 1e-5                     # skipped samples were (numerically) transparent
    assert np.abs(got - img_plain.cpu().numpy()).max() <= 1e-6     # one-leaf blocks do not change the image
    k = 300
    pi = (synth.u64(3, 400, np.arange(k, dtype=np.uint64)) % np.uint64(W)).astype(np.int64)
    pj = (synth.u64(3, 401, np.arange(k, dtype=np.uint64)) % np.uint64(H)).astype(np.int64)
    ij = np.concatenate([np.stack([pi, pj], 1), [[0, 0], [W - 1, 0], [0, H - 1], [W - 1, H - 1], [W // 2, H // 2]]])
    hg = w.host_graph
    pal = oracle.graph_eval(hg["child_a"], hg["child_b"], hg["weight"], hg["n_leaves"], rtf.astype(np.float64))
    flat = np.zeros(w.n_voxels_padded, dtype=np.uint32)
    for l, s0 in enumerate(w.level_start):                          # level 0 from the generator's volume, not from the device
        lv = seg_index if l == 0 else w.host_idx[l]
        flat[s0:s0 + lv.size] = lv.reshape(-1)
    ref, _ = oracle.render_pixels(None, pal, view, ij, flat=(flat, w.level_start, np.array(w.mip_dims)))
    err = np.abs(got[ij[:, 1], ij[:, 0]] - ref).max()
    hit = (ref[:, 3] > 0).mean()
    print(f"render 1600x1200 {w.name}: max|err| on {ij.shape[0]} sampled pixels = {err:.2e} ({hit:.0%} hit the volume); "
          f"samples composited/skipped/from one-leaf blocks: {st[0, :3].tolist()}, without ESS {st[1, :3].tolist()}, "
          f"without the histogram-mipmap flag {st[2, :3].tolist()}")
    assert hit > 0.3 and err <= 5e-6, err


def test_config3_fp16_output_full_size(libs):
    """Same launch configuration with the fp16 output, every voxel of every level: level 0 must hold exactly the fp16
    code of TF[S(v)] (a leaf's colour is the fp32 TF entry, and RN to fp16 of an fp32 value is the same on both sides);
    every other level within 1 fp16 ulp of RN(oracle) on the host-built node indices."""
    mg, workload = libs
    w = workload.make(3, keep_seg=True)
    try:
        tf = w.tf(2)
        nodes, out = _run_update(mg, w, tf, mg.MG_RGBA16F)
        ref_nodes = _check_nodes(w, nodes, tf)
        out4 = out.view(torch.float16).view(-1, 4)
        # level 0: bit-exact against the code table of the TF, indexed by the generator's volume
        ids, seg_index = _leaf_index_chunked(w.seg)
        code = torch.from_numpy(oracle.to_rgba16f(tf.astype(np.float64)).view(np.int16).astype(np.int64)).cuda()   # [n_leaves, 4]
        flat = seg_index.reshape(-1)
        n0, step, bad = w.level_voxels[0], 1 << 26, 0
        o16 = out.view(torch.int16).view(-1, 4)
        for o in range(0, n0, step):
            e = min(n0, o + step)
            s_ = torch.from_numpy(flat[o:e].astype(np.int64)).cuda()
            bad += int((o16[o:e].to(torch.int64) != code[s_]).any(dim=1).sum().item())
        assert bad == 0, f"{bad} level-0 voxels differ from fp16(TF[S(v)])"
        for l, (s0, nv) in enumerate(zip(w.level_start, w.level_voxels)):
            if l == 0:
                continue
            idx_l = w.host_idx[l].reshape(-1)
            chunk = 1 << 23
            for o in range(0, nv, chunk):
                e = min(nv, o + chunk)
                got = out4[s0 + o:s0 + e].cpu().numpy()
                ref = oracle.to_rgba16f(oracle.lookup(idx_l[o:e], ref_nodes))
                gi, ri = got.view(np.int16).astype(np.int64), ref.view(np.int16).astype(np.int64)
                assert (np.abs(gi - ri) <= 1).all(), f"level {l}, voxels {o}..{e}"
    finally:
        w.close()


@pytest.mark.parametrize("cfg_id", [3, 4])
def test_packed_mipmap_full_size(libs, cfg_id):
    """NEXT-3 at full size: the bit-packed mipmap (Table 1 (8), (9), (A)) colourises to EXACTLY the bytes of
    the uint32 path on all voxels of all levels; per-level i_min / r(l) match the oracle's Eq. 15-16 on the
    builder's indices; the device stream of a whole level equals the oracle's stream bit for bit."""
    mg, workload = libs
    w = workload.make(cfg_id)
    try:
        tf = w.tf(3)
        nodes, out = _run_update(mg, w, tf, mg.MG_RGBA8)
        w.pack()
        out_p = torch.full_like(out, 0xAB)
        st = torch.cuda.current_stream().cuda_stream
        w.graph.colorize_packed(w.d_packed, w.packed_levels, nodes, out_p, fmt=mg.MG_RGBA8, stream=st, from_last_propagate=True)
        torch.cuda.synchronize()
        o4, p4 = out.view(-1, 4), out_p.view(-1, 4)
        for s0, nv in zip(w.level_start, w.level_voxels):                      # every voxel of every level
            assert torch.equal(o4[s0:s0 + nv], p4[s0:s0 + nv])
        total_bits = 0
        for l, lv in enumerate(w.packed_levels):
            lo, hi = oracle.index_range(w.host_idx[l])
            assert (lv["i_min"], lv["bits"]) == (lo, oracle.bits_per_voxel(lo, hi)), l
            total_bits += lv["bits"] * lv["n_voxels"]
        assert w.packed_levels[0]["bits"] == oracle.bits_per_voxel(0, w.n_leaves - 1)   # level 0 references leaves only (I5)
        l = 2                                                                  # one whole level, bit for bit
        lv = w.packed_levels[l]
        ref = oracle.pack_level(w.host_idx[l], lv["i_min"], lv["bits"])
        got = w.d_packed[lv["byte_offset"]:lv["byte_offset"] + ref.size].cpu().numpy()
        assert np.array_equal(got, ref)
        print(f"cfg {cfg_id}: packed mipmap {w.packed_bytes / 1e9:.3f} GB = {total_bits / w.n_voxels:.2f} bits/voxel "
              f"(uint32: {4 * w.n_voxels / 1e9:.3f} GB); r(l) = {[lv['bits'] for lv in w.packed_levels]}")
    finally:
        w.close()


@pytest.mark.parametrize("relabel", [True, False], ids=["relabelled_as_bench_does", "callers_numbering"])
def test_config5_dag_stress_full_size(libs, relabel):
    """2^26 nodes, 24 levels, 2^14 leaves, random children; 512^3 random node-index volume: every node and every voxel.
    bench.py loads this config with MG_RELABEL: the library's numbering is then a permutation of the caller's."""
    mg, workload = libs
    w = workload.make(5, relabel=relabel)
    try:
        assert w.graph.info.n_nodes == 1 << 26 and w.graph.info.depth == 23 and w.n_voxels == 512 ** 3
        assert (w.perm is not None) == relabel
        tf = w.tf(0)
        nodes, out = _run_update(mg, w, tf, mg.MG_RGBA8)
        hg = w.host_graph
        ref_nodes = oracle.graph_eval(hg["child_a"], hg["child_b"], hg["weight"], hg["n_leaves"], tf.astype(np.float64))
        got = nodes.cpu().numpy()
        if relabel:
            got = got[w.perm]                                                # caller's node n lives at perm[n]
        assert np.array_equal(got[:hg["n_leaves"]].view(np.uint32), tf.view(np.uint32)), "leaves not bit-exact"
        assert float(np.abs(got - ref_nodes).max()) <= TOL                   # every one of the 2^26 nodes
        del got
        out4 = out.view(-1, 4)
        chunk = 1 << 23                                                      # every one of the 512^3 voxels, chunked
        for o in range(0, w.n_voxels, chunk):
            e = min(w.n_voxels, o + chunk)
            assert _rgba8_close(out4[o:e].cpu().numpy(), oracle.lookup(w.host_idx[0][o:e], ref_nodes)), (o, e)
    finally:
        w.close()


def test_config5_scaled_with_relabel(libs):
    """Config 5 at 1/64 scale loaded with MG_RELABEL (bench.py --relabel): the library's numbering is a
    permutation of the caller's; node colours and colourised voxels must equal the oracle's through it."""
    mg, workload = libs
    w = workload.make(5, scale=1.0 / 64, relabel=True)
    try:
        assert w.perm is not None and w.graph.info.relabelled == 1
        assert np.array_equal(np.sort(w.perm), np.arange(w.perm.size))
        tf = w.tf(0)
        nodes, out = _run_update(mg, w, tf, mg.MG_RGBA8)
        hg = w.host_graph
        ref = oracle.graph_eval(hg["child_a"], hg["child_b"], hg["weight"], hg["n_leaves"], tf.astype(np.float64))
        got = nodes.cpu().numpy()[w.perm]                                    # caller's node n lives at perm[n]
        assert np.array_equal(got[:hg["n_leaves"]].view(np.uint32), tf.view(np.uint32))
        assert float(np.abs(got - ref).max()) <= TOL
        out4 = out.view(-1, 4).cpu().numpy()[:w.n_voxels]
        assert _rgba8_close(out4, oracle.lookup(w.host_idx[0], ref))         # host_idx keeps the caller's numbering
    finally:
        w.close()


def test_config1_every_voxel_every_level(libs):
    """Config 1 (64^3, 16 segments): element-by-element on all 299,593 voxels, unquantised and b = 9,
    both against the same-graph oracle and against the direct histogram (dense O-2)."""
    mg, workload = libs
    for bits, tol_direct in ((0, 1e-5), (9, TOL_DIRECT)):
        w = workload.make(1, keep_seg=True, quant_bits=bits)
        try:
            tf = w.tf(0)
            nodes, out = _run_update(mg, w, tf, mg.MG_RGBA8)
            ref_nodes = _check_nodes(w, nodes, tf)
            ids, seg_index = oracle.leaf_index(w.seg)
            H = oracle.histogram_mipmap(seg_index, ids.size)
            out4 = out.view(-1, 4).cpu().numpy()
            got_nodes = nodes.cpu().numpy().astype(np.float64)
            for l, counts in enumerate(H):
                s0, nv = w.level_start[l], w.level_voxels[l]
                idx = w.host_idx[l].reshape(-1)
                assert _rgba8_close(out4[s0:s0 + nv], oracle.lookup(idx, ref_nodes))
                direct = oracle.direct_colour(counts, l, tf.astype(np.float64)).reshape(-1, 4)
                assert np.abs(got_nodes[idx] - direct).max() <= tol_direct
        finally:
            w.close()


def _sub_dag(hg, targets):
    """The part of the graph below `targets`, renumbered (leaves first, children before parents), for the
    dense oracle: returns (child_a, child_b, weight, sigma, n_sub_leaves, old ids of the sub-nodes)."""
    a, b, nl = hg["child_a"], hg["child_b"], hg["n_leaves"]
    seen, stack = set(), [int(t) for t in targets]
    while stack:
        n = stack.pop()
        if n in seen:
            continue
        seen.add(n)
        if n >= nl:
            stack += [int(a[n]), int(b[n])]
    old = np.array(sorted(seen), dtype=np.int64)                  # library numbering is children-before-parents
    n_sub_leaves = int((old < nl).sum())
    new = {int(o): i for i, o in enumerate(old)}
    sa = np.array([new[int(a[o])] if o >= nl else 0 for o in old], dtype=np.uint32)
    sb = np.array([new[int(b[o])] if o >= nl else 0 for o in old], dtype=np.uint32)
    return sa, sb, hg["weight"][old].astype(np.float64), hg["weight_sigma"][old].astype(np.float64), n_sub_leaves, old


@pytest.mark.parametrize("cfg_id", [3, 4])
def test_mixture_lut_and_range_queries_full_size(libs, cfg_id):
    """NEXT-4 at full size, in bench.py's launch configuration (batches of random cubes, Table 4's sizes).
    The dense oracle cannot hold 1.7 M x 1182 entries, so: sampled rows of the table against the oracle run on
    the sub-DAG below them; every row sums to 1; NAIVE == the plain per-segment voxel count of the generator's
    volume (exact); FA fetch counts == the oracle's decomposition; FA sums to the box volume (L251) and stays
    within 1 % of the volume of the true counts (L251: 'about 0.3 %')."""
    mg, workload = libs
    w = workload.make(cfg_id, keep_seg=True)
    try:
        hg, g = w.host_graph, w.graph
        nl = hg["n_leaves"]
        lut = g.mixture_lut(hg["weight_sigma"])
        rp, leaf, mu, dmu = lut.export()
        n = rp.size - 1
        assert n == hg["child_a"].size and lut.info.nnz == leaf.size == lut.info.capacity     # builder graphs: disjoint children
        sums = np.add.reduceat(mu, rp[:-1].astype(np.int64))
        assert np.abs(sums - 1.0).max() <= 1e-12
        # sampled rows (incl. the root and the deepest nodes) against the dense oracle on their sub-DAG
        pick = np.unique(np.concatenate([(synth.u64(3, 500, np.arange(300, dtype=np.uint64)) % np.uint64(n)).astype(np.int64),
                                         np.arange(n - 40, n)]))
        sa, sb, sw, ssg, snl, old = _sub_dag(hg, pick)
        omu, odmu = oracle.mixture_lut(sa, sb, sw, ssg, snl)
        pos = {int(o): i for i, o in enumerate(old)}
        for t in pick:
            s, e = int(rp[t]), int(rp[t + 1])
            row = pos[int(t)]
            cols = np.array([pos[int(c)] for c in leaf[s:e]])               # sub-leaf index of each stored leaf
            assert (np.flatnonzero(omu[row]) == np.sort(cols)).all()
            np.testing.assert_allclose(mu[s:e], omu[row, cols], rtol=1e-12)
            np.testing.assert_allclose(dmu[s:e], odmu[row, cols], rtol=1e-12, atol=1e-300)

        dims = synth.CONFIGS[cfg_id]["dims"]
        ids, seg_index = _leaf_index_chunked(w.seg)
        desc = w.mip_desc()
        l_max = len(w.mip_dims) - 1
        worst = 0.0
        for side in (16, 64, 256):
            boxes = synth.query_boxes(dims, side, 24, seed=cfg_id)
            nq = len(boxes)
            e_fa = torch.empty((nq, nl), dtype=torch.float64, device="cuda")
            d_fa = torch.empty((nq, nl), dtype=torch.float64, device="cuda")
            f_fa = torch.empty((nq,), dtype=torch.int64, device="cuda")
            e_nv = torch.empty((nq, nl), dtype=torch.float64, device="cuda")
            f_nv = torch.empty((nq,), dtype=torch.int64, device="cuda")
            lut.range_query(w.d_idx, desc, boxes, e_fa, d_fa, f_fa, mode=mg.MG_QUERY_FA)
            lut.range_query(w.d_idx, desc, boxes, e_nv, None, f_nv, mode=mg.MG_QUERY_NAIVE)
            torch.cuda.synchronize()
            e_fa, d_fa, f_fa, e_nv, f_nv = (t.cpu().numpy() for t in (e_fa, d_fa, f_fa, e_nv, f_nv))
            for q, (x0, y0, z0, x1, y1, z1) in enumerate(boxes):
                vol = (x1 - x0) * (y1 - y0) * (z1 - z0)
                truth = np.bincount(seg_index[z0:z1, y0:y1, x0:x1].reshape(-1), minlength=nl)
                assert np.array_equal(e_nv[q], truth) and f_nv[q] == vol
                segs = [oracle.fa_axis(lo, hi, l_max) for lo, hi in ((x0, x1), (y0, y1), (z0, z1))]
                n_fetch = sum(1 << (lx + ly + lz - 3 * min(lx, ly, lz)) for _, lx in segs[0] for _, ly in segs[1] for _, lz in segs[2])
                assert f_fa[q] == n_fetch
                assert abs(e_fa[q].sum() - vol) <= 1e-9 * vol
                assert (e_fa[q] >= 0).all() and (d_fa[q] >= 0).all()
                worst = max(worst, float(np.abs(e_fa[q] - truth).max()) / vol)
        print(f"cfg{cfg_id} range queries: LUT {lut.info.nnz} entries ({lut.info.device_bytes / 1e6:.0f} MB, longest row "
              f"{lut.info.max_row_nnz}); max |FA - true count| / volume = {worst:.2e}")
        assert worst < 0.01, worst
        lut.close()
    finally:
        w.close()


def test_config3_device_mipmap_front_end_full_size(libs):
    """NEXT-4 (second half) at full size: the device-assisted assembly (bench.py --device-mipmap) yields the host
    builder's graph and node-index mipmap bit for bit, on all 1,438,087,061 voxels."""
    mg, workload = libs
    a = workload.make(3)
    try:
        ga = {k: a.host_graph[k].copy() for k in ("child_a", "child_b", "weight", "weight_sigma", "level_offsets", "leaf_segment_id")}
        ref = a.d_idx.clone()
        stats_a = dict(a.stats)
    finally:
        a.close()
    b = workload.make(3, device_mipmap=True)
    try:
        for k, v in ga.items():
            assert np.array_equal(v, b.host_graph[k]), k
        assert torch.equal(ref, b.d_idx)
        print(f"cfg3 setup: host path synth {stats_a['synth_s']:.2f} + builder {stats_a['builder_s']:.2f} + upload "
              f"{stats_a['upload_idx_s']:.2f} s; device front end: synth {b.stats['synth_s']:.2f} + front end "
              f"{b.stats['front_end_s']:.2f} + builder {b.stats['builder_s']:.2f} + upload {b.stats['upload_idx_s']:.2f} s "
              f"({b.stats['n_level1_mixed']} non-pure level-1 parents)")
    finally:
        b.close()


@pytest.mark.parametrize("cfg_id", [3, 4, 2])
def test_device_levels_full_size(libs, cfg_id):
    """NEXT-4 (second half) at full size: the levels >= 1 of the histogram mipmap merged and hash-consed on the device
    (bench.py --device-levels) yield the graph and the node-index mipmap of the level-1 front-end path bit for bit."""
    mg, workload = libs
    a = workload.make(cfg_id, device_mipmap=True)
    try:
        ga = {k: a.host_graph[k].copy() for k in ("child_a", "child_b", "weight", "weight_sigma", "level_offsets", "leaf_segment_id")}
        ref = a.d_idx.clone()
        stats_a = dict(a.stats)
    finally:
        a.close()
    b = workload.make(cfg_id, device_mipmap="levels")
    try:
        for k, v in ga.items():
            assert np.array_equal(v, b.host_graph[k]), k
        assert torch.equal(ref, b.d_idx)
        assert b.stats["n_distinct_mixtures"] == stats_a["n_distinct_mixtures"] and b.stats["nnz_per_voxel"] == stats_a["nnz_per_voxel"]
        print(f"cfg{cfg_id} setup, level-1 front end: front {stats_a['front_end_s']:.2f} + builder {stats_a['builder_s']:.2f} "
              f"(mipmap {stats_a['builder_mipmap_s']:.2f}) + upload {stats_a['upload_idx_s']:.2f} s; device levels 1 .. "
              f"{b.stats['device_levels_done']}: front {b.stats['front_end_s']:.2f} + builder {b.stats['builder_s']:.2f} "
              f"(mipmap {b.stats['builder_mipmap_s']:.2f}) + upload {b.stats['upload_idx_s']:.2f} s; "
              f"{b.stats['n_device_mixtures']} of {b.stats['n_distinct_mixtures']} distinct mixtures found on the device")
    finally:
        b.close()
