"""CPU fp64 oracle of the Mixture Graph TF-propagation path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes/numpy wrapper around ``mg_oracle.c`` (see its header for citations and pins).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from the CUDA library,
the host builder or the input generators; inputs are passed in as numpy arrays.

Function -> passage (PAPER.md line):
  mip_dims             O-1  L80
  leaf_index           Q14  L76, L130 (sources = the segment IDs present)
  histogram_mipmap     O-2  Eq. 4 L78-L80 (integer counts scaled to 8^l)
  direct_colour        O-2  L66 (<m, x>)
  direct_colour_level  O-3c L66 with Eq. 4 unrolled: every voxel of a level, no histogram table
  brute_force_histogram O-3 Eq. 4 unrolled
  brute_force_level    O-3 for every voxel of one level in one pass over the finest voxels
  symbolic_eval_sparse O-5 on a sparse matrix, level by level (full-size graphs; a scipy sparse product per level)
  graph_eval           O-4  L259, L269, L371, Eq. 8
  graph_eval_attr      NEXT-1: any numeric attribute, n_ch channels (L269, L271 (i)-(ii), L277)
  topo_levels          L211
  graph_eval_levels    L213, L373 (the paper's OpenMP CPU baseline shape)
  symbolic_eval        O-5  L321, L375
  lookup               L221, L267
  to_rgba8 / to_rgba16f  Q13 (defined by this repo; not in the paper)
  bits_per_voxel, index_range, pack_level, unpack_level   NEXT-3: Table 1 (8),(9),(A), Eq. 15-16
  pixel_ray, sample_lod, render, render_pixels   NEXT-2: ray-marching the paletted mipmap, readings R1-R6 (L265-L271, L414)
  mixture_lut          NEXT-4: mu and dmu per node, Eq. 17-18 L229-L239, L375 (reading Q19)
  fa_axis, range_query_fa, range_query_naive   NEXT-4: footprint assembly, section 3.6, Table 4 (reading Q20)
All functions are pinned by tests/test_oracle_pins.py / test_oracle_render.py / test_oracle_query.py; none is "parity
unpinned".  The weakest pin is Eq. 18 (mixture_lut's dmu): the paper prints no value for it, so it is tied only to a
hand-worked two-node case, its homogeneity in dw and the zero-sigma case; mu itself is pinned through symbolic_eval.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_lib = C.CDLL(_build())

_u32p = np.ctypeslib.ndpointer(np.uint32, flags="C_CONTIGUOUS")
_u64p = np.ctypeslib.ndpointer(np.uint64, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
_u8p = np.ctypeslib.ndpointer(np.uint8, flags="C_CONTIGUOUS")
_u64 = C.c_uint64
_u32 = C.c_uint32

_lib.mgo_mip_dims.argtypes = [_u64, _u64, _u64, _u64p, C.c_int]
_lib.mgo_mip_dims.restype = C.c_int
_lib.mgo_hist_level0.argtypes = [_u32p, _u64, _u32, _u64p]
_lib.mgo_hist_level0.restype = None
_lib.mgo_hist_next_level.argtypes = [_u64p, _u64, _u64, _u64, _u32, _u64p]
_lib.mgo_hist_next_level.restype = None
_lib.mgo_direct_colour.argtypes = [_u64p, _u64, _u32, _u32, _f64p, _f64p]
_lib.mgo_direct_colour.restype = None
_lib.mgo_brute_force_histogram.argtypes = [_u32p, _u64, _u64, _u64, _u32, _u32, _u64, _u64, _u64, _f64p]
_lib.mgo_brute_force_histogram.restype = None
_lib.mgo_brute_force_level.argtypes = [_u32p, _u64, _u64, _u64, _u32, _u32, _f64p]
_lib.mgo_brute_force_level.restype = None
_lib.mgo_direct_colour_level.argtypes = [_u32p, _u64, _u64, _u64, _f64p, _u32, _u64, _u64, _f64p]
_lib.mgo_direct_colour_level.restype = None
_lib.mgo_graph_eval.argtypes = [_u32p, _u32p, _f64p, _u64, _u64, _f64p, _f64p]
_lib.mgo_graph_eval.restype = None
_lib.mgo_graph_eval_attr.argtypes = [_u32p, _u32p, _f64p, _u64, _u64, _u32, _f64p, _f64p]
_lib.mgo_graph_eval_attr.restype = None
_lib.mgo_topo_levels.argtypes = [_u32p, _u32p, _u64, _u64, _u32p]
_lib.mgo_topo_levels.restype = C.c_int64
_lib.mgo_graph_eval_levels.argtypes = [_u32p, _u32p, _f64p, _u64, _u64p, _u64p, _u32, _f64p, _f64p, C.c_int]
_lib.mgo_graph_eval_levels.restype = C.c_int
_lib.mgo_symbolic_eval.argtypes = [_u32p, _u32p, _f64p, _u64, _u64, _f64p]
_lib.mgo_symbolic_eval.restype = None
_lib.mgo_lookup.argtypes = [_u32p, _u64, _f64p, _f64p, C.c_int]
_lib.mgo_lookup.restype = C.c_int
_lib.mgo_to_rgba8.argtypes = [_f64p, _u64, _u8p]
_lib.mgo_to_rgba8.restype = None
_lib.mgo_colourise_rgba8.argtypes = [_u32p, _u64, _f64p, _u8p, C.c_int]
_lib.mgo_colourise_rgba8.restype = C.c_int


_lib.mgo_bits_per_voxel.argtypes = [_u32, _u32]
_lib.mgo_bits_per_voxel.restype = _u32
_lib.mgo_pack_bits.argtypes = [_u32p, _u64, _u32, _u32, _u8p]
_lib.mgo_pack_bits.restype = None
_lib.mgo_unpack_bits.argtypes = [_u8p, _u64, _u32, _u32, _u32p]
_lib.mgo_unpack_bits.restype = None
_lib.mgo_sample_lod.argtypes = [_u32p, _u64p, _u32p, _u32, _f64p, _f64p, C.c_double, _f64p]
_lib.mgo_sample_lod.restype = None
_lib.mgo_pixel_ray.argtypes = [_f64p, C.c_double, _u32, _u32, _u32, _u32, _f64p]
_lib.mgo_pixel_ray.restype = None
_lib.mgo_render.argtypes = [_u32p, _u64p, _u32p, _u32, _f64p, _f64p, _f64p, _u32, _u32, _f64p, _u64p]
_lib.mgo_render.restype = None
_lib.mgo_render_pixels.argtypes = [_u32p, _u64p, _u32p, _u32, _f64p, _f64p, _f64p, _u32, _u32, _u32p, _u64, _f64p, _u64p]
_lib.mgo_render_pixels.restype = None
_lib.mgo_mixture_lut.argtypes = [_u32p, _u32p, _f64p, _f64p, _u64, _u64, _f64p, _f64p]
_lib.mgo_mixture_lut.restype = None
_lib.mgo_fa_axis.argtypes = [_u64, _u64, _u32, _u64p, _u32p]
_lib.mgo_fa_axis.restype = _u32
_lib.mgo_range_query_fa.argtypes = [_u32p, _u64p, _u32p, _u32, _f64p, _f64p, _u64, _u64p, _f64p, _f64p]
_lib.mgo_range_query_fa.restype = _u64
_lib.mgo_range_query_naive.argtypes = [_u32p, _u32p, _f64p, _u64, _u64p, _f64p]
_lib.mgo_range_query_naive.restype = _u64


def _c(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def mip_dims(dims_xyz):
    """[(X_l, Y_l, Z_l)] for l = 0..l_max (ceil-halving to 1^3, L80)."""
    buf = np.zeros(3 * 64, dtype=np.uint64)
    n = _lib.mgo_mip_dims(int(dims_xyz[0]), int(dims_xyz[1]), int(dims_xyz[2]), buf, 64)
    return [tuple(int(v) for v in buf[3 * l:3 * l + 3]) for l in range(n)]


def leaf_index(S):
    """Sorted distinct segment IDs present in S (they are the sources, L130; background 0 is an
    ordinary segment, Q14) and the per-voxel leaf number.  Returns (ids, seg_index like S)."""
    ids, inv = np.unique(np.asarray(S), return_inverse=True)
    return ids.astype(np.uint32), inv.reshape(np.shape(S)).astype(np.uint32)


def histogram_mipmap(seg_index, n_seg):
    """Dense integer histogram mipmap: list over levels of uint64 [Z_l, Y_l, X_l, n_seg] with
    every voxel's counts summing to 8^l (O-2).  Small volumes only (dense)."""
    seg_index = _c(seg_index, np.uint32)
    Z, Y, X = seg_index.shape
    dims = mip_dims((X, Y, Z))
    lv = np.zeros((Z, Y, X, n_seg), dtype=np.uint64)
    _lib.mgo_hist_level0(seg_index.reshape(-1), seg_index.size, n_seg, lv.reshape(-1))
    out = [lv]
    for l in range(1, len(dims)):
        cx, cy, cz = dims[l - 1]
        px, py, pz = dims[l]
        nxt = np.zeros((pz, py, px, n_seg), dtype=np.uint64)
        _lib.mgo_hist_next_level(out[-1].reshape(-1), cx, cy, cz, n_seg, nxt.reshape(-1))
        out.append(nxt)
    return out


def direct_colour(counts, level, tf):
    """C_dir = (sum_s c_s TF[s]) / 8^l, fp64 [Z_l, Y_l, X_l, 4]."""
    counts = _c(counts, np.uint64)
    n_seg = counts.shape[-1]
    tf = _c(tf, np.float64)
    assert tf.shape == (n_seg, 4)
    out = np.zeros(counts.shape[:-1] + (4,), dtype=np.float64)
    _lib.mgo_direct_colour(counts.reshape(-1), counts.size // n_seg, n_seg, level, tf.reshape(-1),
                           out.reshape(-1))
    return out


def brute_force_histogram(seg_index, n_seg, level, i, j, k):
    """Normalised histogram (sums to 1) of voxel (i,j,k) of ``level`` by the unrolled Eq. 4."""
    seg_index = _c(seg_index, np.uint32)
    Z, Y, X = seg_index.shape
    h = np.zeros(n_seg, dtype=np.float64)
    _lib.mgo_brute_force_histogram(seg_index.reshape(-1), X, Y, Z, n_seg, level, i, j, k, h)
    return h


def brute_force_level(seg_index, n_seg, level):
    """Normalised histograms of EVERY voxel of ``level`` by the unrolled Eq. 4 (one pass over the finest voxels):
    fp64 [Z_l, Y_l, X_l, n_seg], every voxel's histogram summing to 1.  Dense: for the coarse levels of big volumes."""
    seg_index = _c(seg_index, np.uint32)
    Z, Y, X = seg_index.shape
    xl, yl, zl = mip_dims((X, Y, Z))[level]
    h = np.zeros((zl, yl, xl, n_seg), dtype=np.float64)
    _lib.mgo_brute_force_level(seg_index.reshape(-1), X, Y, Z, n_seg, level, h.reshape(-1))
    return h


def direct_colour_level(seg_index, tf, level, k_begin=0, k_end=None):
    """C_dir = sum_s H[s] TF[s] of EVERY voxel of the coarse z-slabs [k_begin, k_end) of ``level``, accumulated finest
    voxel by finest voxel with the unrolled weights of Eq. 4 (O-3c; no histogram table, so it runs at full size):
    fp64 [k_end - k_begin, Y_l, X_l, 4]."""
    seg_index = _c(seg_index, np.uint32)
    tf = _c(tf, np.float64)
    Z, Y, X = seg_index.shape
    xl, yl, zl = mip_dims((X, Y, Z))[level]
    k_end = zl if k_end is None else int(k_end)
    assert 0 <= k_begin <= k_end <= zl and tf.ndim == 2 and tf.shape[1] == 4
    out = np.zeros((k_end - k_begin, yl, xl, 4), dtype=np.float64)
    _lib.mgo_direct_colour_level(seg_index.reshape(-1), X, Y, Z, tf.reshape(-1), level, k_begin, k_end, out.reshape(-1))
    return out


def graph_eval(child_a, child_b, weight, n_leaves, tf):
    """c[n] fp64 [n_nodes, 4]: leaves = tf, then (1-w) c[a] + w c[b] in index order (O-4).
    ``weight`` may be fp32 (converted exactly) or fp64."""
    a, b = _c(child_a, np.uint32), _c(child_b, np.uint32)
    w = _c(weight, np.float64)
    tf = _c(tf, np.float64)
    n = a.size
    assert b.size == n and w.size == n and tf.shape == (n_leaves, 4)
    c = np.zeros((n, 4), dtype=np.float64)
    _lib.mgo_graph_eval(a, b, w, n, n_leaves, tf.reshape(-1), c.reshape(-1))
    return c


def graph_eval_attr(child_a, child_b, weight, n_leaves, attr):
    """NEXT-1: c fp64 [n_nodes, n_ch] for an arbitrary per-leaf attribute ``attr`` [n_leaves, n_ch]
    (opacity alone: n_ch = 1, L271; light contributions, L277; K batched TFs: n_ch = 4 K)."""
    a, b = _c(child_a, np.uint32), _c(child_b, np.uint32)
    w = _c(weight, np.float64)
    attr = _c(attr, np.float64)
    n = a.size
    assert attr.ndim == 2 and attr.shape[0] == n_leaves and b.size == n and w.size == n
    n_ch = attr.shape[1]
    c = np.zeros((n, n_ch), dtype=np.float64)
    _lib.mgo_graph_eval_attr(a, b, w, n, n_leaves, n_ch, attr.reshape(-1), c.reshape(-1))
    return c


def topo_levels(child_a, child_b, n_leaves):
    """(level u32 [n_nodes], depth): sources 0, otherwise max(v1, v2) + 1 (L211)."""
    a, b = _c(child_a, np.uint32), _c(child_b, np.uint32)
    lev = np.zeros(a.size, dtype=np.uint32)
    depth = _lib.mgo_topo_levels(a, b, a.size, n_leaves, lev)
    if depth < 0:
        raise ValueError("child index does not precede its parent (Eq. 8)")
    return lev, int(depth)


def graph_eval_levels(child_a, child_b, weight, n_leaves, tf, n_threads=0):
    """Level-synchronous OpenMP evaluation (the paper's CPU baseline, L213/L373).
    Returns (c fp64 [n_nodes, 4], threads used)."""
    a, b = _c(child_a, np.uint32), _c(child_b, np.uint32)
    w = _c(weight, np.float64)
    tf = _c(tf, np.float64)
    lev, depth = topo_levels(a, b, n_leaves)
    order = np.argsort(lev, kind="stable").astype(np.uint64)
    start = np.searchsorted(lev[order.astype(np.int64)], np.arange(depth + 2)).astype(np.uint64)
    c = np.zeros((a.size, 4), dtype=np.float64)
    used = _lib.mgo_graph_eval_levels(a, b, w, n_leaves, order, start, depth, tf.reshape(-1),
                                      c.reshape(-1), n_threads)
    return c, used


def symbolic_eval(child_a, child_b, weight, n_leaves):
    """mu fp64 [n_nodes, n_leaves]: unit vectors on the leaves, propagated (O-5)."""
    a, b = _c(child_a, np.uint32), _c(child_b, np.uint32)
    w = _c(weight, np.float64)
    mu = np.zeros((a.size, n_leaves), dtype=np.float64)
    _lib.mgo_symbolic_eval(a, b, w, a.size, n_leaves, mu.reshape(-1))
    return mu


def symbolic_eval_sparse(child_a, child_b, weight, n_leaves):
    """O-5 for graphs too large for the dense table: mu as a scipy CSR matrix [n_nodes, n_leaves], fp64.
    Leaves carry unit vectors; the nodes of topological level L (= max + 1, L211) are all
    mu[n] = (1 - w) mu[a] + w mu[b] of rows of lower levels, i.e. ONE sparse product W_L @ mu_below with two
    entries (1 - w, w) per row of W_L -- the same recurrence as symbolic_eval, a level at a time."""
    import scipy.sparse as sp
    a, b = _c(child_a, np.uint32).astype(np.int64), _c(child_b, np.uint32).astype(np.int64)
    w = _c(weight, np.float64)
    n = a.size
    lev, depth = topo_levels(child_a, child_b, n_leaves)
    mu = sp.identity(n_leaves, dtype=np.float64, format="csr")
    mu.resize((n, n_leaves))
    for L in range(1, depth + 1):                                    # (rows of the levels >= L are still empty)
        rows = np.flatnonzero(lev == L)
        k = rows.size
        W = sp.csr_matrix((np.concatenate([1.0 - w[rows], w[rows]]),
                           (np.concatenate([np.arange(k), np.arange(k)]), np.concatenate([a[rows], b[rows]]))),
                          shape=(k, n))
        level_rows = W @ mu
        # scatter the new rows into mu (children of later levels read them)
        sel = sp.csr_matrix((np.ones(k), (rows, np.arange(k))), shape=(n, k))
        mu = mu + sel @ level_rows
    return mu.tocsr()


def lookup(node_idx, c, n_threads=1):
    """C_graph(v) = c[node_idx[v]], fp64 [..., 4]."""
    idx = _c(node_idx, np.uint32)
    c = _c(c, np.float64)
    out = np.zeros(idx.shape + (4,), dtype=np.float64)
    _lib.mgo_lookup(idx.reshape(-1), idx.size, c.reshape(-1), out.reshape(-1), n_threads)
    return out


def to_rgba8(c):
    """uint8 [..., 4]: round_half_even(clamp(fp32(c), 0, 1) * 255), decision in fp32 (Q13)."""
    c = _c(c, np.float64)
    out = np.zeros(c.shape, dtype=np.uint8)
    _lib.mgo_to_rgba8(c.reshape(-1), c.size // 4, out.reshape(-1))
    return out


def to_rgba16f(c):
    """fp16 [..., 4]: RN(fp32(c)) (Q13)."""
    return np.asarray(c, dtype=np.float64).astype(np.float32).astype(np.float16)


def colourise_rgba8(node_idx, c, n_threads=0):
    """lookup + to_rgba8 in one pass (timed CPU baseline of the colourise step)."""
    idx = _c(node_idx, np.uint32)
    c = _c(c, np.float64)
    out = np.zeros(idx.shape + (4,), dtype=np.uint8)
    used = _lib.mgo_colourise_rgba8(idx.reshape(-1), idx.size, c.reshape(-1), out.reshape(-1), n_threads)
    return out, used


# ---- NEXT-3: bit-packed node-ID volumes (Table 1 rows (8), (9), (A); Eq. 15-16) ------------------

def index_range(node_idx):
    """(i_min(l), i_max(l)) of Eq. 15, read per level (Q10): min / max node ID referenced by the level."""
    idx = np.asarray(node_idx)
    return int(idx.min()), int(idx.max())


def bits_per_voxel(i_min, i_max):
    """r(l) = ceil(log2(i_max - i_min + 1)), Eq. 16."""
    return int(_lib.mgo_bits_per_voxel(int(i_min), int(i_max)))


def pack_level(node_idx, i_min, r):
    """uint8 stream of ceil(n r / 8) bytes: voxel v holds (node_idx[v] - i_min) in bits [v r, (v+1) r),
    LSB first (reading Q18)."""
    idx = _c(node_idx, np.uint32).reshape(-1)
    out = np.zeros((idx.size * int(r) + 7) // 8, dtype=np.uint8)
    _lib.mgo_pack_bits(idx, idx.size, int(i_min), int(r), out)
    return out


def unpack_level(stream, n_vox, i_min, r):
    """Inverse of pack_level: uint32 [n_vox]."""
    st = _c(stream, np.uint8).reshape(-1)
    assert st.size * 8 >= int(n_vox) * int(r)
    out = np.zeros(int(n_vox), dtype=np.uint32)
    _lib.mgo_unpack_bits(st, int(n_vox), int(i_min), int(r), out)
    return out


# ---- NEXT-2: ray-marching the paletted mipmap (section 4; readings R1-R6 in mg_oracle.c) ----

def _pyramid(levels):
    """levels: list of uint32 [Z_l, Y_l, X_l] node-index volumes, finest first -> (idx, offsets, dims)."""
    offs, dims, flat, o = [], [], [], 0
    for lv in levels:
        lv = np.asarray(lv)
        offs.append(o)
        dims.append((lv.shape[2], lv.shape[1], lv.shape[0]))
        flat.append(_c(lv, np.uint32).reshape(-1))
        o += lv.size
    return np.concatenate(flat), np.array(offs, dtype=np.uint64), np.array(dims, dtype=np.uint32).reshape(-1)


def _cam_par(view):
    cam = np.concatenate([np.asarray(view[k], dtype=np.float64).reshape(3) for k in ("eye", "right", "up", "forward")])
    par = np.array([view["tan_half_fov"], *np.asarray(view["spacing"], dtype=np.float64).reshape(3), view["step_voxels"],
                    view["ref_step_voxels"], view["lod_bias"], view["ess_threshold"], view["alpha_cutoff"]], dtype=np.float64)
    return np.ascontiguousarray(cam), par


def pixel_ray(view, i, j):
    """R1: unit direction of pixel (i, j) (j = row from the top)."""
    cam, par = _cam_par(view)
    d = np.zeros(3)
    _lib.mgo_pixel_ray(cam, par[0], int(view["width"]), int(view["height"]), int(i), int(j), d)
    return d


def sample_lod(levels, palette, p_vox, lam):
    """R3: trilinear + inter-level blend at p_vox (level-0 voxel coordinates) for fractional level lam."""
    idx, offs, dims = _pyramid(levels)
    out = np.zeros(4)
    _lib.mgo_sample_lod(idx, offs, dims, len(levels), _c(palette, np.float64).reshape(-1),
                        np.ascontiguousarray(p_vox, dtype=np.float64), float(lam), out)
    return out


def render(levels, palette, view):
    """R1-R6: fp64 image [H, W, 4] = (C_rgb associated, A) and (samples evaluated, samples skipped)."""
    idx, offs, dims = _pyramid(levels)
    cam, par = _cam_par(view)
    W, H = int(view["width"]), int(view["height"])
    out = np.zeros((H, W, 4), dtype=np.float64)
    stats = np.zeros(2, dtype=np.uint64)
    _lib.mgo_render(idx, offs, dims, len(levels), _c(palette, np.float64).reshape(-1), cam, par, W, H,
                    out.reshape(-1), stats)
    return out, (int(stats[0]), int(stats[1]))


def render_pixels(levels, palette, view, pixels_ij, flat=None):
    """The same rays as ``render`` for selected pixels only: pixels_ij = [(column i, row j)] -> fp64 [n, 4] and
    the (evaluated, skipped) counters.  ``flat`` = (node_idx, level_offset, level_dim_xyz) passes an already
    concatenated pyramid (full-size volumes) instead of ``levels``."""
    if flat is None:
        idx, offs, dims = _pyramid(levels)
    else:
        idx = _c(flat[0], np.uint32).reshape(-1)
        offs = np.ascontiguousarray(flat[1], dtype=np.uint64)
        dims = np.ascontiguousarray(flat[2], dtype=np.uint32).reshape(-1)
    cam, par = _cam_par(view)
    ij = np.ascontiguousarray(pixels_ij, dtype=np.uint32).reshape(-1, 2)
    out = np.zeros((ij.shape[0], 4), dtype=np.float64)
    stats = np.zeros(2, dtype=np.uint64)
    _lib.mgo_render_pixels(idx, offs, dims, offs.size, _c(palette, np.float64).reshape(-1), cam, par,
                           int(view["width"]), int(view["height"]), ij.reshape(-1), ij.shape[0], out.reshape(-1), stats)
    return out, (int(stats[0]), int(stats[1]))


# ---- NEXT-4: mixture lookup table with Eq. 18 errors; footprint-assembly range queries (sections 3.5-3.6) ----

def mixture_lut(child_a, child_b, weight, weight_sigma, n_leaves):
    """(mu, dmu) fp64 [n_nodes, n_leaves]: e_i with error 0 on leaf i, propagated with Eq. 18 (L375)."""
    a, b = _c(child_a, np.uint32), _c(child_b, np.uint32)
    w, sg = _c(weight, np.float64), _c(weight_sigma, np.float64)
    mu = np.zeros((a.size, n_leaves), dtype=np.float64)
    dmu = np.zeros((a.size, n_leaves), dtype=np.float64)
    _lib.mgo_mixture_lut(a, b, w, sg, a.size, n_leaves, mu.reshape(-1), dmu.reshape(-1))
    return mu, dmu


def fa_axis(lo, hi, max_level):
    """1D decomposition of [lo, hi) into aligned power-of-two pieces (section 3.6): [(start, level)]."""
    start = np.zeros(130, dtype=np.uint64)
    level = np.zeros(130, dtype=np.uint32)
    n = _lib.mgo_fa_axis(int(lo), int(hi), int(max_level), start, level)
    return [(int(start[i]), int(level[i])) for i in range(n)]


def range_query_fa(levels, mu, dmu, box):
    """Footprint assembly over box = (x0, y0, z0, x1, y1, z1): (expected voxels per leaf, error per leaf, fetches)."""
    idx, offs, dims = _pyramid(levels)
    mu, dmu = _c(mu, np.float64), _c(dmu, np.float64)
    nl = mu.shape[1]
    e, d = np.zeros(nl), np.zeros(nl)
    n = _lib.mgo_range_query_fa(idx, offs, dims, len(levels), mu.reshape(-1), dmu.reshape(-1), nl,
                                np.ascontiguousarray(box, dtype=np.uint64), e, d)
    return e, d, int(n)


def range_query_naive(level0, mu, box):
    """Sum of mu over every finest-level voxel of the box (L377): (expected voxels per leaf, fetches)."""
    l0 = _c(level0, np.uint32)
    dims = np.array([l0.shape[2], l0.shape[1], l0.shape[0]], dtype=np.uint32)
    mu = _c(mu, np.float64)
    e = np.zeros(mu.shape[1])
    n = _lib.mgo_range_query_naive(l0.reshape(-1), dims, mu.reshape(-1), mu.shape[1],
                                   np.ascontiguousarray(box, dtype=np.uint64), e)
    return e, int(n)
