"""Seeded synthetic inputs shaped like the paper's workloads.

This module holds NONE of the method's arithmetic (no histogram, no factorisation, no lerp):
it only draws segmentation volumes, transfer functions and random DAGs from a counter-based
generator, so that the CPU oracle (``oracle/``) and the CUDA path can be fed the same arrays.
It imports neither of them.

The paper's data sets (Hippocampus, Neocortex, Polymer; Table 2) are not
available; the volumes below take only their resolution, segment count, anisotropy (1:1:7,
L277) and background share.

Generator: ``u64(seed, stream, i) = splitmix64(splitmix64((seed << 32) ^ stream) + i)``;
floats are the top 24 bits / 2^24 (exactly representable in fp32, in [0, 1)).
All volume arithmetic is exact integer arithmetic so that a GPU implementation of the same
recipe (``csrc/synth_kernels.cu``) is bit-identical; tests compare the two on crops.
"""

from __future__ import annotations

import numpy as np

_U64 = np.uint64
_GOLD = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)


def splitmix64(x):
    """One splitmix64 step (add the golden constant, then the finaliser) on uint64 arrays."""
    with np.errstate(over="ignore"):
        z = np.asarray(x, dtype=_U64) + _GOLD
        z = (z ^ (z >> _U64(30))) * _M1
        z = (z ^ (z >> _U64(27))) * _M2
        return z ^ (z >> _U64(31))


def stream_key(seed: int, stream: int) -> np.uint64:
    return splitmix64(np.array([(int(seed) << 32) ^ int(stream)], dtype=_U64))[0]


def u64(seed: int, stream: int, i) -> np.ndarray:
    """Counter-based draw number ``i`` (array or scalar) of stream ``stream`` of ``seed``."""
    key = stream_key(seed, stream)
    with np.errstate(over="ignore"):
        return splitmix64(key + np.asarray(i, dtype=_U64))


def uniform01(seed: int, stream: int, i) -> np.ndarray:
    """fp32 in [0,1): top 24 bits of the 64-bit draw / 2^24."""
    return ((u64(seed, stream, i) >> _U64(40)).astype(np.float32)) * np.float32(1.0 / (1 << 24))


# ----------------------------------------------------------------------------------------------
# transfer functions
# ----------------------------------------------------------------------------------------------

def random_tf(n_segments: int, seed: int, update: int = 0, alpha_zero_frac: float = 0.0) -> np.ndarray:
    """fp32 [n_segments, 4] uniform RGBA in [0,1) (configs 1-5).

    ``update`` selects an independent TF (config 2: "100 consecutive random TF updates").
    ``alpha_zero_frac`` > 0 zeroes ONLY the A channel of the segments whose extra draw is below
    it (config 3: 30 % of segments alpha = 0)."""
    i = np.arange(n_segments * 4, dtype=np.uint64)
    tf = uniform01(seed, 100 + 2 * update, i).reshape(n_segments, 4).copy()
    if alpha_zero_frac > 0.0:
        extra = uniform01(seed, 101 + 2 * update, np.arange(n_segments, dtype=np.uint64))
        tf[extra < np.float32(alpha_zero_frac), 3] = 0.0
    return tf


def random_attr(n_segments: int, n_channels: int, seed: int, lo: float = 0.0, hi: float = 1.0) -> np.ndarray:
    """fp32 [n_segments, n_channels] uniform in [lo, hi): a generic per-segment attribute
    (opacity alone, light contributions, K batched TFs as 4 K channels; NEXT-1)."""
    i = np.arange(n_segments * n_channels, dtype=np.uint64)
    u = uniform01(seed, 300 + n_channels, i).reshape(n_segments, n_channels)
    return (np.float32(lo) + u * np.float32(hi - lo)).astype(np.float32)


def orbit_view(dims_xyz, spacing=(1.0, 1.0, 1.0), azimuth_deg: float = 30.0, elevation_deg: float = 20.0,
               distance: float = 1.6, fov_deg: float = 40.0, width: int = 64, height: int = 48,
               step_voxels: float = 0.5, ref_step_voxels: float = 1.0, lod_bias: float = 0.0,
               ess_threshold: float = 1e-8, alpha_cutoff: float = 1.0) -> dict:
    """A pinhole view of the volume for the ray-marcher (NEXT-2): the eye orbits the volume's centre at
    ``distance`` x the box diagonal, looking at the centre.  Pure input construction (an orthonormal
    camera basis); the meaning of every field is defined by the renderer (include/mg.h, oracle R1-R6).
    The paper renders 1600 x 1200 at 0.5-voxel steps (L414) with an ESS threshold of 1e-8 (L271)."""
    ext = np.asarray(dims_xyz, dtype=np.float64) * np.asarray(spacing, dtype=np.float64)
    centre = 0.5 * ext
    az, el = np.deg2rad(azimuth_deg), np.deg2rad(elevation_deg)
    back = np.array([np.cos(el) * np.cos(az), np.cos(el) * np.sin(az), np.sin(el)])
    eye = centre + back * distance * float(np.linalg.norm(ext))
    forward = -back
    world_up = np.array([0.0, 0.0, 1.0]) if abs(back[2]) < 0.99 else np.array([0.0, 1.0, 0.0])
    right = np.cross(forward, world_up)
    right /= np.linalg.norm(right)
    up = np.cross(right, forward)
    return dict(width=int(width), height=int(height), eye=eye, right=right, up=up, forward=forward,
                tan_half_fov=float(np.tan(np.deg2rad(fov_deg) / 2)), spacing=np.asarray(spacing, dtype=np.float64),
                step_voxels=float(step_voxels), ref_step_voxels=float(ref_step_voxels), lod_bias=float(lod_bias),
                ess_threshold=float(ess_threshold), alpha_cutoff=float(alpha_cutoff))


RENDER_ALPHA_SCALE = 0.04      # render inputs: TF opacities scaled so that rays travel ~25+ voxels before saturating


def render_view(c: dict, width: int = 1600, height: int = 1200, **overrides) -> dict:
    """The view bench.py and the full-size parity test render a config with: the paper's 1600 x 1200
    viewport at 0.5-voxel steps (L414), ESS threshold 1e-8 (L271), voxel spacing 1 : 1 : zscale (L277),
    the volume filling most of the frame."""
    kw = dict(azimuth_deg=35.0, elevation_deg=30.0, distance=0.75, fov_deg=45.0)
    kw.update(overrides)
    v = orbit_view(c["dims"], spacing=(1.0, 1.0, float(c.get("zscale", 1))), width=width, height=height, **kw)
    v["flags"] = 1          # MG_VIEW_HISTOGRAM_MIPMAP: the configs' mipmaps come from the builder
    return v


def render_tf(tf: np.ndarray) -> np.ndarray:
    """The config's TF with its opacities scaled by RENDER_ALPHA_SCALE (exact zeros stay zero)."""
    out = tf.copy()
    out[:, 3] *= np.float32(RENDER_ALPHA_SCALE)
    return out


def query_boxes(dims_xyz, side: int, n: int, seed: int) -> list:
    """``n`` randomly aligned range queries of (up to) side^3 voxels inside the volume (Table 4: "randomly-
    aligned range queries covering between 16^3 to 256^3 voxels"): [x0, y0, z0, x1, y1, z1], half-open.  An
    axis shorter than ``side`` is covered whole."""
    out = []
    for q in range(n):
        r = u64(seed, 600 + side, np.arange(3 * q, 3 * q + 3, dtype=np.uint64))
        ext = [min(int(side), int(d)) for d in dims_xyz]
        lo = [int(r[a] % np.uint64(int(dims_xyz[a]) - ext[a] + 1)) for a in range(3)]
        out.append(lo + [lo[a] + ext[a] for a in range(3)])
    return out


def single_segment_update(tf: np.ndarray, seed: int, update: int) -> np.ndarray:
    """Config 4: each update re-draws ONE random segment's RGBA; returns a new array."""
    out = tf.copy()
    n = tf.shape[0]
    s = int(u64(seed, 200, update) % _U64(n))
    out[s] = uniform01(seed, 201, np.arange(4 * update, 4 * update + 4, dtype=np.uint64))
    return out


# ----------------------------------------------------------------------------------------------
# Voronoi segmentations (configs 1-3)
# ----------------------------------------------------------------------------------------------

def voronoi_seeds(dims_xyz, n_seeds: int, seed: int) -> np.ndarray:
    """``n_seeds`` DISTINCT integer points, int32 [n_seeds, 3] as (x, y, z)."""
    X, Y, Z = (int(d) for d in dims_xyz)
    if n_seeds > X * Y * Z:
        raise ValueError("more seeds than voxels")
    pts, seen, c = [], set(), 0
    while len(pts) < n_seeds:
        r = u64(seed, 1, np.arange(3 * c, 3 * c + 3, dtype=np.uint64))
        p = (int(r[0] % _U64(X)), int(r[1] % _U64(Y)), int(r[2] % _U64(Z)))
        c += 1
        if p not in seen:
            seen.add(p)
            pts.append(p)
    return np.asarray(pts, dtype=np.int32)


def voxel_jitter(seed: int, lin: np.ndarray, amp: int):
    """Per-voxel jitter in {-amp..amp}^3 from a hash of the linear voxel index (config 2)."""
    h = u64(seed, 2, lin)
    m = _U64(2 * amp + 1)
    jx = (h % m).astype(np.int64) - amp
    jy = ((h >> _U64(16)) % m).astype(np.int64) - amp
    jz = ((h >> _U64(32)) % m).astype(np.int64) - amp
    return jx, jy, jz


def voronoi_volume(dims_xyz, seeds_xyz: np.ndarray, zscale: int = 1, jitter: int = 0,
                   seed: int = 0, region=None) -> np.ndarray:
    """uint32 [Z, Y, X] (x fastest): label = argmin_k dx^2 + dy^2 + (zscale*dz)^2 in exact integer
    arithmetic, ties -> lowest seed index.  With ``jitter`` > 0 the query point of voxel x is
    clamp(x + j(x)) (config 2's "3-voxel boundary jitter").  ``region`` = (z0, z1, y0, y1, x0, x1)
    evaluates only that sub-box (global coordinates), for crop checks of the GPU generator."""
    X, Y, Z = (int(d) for d in dims_xyz)
    z0, z1, y0, y1, x0, x1 = region if region is not None else (0, Z, 0, Y, 0, X)
    sx = seeds_xyz[:, 0].astype(np.int64)[:, None, None]
    sy = seeds_xyz[:, 1].astype(np.int64)[:, None, None]
    sz = seeds_xyz[:, 2].astype(np.int64)[:, None, None]
    out = np.empty((z1 - z0, y1 - y0, x1 - x0), dtype=np.uint32)
    yy, xx = np.meshgrid(np.arange(y0, y1, dtype=np.int64), np.arange(x0, x1, dtype=np.int64),
                         indexing="ij")
    for z in range(z0, z1):
        qx, qy, qz = xx, yy, np.full_like(xx, z)
        if jitter > 0:
            lin = ((z * Y + yy) * X + xx).astype(np.uint64)
            jx, jy, jz = voxel_jitter(seed, lin, jitter)
            qx = np.clip(xx + jx, 0, X - 1)
            qy = np.clip(yy + jy, 0, Y - 1)
            qz = np.clip(qz + jz, 0, Z - 1)
        d = (qx[None] - sx) ** 2 + (qy[None] - sy) ** 2 + (zscale * (qz[None] - sz)) ** 2
        out[z - z0] = np.argmin(d, axis=0).astype(np.uint32)   # first minimum = lowest index
    return out


# ----------------------------------------------------------------------------------------------
# random cylinders over background 0 (config 4)
# ----------------------------------------------------------------------------------------------

def cylinder_params(dims_xyz, n_cyl: int, seed: int) -> np.ndarray:
    """int64 [n_cyl, 8]: cx, cy, cz, ax, ay, az, r16, L.

    Centre uniform in the box (integer voxel); axis = an integer vector drawn uniformly from the
    ball 0 < |a|^2 <= 1024^2 by rejection (=> direction uniform on the sphere, integers only);
    radius r = r16/16 in [2, 5] voxels; length L in [20, 200] voxels, flat caps."""
    X, Y, Z = (int(d) for d in dims_xyz)
    out = np.empty((n_cyl, 8), dtype=np.int64)
    c = 0
    for k in range(n_cyl):
        r = u64(seed, 3, np.arange(5 * k, 5 * k + 5, dtype=np.uint64))
        out[k, 0] = int(r[0] % _U64(X))
        out[k, 1] = int(r[1] % _U64(Y))
        out[k, 2] = int(r[2] % _U64(Z))
        out[k, 6] = 32 + int(r[3] % _U64(49))       # 32..80 sixteenths = 2..5 voxels
        out[k, 7] = 20 + int(r[4] % _U64(181))      # 20..200 voxels
        while True:
            a = u64(seed, 4, np.arange(3 * c, 3 * c + 3, dtype=np.uint64))
            c += 1
            ax, ay, az = (int(v % _U64(2049)) - 1024 for v in a)
            n2 = ax * ax + ay * ay + az * az
            if 0 < n2 <= 1024 * 1024:
                out[k, 3:6] = (ax, ay, az)
                break
    return out


def cylinder_volume(dims_xyz, params: np.ndarray, region=None) -> np.ndarray:
    """uint32 [Z, Y, X]: voxel p belongs to cylinder k (label k+1) iff, with d = p - c, t = d.a:
    4 t^2 <= L^2 |a|^2  and  256 (|d|^2 |a|^2 - t^2) <= r16^2 |a|^2   (exact int64);
    later cylinders overwrite earlier ones; everything else is background 0."""
    X, Y, Z = (int(d) for d in dims_xyz)
    z0, z1, y0, y1, x0, x1 = region if region is not None else (0, Z, 0, Y, 0, X)
    out = np.zeros((z1 - z0, y1 - y0, x1 - x0), dtype=np.uint32)
    for k in range(params.shape[0]):
        cx, cy, cz, ax, ay, az, r16, L = (int(v) for v in params[k])
        a2 = ax * ax + ay * ay + az * az
        nrm = float(a2) ** 0.5
        r = r16 / 16.0
        ext = [int(0.5 * L * abs(a) / nrm + r) + 2 for a in (ax, ay, az)]   # conservative bbox
        bx0, bx1 = max(x0, cx - ext[0]), min(x1, cx + ext[0] + 1)
        by0, by1 = max(y0, cy - ext[1]), min(y1, cy + ext[1] + 1)
        bz0, bz1 = max(z0, cz - ext[2]), min(z1, cz + ext[2] + 1)
        if bx0 >= bx1 or by0 >= by1 or bz0 >= bz1:
            continue
        dz, dy, dx = np.meshgrid(np.arange(bz0, bz1, dtype=np.int64) - cz,
                                 np.arange(by0, by1, dtype=np.int64) - cy,
                                 np.arange(bx0, bx1, dtype=np.int64) - cx, indexing="ij")
        t = dx * ax + dy * ay + dz * az
        d2 = dx * dx + dy * dy + dz * dz
        inside = (4 * t * t <= L * L * a2) & (256 * (d2 * a2 - t * t) <= r16 * r16 * a2)
        sub = out[bz0 - z0:bz1 - z0, by0 - y0:by1 - y0, bx0 - x0:bx1 - x0]
        sub[inside] = k + 1
    return out


# ----------------------------------------------------------------------------------------------
# config 5: synthetic DAG stress + random node-index volume
# ----------------------------------------------------------------------------------------------

def random_dag_levels(level_sizes, seed: int):
    """Random binary-lerp DAG with the given number of nodes per topological level
    (level_sizes[0] = number of leaves).  ``child_a`` is uniform in level L-1 (so the topological
    level of the node is exactly L), ``child_b`` uniform over all levels < L, redrawn (next
    stream) while equal to ``child_a``; ``weight`` = fp32 U(0,1) with 0 excluded.
    Returns (child_a u32, child_b u32, weight f32, level_offsets u64 [n_levels+1]); entries of
    the leaves in child/weight are 0."""
    n_levels = len(level_sizes)
    off = np.zeros(n_levels + 1, dtype=np.uint64)
    off[1:] = np.cumsum(np.asarray(level_sizes, dtype=np.uint64))
    n_nodes = int(off[-1])
    a = np.zeros(n_nodes, dtype=np.uint32)
    b = np.zeros(n_nodes, dtype=np.uint32)
    w = np.zeros(n_nodes, dtype=np.float32)
    for L in range(1, n_levels):
        lo, hi = int(off[L]), int(off[L + 1])
        plo = int(off[L - 1])
        idx = np.arange(lo, hi, dtype=np.uint64)
        ca = (u64(seed, 10, idx) % _U64(lo - plo)).astype(np.int64) + plo
        cb = (u64(seed, 11, idx) % _U64(lo)).astype(np.int64)
        rnd = 1
        while True:
            eq = np.nonzero(cb == ca)[0]
            if eq.size == 0:
                break
            cb[eq] = (u64(seed, 11 + 16 * rnd, idx[eq]) % _U64(lo)).astype(np.int64)
            rnd += 1
        ww = uniform01(seed, 12, idx)
        ww[ww == 0.0] = np.float32(2.0 ** -24)
        a[lo:hi], b[lo:hi], w[lo:hi] = ca, cb, ww
    return a, b, w, off


def random_dag(n_nodes: int, n_levels: int, n_leaves: int, seed: int):
    """Config 5 recipe at any size: level 0 = ``n_leaves`` leaves; levels 1..n_levels-1 share the
    remaining nodes equally (the remainder goes to the last level).  See random_dag_levels."""
    per = (n_nodes - n_leaves) // (n_levels - 1)
    sizes = [n_leaves] + [per] * (n_levels - 1)
    sizes[-1] += n_nodes - sum(sizes)
    return random_dag_levels(sizes, seed)


def random_node_idx(n_voxels: int, n_nodes: int, seed: int, chunk: int = 1 << 24) -> np.ndarray:
    """uint32 [n_voxels] uniform in [0, n_nodes) (config 5's 512^3 volume)."""
    out = np.empty(n_voxels, dtype=np.uint32)
    for s in range(0, n_voxels, chunk):
        e = min(n_voxels, s + chunk)
        out[s:e] = (u64(seed, 20, np.arange(s, e, dtype=np.uint64)) % _U64(n_nodes)).astype(np.uint32)
    return out


# ----------------------------------------------------------------------------------------------
# the five BASELINE.json configs
# ----------------------------------------------------------------------------------------------

CONFIGS = {
    1: dict(name="cfg1_64cube_16seg", dims=(64, 64, 64), n_segments=16, seed=1, kind="voronoi",
            zscale=1, jitter=0, alpha_zero_frac=0.0),
    # tf_sequence / n_updates: the TF-update sequence BASELINE.json names for the config (Workload.tf(u) is update u of it):
    # "random" = an independent TF per update (config 2: "100 consecutive random TF updates"), "single_segment" = update u
    # re-draws one random segment of update u - 1 (config 4: "per-update TF changes one random segment").
    # quant_bits: the builder's weight bitrate for this config when the caller names none: the smallest b whose quantised
    # graph stays inside north_star's 2e-3 of the direct histogram colour on EVERY voxel of every level at full size.  The
    # paper's b = 9 (L305) does on config 3 (1.85e-3); on config 2 it reaches 2.20e-3 (level 3; the per-level samples of
    # earlier rounds had shown 1.63e-3) and on config 4, whose 15,918-component root sits 14 lerps deep, 2.05e-3 -- both
    # run at b = 10 (Table 2's max l1 error 0.005 at b = 9 allows 2.5e-3 in colour).
    2: dict(name="cfg2_hippocampus_shaped", dims=(1178, 1125, 789), n_segments=353, seed=2,
            kind="voronoi", zscale=1, jitter=3, alpha_zero_frac=0.0, quant_bits=10, tf_sequence="random", n_updates=100),
    3: dict(name="cfg3_neocortex_shaped", dims=(2048, 2048, 300), n_segments=1182, seed=3,
            kind="voronoi", zscale=7, jitter=0, alpha_zero_frac=0.3, tf_sequence="random", n_updates=100),
    4: dict(name="cfg4_polymer_shaped", dims=(614, 961, 600), n_segments=15917, seed=4,
            kind="cylinders", alpha_zero_frac=0.0, quant_bits=10, tf_sequence="single_segment", n_updates=100),
    5: dict(name="cfg5_dag_stress", n_nodes=1 << 26, n_levels=24, n_leaves=1 << 14, seed=5,
            kind="dag", volume_voxels=512 ** 3),
}


def scaled_config(cfg: int, scale: float) -> dict:
    """A geometrically similar, smaller instance of config 2-4 (dims * scale, segment count
    * scale^3, at least 4) for CPU-sized tests; scale = 1 returns the config itself."""
    c = dict(CONFIGS[cfg])
    if scale != 1.0:
        c["dims"] = tuple(max(2, int(round(d * scale))) for d in c["dims"])
        c["n_segments"] = max(4, int(round(c["n_segments"] * scale ** 3)))
        c["name"] += f"_x{scale:g}"
    return c


def make_volume(c: dict, region=None) -> np.ndarray:
    """The uint32 segmentation volume [Z, Y, X] of a (possibly scaled) config dict, on the CPU."""
    if c["kind"] == "voronoi":
        seeds = voronoi_seeds(c["dims"], c["n_segments"], c["seed"])
        return voronoi_volume(c["dims"], seeds, c["zscale"], c["jitter"], c["seed"], region)
    if c["kind"] == "cylinders":
        return cylinder_volume(c["dims"], cylinder_params(c["dims"], c["n_segments"], c["seed"]), region)
    raise ValueError(c["kind"])
