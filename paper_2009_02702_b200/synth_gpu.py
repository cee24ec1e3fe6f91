"""GPU versions of the synth.py volume generators (ctypes binding of libmg_synth.so).

Input generation only -- none of the method's arithmetic.  The recipes, the counter-based
generator and the exact integer predicates are those of ``synth.py``; the results are
bit-identical (tests/test_synth_gpu.py compares crops).  Needed because configs 2-4 take ~10^12
distance evaluations at full size.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import synth

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmg_synth.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2009_02702_b200.build`")
lib = C.CDLL(LIB_PATH)

_vp = C.c_void_p
lib.mgs_voronoi.argtypes = [_vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_uint64,
                            _vp, _vp, _vp]
lib.mgs_voronoi.restype = C.c_int
lib.mgs_cylinders.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp]
lib.mgs_cylinders.restype = C.c_int
lib.mgs_tile_size.argtypes = []
lib.mgs_tile_size.restype = C.c_int

SYMBOLS = ["mgs_voronoi", "mgs_cylinders", "mgs_tile_size"]


def _region(dims_xyz, region):
    X, Y, Z = (int(d) for d in dims_xyz)
    r = region if region is not None else (0, Z, 0, Y, 0, X)
    return np.asarray(r, dtype=np.int32)


def voronoi_volume(dims_xyz, seeds_xyz: np.ndarray, zscale: int = 1, jitter: int = 0, seed: int = 0,
                   region=None, device="cuda"):
    """torch uint32-valued int32 tensor [Z, Y, X] on ``device``; same result as synth.voronoi_volume."""
    import torch
    X, Y, Z = (int(d) for d in dims_xyz)
    reg = _region(dims_xyz, region)
    s4 = np.zeros((seeds_xyz.shape[0], 4), dtype=np.int32)
    s4[:, :3] = seeds_xyz
    d_seeds = torch.from_numpy(s4).to(device)
    shape = (int(reg[1] - reg[0]), int(reg[3] - reg[2]), int(reg[5] - reg[4]))
    out = torch.empty(shape, dtype=torch.int32, device=device)
    key = int(synth.stream_key(seed, 2))
    rc = lib.mgs_voronoi(d_seeds.data_ptr(), s4.shape[0], X, Y, Z, int(zscale), int(jitter), key,
                         reg.ctypes.data, out.data_ptr(), torch.cuda.current_stream().cuda_stream or None)
    if rc != 0:
        raise RuntimeError(f"mgs_voronoi failed: cudaError {-rc}")
    return out


def cylinder_tiles(params: np.ndarray, reg: np.ndarray, tile: int):
    """CSR lists (tile -> ascending cylinder numbers) from conservative bounding boxes."""
    z0, z1, y0, y1, x0, x1 = (int(v) for v in reg)
    tx, ty, tz = (-(-(x1 - x0) // tile), -(-(y1 - y0) // tile), -(-(z1 - z0) // tile))
    p = params.astype(np.float64)
    nrm = np.sqrt(p[:, 3] ** 2 + p[:, 4] ** 2 + p[:, 5] ** 2)
    r = p[:, 6] / 16.0
    tiles, cyls = [], []
    for k in range(params.shape[0]):
        ext = [int(0.5 * p[k, 7] * abs(p[k, 3 + d]) / nrm[k] + r[k]) + 2 for d in range(3)]
        lo = [int(params[k, d]) - ext[d] for d in range(3)]
        hi = [int(params[k, d]) + ext[d] for d in range(3)]
        bx0, bx1 = max(x0, lo[0]) - x0, min(x1 - 1, hi[0]) - x0
        by0, by1 = max(y0, lo[1]) - y0, min(y1 - 1, hi[1]) - y0
        bz0, bz1 = max(z0, lo[2]) - z0, min(z1 - 1, hi[2]) - z0
        if bx0 > bx1 or by0 > by1 or bz0 > bz1:
            continue
        gx = np.arange(bx0 // tile, bx1 // tile + 1)
        gy = np.arange(by0 // tile, by1 // tile + 1)
        gz = np.arange(bz0 // tile, bz1 // tile + 1)
        t = (gz[:, None, None] * ty + gy[None, :, None]) * tx + gx[None, None, :]
        tiles.append(t.reshape(-1))
        cyls.append(np.full(t.size, k, dtype=np.uint32))
    n_tiles = tx * ty * tz
    off = np.zeros(n_tiles + 1, dtype=np.uint32)
    if not tiles:
        return off, np.zeros(1, dtype=np.uint32)
    tiles = np.concatenate(tiles)
    cyls = np.concatenate(cyls)
    order = np.argsort(tiles, kind="stable")          # stable: cylinders stay ascending inside a tile
    off[1:] = np.cumsum(np.bincount(tiles, minlength=n_tiles))
    return off, cyls[order]


def cylinder_volume(dims_xyz, params: np.ndarray, region=None, device="cuda"):
    """torch int32 tensor [Z, Y, X] on ``device``; same result as synth.cylinder_volume."""
    import torch
    reg = _region(dims_xyz, region)
    off, lst = cylinder_tiles(params, reg, lib.mgs_tile_size())
    d_par = torch.from_numpy(np.ascontiguousarray(params, dtype=np.int64)).to(device)
    d_off = torch.from_numpy(off.view(np.int32)).to(device)
    d_lst = torch.from_numpy(lst.view(np.int32)).to(device)
    shape = (int(reg[1] - reg[0]), int(reg[3] - reg[2]), int(reg[5] - reg[4]))
    out = torch.empty(shape, dtype=torch.int32, device=device)
    rc = lib.mgs_cylinders(d_par.data_ptr(), d_off.data_ptr(), d_lst.data_ptr(), reg.ctypes.data, out.data_ptr(),
                           torch.cuda.current_stream().cuda_stream or None)
    if rc != 0:
        raise RuntimeError(f"mgs_cylinders failed: cudaError {-rc}")
    torch.cuda.current_stream().synchronize()          # d_par / d_off / d_lst go out of scope
    return out


def make_volume(c: dict, region=None, device="cuda"):
    """GPU counterpart of synth.make_volume."""
    if c["kind"] == "voronoi":
        seeds = synth.voronoi_seeds(c["dims"], c["n_segments"], c["seed"])
        return voronoi_volume(c["dims"], seeds, c["zscale"], c["jitter"], c["seed"], region, device)
    if c["kind"] == "cylinders":
        return cylinder_volume(c["dims"], synth.cylinder_params(c["dims"], c["n_segments"], c["seed"]), region, device)
    raise ValueError(c["kind"])
