"""ctypes binding of the host-side graph builder (include/mg_builder.h): argument marshalling only.

Histogram mipmap (a0), factorisation + node re-use + quantisation (a1) and topological relabelling
(a2) all run in libmg_builder.so (host C++/OpenMP); nothing here computes.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmg_builder.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2009_02702_b200.build`")
lib = C.CDLL(LIB_PATH)

MGB_OK = 0
PICK_SMALLEST_INDEX, PICK_SMALLEST_MASS = 0, 1

SYMBOLS = ["mgb_default_params", "mgb_build", "mgb_build_from_level1", "mgb_build_from_levels", "mgb_get_front_mixture_nodes",
           "mgb_build_from_mixtures", "mgb_free", "mgb_get_info",
           "mgb_mip_dims", "mgb_mip_chain", "mgb_get_graph", "mgb_node_idx_ptr", "mgb_get_node_idx", "mgb_get_codebook",
           "mgb_get_weight_sigma", "mgb_last_error"]


class Params(C.Structure):
    _fields_ = [("quant_bits", C.c_uint32), ("tau", C.c_uint32), ("big_cutoff", C.c_uint32),
                ("pick_order", C.c_uint32), ("n_threads", C.c_uint32), ("relabel", C.c_uint32),
                ("phi2_exact_budget", C.c_uint64)]


class Info(C.Structure):
    _fields_ = [("dims", C.c_uint64 * 3), ("n_mip_levels", C.c_uint32), ("n_leaves", C.c_uint32),
                ("n_voxels_total", C.c_uint64), ("n_nodes", C.c_uint64), ("depth", C.c_uint32),
                ("quant_bits", C.c_uint32), ("n_distinct_mixtures", C.c_uint64), ("nnz_total", C.c_uint64),
                ("n_stage1", C.c_uint64), ("n_stage2", C.c_uint64), ("n_big", C.c_uint64),
                ("phi2_exact", C.c_uint32), ("reserved", C.c_uint32), ("max_bin_sigma", C.c_double),
                ("seconds_mipmap", C.c_double), ("seconds_factorise", C.c_double),
                ("seconds_finalise", C.c_double)]


_vp = C.c_void_p
lib.mgb_default_params.argtypes = [C.POINTER(Params)]
lib.mgb_default_params.restype = None
lib.mgb_build.argtypes = [_vp, C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(Params), C.POINTER(_vp)]
lib.mgb_build.restype = C.c_int
lib.mgb_build_from_mixtures.argtypes = [C.c_uint32, C.c_uint64, _vp, _vp, _vp, C.POINTER(Params), C.POINTER(_vp)]
lib.mgb_build_from_mixtures.restype = C.c_int
lib.mgb_free.argtypes = [_vp]
lib.mgb_free.restype = None
lib.mgb_get_info.argtypes = [_vp, C.POINTER(Info)]
lib.mgb_get_info.restype = C.c_int
lib.mgb_mip_dims.argtypes = [_vp, _vp]
lib.mgb_mip_dims.restype = C.c_int
lib.mgb_mip_chain.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, _vp, C.c_uint32]
lib.mgb_mip_chain.restype = C.c_uint32
lib.mgb_get_graph.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp]
lib.mgb_get_graph.restype = C.c_int
lib.mgb_node_idx_ptr.argtypes = [_vp, C.c_uint32]
lib.mgb_node_idx_ptr.restype = _vp
lib.mgb_get_node_idx.argtypes = [_vp, C.c_uint32, _vp]
lib.mgb_get_node_idx.restype = C.c_int
lib.mgb_build_from_level1.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, _vp, C.c_uint32, _vp, _vp, _vp, C.c_uint64,
                                      C.POINTER(Params), C.POINTER(_vp)]
lib.mgb_build_from_level1.restype = C.c_int
lib.mgb_build_from_levels.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, _vp, C.c_uint32, C.c_uint32, _vp, C.c_uint64, _vp, _vp, _vp, _vp,
                                      _vp, _vp, C.c_uint64, C.c_uint64, C.POINTER(Params), C.POINTER(_vp)]
lib.mgb_build_from_levels.restype = C.c_int
lib.mgb_get_front_mixture_nodes.argtypes = [_vp, _vp]
lib.mgb_get_front_mixture_nodes.restype = C.c_int
lib.mgb_get_weight_sigma.argtypes = [_vp, _vp]
lib.mgb_get_weight_sigma.restype = C.c_int
lib.mgb_get_codebook.argtypes = [_vp, _vp, _vp, _vp]
lib.mgb_get_codebook.restype = C.c_int
lib.mgb_last_error.argtypes = []
lib.mgb_last_error.restype = C.c_char_p


class BuilderError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where} failed with {code}: {lib.mgb_last_error().decode()}")


def _check(rc: int, where: str) -> None:
    if rc != MGB_OK:
        raise BuilderError(rc, where)


def mip_chain(dims_xyz) -> list:
    """[(X_l, Y_l, Z_l)] of the mipmap of a volume that has not been built yet (mgb_mip_chain: the rule of L80)."""
    d = np.zeros(3 * 64, dtype=np.uint64)
    n = int(lib.mgb_mip_chain(int(dims_xyz[0]), int(dims_xyz[1]), int(dims_xyz[2]), d.ctypes.data, 64))
    return [tuple(int(v) for v in d[3 * l:3 * l + 3]) for l in range(n)]


def default_params(**overrides) -> Params:
    p = Params()
    lib.mgb_default_params(C.byref(p))
    for k, v in overrides.items():
        if not hasattr(p, k):
            raise TypeError(f"unknown builder parameter {k!r}")
        setattr(p, k, v)
    return p


class Result:
    """Handle of a built Mixture Graph (mgb_build ... mgb_free)."""

    def __init__(self, handle):
        self._h = handle
        self.info = Info()
        _check(lib.mgb_get_info(self._h, C.byref(self.info)), "mgb_get_info")
        d = np.zeros(3 * self.info.n_mip_levels, dtype=np.uint64)
        _check(lib.mgb_mip_dims(self._h, d.ctypes.data), "mgb_mip_dims")
        self.mip_dims = [tuple(int(v) for v in d[3 * l:3 * l + 3]) for l in range(self.info.n_mip_levels)]

    def close(self) -> None:
        if self._h is not None:
            lib.mgb_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def graph(self) -> dict:
        """child_a, child_b (u32), weight (f32), weight_exact (f64), level_offsets (u64), leaf_segment_id."""
        n = int(self.info.n_nodes)
        out = dict(child_a=np.zeros(n, np.uint32), child_b=np.zeros(n, np.uint32), weight=np.zeros(n, np.float32),
                   weight_exact=np.zeros(n, np.float64), level_offsets=np.zeros(self.info.depth + 2, np.uint64),
                   leaf_segment_id=np.zeros(self.info.n_leaves, np.uint32))
        _check(lib.mgb_get_graph(self._h, *(out[k].ctypes.data for k in
                                            ("child_a", "child_b", "weight", "weight_exact", "level_offsets",
                                             "leaf_segment_id"))), "mgb_get_graph")
        out["n_leaves"] = int(self.info.n_leaves)
        out["weight_sigma"] = np.zeros(n, np.float32)
        _check(lib.mgb_get_weight_sigma(self._h, out["weight_sigma"].ctypes.data), "mgb_get_weight_sigma")
        return out

    def n_voxels(self, level: int) -> int:
        x, y, z = self.mip_dims[level]
        return x * y * z

    def node_idx(self, level: int, copy: bool = True) -> np.ndarray:
        """uint32 [Z_l, Y_l, X_l]; copy=False returns a view of the builder-owned array (valid until close())."""
        x, y, z = self.mip_dims[level]
        n = x * y * z
        if copy:
            out = np.zeros(n, dtype=np.uint32)
            _check(lib.mgb_get_node_idx(self._h, level, out.ctypes.data), "mgb_get_node_idx")
        else:
            p = lib.mgb_node_idx_ptr(self._h, level)
            if not p:
                raise BuilderError(-1, "mgb_node_idx_ptr")
            out = np.ctypeslib.as_array(C.cast(p, C.POINTER(C.c_uint32)), shape=(n,))
        return out.reshape(z, y, x)

    def codebook(self):
        nb = 1 << int(self.info.quant_bits)
        cw, sg, cnt = np.zeros(nb, np.float32), np.zeros(nb, np.float32), np.zeros(nb, np.uint64)
        _check(lib.mgb_get_codebook(self._h, cw.ctypes.data, sg.ctypes.data, cnt.ctypes.data), "mgb_get_codebook")
        return cw, sg, cnt


def build(seg: np.ndarray, params: Params | None = None, **overrides) -> Result:
    """Build from a uint32 segment-ID volume [Z, Y, X]."""
    seg = np.ascontiguousarray(seg, dtype=np.uint32)
    if seg.ndim != 3:
        raise ValueError("seg must be [Z, Y, X]")
    p = params if params is not None else default_params(**overrides)
    h = _vp()
    Z, Y, X = seg.shape
    _check(lib.mgb_build(seg.ctypes.data, X, Y, Z, C.byref(p), C.byref(h)), "mgb_build")
    return Result(h)


def build_from_level1(dims_xyz, leaf_segment_id, level1, mixed_voxel, mixed_children, params: Params | None = None,
                      **overrides) -> Result:
    """Build from levels 0 / 1 classified by a front end (mg.mipmap_leaf_index + mg.mipmap_front_level1, or any
    equivalent): ``level1`` uint32 [Z_1, Y_1, X_1] (leaf number of a pure parent, 0xFFFFFFFF otherwise),
    ``mixed_voxel`` uint32 [n], ``mixed_children`` uint32 [n, 8].  Level 0's node index is not stored."""
    X, Y, Z = (int(d) for d in dims_xyz)
    ids = np.ascontiguousarray(leaf_segment_id, dtype=np.uint32)
    l1 = np.ascontiguousarray(level1, dtype=np.uint32).reshape(-1)
    mv = np.ascontiguousarray(mixed_voxel, dtype=np.uint32).reshape(-1)
    mc = np.ascontiguousarray(mixed_children, dtype=np.uint32).reshape(-1, 8)
    if mc.shape[0] != mv.size:
        raise ValueError("mixed_children must be [n_mixed, 8]")
    n1 = -(-X // 2) * -(-Y // 2) * -(-Z // 2)
    if (X, Y, Z) != (1, 1, 1) and l1.size != n1:
        raise ValueError(f"level1 must have {n1} voxels")
    p = params if params is not None else default_params(**overrides)
    h = _vp()
    _check(lib.mgb_build_from_level1(X, Y, Z, ids.ctypes.data, ids.size, l1.ctypes.data if l1.size else None,
                                     mv.ctypes.data if mv.size else None, mc.ctypes.data if mv.size else None, mv.size,
                                     C.byref(p), C.byref(h)), "mgb_build_from_level1")
    return Result(h)


def build_from_levels(dims_xyz, leaf_segment_id, level_done: int, handles, mixtures: dict, nnz_levels: int,
                      params: Params | None = None, **overrides):
    """Build from the levels 0 .. ``level_done`` of the histogram mipmap built elsewhere (mg.MixtureTable):
    ``handles`` uint32 of level ``level_done``, ``mixtures`` = MixtureTable.export().  Returns (Result, node_of_mixture
    uint32 [n listed mixtures])."""
    p = params if params is not None else default_params(**overrides)
    ids = np.ascontiguousarray(leaf_segment_id, dtype=np.uint32)
    h = np.ascontiguousarray(handles, dtype=np.uint32).reshape(-1)
    m = {k: np.ascontiguousarray(v) for k, v in mixtures.items()}
    X, Y, Z = (int(d) for d in dims_xyz)
    out = _vp()
    _check(lib.mgb_build_from_levels(X, Y, Z, ids.ctypes.data, ids.size, int(level_done), h.ctypes.data, m["k"].size,
                                     m["offset"].ctypes.data, m["k"].ctypes.data, m["tlog"].ctypes.data, m["first_pos"].ctypes.data,
                                     m["leaf"].ctypes.data, m["count"].ctypes.data, m["leaf"].size, int(nnz_levels), C.byref(p),
                                     C.byref(out)), "mgb_build_from_levels")
    r = Result(out)
    nodes = np.zeros(m["k"].size, dtype=np.uint32)
    _check(lib.mgb_get_front_mixture_nodes(out, nodes.ctypes.data), "mgb_get_front_mixture_nodes")
    return r, nodes


def build_from_mixtures(n_leaves: int, mixtures, params: Params | None = None, **overrides) -> Result:
    """``mixtures``: list of lists of (leaf, integer count)."""
    off = np.zeros(len(mixtures) + 1, dtype=np.uint64)
    leaf, cnt = [], []
    for m, e in enumerate(mixtures):
        for l, c in e:
            leaf.append(l)
            cnt.append(c)
        off[m + 1] = len(leaf)
    leaf = np.asarray(leaf, dtype=np.uint32)
    cnt = np.asarray(cnt, dtype=np.uint64)
    p = params if params is not None else default_params(**overrides)
    h = _vp()
    _check(lib.mgb_build_from_mixtures(int(n_leaves), len(mixtures), off.ctypes.data,
                                       leaf.ctypes.data if leaf.size else None,
                                       cnt.ctypes.data if cnt.size else None, C.byref(p), C.byref(h)),
           "mgb_build_from_mixtures")
    return Result(h)
