"""ctypes binding of the C-ABI library (include/mg.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used by callers for device
memory (``tensor.data_ptr()``) and streams (``torch.cuda.current_stream().cuda_stream``).  There is
no CPU fallback: if ``libmg.so`` is missing this module raises at import time.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmg.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2009_02702_b200.build` "
                      "(there is no CPU fallback for the CUDA path)")
lib = C.CDLL(LIB_PATH)

MG_OK, MG_ERR_INVALID_ARG, MG_ERR_INVALID_GRAPH, MG_ERR_CUDA, MG_ERR_OOM = 0, -1, -2, -3, -4
MG_RELABEL, MG_NO_PALETTES = 1, 2
MG_RGBA8, MG_RGBA16F, MG_BOTH, MG_FORCE_CONVERT, MG_PALETTE_FROM_LAST_PROPAGATE = 1, 2, 3, 16, 32
ALL_LEVELS = 0xFFFFFFFF

# every symbol include/mg.h declares (tests check that the library exports all of them)
SYMBOLS = ["mg_load_graph", "mg_free_graph", "mg_graph_info", "mg_level_offsets", "mg_node_permutation",
           "mg_relabel_indices", "mg_check_indices", "mg_propagate", "mg_propagate_host", "mg_colorize", "mg_tf_update_host",
           "mg_last_error", "mg_kernel_launch_count",
           "mg_bits_per_voxel", "mg_packed_stream_bytes", "mg_index_range", "mg_index_ranges_static", "mg_pack_indices",
           "mg_colorize_packed",
           "mg_propagate_attr", "mg_render", "mg_render_ex", "mg_ess_mask_build",
           "mg_mixture_lut_build", "mg_mixture_lut_free", "mg_mixture_lut_info", "mg_mixture_lut_export", "mg_range_query",
           "mg_mipmap_leaf_index", "mg_mipmap_front_level1", "mg_mipmap_levels_build", "mg_mipmap_levels_build_ex",
           "mg_mixture_table_free",
           "mg_mixture_table_info", "mg_mixture_table_export", "mg_mipmap_remap_handles"]


class MgInfo(C.Structure):
    _fields_ = [("n_nodes", C.c_uint64), ("n_internal", C.c_uint64), ("n_leaves", C.c_uint32),
                ("depth", C.c_uint32), ("n_topo_levels", C.c_uint32), ("first_fused_level", C.c_uint32),
                ("n_launches_propagate", C.c_uint32), ("relabelled", C.c_uint32), ("device_bytes", C.c_uint64)]


class MgPackedLevel(C.Structure):
    _fields_ = [("n_voxels", C.c_uint64), ("out_offset", C.c_uint64), ("byte_offset", C.c_uint64),
                ("bits", C.c_uint32), ("i_min", C.c_uint32)]


MG_MAX_PACKED_LEVELS = 32
_vp = C.c_void_p
lib.mg_load_graph.argtypes = [_vp, _vp, _vp, C.c_uint64, C.c_uint32, _vp, C.c_uint32, _vp, C.c_uint32, C.POINTER(_vp)]
lib.mg_load_graph.restype = C.c_int
lib.mg_free_graph.argtypes = [_vp]
lib.mg_free_graph.restype = None
lib.mg_graph_info.argtypes = [_vp, C.POINTER(MgInfo)]
lib.mg_graph_info.restype = C.c_int
lib.mg_level_offsets.argtypes = [_vp, _vp]
lib.mg_level_offsets.restype = C.c_int
lib.mg_node_permutation.argtypes = [_vp, _vp]
lib.mg_node_permutation.restype = C.c_int
lib.mg_relabel_indices.argtypes = [_vp, _vp, C.c_uint64, _vp]
lib.mg_relabel_indices.restype = C.c_int
lib.mg_check_indices.argtypes = [_vp, _vp, C.c_uint64, C.POINTER(C.c_uint64), _vp]
lib.mg_check_indices.restype = C.c_int
lib.mg_propagate.argtypes = [_vp, _vp, _vp, _vp]
lib.mg_propagate.restype = C.c_int
lib.mg_propagate_host.argtypes = [_vp, _vp, _vp, _vp]
lib.mg_propagate_host.restype = C.c_int
lib.mg_colorize.argtypes = [_vp, C.c_uint32, _vp, C.c_uint64, _vp, _vp, _vp, C.c_uint32, _vp]
lib.mg_colorize.restype = C.c_int
lib.mg_tf_update_host.argtypes = [_vp, _vp, _vp, _vp, C.c_uint64, _vp, _vp, C.c_uint32, _vp]
lib.mg_tf_update_host.restype = C.c_int
lib.mg_last_error.argtypes = []
lib.mg_last_error.restype = C.c_char_p
lib.mg_kernel_launch_count.argtypes = []
lib.mg_kernel_launch_count.restype = C.c_uint64


lib.mg_bits_per_voxel.argtypes = [C.c_uint32, C.c_uint32]
lib.mg_bits_per_voxel.restype = C.c_uint32
lib.mg_packed_stream_bytes.argtypes = [C.c_uint64, C.c_uint32]
lib.mg_packed_stream_bytes.restype = C.c_uint64
lib.mg_index_range.argtypes = [_vp, C.c_uint64, C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), _vp]
lib.mg_index_range.restype = C.c_int
MG_INDEX_RANGES_STATIC_MAX_LEVELS = 32
lib.mg_index_ranges_static.argtypes = [_vp, _vp, C.c_uint32, _vp, _vp, _vp]
lib.mg_index_ranges_static.restype = C.c_int
lib.mg_pack_indices.argtypes = [_vp, C.c_uint64, C.c_uint32, C.c_uint32, _vp, _vp]
lib.mg_pack_indices.restype = C.c_int
lib.mg_colorize_packed.argtypes = [_vp, _vp, C.POINTER(MgPackedLevel), C.c_uint32, _vp, _vp, _vp, C.c_uint32, _vp]
lib.mg_colorize_packed.restype = C.c_int


MG_MAX_ATTR_CHANNELS = 64
lib.mg_propagate_attr.argtypes = [_vp, _vp, _vp, C.c_uint32, _vp]
lib.mg_propagate_attr.restype = C.c_int


MG_MAX_MIP_LEVELS = 24
MG_VIEW_HISTOGRAM_MIPMAP = 1


class MgMipmapDesc(C.Structure):
    _fields_ = [("n_levels", C.c_uint32), ("reserved", C.c_uint32), ("level_offset", C.c_uint64 * MG_MAX_MIP_LEVELS),
                ("level_dim", (C.c_uint32 * 3) * MG_MAX_MIP_LEVELS)]


class MgView(C.Structure):
    _fields_ = [("eye", C.c_double * 3), ("right", C.c_double * 3), ("up", C.c_double * 3), ("forward", C.c_double * 3),
                ("tan_half_fov", C.c_double), ("spacing", C.c_double * 3), ("step_voxels", C.c_double),
                ("ref_step_voxels", C.c_double), ("lod_bias", C.c_double), ("ess_threshold", C.c_double),
                ("alpha_cutoff", C.c_double), ("width", C.c_uint32), ("height", C.c_uint32), ("flags", C.c_uint32),
                ("reserved", C.c_uint32)]


lib.mg_render.argtypes = [_vp, _vp, C.POINTER(MgMipmapDesc), _vp, C.POINTER(MgView), _vp, _vp, _vp]
lib.mg_render.restype = C.c_int


class MgRenderAux(C.Structure):
    _fields_ = [("ess_mask", _vp), ("reserved", _vp)]


lib.mg_render_ex.argtypes = [_vp, _vp, C.POINTER(MgMipmapDesc), _vp, C.POINTER(MgView), C.POINTER(MgRenderAux), _vp, _vp, _vp]
lib.mg_render_ex.restype = C.c_int
lib.mg_ess_mask_build.argtypes = [_vp, _vp, C.POINTER(MgMipmapDesc), _vp, C.c_double, _vp, _vp]
lib.mg_ess_mask_build.restype = C.c_int


class MgLutInfo(C.Structure):
    _fields_ = [("n_nodes", C.c_uint64), ("nnz", C.c_uint64), ("capacity", C.c_uint64), ("device_bytes", C.c_uint64),
                ("n_leaves", C.c_uint32), ("max_row_nnz", C.c_uint32)]


MG_QUERY_FA, MG_QUERY_NAIVE, MG_QUERY_FA_WALK = 0, 1, 2
lib.mg_mixture_lut_build.argtypes = [_vp, _vp, C.POINTER(_vp), _vp]
lib.mg_mixture_lut_build.restype = C.c_int
lib.mg_mixture_lut_free.argtypes = [_vp]
lib.mg_mixture_lut_free.restype = None
lib.mg_mixture_lut_info.argtypes = [_vp, C.POINTER(MgLutInfo)]
lib.mg_mixture_lut_info.restype = C.c_int
lib.mg_mixture_lut_export.argtypes = [_vp, _vp, _vp, _vp, _vp]
lib.mg_mixture_lut_export.restype = C.c_int
lib.mg_range_query.argtypes = [_vp, _vp, C.POINTER(MgMipmapDesc), _vp, C.c_uint32, _vp, _vp, _vp, C.c_uint32, _vp]
lib.mg_range_query.restype = C.c_int


lib.mg_mipmap_leaf_index.argtypes = [_vp, C.c_uint64, _vp, _vp, C.c_uint32, C.POINTER(C.c_uint32), _vp]
lib.mg_mipmap_leaf_index.restype = C.c_int
lib.mg_mipmap_front_level1.argtypes = [_vp, C.c_uint64, C.c_uint64, C.c_uint64, _vp, _vp, _vp, C.c_uint64,
                                       C.POINTER(C.c_uint64), _vp]
lib.mg_mipmap_front_level1.restype = C.c_int


class MgMixtureTableInfo(C.Structure):
    _fields_ = [("n_mixtures", C.c_uint64), ("n_entries", C.c_uint64), ("nnz_levels", C.c_uint64), ("device_bytes", C.c_uint64),
                ("levels_done", C.c_uint32), ("n_leaves", C.c_uint32)]


lib.mg_mipmap_levels_build.argtypes = [_vp, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint32, _vp, _vp, C.c_uint32, C.POINTER(_vp), _vp]
lib.mg_mipmap_levels_build.restype = C.c_int
lib.mg_mipmap_levels_build_ex.argtypes = [_vp, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint32, _vp, _vp, C.c_uint32, C.c_uint64, C.c_uint64,
                                          C.POINTER(_vp), _vp]
lib.mg_mipmap_levels_build_ex.restype = C.c_int
lib.mg_mixture_table_free.argtypes = [_vp]
lib.mg_mixture_table_free.restype = None
lib.mg_mixture_table_info.argtypes = [_vp, C.POINTER(MgMixtureTableInfo)]
lib.mg_mixture_table_info.restype = C.c_int
lib.mg_mixture_table_export.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp]
lib.mg_mixture_table_export.restype = C.c_int
lib.mg_mipmap_remap_handles.argtypes = [_vp, C.c_uint64, _vp, C.c_uint32, _vp]
lib.mg_mipmap_remap_handles.restype = C.c_int


class MgError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where} failed with {code}: {lib.mg_last_error().decode()}")


def _check(rc: int, where: str) -> None:
    if rc != MG_OK:
        raise MgError(rc, where)


def _ptr(x) -> int | None:
    """Address of a torch tensor / numpy array / raw int (None -> NULL)."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()          # torch.Tensor


def _np(a, dt):
    return None if a is None else np.ascontiguousarray(a, dtype=dt)


def kernel_launch_count() -> int:
    return int(lib.mg_kernel_launch_count())


def bits_per_voxel(i_min: int, i_max: int) -> int:
    return int(lib.mg_bits_per_voxel(int(i_min), int(i_max)))


def packed_stream_bytes(n_voxels: int, bits: int) -> int:
    return int(lib.mg_packed_stream_bytes(int(n_voxels), int(bits)))


def index_range(idx_device, n: int, stream: int = 0):
    lo, hi = C.c_uint32(), C.c_uint32()
    _check(lib.mg_index_range(_ptr(idx_device), int(n), C.byref(lo), C.byref(hi), stream or None), "mg_index_range")
    return int(lo.value), int(hi.value)


def index_ranges_static(idx_device, level_offsets, stream: int = 0):
    """(i_min[l], i_max[l]) of every level of a device index buffer through mg_index_ranges_static, the entry point for
    callers that must not allocate device memory (their own arena owns it all, or a cudaFree stall is not affordable):
    its scratch is a fixed array inside libmg.so, good for up to MG_INDEX_RANGES_STATIC_MAX_LEVELS levels.
    ``level_offsets`` has one more entry than there are levels.  Synchronises ``stream``."""
    off = np.ascontiguousarray(level_offsets, dtype=np.uint64)
    n_levels = off.size - 1
    lo, hi = np.empty(max(n_levels, 1), np.uint32), np.empty(max(n_levels, 1), np.uint32)
    _check(lib.mg_index_ranges_static(_ptr(idx_device), off.ctypes.data, n_levels, lo.ctypes.data, hi.ctypes.data,
                                      stream or None), "mg_index_ranges_static")
    return lo[:n_levels], hi[:n_levels]


def pack_indices(idx_device, n: int, i_min: int, bits: int, packed_device, stream: int = 0) -> None:
    _check(lib.mg_pack_indices(_ptr(idx_device), int(n), int(i_min), int(bits), _ptr(packed_device), stream or None),
           "mg_pack_indices")


def packed_levels(levels) -> "C.Array":
    """ctypes array of MgPackedLevel from dicts / tuples (n_voxels, out_offset, byte_offset, bits, i_min)."""
    arr = (MgPackedLevel * len(levels))()
    for i, l in enumerate(levels):
        if isinstance(l, dict):
            l = (l["n_voxels"], l["out_offset"], l["byte_offset"], l["bits"], l["i_min"])
        arr[i] = MgPackedLevel(*[int(x) for x in l])
    return arr


def mipmap_leaf_index(seg_device, n_voxels: int, level0_device, capacity: int = 1 << 20, stream: int = 0) -> np.ndarray:
    """NEXT-4 front end, level 0: writes leaf numbers to level0_device, returns the sorted distinct segment IDs."""
    ids = np.zeros(int(capacity), dtype=np.uint32)
    n = C.c_uint32(0)
    _check(lib.mg_mipmap_leaf_index(_ptr(seg_device), int(n_voxels), _ptr(level0_device), ids.ctypes.data, int(capacity),
                                    C.byref(n), stream or None), "mg_mipmap_leaf_index")
    return ids[:n.value].copy()


def mipmap_front_level1(level0_device, dims_xyz, level1_device, mixed_voxel_device, mixed_children_device, capacity: int,
                        stream: int = 0) -> int:
    """NEXT-4 front end, level 1: fills level1_device and the list of non-pure parents; returns their number
    (entries beyond ``capacity`` are dropped: call again with larger lists if it is exceeded)."""
    n = C.c_uint64(0)
    X, Y, Z = (int(d) for d in dims_xyz)
    _check(lib.mg_mipmap_front_level1(_ptr(level0_device), X, Y, Z, _ptr(level1_device), _ptr(mixed_voxel_device),
                                      _ptr(mixed_children_device), int(capacity), C.byref(n), stream or None),
           "mg_mipmap_front_level1")
    return int(n.value)


class MixtureTable:
    """Device mixture store of mg_mipmap_levels_build (the levels >= 1 of the histogram mipmap built on the device)."""

    def __init__(self, level0_device, dims_xyz, n_leaves: int, levels_device, level_offsets, stream: int = 0,
                 cap_mixtures: int = 0, cap_entries: int = 0):
        X, Y, Z = (int(d) for d in dims_xyz)
        off = np.ascontiguousarray(level_offsets, dtype=np.uint64)
        h = _vp()
        self._h = None
        if cap_mixtures or cap_entries:
            _check(lib.mg_mipmap_levels_build_ex(_ptr(level0_device), X, Y, Z, int(n_leaves), _ptr(levels_device), off.ctypes.data,
                                                 int(off.size), int(cap_mixtures), int(cap_entries), C.byref(h), stream or None),
                   "mg_mipmap_levels_build_ex")
        else:
            _check(lib.mg_mipmap_levels_build(_ptr(level0_device), X, Y, Z, int(n_leaves), _ptr(levels_device), off.ctypes.data,
                                              int(off.size), C.byref(h), stream or None), "mg_mipmap_levels_build")
        self._h = h
        self.info = MgMixtureTableInfo()
        _check(lib.mg_mixture_table_info(self._h, C.byref(self.info)), "mg_mixture_table_info")

    def export(self) -> dict:
        """Host copy: offset u64, k u32, tlog u32, first_pos u64 per mixture; leaf u32, count u64 per entry."""
        n, e = int(self.info.n_mixtures), int(self.info.n_entries)
        out = dict(offset=np.zeros(n, np.uint64), k=np.zeros(n, np.uint32), tlog=np.zeros(n, np.uint32),
                   first_pos=np.zeros(n, np.uint64), leaf=np.zeros(e, np.uint32), count=np.zeros(e, np.uint64))
        _check(lib.mg_mixture_table_export(self._h, *(out[k].ctypes.data for k in ("offset", "k", "tlog", "first_pos", "leaf", "count"))),
               "mg_mixture_table_export")
        return out

    def close(self) -> None:
        if getattr(self, "_h", None):
            lib.mg_mixture_table_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def mipmap_remap_handles(handles_device, n: int, node_of_mixture_device, n_mixtures: int, stream: int = 0) -> None:
    _check(lib.mg_mipmap_remap_handles(_ptr(handles_device), int(n), _ptr(node_of_mixture_device), int(n_mixtures), stream or None),
           "mg_mipmap_remap_handles")


def mipmap_desc(level_offsets, level_dims_xyz) -> MgMipmapDesc:
    """level_offsets[l] = first voxel of level l, level_dims_xyz[l] = (X_l, Y_l, Z_l)."""
    d = MgMipmapDesc()
    d.n_levels = len(level_offsets)
    if d.n_levels > MG_MAX_MIP_LEVELS:
        raise ValueError(f"at most {MG_MAX_MIP_LEVELS} mip levels")
    for l, (o, dims) in enumerate(zip(level_offsets, level_dims_xyz)):
        d.level_offset[l] = int(o)
        for a in range(3):
            d.level_dim[l][a] = int(dims[a])
    return d


def view_struct(view: dict) -> MgView:
    """Marshal a view dictionary (the fields of mg_view; synth.orbit_view builds one)."""
    v = MgView()
    for k in ("eye", "right", "up", "forward", "spacing"):
        for a in range(3):
            getattr(v, k)[a] = float(view[k][a])
    for k in ("tan_half_fov", "step_voxels", "ref_step_voxels", "lod_bias", "ess_threshold", "alpha_cutoff"):
        setattr(v, k, float(view[k]))
    v.width, v.height = int(view["width"]), int(view["height"])
    v.flags = int(view.get("flags", 0))
    return v


class Graph:
    """Handle of a loaded Mixture Graph (mg_load_graph ... mg_free_graph)."""

    def __init__(self, child_a, child_b, weight, n_leaves: int, level_offsets=None,
                 leaf_segment_id=None, flags: int = 0):
        a, b = _np(child_a, np.uint32), _np(child_b, np.uint32)
        w = _np(weight, np.float32)
        off = _np(level_offsets, np.uint64)
        seg = _np(leaf_segment_id, np.uint32)
        n_nodes = int(a.size)
        n_topo = 0 if off is None else int(off.size) - 1
        h = _vp()
        self._h = None
        _check(lib.mg_load_graph(_ptr(a), _ptr(b), _ptr(w), n_nodes, int(n_leaves), _ptr(off), n_topo,
                                 _ptr(seg), int(flags), C.byref(h)), "mg_load_graph")
        self._h = h

    def close(self) -> None:
        if self._h is not None:
            lib.mg_free_graph(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def info(self) -> MgInfo:
        i = MgInfo()
        _check(lib.mg_graph_info(self._h, C.byref(i)), "mg_graph_info")
        return i

    def level_offsets(self) -> np.ndarray:
        out = np.zeros(self.info.n_topo_levels + 1, dtype=np.uint64)
        _check(lib.mg_level_offsets(self._h, _ptr(out)), "mg_level_offsets")
        return out

    def node_permutation(self) -> np.ndarray:
        out = np.zeros(self.info.n_nodes, dtype=np.uint32)
        _check(lib.mg_node_permutation(self._h, _ptr(out)), "mg_node_permutation")
        return out

    def relabel_indices(self, idx_device, n: int, stream: int = 0) -> None:
        _check(lib.mg_relabel_indices(self._h, _ptr(idx_device), int(n), stream or None), "mg_relabel_indices")

    def check_indices(self, node_idx_device, n: int, stream: int = 0) -> int:
        """Number of entries of a device index volume that name no node of this graph (mg_check_indices)."""
        bad = C.c_uint64(0)
        _check(lib.mg_check_indices(self._h, _ptr(node_idx_device), int(n), C.byref(bad), stream or None), "mg_check_indices")
        return int(bad.value)

    def propagate(self, tf_device, node_rgba_device, stream: int = 0) -> None:
        _check(lib.mg_propagate(self._h, _ptr(tf_device), _ptr(node_rgba_device), stream or None), "mg_propagate")

    def propagate_host(self, tf_host, node_rgba_device, stream: int = 0) -> None:
        _check(lib.mg_propagate_host(self._h, _ptr(tf_host), _ptr(node_rgba_device), stream or None),
               "mg_propagate_host")

    def propagate_attr(self, leaf_attr_device, node_attr_device, n_channels: int, stream: int = 0) -> None:
        _check(lib.mg_propagate_attr(self._h, _ptr(leaf_attr_device), _ptr(node_attr_device), int(n_channels),
                                     stream or None), "mg_propagate_attr")

    def colorize(self, node_idx_device, n_voxels: int, node_rgba_device, out, out_aux=None,
                 fmt: int = MG_RGBA8, mip_level: int = ALL_LEVELS, stream: int = 0,
                 from_last_propagate: bool = False) -> None:
        """``from_last_propagate`` adds MG_PALETTE_FROM_LAST_PROPAGATE to ``fmt`` (see include/mg.h)."""
        f = int(fmt) | (MG_PALETTE_FROM_LAST_PROPAGATE if from_last_propagate else 0)
        _check(lib.mg_colorize(self._h, int(mip_level), _ptr(node_idx_device), int(n_voxels),
                               _ptr(node_rgba_device), _ptr(out), _ptr(out_aux), f, stream or None),
               "mg_colorize")

    def colorize_packed(self, packed_device, levels, node_rgba_device, out, out_aux=None, fmt: int = MG_RGBA8,
                        stream: int = 0, from_last_propagate: bool = False) -> None:
        arr = levels if isinstance(levels, C.Array) else packed_levels(levels)
        f = int(fmt) | (MG_PALETTE_FROM_LAST_PROPAGATE if from_last_propagate else 0)
        _check(lib.mg_colorize_packed(self._h, _ptr(packed_device), arr, len(arr), _ptr(node_rgba_device), _ptr(out),
                                      _ptr(out_aux), f, stream or None), "mg_colorize_packed")

    def tf_update_host(self, tf_host, node_rgba_device, node_idx_device, n_voxels: int, out_device,
                       out_host=None, fmt: int = MG_RGBA8, stream: int = 0) -> None:
        _check(lib.mg_tf_update_host(self._h, _ptr(tf_host), _ptr(node_rgba_device), _ptr(node_idx_device),
                                     int(n_voxels), _ptr(out_device), _ptr(out_host), int(fmt), stream or None),
               "mg_tf_update_host")

    def render(self, node_idx_device, mip, node_rgba_device, view, out_rgba_device, stats_device=None,
               stream: int = 0, ess_mask_device=None) -> None:
        """mg_render, or mg_render_ex when ``ess_mask_device`` (from ess_mask_build) is given."""
        m = mip if isinstance(mip, MgMipmapDesc) else mipmap_desc(*mip)
        v = view if isinstance(view, MgView) else view_struct(view)
        if ess_mask_device is None:
            _check(lib.mg_render(self._h, _ptr(node_idx_device), C.byref(m), _ptr(node_rgba_device), C.byref(v),
                                 _ptr(out_rgba_device), _ptr(stats_device), stream or None), "mg_render")
        else:
            aux = MgRenderAux(_ptr(ess_mask_device), None)
            _check(lib.mg_render_ex(self._h, _ptr(node_idx_device), C.byref(m), _ptr(node_rgba_device), C.byref(v),
                                    C.byref(aux), _ptr(out_rgba_device), _ptr(stats_device), stream or None), "mg_render_ex")

    def ess_mask_build(self, node_idx_device, mip, node_rgba_device, ess_threshold: float, ess_mask_device,
                       stream: int = 0) -> None:
        """Fill ``ess_mask_device`` (uint16 per voxel of mip level 2) for mg_render_ex."""
        m = mip if isinstance(mip, MgMipmapDesc) else mipmap_desc(*mip)
        _check(lib.mg_ess_mask_build(self._h, _ptr(node_idx_device), C.byref(m), _ptr(node_rgba_device),
                                     float(ess_threshold), _ptr(ess_mask_device), stream or None), "mg_ess_mask_build")

    def mixture_lut(self, weight_sigma=None, stream: int = 0) -> "MixtureLut":
        """NEXT-4: build the mixture lookup table (mu, dmu per node) of this graph on the device."""
        return MixtureLut(self, weight_sigma, stream)


class MixtureLut:
    """Handle of a device mixture lookup table (mg_mixture_lut_build ... mg_mixture_lut_free)."""

    def __init__(self, graph: Graph, weight_sigma=None, stream: int = 0):
        sg = _np(weight_sigma, np.float32)
        if sg is not None and sg.size != graph.info.n_nodes:
            raise ValueError("weight_sigma must have n_nodes entries")
        h = _vp()
        _check(lib.mg_mixture_lut_build(graph._h, _ptr(sg), C.byref(h), stream or None), "mg_mixture_lut_build")
        self._h = h
        self.info = MgLutInfo()
        _check(lib.mg_mixture_lut_info(self._h, C.byref(self.info)), "mg_mixture_lut_info")

    def close(self) -> None:
        if getattr(self, "_h", None):
            lib.mg_mixture_lut_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def export(self):
        """(row_ptr u64 [n_nodes + 1], leaf u32 [nnz], mu f64 [nnz], dmu f64 [nnz]) on the host."""
        n, nnz = int(self.info.n_nodes), int(self.info.nnz)
        rp, leaf = np.zeros(n + 1, np.uint64), np.zeros(nnz, np.uint32)
        mu, dmu = np.zeros(nnz, np.float64), np.zeros(nnz, np.float64)
        _check(lib.mg_mixture_lut_export(self._h, rp.ctypes.data, leaf.ctypes.data, mu.ctypes.data, dmu.ctypes.data),
               "mg_mixture_lut_export")
        return rp, leaf, mu, dmu

    def range_query(self, node_idx_device, mip, boxes, expect_device, err_device=None, fetches_device=None,
                    mode: int = MG_QUERY_FA, stream: int = 0) -> None:
        m = mip if isinstance(mip, MgMipmapDesc) else mipmap_desc(*mip)
        b = np.ascontiguousarray(boxes, dtype=np.uint64).reshape(-1, 6)
        _check(lib.mg_range_query(self._h, _ptr(node_idx_device), C.byref(m), b.ctypes.data, b.shape[0],
                                  _ptr(expect_device), _ptr(err_device), _ptr(fetches_device), int(mode), stream or None),
               "mg_range_query")
