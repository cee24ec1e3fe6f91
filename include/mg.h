/*
 * mg.h -- C ABI of the B200-native Mixture Graph transfer-function propagation library.
 *
 * Implements the hot path of "The Mixture Graph" (arXiv 2009.02702; "L<n>" = line n of PAPER.md):
 *   a4  leaf assignment        c[k] = TF[k], bit-exact                         (L371)
 *   a5  propagation            c[n] = (1 - w[n]) c[a[n]] + w[n] c[b[n]]        (L259, L269, L371)
 *                              level-synchronous over the topological levels   (L211-L213)
 *   a6  colourise              out[v] = convert(c[node_idx[v]])                (L221, L267)
 *
 * Conventions
 *   - every call returns int: MG_OK (0) or a negative MG_ERR_*; mg_last_error() gives a
 *     thread-local message for the last failing call on this thread.  No exceptions, no aborts.
 *   - "host" / "device" is stated per pointer.  Device pointers must belong to the CUDA device that
 *     was current when mg_load_graph was called.  `stream` is a cudaStream_t passed as void*
 *     (NULL = the legacy default stream).
 *   - mg_propagate / mg_colorize only ENQUEUE work on `stream`: no synchronisation and no
 *     allocation (the first call on a graph may create cached launch state).
 *     Caller-owned buffers must outlive the enqueued work.
 *   - the library owns only its device copy of the graph (and per-graph scratch: 8-bit / 16-bit
 *     palettes, a TF staging buffer), released by mg_free_graph.
 *   - a graph handle is not thread-safe: calls on ONE handle must be serialised by the caller
 *     (different handles are independent).  Every call that launches work checks that the graph's
 *     device is the current one and fails with MG_ERR_INVALID_ARG otherwise.
 *   - there is no CPU fallback: without a CUDA device every compute call fails with MG_ERR_CUDA.
 */
#ifndef MG_H_
#define MG_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mg_graph mg_graph;

enum {
    MG_OK = 0,
    MG_ERR_INVALID_ARG = -1,   /* NULL pointer, bad enum, misaligned buffer ...            */
    MG_ERR_INVALID_GRAPH = -2, /* the arrays do not describe a valid Mixture Graph         */
    MG_ERR_CUDA = -3,          /* a CUDA runtime call failed (message has the CUDA error)  */
    MG_ERR_OOM = -4            /* host or device allocation failed                         */
};

/* mg_load_graph flags */
enum {
    MG_RELABEL = 1u, /* input is only children-before-parents (Eq. 8), not level-contiguous:
                       the library computes the topological levels (L211), permutes the nodes so
                       that every level is contiguous (leaves keep their numbers; inside a level
                       nodes are ordered by their children's new numbers for L2 locality) and
                       exposes the permutation through mg_node_permutation.                      */
    MG_NO_PALETTES = 2u /* mg_propagate writes node_rgba only, not the 8-bit / 16-bit palettes (12 B per
                           node less traffic for callers that only want the fp32 palette, e.g. for
                           mg_render); mg_colorize then always derives them itself and rejects
                           MG_PALETTE_FROM_LAST_PROPAGATE.                                           */
};

/* mg_colorize output formats (bit mask) */
enum {
    MG_RGBA8 = 1u,         /* 4 x uint8 per voxel, R in byte 0: round_half_even(clamp(c,0,1)*255)  */
    MG_RGBA16F = 2u,       /* 4 x IEEE fp16 per voxel (round to nearest even)                      */
    MG_BOTH = 3u,          /* both; RGBA8 to out_rgba, fp16 to out_rgba_aux                        */
    MG_FORCE_CONVERT = 16u, /* derive the palettes from node_rgba: this IS the default since the palette
                               contract became explicit; the flag is accepted and changes nothing      */
    MG_PALETTE_FROM_LAST_PROPAGATE = 32u /* gather from the palettes the last mg_propagate derived (see
                                            mg_colorize): no conversion kernel                         */
};

typedef struct mg_info {
    uint64_t n_nodes;       /* leaves + internal nodes                                        */
    uint64_t n_internal;    /* n_nodes - n_leaves                                             */
    uint32_t n_leaves;      /* sources = segment IDs (L130)                                   */
    uint32_t depth;         /* topological depth = number of synchronisation points (L211)    */
    uint32_t n_topo_levels; /* depth + 1                                                      */
    uint32_t first_fused_level; /* levels >= this run inside ONE persistent CTA (0 = none)    */
    uint32_t n_launches_propagate; /* kernel launches one mg_propagate enqueues               */
    uint32_t relabelled;    /* 1 if the library permuted the nodes (MG_RELABEL)               */
    uint64_t device_bytes;  /* device memory owned by the graph object                        */
} mg_info;

/*
 * mg_load_graph -- validate a Mixture Graph given as HOST SoA arrays and copy it to the device.
 *
 *   child_a, child_b  host uint32[n_nodes]: the two predecessors of each node (stored as incoming
 *                     edges, L140).  Entries of the leaves [0, n_leaves) are ignored.
 *   weight            host float[n_nodes]: w of the triple (a, b, w) = (1-w) s_a + w s_b (L259):
 *                     the weight multiplies child_b.  Must satisfy 0 < w < 1 (L176).
 *   n_nodes, n_leaves leaves are nodes 0 .. n_leaves-1, in leaf_segment_id order; n_nodes < 2^32.
 *   level_offsets     host uint64[n_topo_levels + 1], [0] = 0, [1] = n_leaves, [last] = n_nodes;
 *                     nodes of topological level L occupy [off[L], off[L+1]) and both children of
 *                     such a node lie below off[L], at least one of them at or above off[L-1]
 *                     (level = max + 1, L211).  May be NULL together with flags & MG_RELABEL.
 *   n_topo_levels     depth + 1 (ignored with MG_RELABEL when level_offsets is NULL).
 *   leaf_segment_id   host uint32[n_leaves] or NULL: the segment ID of each leaf (kept for
 *                     mg_graph_info consumers; strictly increasing if given).
 *   flags             0, MG_RELABEL, MG_NO_PALETTES or both.
 *   out               receives the graph handle.
 *
 * All arrays are caller-owned and copied.  Errors: MG_ERR_INVALID_ARG (NULL, n_leaves = 0,
 * n_nodes >= 2^32), MG_ERR_INVALID_GRAPH (a == b, child not below its level, level not max+1,
 * w outside (0,1) or not finite, offsets not increasing), MG_ERR_OOM, MG_ERR_CUDA.
 */
int mg_load_graph(const uint32_t *child_a, const uint32_t *child_b, const float *weight,
                  uint64_t n_nodes, uint32_t n_leaves, const uint64_t *level_offsets,
                  uint32_t n_topo_levels, const uint32_t *leaf_segment_id, uint32_t flags,
                  mg_graph **out);

/* Release the handle and every device buffer it owns.  NULL is allowed. */
void mg_free_graph(mg_graph *g);

/* Fill *info.  Host only. */
int mg_graph_info(const mg_graph *g, mg_info *info);

/* level_offsets of the loaded (possibly relabelled) graph: host uint64[n_topo_levels + 1]. */
int mg_level_offsets(const mg_graph *g, uint64_t *level_offsets_host);

/* new_of_old_host: host uint32[n_nodes]; node `old` of the arrays given to mg_load_graph is node
 * new_of_old[old] of the library's numbering (identity unless MG_RELABEL permuted the graph). */
int mg_node_permutation(const mg_graph *g, uint32_t *new_of_old_host);

/* One-off: rewrite a DEVICE array of n node indices in place from the caller's numbering to the
 * library's (idx[i] = new_of_old[idx[i]]), so that builder-numbered node_idx volumes can be passed
 * to mg_colorize.  No-op for a graph that was not relabelled. */
int mg_relabel_indices(mg_graph *g, uint32_t *idx_device, uint64_t n, void *stream);

/*
 * mg_propagate -- one full transfer-function update (the paper performs full updates only, L221).
 *
 *   tf_rgba    DEVICE float[n_leaves][4], leaf order.  16-byte aligned.
 *   node_rgba  DEVICE float[n_nodes][4], caller-allocated, 16-byte aligned.  On completion
 *              node_rgba[k] == tf_rgba[k] bit-for-bit for k < n_leaves and every other entry holds
 *              fma(w, c_b, fma(-w, c_a, c_a)) per channel in fp32, in the library's numbering.
 *
 * Enqueues: one kernel per large topological level (leaf copy fused into the first) and one
 * persistent single-CTA kernel for the small top levels.  Every kernel also writes the 8-bit and
 * 16-bit palettes that mg_colorize gathers from.
 */
int mg_propagate(mg_graph *g, const float *tf_rgba, float *node_rgba, void *stream);

/* Same, with the TF in HOST memory (pinned for a truly asynchronous copy): enqueues the
 * host-to-device copy of n_leaves float4 into a graph-owned staging buffer first -- the quantity
 * the paper times ("GPU timings include the data upload of one float4 color per source", L371). */
int mg_propagate_host(mg_graph *g, const float *tf_rgba_host, float *node_rgba, void *stream);

/*
 * mg_colorize -- materialise (part of) the pre-filtered RGBA mipmap: out[v] = convert(c[idx[v]]).
 *
 *   mip_level        informational (the operation is the same for every level); pass 0xFFFFFFFF
 *                    when one call covers several concatenated levels.
 *   node_idx_volume  DEVICE uint32[n_voxels], x fastest, values < n_nodes in the LIBRARY's
 *                    numbering (see mg_relabel_indices).  4-byte aligned; the fast path needs the
 *                    index and output pointers to have the same offset modulo 16 bytes in units of
 *                    voxels (true for any two cudaMalloc'ed buffers indexed at the same voxel).
 *   n_voxels         number of voxels; authoritative.  0 is allowed (no work).
 *   node_rgba        DEVICE float[n_nodes][4], 16-byte aligned: THE palette ("one vec4 colour entry
 *                    per node", L267), in the library's numbering.  By default the call first derives
 *                    the 8-bit / 16-bit palette of the requested format from this buffer (one extra
 *                    kernel on `stream`, 20-24 B per node), so the output always reflects the buffer
 *                    as it is on `stream` at this point -- whoever wrote it (mg_propagate,
 *                    mg_propagate_attr with 4 channels, the caller's own kernels).
 *   out_rgba         DEVICE output, n_voxels * 4 bytes (MG_RGBA8, MG_BOTH) or * 8 (MG_RGBA16F).
 *   out_rgba_aux     DEVICE fp16 output for MG_BOTH, else ignored (may be NULL).
 *   format           MG_RGBA8 | MG_RGBA16F | MG_BOTH, optionally | MG_PALETTE_FROM_LAST_PROPAGATE:
 *                    the caller states that node_rgba is the buffer the most recent mg_propagate /
 *                    mg_propagate_host on this graph filled, that nothing has written it since, and
 *                    that this call is ordered after that propagation (same stream, or an event).
 *                    The palettes that propagation derived are then gathered as they are (no
 *                    conversion kernel: a TF update is mg_propagate's launches + ONE colourise launch).
 *                    The library can only check what it sees: the flag is rejected with
 *                    MG_ERR_INVALID_ARG when node_rgba is not that buffer, when a library call has
 *                    written into it since (mg_propagate_attr), when an unflagged colourise has
 *                    re-derived the palettes since, or on a MG_NO_PALETTES graph.  Writes by the
 *                    caller's own kernels are the caller's to declare -- by NOT passing the flag.
 *
 * An RGBA8 palette beyond what the L2 serves for random gathers (more than 88 MB = 23 M nodes, up to 4 x that) is
 * gathered tile by tile: the call then enqueues one sweep over the indices per palette tile (MG_COLORIZE_TILE_BYTES
 * in the environment of mg_load_graph overrides the 88-MB tile size for that graph; it is not consulted afterwards),
 * each merging its voxels into out_rgba, so out_rgba is READ as
 * well as written between the sweeps and must not be touched by another stream's work meanwhile.
 */
int mg_colorize(mg_graph *g, uint32_t mip_level, const uint32_t *node_idx_volume,
                uint64_t n_voxels, const float *node_rgba, void *out_rgba, void *out_rgba_aux,
                uint32_t format, void *stream);

/* Count the entries of a DEVICE node-index volume that name no node of g (>= n_nodes): mg_colorize, mg_render and
 * mg_range_query gather through the indices unchecked, so a caller that did not build them with this library's
 * builder can validate them once (compute-sanitizer being unavailable on some pools, this is the bounds check a
 * memcheck run would make).  *n_bad_host receives the count; synchronises `stream`. */
int mg_check_indices(const mg_graph *g, const uint32_t *node_idx_device, uint64_t n, uint64_t *n_bad_host,
                     void *stream);

/*
 * mg_tf_update_host -- the whole per-update path with HOST buffers at both ends:
 * H2D of the TF, mg_propagate, mg_colorize over n_voxels (typically every mip level,
 * concatenated), and -- if out_host is not NULL -- D2H of the colourised output.
 * out_device is the DEVICE buffer the mipmap is materialised in (what a renderer would sample);
 * out_host, if given, must hold n_voxels * 4 (MG_RGBA8) or * 8 (MG_RGBA16F) bytes (MG_BOTH is not
 * accepted here).  Enqueue-only, like the calls it is made of.
 */
int mg_tf_update_host(mg_graph *g, const float *tf_rgba_host, float *node_rgba,
                      const uint32_t *node_idx_volume, uint64_t n_voxels, void *out_device,
                      void *out_host, uint32_t format, void *stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-3: bit-packed node-ID volumes (Table 1 rows (8), (9), (A); Eq. 15-16).
 *
 * Per mip level l the paper stores i_min(l) and, for every voxel, (node ID - i_min(l)) at the fixed
 * bitrate r(l) = ceil(log2(i_max(l) - i_min(l) + 1)); the shader addresses the stream by bit address
 * (L267).  Bit order (not fixed by the paper; reading Q18): voxel v of the level occupies
 * stream bits [v r, (v+1) r), stream bit q is bit (q mod 8) of byte q / 8, value bit k goes to
 * stream bit v r + k (LSB first, little endian).
 * ------------------------------------------------------------------------------------------------ */
#define MG_MAX_PACKED_LEVELS 32

typedef struct mg_packed_level {
    uint64_t n_voxels;    /* voxels of the level (0 = skip)                                          */
    uint64_t out_offset;  /* first voxel of the level in the output buffers; multiple of 4            */
    uint64_t byte_offset; /* start of the level's stream inside the packed buffer; multiple of 16     */
    uint32_t bits;        /* r(l), 0 .. 32 (0: every voxel is node i_min)                             */
    uint32_t i_min;       /* i_min(l)                                                                 */
} mg_packed_level;

/* r = ceil(log2(i_max - i_min + 1)), Eq. 16.  Host only. */
uint32_t mg_bits_per_voxel(uint32_t i_min, uint32_t i_max);

/* Bytes to allocate for the stream of one level: ceil(n r / 8) rounded up to 16, plus 16.  Host only. */
uint64_t mg_packed_stream_bytes(uint64_t n_voxels, uint32_t bits);

/* i_min / i_max of Eq. 15 for a DEVICE index volume (n > 0).  Returns the two values to the HOST:
 * this call synchronises `stream`. */
int mg_index_range(const uint32_t *idx_device, uint64_t n, uint32_t *i_min, uint32_t *i_max, void *stream);

/*
 * mg_index_ranges_static -- i_min(l) / i_max(l) of Eq. 15 for EVERY level of a mipmap in one call that allocates
 * nothing (no cudaMalloc, no cudaFree, no allocating library routine).
 *
 * Who needs it: mg_index_range gets its scratch words from cudaMalloc and returns them with cudaFree on each call.
 * A host application that has given the device's whole memory to an arena of its own (a renderer's resource pool, a
 * framework's caching allocator) may find the driver has nothing left to give, and a frame loop cannot take
 * cudaFree's wait on all of the device's streams between a TF update and the next frame.  Here the scratch -- one
 * (min, max) pair per level -- is a fixed 256-byte array inside the library image instead; every GPU that loads
 * libmg.so holds it until the process exits.
 *
 *   idx_device          DEVICE uint32 indices, the levels back to back or with gaps, 4-byte aligned.
 *   level_offsets_host  HOST uint64[n_levels + 1], non-decreasing: level l is idx_device[off[l] .. off[l + 1]).
 *   n_levels            1 .. MG_INDEX_RANGES_STATIC_MAX_LEVELS; more is refused with MG_ERR_INVALID_ARG (the array
 *                       has no room: call mg_index_range per level instead).
 *   i_min_host, i_max_host  HOST uint32[n_levels], caller-owned: receive the ranges, the same values
 *                       mg_index_range returns level by level.  An empty level reports i_min = 0xFFFFFFFF, i_max = 0.
 *
 * Enqueues two kernels and an 8 n_levels-byte copy to the host on `stream`, then synchronises `stream` (like
 * mg_index_range, it returns values to the host).  The first call on each device also asks the runtime for the
 * device address of the array (cudaGetSymbolAddress, with that device current; at most 64 devices): make that
 * first call before any stream capture begins.  All calls on a device share the one array, which keeps whatever the
 * previous call left; each call resets the pairs it uses first, so calls one after another are independent, but
 * two calls whose kernels overlap on the same GPU (from two host threads or two streams) race on it and must be
 * serialised by the caller.  Errors: MG_ERR_INVALID_ARG (NULL, n_levels out of range, decreasing offsets, device
 * ordinal >= 64), MG_ERR_CUDA.
 */
#define MG_INDEX_RANGES_STATIC_MAX_LEVELS 32
int mg_index_ranges_static(const uint32_t *idx_device, const uint64_t *level_offsets_host, uint32_t n_levels,
                           uint32_t *i_min_host, uint32_t *i_max_host, void *stream);

/* One-off encoder step (Table 1 row (A)): pack DEVICE uint32 indices (every value in
 * [i_min, i_min + 2^bits); a value outside is reduced modulo 2^bits and never touches its neighbours'
 * bits) into the DEVICE stream `packed_device` (16-byte aligned,
 * mg_packed_stream_bytes(n, bits) bytes, fully written incl. zero padding).  Enqueue-only. */
int mg_pack_indices(const uint32_t *idx_device, uint64_t n, uint32_t i_min, uint32_t bits,
                    void *packed_device, void *stream);

/* mg_colorize with packed input, ALL levels in one launch: for every level l and voxel v < n_voxels,
 * out[out_offset + v] = convert(c[i_min + bits(v)]).  `levels` is a HOST array of n_levels
 * (<= MG_MAX_PACKED_LEVELS) descriptors, copied at enqueue.  packed_device, out_rgba, out_rgba_aux
 * are DEVICE, 16-byte aligned.  node_rgba and the palette contract are those of mg_colorize: the palettes
 * are derived from node_rgba first unless format carries MG_PALETTE_FROM_LAST_PROPAGATE.  Unpacked indices
 * are clamped to n_nodes - 1 (a stale (i_min, bits) pair cannot gather out of bounds).
 * format: MG_RGBA8 | MG_RGBA16F | MG_BOTH [| MG_PALETTE_FROM_LAST_PROPAGATE].  Enqueue-only. */
int mg_colorize_packed(mg_graph *g, const void *packed_device, const mg_packed_level *levels,
                       uint32_t n_levels, const float *node_rgba, void *out_rgba, void *out_rgba_aux,
                       uint32_t format, void *stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-1: propagation of any numeric segment attribute ("the Mixture Graph allows the
 * efficient computation of any kind of numeric segmentation attribute"): opacity alone for
 * empty-space skipping (L271 (i)-(ii)), diffuse / specular light contributions (L277), or K transfer
 * functions batched as 4 K channels -- one pass over the graph arrays for all channels.
 *
 *   leaf_attr   DEVICE float[n_leaves][n_channels], leaf order, channel fastest.
 *   node_attr   DEVICE float[n_nodes][n_channels], caller-allocated, must not alias leaf_attr.
 *               On completion node_attr[k][:] == leaf_attr[k][:] bit-for-bit for k < n_leaves; every
 *               other entry holds fma(w, x_b, fma(-w, x_a, x_a)) per channel in fp32 (the arithmetic
 *               of mg_propagate), in the library's numbering.
 *   n_channels  1 .. MG_MAX_ATTR_CHANNELS.  Both buffers 4-byte aligned; 16-byte (8-byte) aligned
 *               buffers with n_channels % 4 == 0 (% 2 == 0) take the vectorised path.
 *
 * Enqueue-only, no allocation.  Does not write the 8/16-bit palettes of mg_propagate; if node_attr
 * overlaps the node_rgba those palettes mirror, MG_PALETTE_FROM_LAST_PROPAGATE is refused from here on
 * (mg_colorize on a 4-channel node_attr derives its palettes from it, as for any node_rgba).
 * Errors: MG_ERR_INVALID_ARG (NULL, aliasing, misalignment, n_channels out of range), MG_ERR_CUDA.
 * ------------------------------------------------------------------------------------------------ */
#define MG_MAX_ATTR_CHANNELS 64
int mg_propagate_attr(mg_graph *g, const float *leaf_attr, float *node_attr, uint32_t n_channels,
                      void *stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-2: headless ray-marcher over the paletted histogram mipmap (section 4,
 * L414): "rendering from the Mixture Graph is the same as rendering from a paletted texture" (L267);
 * "we still have to perform the computation of the mip level as well as the interpolation in the
 * shader manually" (L269).  The paper gives the ingredients, not formulas; the readings R1-R6 are
 * listed in DESIGN.md section 3:
 *   R1 pinhole camera: pixel (i, j) (j = row from the top) looks along
 *      normalise(forward + u right + v up), u = (2 (i + 1/2) / W - 1) tan_half_fov W / H,
 *      v = (1 - 2 (j + 1/2) / H) tan_half_fov; voxel (x, y, z) of level 0 occupies
 *      [x sx, (x + 1) sx] x ... in world units (anisotropic spacing, L277).
 *   R2 LOD linear in view depth (L269): rho = z_view (2 tan_half_fov / H) / s_ref, s_ref = min spacing,
 *      lambda = clamp(log2(rho) + lod_bias, 0, l_max).
 *   R3 manual trilinear interpolation of palette colours on levels floor(lambda) and floor(lambda)+1
 *      (voxel i of level l centred at (i + 1/2) 2^l, indices clamped to the level), blended by frac(lambda).
 *   R4 step Delta = step_voxels s_ref 2^lambda with opacity correction
 *      alpha' = 1 - (1 - alpha)^(Delta / (ref_step_voxels s_ref)) (L269; 0.5-voxel steps, L414).
 *   R5 front-to-back compositing from the entry of the volume's box, sample at the interval mid-point,
 *      last interval clipped to the exit, stop at A >= alpha_cutoff.
 *   R6 hierarchical empty-space skipping (L271): a ray is in "empty mode" when it enters the volume and after
 *      every sample that was skipped or whose interpolated opacity was < ess_threshold.  In empty mode, before
 *      a sample is fetched, climb from level floor(lambda)+2 upwards while the parent voxel's palette opacity
 *      is < ess_threshold; samples whose whole 2 x 8-voxel footprint lies in the largest such block are not
 *      fetched.  ess_threshold < 0 disables it.
 * Arithmetic: ray parameter, step and sample position in fp64 (positions then in 32.32 fixed point for the per-level
 * voxel indices, fractions and block tests); fractional LOD, interpolation weights, colours and opacity correction in
 * fp32; compositing sums in fp64.
 * ------------------------------------------------------------------------------------------------ */
#define MG_MAX_MIP_LEVELS 24

typedef struct mg_mipmap_desc {
    uint32_t n_levels;                             /* 1 .. MG_MAX_MIP_LEVELS                              */
    uint32_t reserved;                             /* 0                                                   */
    uint64_t level_offset[MG_MAX_MIP_LEVELS];      /* first voxel of level l in node_idx_mipmap           */
    uint32_t level_dim[MG_MAX_MIP_LEVELS][3];      /* X_l, Y_l, Z_l; level l+1 = ceil(level l / 2), L80   */
} mg_mipmap_desc;

typedef struct mg_view {
    double eye[3], right[3], up[3], forward[3];    /* world units; right/up/forward orthonormal           */
    double tan_half_fov;                           /* vertical half field of view                         */
    double spacing[3];                             /* world size of a level-0 voxel along x, y, z (> 0)    */
    double step_voxels;                            /* > 0; step at full resolution in units of s_ref       */
    double ref_step_voxels;                        /* > 0; step the TF opacities refer to                  */
    double lod_bias;
    double ess_threshold;                          /* < 0: no empty-space skipping (paper: 1e-8)           */
    double alpha_cutoff;                           /* early ray termination (1.0 = never)                  */
    uint32_t width, height;                        /* image size in pixels (> 0)                           */
    uint32_t flags;                                /* 0 or MG_VIEW_HISTOGRAM_MIPMAP                        */
    uint32_t reserved;                             /* 0                                                    */
} mg_view;

/* mg_view.flags */
enum {
    MG_VIEW_HISTOGRAM_MIPMAP = 1u /* the caller asserts that node_idx_mipmap is the histogram mipmap of THIS graph
                                     (Eq. 4; what the builder emits): a voxel whose node is a leaf (< n_leaves) holds
                                     a pure mixture e_k, hence every voxel below it names the same leaf (L223).  The
                                     marcher then fetches the coarse level of a sample first; if its 8 voxels name
                                     one leaf, the 8 voxels of the fine level (their children) do too and the sample
                                     takes that leaf's palette colour without the second fetch.  The image is
                                     unchanged up to rounding (the 16 taps would all return that colour). */
};

/*
 * mg_render -- one image.  Enqueue-only, no allocation, one kernel launch.
 *   node_idx_mipmap  DEVICE uint32, every level concatenated as `mip` describes, x fastest, values
 *                    < n_nodes in the library's numbering (not checked).
 *   mip, view        HOST, copied at enqueue.
 *   node_rgba        DEVICE float[n_nodes][4], 16-byte aligned: the palette (any mg_propagate output).
 *   out_rgba         DEVICE float[height][width][4], 16-byte aligned: (C_r, C_g, C_b, A), associated
 *                    colour over a transparent background; rays missing the volume give zeros.
 *   stats_device     DEVICE uint64[4] or NULL (the caller zeroes it): [0] += samples composited,
 *                    [1] += samples skipped by R6, [2] += those of [0] whose coarse level named one leaf
 *                    (MG_VIEW_HISTOGRAM_MIPMAP: fine level not fetched), [3] unused.
 * Errors: MG_ERR_INVALID_ARG (NULL, misalignment, bad sizes, level dims that are not the ceil-halving
 * chain of L80, offsets overlapping, a step so small that a ray would need more than 2^24 of them), MG_ERR_CUDA.
 */
int mg_render(mg_graph *g, const uint32_t *node_idx_mipmap, const mg_mipmap_desc *mip,
              const float *node_rgba, const mg_view *view, float *out_rgba, uint64_t *stats_device,
              void *stream);

/*
 * Hierarchical empty-space skipping without the per-probe climb (R6; PAPER.md L271 (i)-(iii)).  The climb of R6
 * reads, per probe, the palette opacity of the parent voxels from level floor(lambda) + 2 upwards -- a chain of
 * dependent gathers.  Those comparisons depend only on the voxel, the palette and the threshold, so they can be
 * made once per TF update: mg_ess_mask_build writes, for every voxel of mip level 2, a 16-bit mask whose bit k says
 * "the ancestor of this voxel on level 2 + k has opacity < ess_threshold" (bit 0: the voxel itself).  A probe of
 * mg_render_ex is then ONE 2-byte load: the run of set bits from level floor(lambda) + 2 on is exactly the climb.
 * Same blocks, same skipped samples, same image as mg_render.
 *   ess_mask        DEVICE uint16[X_2 Y_2 Z_2] (level 2 of `mip`, x fastest), caller-allocated
 *   ess_threshold   the mg_view.ess_threshold the mask will be used with
 * Needs 3 <= n_levels <= 18.  Must be rebuilt after every change of node_rgba or of the threshold (the library
 * cannot see a stale mask: with one, skipped samples are no longer provably transparent).  Enqueue-only, one launch.
 */
int mg_ess_mask_build(mg_graph *g, const uint32_t *node_idx_mipmap, const mg_mipmap_desc *mip,
                      const float *node_rgba, double ess_threshold, uint16_t *ess_mask, void *stream);

/* Optional acceleration data of mg_render_ex; every pointer may be NULL (then the plain path of mg_render is taken). */
typedef struct mg_render_aux {
    const uint16_t *ess_mask;   /* DEVICE, from mg_ess_mask_build on THIS mipmap, palette and view->ess_threshold */
    const void *reserved;       /* NULL */
} mg_render_aux;

/* mg_render with acceleration data (aux may be NULL: identical to mg_render). */
int mg_render_ex(mg_graph *g, const uint32_t *node_idx_mipmap, const mg_mipmap_desc *mip,
                 const float *node_rgba, const mg_view *view, const mg_render_aux *aux, float *out_rgba,
                 uint64_t *stats_device, void *stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-4: mixture lookup table with error propagation and sub-volume (range) queries
 * (section 3.5 Eq. 17-18, section 3.6, Table 4).
 *
 * The table stores, per node, the sparse mixture mu (expected share of every leaf / segment) and its
 * uncertainty dmu: leaf i holds e_i with error 0; an internal node (a, b, w +- dw) holds
 *   mu_i = (1 - w) a_i + w b_i,   dmu_i = sqrt(mu_i^2 ((da_i / a_i)^2 + (db_i / b_i)^2 + 2 (dw / w)^2))   (Eq. 18)
 * where a ratio with a zero denominator (component absent from that child) is dropped (reading Q19) and
 * dw is the standard deviation of the weight's quantiser bin (L176).  fp64 throughout, w = (double) of
 * the graph's fp32 weight.  Device layout: CSR rows sorted by leaf index.
 *
 * A range query returns, for a box of the level-0 grid, the expected number of voxels of every leaf and
 * its error.  MG_QUERY_FA is the paper's footprint assembly: each axis range is cut into the largest
 * aligned power-of-two pieces, every box of the tensor product is tesselated by cubes whose side is its
 * shortest extent, each cube is ONE sample of the histogram mipmap at level log2(side), denormalised by
 * side^3; errors add in quadrature (Eq. 17).  MG_QUERY_NAIVE adds every level-0 voxel of the box (L377).
 * ------------------------------------------------------------------------------------------------ */
typedef struct mg_mixture_lut mg_mixture_lut;

typedef struct mg_lut_info {
    uint64_t n_nodes;      /* rows                                                        */
    uint64_t nnz;          /* stored (leaf, mu, dmu) entries                              */
    uint64_t capacity;     /* entries allocated (an upper bound computed before the build) */
    uint64_t device_bytes; /* device memory owned by the table                            */
    uint32_t n_leaves;
    uint32_t max_row_nnz;  /* longest row                                                 */
} mg_lut_info;

enum {
    MG_QUERY_FA = 0u,      /* footprint assembly                                                               */
    MG_QUERY_NAIVE = 1u,   /* every level-0 voxel                                                              */
    MG_QUERY_FA_WALK = 2u  /* footprint assembly with the work distribution used for queries of > 4096 boxes   */
                           /* (every warp walks all boxes); same result, exposed so that it can be tested       */
};

/* Build the table for a loaded graph.  weight_sigma: HOST float[n_nodes] in the library's numbering
 * (entries of the leaves ignored), or NULL for dw = 0 everywhere.  Allocates device memory and
 * synchronises `stream` (a one-off at load time, L375).  Errors: MG_ERR_INVALID_ARG, MG_ERR_OOM
 * (the entry bound sum_n min(n_leaves, nnz(a) + nnz(b)) does not fit), MG_ERR_CUDA. */
int mg_mixture_lut_build(mg_graph *g, const float *weight_sigma, mg_mixture_lut **out, void *stream);
void mg_mixture_lut_free(mg_mixture_lut *lut);
int mg_mixture_lut_info(const mg_mixture_lut *lut, mg_lut_info *info);

/* Copy the table to the HOST (tests, export): row_ptr uint64[n_nodes + 1], then leaf uint32[nnz],
 * mu double[nnz], dmu double[nnz] in row order.  Any pointer may be NULL.  Synchronises. */
int mg_mixture_lut_export(const mg_mixture_lut *lut, uint64_t *row_ptr, uint32_t *leaf, double *mu, double *dmu);

/*
 * mg_range_query -- n_queries boxes in two launches: one zeroes the results, the other accumulates and -- in the last
 * CTA of every query to finish -- takes the square roots of Eq. 17 (no memsets, no separate finishing kernel).
 *   node_idx_mipmap  DEVICE uint32, all levels as `mip` describes (MG_QUERY_NAIVE reads level 0 only).
 *   boxes            HOST uint64[n_queries][6] = x0, y0, z0, x1, y1, z1, half-open, non-empty, inside
 *                    level 0 (validated).  Up to 64 boxes travel in the kernel parameters; larger batches are
 *                    copied into a table-owned staging buffer at enqueue (it grows, i.e. allocates, when
 *                    n_queries exceeds every earlier call's).
 *   expect, err      DEVICE double[n_queries][n_leaves]: expected voxels per leaf and its error
 *                    (err may be NULL).  sum_i expect[q][i] = volume of box q (L251).
 *   fetches          DEVICE uint64[n_queries] or NULL: samples fetched per query (Table 4).
 *   mode             MG_QUERY_FA, MG_QUERY_NAIVE or MG_QUERY_FA_WALK.
 * Enqueue-only apart from the staging copy of large batches.  Accumulation uses fp64 atomics: the result is the oracle's
 * up to summation order.
 */
int mg_range_query(mg_mixture_lut *lut, const uint32_t *node_idx_mipmap, const mg_mipmap_desc *mip,
                   const uint64_t *boxes, uint32_t n_queries, double *expect, double *err,
                   uint64_t *fetches, uint32_t mode, void *stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-4 (second half): device front end of the histogram mipmap (a0; Eq. 4).
 * The two finest levels hold 98 % of the mipmap's voxels and almost all of them are pure (Table 2);
 * classifying them is a stream over the volume.  These two calls do that on the device; the host builder
 * continues from their output (mgb_build_from_level1 of include/mg_builder.h) and produces the same graph and
 * node indices as mgb_build on the same volume.  Both calls allocate small temporaries and synchronise `stream`.
 * ------------------------------------------------------------------------------------------------ */

/* Level 0: H(., 0) = e_S (Eq. 4).  The sorted distinct segment IDs present in the volume become the leaves
 * (reading Q14: background is an ordinary segment).
 *   seg_device        DEVICE uint32[n_voxels] segment IDs (all < 2^28, else MG_ERR_INVALID_ARG: use mgb_build)
 *   level0_device     DEVICE uint32[n_voxels] receives the leaf number of every voxel; may be seg_device itself
 *   leaf_segment_id   HOST uint32[capacity] receives the sorted distinct IDs
 *   n_leaves          HOST: their number (also set when it exceeds capacity, which is MG_ERR_INVALID_ARG) */
int mg_mipmap_leaf_index(const uint32_t *seg_device, uint64_t n_voxels, uint32_t *level0_device,
                         uint32_t *leaf_segment_id, uint32_t capacity, uint32_t *n_leaves, void *stream);

/* Level 1: H(i, j, k, 1) = the average of the existing children (Eq. 4, reading Q2).  A parent whose existing
 * children are one leaf is that leaf; every other parent is listed with its children for the host builder.
 *   level0_device          DEVICE uint32[Z][Y][X] leaf numbers (x fastest)
 *   level1_device          DEVICE uint32[ceil(Z/2)][ceil(Y/2)][ceil(X/2)]: the leaf, or 0xFFFFFFFF for a listed parent
 *   mixed_voxel_device     DEVICE uint32[capacity]: level-1 voxel index of each listed parent (order unspecified)
 *   mixed_children_device  DEVICE uint32[capacity][8], 16-byte aligned: its children at [4 dz + 2 dy + dx],
 *                          0xFFFFFFFF for a child outside the volume
 *   n_mixed                HOST: number of listed parents; entries beyond `capacity` are dropped, so a caller seeing
 *                          n_mixed > capacity calls again with larger lists (level1_device is complete either way) */
int mg_mipmap_front_level1(const uint32_t *level0_device, uint64_t X, uint64_t Y, uint64_t Z,
                           uint32_t *level1_device, uint32_t *mixed_voxel_device, uint32_t *mixed_children_device,
                           uint64_t capacity, uint64_t *n_mixed, void *stream);

/*
 * The levels >= 1 on the device (second half of NEXT-4, continued; Eq. 4: only DISTINCT mixtures
 * reach the factorisation).  For l = 1, 2, ...: a parent whose existing children carry one mixture inherits it; every
 * other parent merges its children's sparse integer mixtures (each child weighing 1/N, reading Q2), divides by the common
 * power of two and hash-conses the result (64-bit hash, contents verified).  A HANDLE is a leaf number (< 2^31) or
 * 0x80000000 | mixture number (numbers in creation order: arbitrary).  A level in which one parent's children hold more
 * than 256 entries in total is left to the host together with the levels above it (the few thousand voxels whose
 * mixtures hold hundreds of segments): mgb_build_from_levels (include/mg_builder.h) continues from the last finished
 * level and yields the same graph and node indices as mgb_build on the same volume.
 *   level0_device   DEVICE uint32[Z][Y][X] leaf numbers (mg_mipmap_leaf_index)
 *   levels_device   DEVICE uint32 buffer; level l >= 1 is written at levels_device + level_offset[l] (handles, x fastest)
 *   level_offset    HOST uint64[n_levels] in voxels ([0] is not used); n_levels = length of the ceil-halving chain (L80)
 *   out             the mixture store (device memory owned by the table; mg_mixture_table_free)
 * Allocates (stores sized once, from the number of level-1 merges: 1.5 merges + 2^20 mixtures, 12 per merge + 2^22
 * entries) and synchronises `stream` several times per level.  A level whose mixtures do not fit the stores is not an
 * error: like a level with oversized mixtures it is left to the host together with the levels above it (a
 * nearest-neighbour-upsampled volume, whose level 1 is pure and whose level 2 holds all the merges, is such a case).
 * Everything in levels_device at or above level levels_done + 1 is scratch on return (half-written handles).
 * Errors: MG_ERR_INVALID_ARG (NULL, dims / n_levels mismatch, level 1 with >= 2^32 voxels, a 64-bit hash collision
 * between different mixtures), MG_ERR_OOM (a device allocation failed), MG_ERR_CUDA.
 *
 * mg_mipmap_levels_build_ex is the same call with the store capacities stated by the caller (cap_mixtures distinct
 * mixtures, cap_entries (leaf, count) entries; 0 = the default sizing above) -- to reserve more for data whose upper
 * levels are known to keep merging, or to bound the device memory the table may take (24 B per mixture + 40 B per
 * hash slot, 2 .. 4 slots per mixture; 12 B per entry).
 */
typedef struct mg_mixture_table mg_mixture_table;

typedef struct mg_mixture_table_info_t {
    uint64_t n_mixtures;    /* distinct mixtures with >= 2 non-zeros                                     */
    uint64_t n_entries;     /* their (leaf, count) entries                                              */
    uint64_t nnz_levels;    /* non-zeros summed over every voxel of the finished levels 1 .. levels_done */
    uint64_t device_bytes;  /* device memory owned by the table                                         */
    uint32_t levels_done;   /* last level built on the device (0: none)                                  */
    uint32_t n_leaves;
} mg_mixture_table_info_t;

int mg_mipmap_levels_build(const uint32_t *level0_device, uint64_t X, uint64_t Y, uint64_t Z, uint32_t n_leaves,
                           uint32_t *levels_device, const uint64_t *level_offset, uint32_t n_levels,
                           mg_mixture_table **out, void *stream);
int mg_mipmap_levels_build_ex(const uint32_t *level0_device, uint64_t X, uint64_t Y, uint64_t Z, uint32_t n_leaves,
                              uint32_t *levels_device, const uint64_t *level_offset, uint32_t n_levels,
                              uint64_t cap_mixtures, uint64_t cap_entries, mg_mixture_table **out, void *stream);
void mg_mixture_table_free(mg_mixture_table *t);
int mg_mixture_table_info(const mg_mixture_table *t, mg_mixture_table_info_t *info);

/* Copy the store to the HOST: per mixture its first entry (offset), non-zeros k, tlog (the reduced counts sum to
 * 2^tlog) and first occurrence (level << 40 | voxel: the scanline order of L257); then the entries (leaf ascending
 * inside a mixture, count).  Any pointer may be NULL.  Synchronises. */
int mg_mixture_table_export(const mg_mixture_table *t, uint64_t *offset, uint32_t *k, uint32_t *tlog,
                            uint64_t *first_pos, uint32_t *leaf, uint64_t *count);

/* handles[i] = node_of_mixture[id] for every handle 0x80000000 | id (leaf handles are node numbers already): turns the
 * device-built levels into node-index volumes once the host has numbered the mixtures' nodes.  DEVICE buffers.  Enqueue-only. */
int mg_mipmap_remap_handles(uint32_t *handles_device, uint64_t n, const uint32_t *node_of_mixture_device,
                            uint32_t n_mixtures, void *stream);

/* Thread-local description of the last error returned on this thread ("" if none). */
const char *mg_last_error(void);

/* Number of kernels the library has launched since it was loaded (for gpu_launches accounting). */
uint64_t mg_kernel_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* MG_H_ */
