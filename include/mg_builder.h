/*
 * mg_builder.h -- C ABI of the host-side Mixture Graph builder (pure host code, no CUDA).
 *
 * Builds, from a segment-ID volume, everything mg_load_graph / mg_colorize (include/mg.h) consume
 * (arXiv 2009.02702; "L<n>" = line n of PAPER.md):
 *   a0  normalised histogram mipmap, Eq. 4 (L76-L80): average of the existing children, dims
 *       ceil-halved down to 1^3.  Mixtures are kept as exact integer counts (every entry is a
 *       dyadic rational because N is 1, 2, 4 or 8) and hash-consed, so only DISTINCT mixtures are
 *       factorised.
 *   a1  factorisation into binary lerps, Eq. 5-7 (L88-L98), greedy max-reduction phi_2, Eq. 13-14
 *       (L162-L176), with the tau two-stage schedule (L257), node re-use keyed on
 *       (min child, max child, weight bin) (L130, L144, L361), scalar quantisation of the weights
 *       into 2^b uniform bins of (0,1) with centroid codewords and per-bin sigma (L176), and the
 *       interpolation symmetry (i,j,w) == (j,i,1-w) used to keep the lower-error side (L259).
 *   a2  topological levels (L211) and a relabelling that makes every level contiguous.
 *
 * Where the paper is silent the readings of DESIGN.md ("Readings") apply; in particular any
 * factorisation is valid (L144 "not unique") and the relaxations this builder makes for speed
 * (L319 anticipates them) are: mixtures with more than `big_cutoff` non-zeros are factorised as a
 * balanced tournament without the phi_2 search, and phi_2 falls back to frozen norms when the
 * exact score maintenance would exceed `phi2_exact_budget` updates.
 *
 * Conventions: all pointers are HOST pointers; volumes are [Z][Y][X] with x fastest; every call
 * returns 0 (MGB_OK) or a negative code, with a thread-local message from mgb_last_error().
 * The result handle owns its arrays; getters copy into caller-owned buffers (NULL = skip).
 */
#ifndef MG_BUILDER_H_
#define MG_BUILDER_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mgb_result mgb_result;

enum { MGB_OK = 0, MGB_ERR_INVALID_ARG = -1, MGB_ERR_OOM = -4, MGB_ERR_LIMIT = -5 };

enum { MGB_PICK_SMALLEST_INDEX = 0, /* stage 2 pairs the two smallest node indices (FIFO tournament,
                                       depth ceil(log2 k)); default                                   */
       MGB_PICK_SMALLEST_MASS = 1   /* pairs the two smallest masses (the order Fig. 2 shows)         */ };

typedef struct mgb_params {
    uint32_t quant_bits;        /* b in [1,16] (L189); 0 = unquantised: exact ratios, no merging      */
    uint32_t tau;               /* stage-1 cutoff (L257); paper: 3                                     */
    uint32_t big_cutoff;        /* mixtures with more non-zeros skip phi_2 (balanced tournament); 0 = never */
    uint32_t pick_order;        /* MGB_PICK_*                                                          */
    uint32_t n_threads;         /* 0 = all cores                                                       */
    uint32_t relabel;           /* 1 = output level-contiguous numbering (a2); 0 = creation order      */
    uint64_t phi2_exact_budget; /* max score updates for exact phi_2; above it norms are frozen        */
} mgb_params;

typedef struct mgb_info {
    uint64_t dims[3];            /* X, Y, Z of level 0                                                 */
    uint32_t n_mip_levels;       /* l_max + 1                                                          */
    uint32_t n_leaves;           /* distinct segment IDs present (background included, Q14)            */
    uint64_t n_voxels_total;     /* voxels of all mip levels                                           */
    uint64_t n_nodes;            /* leaves + internal nodes                                            */
    uint32_t depth;              /* topological depth (L211)                                           */
    uint32_t quant_bits;
    uint64_t n_distinct_mixtures;/* hash-consed mixtures with >= 2 non-zeros                           */
    uint64_t nnz_total;          /* sum over all voxels of all levels of ||H||_0 (Table 2 "non-zeros") */
    uint64_t n_stage1;           /* mixtures factorised by the phi_2 search (tau < k <= big_cutoff)    */
    uint64_t n_stage2;           /* mixtures with k <= tau (scanline stage)                            */
    uint64_t n_big;              /* mixtures above big_cutoff                                          */
    uint32_t phi2_exact;         /* 1 if the exact phi_2 maintenance was used                          */
    uint32_t reserved;
    double max_bin_sigma;        /* max over bins of the empirical rms deviation (Table 3 "error")     */
    double seconds_mipmap, seconds_factorise, seconds_finalise;
} mgb_info;

/* Defaults: b = 9 (L305), tau = 3 (L257), big_cutoff = 32, smallest-index order, all cores,
 * relabel = 1, phi2_exact_budget = 2e9. */
void mgb_default_params(mgb_params *p);

/* Build from a segment-ID volume seg[Z][Y][X] (uint32; IDs may be sparse; every distinct ID present
 * becomes one leaf, in increasing ID order). */
int mgb_build(const uint32_t *seg, uint64_t X, uint64_t Y, uint64_t Z, const mgb_params *params,
              mgb_result **out);

/*
 * mgb_build_from_level1 -- mgb_build for a volume whose two finest levels were classified elsewhere (the device
 * front end mg_mipmap_leaf_index / mg_mipmap_front_level1 of include/mg.h: level 0 is 87 % of the mipmap and the
 * classification is a pure stream).  The result is identical to mgb_build on the same volume, except that the node
 * index of level 0 is not stored: it is the leaf number, which the caller already has (mgb_get_node_idx(level 0)
 * fails, mgb_node_idx_ptr returns NULL).
 *   X, Y, Z          dimensions of level 0
 *   leaf_segment_id  uint32[n_leaves] sorted distinct segment IDs present (Q14)
 *   level1           uint32[X_1 Y_1 Z_1] (ceil-halved dims): the leaf number of every parent whose existing children
 *                    are one segment, 0xFFFFFFFF for every other parent; may be NULL for a 1 x 1 x 1 volume
 *   mixed_voxel      uint32[n_mixed] level-1 voxel index of every 0xFFFFFFFF parent, each exactly once, any order
 *   mixed_children   uint32[n_mixed][8] leaf numbers of its existing children (2, 4 or 8 of them, Eq. 4 / Q2),
 *                    0xFFFFFFFF for children outside the volume; their order does not matter
 * Errors: MGB_ERR_INVALID_ARG when the three arrays are inconsistent.
 */
int mgb_build_from_level1(uint64_t X, uint64_t Y, uint64_t Z, const uint32_t *leaf_segment_id, uint32_t n_leaves,
                          const uint32_t *level1, const uint32_t *mixed_voxel, const uint32_t *mixed_children,
                          uint64_t n_mixed, const mgb_params *params, mgb_result **out);

/*
 * mgb_build_from_levels -- mgb_build for a volume whose levels 0 .. level_done of the histogram mipmap were built
 * elsewhere (mg_mipmap_leaf_index + mg_mipmap_levels_build of include/mg.h).  The caller lists the distinct mixtures
 * found there and passes the handles of the last finished level; the host continues with Eq. 4 from level_done + 1,
 * then factorises.  Same graph, same node numbering as mgb_build on the same volume.  The node indices of the levels
 * 0 .. level_done - 1 are not stored (mgb_get_node_idx fails for them): they follow from the caller's handles through
 * mgb_get_front_mixture_nodes (mg_mipmap_remap_handles applies it on the device).
 *   level_done      1 .. l_max
 *   handles         uint32[voxels of level_done]: a leaf number, or 0x80000000 | q for the q-th listed mixture
 *   mix_offset/k/tlog/first_pos   per listed mixture: first entry, non-zeros (>= 2), log2 of the sum of its counts,
 *                   first occurrence level << 40 | voxel (the scanline order the canonical numbering sorts by, L257)
 *   leaf, count     entries (leaves ascending inside a mixture; counts reduced: not all even)
 *   nnz_levels      non-zeros summed over every voxel of the levels 1 .. level_done (statistics only)
 * Errors: MGB_ERR_INVALID_ARG for malformed mixtures or handles.
 */
int mgb_build_from_levels(uint64_t X, uint64_t Y, uint64_t Z, const uint32_t *leaf_segment_id, uint32_t n_leaves,
                          uint32_t level_done, const uint32_t *handles, uint64_t n_mixtures, const uint64_t *mix_offset,
                          const uint32_t *mix_k, const uint32_t *mix_tlog, const uint64_t *mix_first_pos,
                          const uint32_t *leaf, const uint64_t *count, uint64_t n_entries, uint64_t nnz_levels,
                          const mgb_params *params, mgb_result **out);

/* node_of_mixture[q] = node (final numbering) of the q-th mixture listed to mgb_build_from_levels. */
int mgb_get_front_mixture_nodes(const mgb_result *r, uint32_t *node_of_mixture);

/* Build from explicit mixtures instead of a volume (tests, Fig. 2): mixture m has entries
 * [offsets[m], offsets[m+1]) of (leaf[], count[]) with strictly increasing leaf numbers < n_leaves
 * and positive integer counts (any scale).  The result has one "mip level" holding n_mixtures
 * "voxels": node index of each mixture. */
int mgb_build_from_mixtures(uint32_t n_leaves, uint64_t n_mixtures, const uint64_t *offsets,
                            const uint32_t *leaf, const uint64_t *count, const mgb_params *params,
                            mgb_result **out);

void mgb_free(mgb_result *r);
int mgb_get_info(const mgb_result *r, mgb_info *info);

/* dims_out: uint64[3 * n_mip_levels] = X_l, Y_l, Z_l per level. */
int mgb_mip_dims(const mgb_result *r, uint64_t *dims_out);

/* The ceil-halving chain of L80 for a volume that has not been built yet: "we round up the resolution of each
 * subsequent level ... until we reach l = l_max with a resolution of 1^3 voxels".  Writes X_l, Y_l, Z_l of at most
 * max_levels levels and returns the number of levels l_max + 1 (0 for a zero dimension).  Host only. */
uint32_t mgb_mip_chain(uint64_t X, uint64_t Y, uint64_t Z, uint64_t *dims_out, uint32_t max_levels);

/* Copy the graph out.  child_a/child_b/weight/weight_exact have n_nodes entries (leaves' entries 0),
 * level_offsets depth + 2, leaf_segment_id n_leaves.  weight = fp32 codeword (or fp32 of the exact
 * ratio when unquantised), weight_exact = mean of the exact ratios merged into the node (fp64),
 * oriented like weight (it multiplies child_b). */
int mgb_get_graph(const mgb_result *r, uint32_t *child_a, uint32_t *child_b, float *weight,
                  double *weight_exact, uint64_t *level_offsets, uint32_t *leaf_segment_id);

/* delta w of Eq. 18 per node: float[n_nodes], the empirical standard deviation of the quantiser bin the
 * node's codeword was taken from (L176: "we store an empirical standard deviation sigma for each bin to
 * facilitate estimating the error"); 0 for leaves and for unquantised builds. */
int mgb_get_weight_sigma(const mgb_result *r, float *weight_sigma);

/* Node index (in the numbering of mgb_get_graph) of every voxel of one mip level:
 * uint32[Z_l * Y_l * X_l].  mgb_node_idx_ptr returns the builder-owned array (valid until
 * mgb_free), mgb_get_node_idx copies it. */
const uint32_t *mgb_node_idx_ptr(const mgb_result *r, uint32_t level);
int mgb_get_node_idx(const mgb_result *r, uint32_t level, uint32_t *out);

/* Scalar quantiser codebook: 2^b fp32 codewords and per-bin sigma (L176); count[] = weights merged
 * into the bin.  Unquantised builds have no codebook (returns MGB_ERR_INVALID_ARG). */
int mgb_get_codebook(const mgb_result *r, float *codeword, float *sigma, uint64_t *count);

const char *mgb_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MG_BUILDER_H_ */
