/*
 * mg_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU implementation (fp64, integer-exact histograms) of what the
 * Mixture Graph's transfer-function propagation path computes.  Written from the paper only
 * ("L<n>" = line n of PAPER.md, arXiv 2009.02702); it shares no code, header, table or helper
 * with the CUDA library or the host builder and includes none of their files.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load it.  No blocking, fusion or reordering beyond what each cited definition states.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Table 2 voxel totals (O-1), brute force vs
 * recursion and the textbook box filter (O-2/O-3), Fig. 2 / Fig. 4 worked examples and closed-form
 * chains (O-4), mu . TF == colour and row sums (O-5), known values for the output conversions.
 *
 * Layout conventions: volumes are [Z][Y][X], x fastest; colours are 4 doubles (R,G,B,A) per entry.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- O-1: mip dimensions.  "we round up the resolution of each subsequent level ... until we
 * reach l = l_max with a resolution of 1^3 voxels" (L80).  dims_out[l] = {X_l, Y_l, Z_l}.
 * Returns the number of levels l_max + 1 (at most max_levels are written). */
int mgo_mip_dims(uint64_t x, uint64_t y, uint64_t z, uint64_t *dims_out, int max_levels)
{
    int l = 0;
    for (;;) {
        if (l < max_levels) {
            dims_out[3 * l + 0] = x;
            dims_out[3 * l + 1] = y;
            dims_out[3 * l + 2] = z;
        }
        l++;
        if (x == 1 && y == 1 && z == 1)
            return l;
        x = (x + 1) / 2;
        y = (y + 1) / 2;
        z = (z + 1) / 2;
    }
}

/* ---- O-2, level 0: H(i,j,k,0) = e_{S(i,j,k)} (Eq. 4 first line, L78).  Dense integer counts
 * counts[v][s], scaled so that every voxel's counts sum to 8^l (here 8^0 = 1).  seg_index[v] is
 * the leaf number (position in the sorted list of distinct IDs) of S(v). */
void mgo_hist_level0(const uint32_t *seg_index, uint64_t n_vox, uint32_t n_seg, uint64_t *counts)
{
    memset(counts, 0, (size_t)n_vox * n_seg * sizeof(uint64_t));
    for (uint64_t v = 0; v < n_vox; v++)
        counts[v * n_seg + seg_index[v]] = 1;
}

/* ---- O-2, level l from level l-1: H(i,j,k,l) = (1/N) sum over the EXISTING children
 * u in {2i,2i+1}, v in {2j,2j+1}, w in {2k,2k+1} of H(u,v,w,l-1), N = number of existing children
 * (Eq. 4 second line L78, with the garbled lower limit read as v = 2j; N per L80: "typically 8,
 * but potentially less than 8 at the borders"; reading Q2: N counts children).
 * N is 1, 2, 4 or 8, so with counts scaled to 8^l:  c(parent) = sum (8/N) c(child)  -- exact. */
void mgo_hist_next_level(const uint64_t *child, uint64_t cx, uint64_t cy, uint64_t cz,
                         uint32_t n_seg, uint64_t *parent)
{
    uint64_t px = (cx + 1) / 2, py = (cy + 1) / 2, pz = (cz + 1) / 2;
    for (uint64_t k = 0; k < pz; k++)
        for (uint64_t j = 0; j < py; j++)
            for (uint64_t i = 0; i < px; i++) {
                uint64_t *p = parent + ((k * py + j) * px + i) * n_seg;
                uint64_t n = 0;
                for (uint32_t s = 0; s < n_seg; s++)
                    p[s] = 0;
                for (uint64_t w = 2 * k; w <= 2 * k + 1; w++)
                    for (uint64_t v = 2 * j; v <= 2 * j + 1; v++)
                        for (uint64_t u = 2 * i; u <= 2 * i + 1; u++) {
                            if (u >= cx || v >= cy || w >= cz)
                                continue;
                            const uint64_t *c = child + ((w * cy + v) * cx + u) * n_seg;
                            for (uint32_t s = 0; s < n_seg; s++)
                                p[s] += c[s];
                            n++;
                        }
                for (uint32_t s = 0; s < n_seg; s++)
                    p[s] *= 8 / n;
            }
}

/* ---- O-2, direct colour: C_dir(v,l) = <H(v,l), TF> = (sum_s c_s TF[s]) / 8^l  -- the scalar
 * product of a mixture with the data vector (L66), summed in ascending segment order. */
void mgo_direct_colour(const uint64_t *counts, uint64_t n_vox, uint32_t n_seg, uint32_t level,
                       const double *tf, double *out)
{
    double scale = ldexp(1.0, -3 * (int)level); /* 1 / 8^l, exact */
    for (uint64_t v = 0; v < n_vox; v++)
        for (int ch = 0; ch < 4; ch++) {
            double acc = 0.0;
            for (uint32_t s = 0; s < n_seg; s++)
                acc += (double)counts[v * n_seg + s] * tf[4 * s + ch];
            out[4 * v + ch] = acc * scale;
        }
}

/* ---- O-3: brute force, non-recursive form of Eq. 4 for ONE voxel (i,j,k) of level l.
 * Unrolling the recursion, a finest voxel (x,y,z) with x>>l == i, y>>l == j, z>>l == k contributes
 * wx(x) wy(y) wz(z) to H(i,j,k,l)[S(x,y,z)], where along one axis w(x) = prod_{m=1..l} 1/n_m and
 * n_m = number of existing children (1 or 2) of x's ancestor at level m, i.e. of (x >> m) among
 * positions {2(x>>m), 2(x>>m)+1} of the level-(m-1) axis of size ceil(X0 / 2^(m-1)).
 * For power-of-two volumes every w is 2^-l and this is the textbook box filter count / 8^l. */
static double axis_weight(uint64_t x, uint64_t x0, uint32_t l)
{
    double w = 1.0;
    uint64_t size = x0; /* axis size at level m-1 */
    for (uint32_t m = 1; m <= l; m++) {
        uint64_t parent = x >> m;
        uint64_t n = (2 * parent + 1 < size) ? 2 : 1;
        w /= (double)n;
        size = (size + 1) / 2;
    }
    return w;
}

void mgo_brute_force_histogram(const uint32_t *seg_index, uint64_t x0, uint64_t y0, uint64_t z0,
                               uint32_t n_seg, uint32_t l, uint64_t i, uint64_t j, uint64_t k,
                               double *hist)
{
    for (uint32_t s = 0; s < n_seg; s++)
        hist[s] = 0.0;
    for (uint64_t z = 0; z < z0; z++) {
        if ((z >> l) != k)
            continue;
        for (uint64_t y = 0; y < y0; y++) {
            if ((y >> l) != j)
                continue;
            for (uint64_t x = 0; x < x0; x++) {
                if ((x >> l) != i)
                    continue;
                hist[seg_index[(z * y0 + y) * x0 + x]] +=
                    axis_weight(x, x0, l) * axis_weight(y, y0, l) * axis_weight(z, z0, l);
            }
        }
    }
}

/* ---- O-4: graph evaluation.  "assign colors to the source leaf nodes ... For each node, we
 * fetch data from its children and perform one interpolation" (L371); a triple (i, j, w) denotes
 * (1 - w) s_i + w s_j (L259) -- the weight multiplies the SECOND child; nodes are visited in index
 * order, valid because children precede parents (Eq. 8).  Leaves are nodes 0..n_leaves-1. */
void mgo_graph_eval(const uint32_t *child_a, const uint32_t *child_b, const double *weight,
                    uint64_t n_nodes, uint64_t n_leaves, const double *tf, double *c)
{
    for (uint64_t n = 0; n < n_leaves; n++)
        for (int ch = 0; ch < 4; ch++)
            c[4 * n + ch] = tf[4 * n + ch];
    for (uint64_t n = n_leaves; n < n_nodes; n++) {
        double w = weight[n];
        const double *ca = c + 4 * (uint64_t)child_a[n];
        const double *cb = c + 4 * (uint64_t)child_b[n];
        for (int ch = 0; ch < 4; ch++)
            c[4 * n + ch] = (1.0 - w) * ca[ch] + w * cb[ch];
    }
}

/* ---- NEXT-1: the same evaluation for ANY numeric segment attribute with n_ch channels per node.
 * "the Mixture Graph allows the efficient computation of any kind of numeric segmentation
 * attribute" (L269); the paper's own uses besides RGBA: opacity alone for empty-space skipping
 * (L271 (i)-(ii): "assigns opacity values of the current transfer function to the leafs,
 * propagates these values through the Mixture Graph") and diffuse / specular light contributions
 * (L277).  attr and c are [node][n_ch], channel fastest.  Same recurrence as mgo_graph_eval. */
void mgo_graph_eval_attr(const uint32_t *child_a, const uint32_t *child_b, const double *weight,
                         uint64_t n_nodes, uint64_t n_leaves, uint32_t n_ch, const double *attr,
                         double *c)
{
    for (uint64_t n = 0; n < n_leaves; n++)
        for (uint32_t ch = 0; ch < n_ch; ch++)
            c[n * n_ch + ch] = attr[n * n_ch + ch];
    for (uint64_t n = n_leaves; n < n_nodes; n++) {
        double w = weight[n];
        const double *ca = c + (uint64_t)child_a[n] * n_ch;
        const double *cb = c + (uint64_t)child_b[n] * n_ch;
        for (uint32_t ch = 0; ch < n_ch; ch++)
            c[n * n_ch + ch] = (1.0 - w) * ca[ch] + w * cb[ch];
    }
}

/* ---- Topological level (L211): sources 0; a node with predecessor values v1, v2 gets
 * max(v1, v2) + 1; "this amounts to a linear scan of all nodes".  Returns the depth (max level),
 * or -1 if a child index does not precede its parent (Eq. 8 violated). */
int64_t mgo_topo_levels(const uint32_t *child_a, const uint32_t *child_b, uint64_t n_nodes,
                        uint64_t n_leaves, uint32_t *level)
{
    int64_t depth = 0;
    for (uint64_t n = 0; n < n_leaves; n++)
        level[n] = 0;
    for (uint64_t n = n_leaves; n < n_nodes; n++) {
        if (child_a[n] >= n || child_b[n] >= n)
            return -1;
        uint32_t v1 = level[child_a[n]], v2 = level[child_b[n]];
        level[n] = (v1 > v2 ? v1 : v2) + 1;
        if ((int64_t)level[n] > depth)
            depth = level[n];
    }
    return depth;
}

/* ---- The paper's CPU baseline shape (L213, L373): "nodes with identical values can be processed
 * without synchronization" -- one OpenMP parallel-for per topological level, levels in ascending
 * order.  Same per-node arithmetic as mgo_graph_eval (results are bit-identical; tested).
 * order[] lists the internal nodes sorted by (level, index); level_start[L] .. level_start[L+1]
 * delimits level L (L = 1..depth) inside order[].  Returns the number of threads used. */
int mgo_graph_eval_levels(const uint32_t *child_a, const uint32_t *child_b, const double *weight,
                          uint64_t n_leaves, const uint64_t *order, const uint64_t *level_start,
                          uint32_t depth, const double *tf, double *c, int n_threads)
{
    int used = 1;
#ifdef _OPENMP
    if (n_threads > 0)
        omp_set_num_threads(n_threads);
    used = omp_get_max_threads();
#endif
    for (uint64_t n = 0; n < n_leaves; n++)
        for (int ch = 0; ch < 4; ch++)
            c[4 * n + ch] = tf[4 * n + ch];
    for (uint32_t L = 1; L <= depth; L++) {
        int64_t lo = (int64_t)level_start[L], hi = (int64_t)level_start[L + 1];
#pragma omp parallel for schedule(static)
        for (int64_t q = lo; q < hi; q++) {
            uint64_t n = order[q];
            double w = weight[n];
            const double *ca = c + 4 * (uint64_t)child_a[n];
            const double *cb = c + 4 * (uint64_t)child_b[n];
            for (int ch = 0; ch < 4; ch++)
                c[4 * n + ch] = (1.0 - w) * ca[ch] + w * cb[ch];
        }
    }
    return used;
}

/* ---- O-5: symbolic evaluation -- "assigning unit vectors e_i to leafs i followed by
 * propagation" (L321), the mixture lookup table of L375.  Dense mu[n][n_leaves]. */
void mgo_symbolic_eval(const uint32_t *child_a, const uint32_t *child_b, const double *weight,
                       uint64_t n_nodes, uint64_t n_leaves, double *mu)
{
    memset(mu, 0, (size_t)n_nodes * n_leaves * sizeof(double));
    for (uint64_t n = 0; n < n_leaves; n++)
        mu[n * n_leaves + n] = 1.0;
    for (uint64_t n = n_leaves; n < n_nodes; n++) {
        double w = weight[n];
        const double *ma = mu + (uint64_t)child_a[n] * n_leaves;
        const double *mb = mu + (uint64_t)child_b[n] * n_leaves;
        for (uint64_t s = 0; s < n_leaves; s++)
            mu[n * n_leaves + s] = (1.0 - w) * ma[s] + w * mb[s];
    }
}

/* ---- Palette lookup (L221 "essentially a paletted texture", L267 "The node ID is a direct
 * reference into the color lookup table"): C_graph(v) = c[node_idx[v]].
 * OpenMP over voxels only for the timed CPU baseline (independent iterations). */
int mgo_lookup(const uint32_t *node_idx, uint64_t n_vox, const double *c, double *out, int n_threads)
{
    int used = 1;
#ifdef _OPENMP
    if (n_threads > 0)
        omp_set_num_threads(n_threads);
    used = omp_get_max_threads();
#endif
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < (int64_t)n_vox; v++)
        for (int ch = 0; ch < 4; ch++)
            out[4 * v + ch] = c[4 * (uint64_t)node_idx[v] + ch];
    return used;
}

/* ---- Output conversion to RGBA8 (not in the paper, whose palette is vec4 float; defined by this
 * repo, reading Q13): clamp to [0,1], times 255, round half to even, R in byte 0.
 * The rounding DECISION is taken in fp32 like the kernel does (the colour is first rounded to
 * fp32, the product formed in fp32), so that both sides decide the integer in one precision. */
void mgo_to_rgba8(const double *c, uint64_t n, uint8_t *out)
{
    for (uint64_t i = 0; i < 4 * n; i++) {
        float f = (float)c[i];
        if (!(f > 0.0f))
            f = 0.0f; /* also maps NaN to 0 */
        if (f > 1.0f)
            f = 1.0f;
        float p = f * 255.0f;
        out[i] = (uint8_t)lrintf(p); /* default rounding mode: to nearest, ties to even */
    }
}

/* Same lookup + conversion as one pass, for the timed CPU baseline of the colourise step. */
int mgo_colourise_rgba8(const uint32_t *node_idx, uint64_t n_vox, const double *c, uint8_t *out,
                        int n_threads)
{
    int used = 1;
#ifdef _OPENMP
    if (n_threads > 0)
        omp_set_num_threads(n_threads);
    used = omp_get_max_threads();
#endif
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < (int64_t)n_vox; v++)
        mgo_to_rgba8(c + 4 * (uint64_t)node_idx[v], 1, out + 4 * v);
    return used;
}

/* ==== NEXT-3: bit-packed node-ID volumes (Table 1 rows (8), (9), (A); Eq. 15-16) ====
 *
 * "For each level of H, we compute the minimum and maximum ID of all nodes referenced in this
 * level ... We store i_min(l) in the bitstream's header for each l.  For each voxel, we then store
 * its node ID minus the minimum node ID of that level, again, using a fixed bitrate of
 * r(l) = ceil(log2(i_max(l) - i_min(l) + 1)) for each voxel in this level" (Eq. 15 read per level,
 * Q10; Eq. 16).  The shader addresses the stream by BIT address with 64-bit arithmetic (L267).
 * The paper does not fix the bit order; reading Q18: voxel v of the level occupies bits
 * [v r, (v+1) r) of the level's stream, bit q of the stream is bit (q mod 8) of byte q / 8 (LSB
 * first, little endian), and bit k of the stored value goes to stream bit v r + k. */

/* Eq. 16.  r = 0 when the level references a single node. */
uint32_t mgo_bits_per_voxel(uint32_t i_min, uint32_t i_max)
{
    uint64_t range = (uint64_t)i_max - (uint64_t)i_min + 1; /* number of representable IDs needed */
    uint32_t r = 0;
    while (((uint64_t)1 << r) < range)
        r++;
    return r;
}

/* Write value - i_min of every voxel, one bit at a time.  stream must be zero-initialised and hold
 * at least ceil(n r / 8) bytes. */
void mgo_pack_bits(const uint32_t *node_idx, uint64_t n_vox, uint32_t i_min, uint32_t r, uint8_t *stream)
{
    for (uint64_t v = 0; v < n_vox; v++) {
        uint32_t val = node_idx[v] - i_min;
        for (uint32_t k = 0; k < r; k++) {
            uint64_t q = v * (uint64_t)r + k;
            if ((val >> k) & 1u)
                stream[q >> 3] |= (uint8_t)(1u << (q & 7));
        }
    }
}

/* Inverse: node_idx[v] = i_min + the r-bit value at bit address v r. */
void mgo_unpack_bits(const uint8_t *stream, uint64_t n_vox, uint32_t i_min, uint32_t r, uint32_t *node_idx)
{
    for (uint64_t v = 0; v < n_vox; v++) {
        uint32_t val = 0;
        for (uint32_t k = 0; k < r; k++) {
            uint64_t q = v * (uint64_t)r + k;
            if ((stream[q >> 3] >> (q & 7)) & 1u)
                val |= 1u << k;
        }
        node_idx[v] = i_min + val;
    }
}
