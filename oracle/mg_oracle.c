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
 * recursion and the textbook box filter (O-2/O-3/O-3c), Fig. 2 / Fig. 4 worked examples and closed-form
 * chains (O-4), mu . TF == colour and row sums (O-5), known values for the output conversions;
 * hand-worked rays / scipy map_coordinates / Beer-Lambert closed forms (ray-marcher, R1-R6); Table 4's fetch
 * counts, brute-force tilings, np.bincount and the sum-to-volume identity (range queries); a hand-worked
 * case for Eq. 18 (the only pin it has).
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

/* ---- O-3 for EVERY voxel of level l at once: the same unrolled Eq. 4 as mgo_brute_force_histogram, visited in
 * the order of the finest voxels instead of once per coarse voxel -- finest voxel (x,y,z) adds
 * wx(x) wy(y) wz(z) to H(x>>l, y>>l, z>>l, l)[S(x,y,z)].  The three axis weights are tabulated first (axis_weight
 * of every coordinate), nothing else differs.  hist is dense [Z_l][Y_l][X_l][n_seg], Z_l = ceil-halved l times.
 * Pins: mgo_brute_force_histogram voxel by voxel, the recursion (O-2) on ragged volumes, count / 8^l on
 * power-of-two ones (tests/test_oracle_pins.py). */
void mgo_brute_force_level(const uint32_t *seg_index, uint64_t x0, uint64_t y0, uint64_t z0,
                           uint32_t n_seg, uint32_t l, double *hist)
{
    uint64_t xl = x0, yl = y0, zl = z0;
    for (uint32_t m = 0; m < l; m++) {
        xl = (xl + 1) / 2;
        yl = (yl + 1) / 2;
        zl = (zl + 1) / 2;
    }
    double *wx = (double *)malloc(x0 * sizeof(double));
    double *wy = (double *)malloc(y0 * sizeof(double));
    double *wz = (double *)malloc(z0 * sizeof(double));
    for (uint64_t x = 0; x < x0; x++) wx[x] = axis_weight(x, x0, l);
    for (uint64_t y = 0; y < y0; y++) wy[y] = axis_weight(y, y0, l);
    for (uint64_t z = 0; z < z0; z++) wz[z] = axis_weight(z, z0, l);
    memset(hist, 0, (size_t)(xl * yl * zl) * n_seg * sizeof(double));
    /* coarse z-slabs are independent: one thread per k, every thread walks its own finest z range in order */
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < (int64_t)zl; k++) {
        for (uint64_t z = (uint64_t)k << l; z < z0 && (z >> l) == (uint64_t)k; z++)
            for (uint64_t y = 0; y < y0; y++) {
                double *row = hist + (((uint64_t)k * yl + (y >> l)) * xl) * n_seg;
                const uint32_t *s = seg_index + (z * y0 + y) * x0;
                double wzy = wz[z] * wy[y];
                for (uint64_t x = 0; x < x0; x++)
                    row[(x >> l) * n_seg + s[x]] += wx[x] * wzy;
            }
    }
    free(wx);
    free(wy);
    free(wz);
}

/* ---- O-3c: the COLOUR of every voxel of level l straight from the definition, for volumes whose dense histogram
 * table would not fit: C_dir(i,j,k,l) = <H(i,j,k,l), TF> = sum_s H(i,j,k,l)[s] TF[s] (L66 with the histogram of Eq. 4,
 * L78-L80).  With H unrolled as in O-3 -- finest voxel (x,y,z) contributes wx(x) wy(y) wz(z) to bin S(x,y,z) of its
 * level-l ancestor -- the sum over bins becomes a sum over the ancestor's finest voxels,
 *     C_dir(i,j,k,l) = sum_{(x,y,z): x>>l == i, y>>l == j, z>>l == k}  wx(x) wy(y) wz(z) TF[S(x,y,z)],
 * which is what is accumulated here, one finest voxel after the other; no histogram is formed.  Only the coarse
 * z-slabs k_begin <= k < k_end are computed (the caller bounds the memory): out is [k_end - k_begin][Y_l][X_l][4].
 * Pins (tests/test_oracle_pins.py): direct_colour of the recursion's integer histograms (O-2) on a ragged volume,
 * slab by slab; numpy's box mean of TF[S] on a power-of-two volume; exact fractions on the 5 x 1 x 1 border case. */
void mgo_direct_colour_level(const uint32_t *seg_index, uint64_t x0, uint64_t y0, uint64_t z0,
                             const double *tf, uint32_t l, uint64_t k_begin, uint64_t k_end, double *out)
{
    uint64_t xl = x0, yl = y0;
    for (uint32_t m = 0; m < l; m++) {
        xl = (xl + 1) / 2;
        yl = (yl + 1) / 2;
    }
    double *wx = (double *)malloc(x0 * sizeof(double));
    double *wy = (double *)malloc(y0 * sizeof(double));
    double *wz = (double *)malloc(z0 * sizeof(double));
    for (uint64_t x = 0; x < x0; x++) wx[x] = axis_weight(x, x0, l);
    for (uint64_t y = 0; y < y0; y++) wy[y] = axis_weight(y, y0, l);
    for (uint64_t z = 0; z < z0; z++) wz[z] = axis_weight(z, z0, l);
    memset(out, 0, (size_t)((k_end - k_begin) * yl * xl) * 4 * sizeof(double));
    /* the coarse rows (k, j) are independent: one thread per row, walking its own finest voxels in (z, y, x) order */
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
    for (int64_t k = (int64_t)k_begin; k < (int64_t)k_end; k++)
        for (int64_t j = 0; j < (int64_t)yl; j++) {
            double *row = out + ((((uint64_t)k - k_begin) * yl + (uint64_t)j) * xl) * 4;
            for (uint64_t z = (uint64_t)k << l; z < z0 && (z >> l) == (uint64_t)k; z++)
                for (uint64_t y = (uint64_t)j << l; y < y0 && (y >> l) == (uint64_t)j; y++) {
                    const uint32_t *s = seg_index + (z * y0 + y) * x0;
                    double wzy = wz[z] * wy[y];
                    for (uint64_t x = 0; x < x0; x++) {
                        double w = wx[x] * wzy;
                        const double *c = tf + 4 * (uint64_t)s[x];
                        double *o = row + 4 * (x >> l);
                        for (int ch = 0; ch < 4; ch++)
                            o[ch] += w * c[ch];
                    }
                }
        }
    free(wx);
    free(wy);
    free(wz);
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

/* ==== NEXT-2: ray-marching the paletted histogram mipmap (section 4) ====
 *
 * "rendering from the Mixture Graph is the same as rendering from a paletted texture" (L267): a
 * sample fetches node IDs, looks their colours up in the palette, and "we still have to perform the
 * computation of the mip level as well as the interpolation in the shader manually" (L269).
 * The paper gives the ingredients, not formulas; the readings (R1-R8) are:
 *  R1 camera     pinhole; pixel (i, j) of a W x H image looks along
 *                d = normalise(forward + u right + v up), u = (2 (i + 1/2) / W - 1) tan_half_fov W / H,
 *                v = (1 - 2 (j + 1/2) / H) tan_half_fov; world units, voxel (x,y,z) of level 0
 *                occupies [x sx, (x+1) sx] x ... (spacing s; "anisotropic voxels up to 1:1:7", L277).
 *  R2 LOD        "the pixel coverage of a voxel is linear in viewspace depth z" (L269, GL 4.5 8.14):
 *                rho = z_view (2 tan_half_fov / H) / s_ref voxels per pixel, s_ref = min spacing,
 *                lambda = clamp(log2(rho) + lod_bias, 0, l_max).
 *  R3 sample     GL_LINEAR_MIPMAP_LINEAR by hand: l0 = floor(lambda), f = lambda - l0, l1 = min(l0+1, l_max);
 *                colour = (1 - f) tri(l0) + f tri(l1); tri(l) = trilinear interpolation of the 8
 *                palette colours around p, voxel i of level l centred at (i + 1/2) 2^l level-0 voxels,
 *                indices clamped to the level's extent; the four floats are interpolated as given (Q11).
 *  R4 step       "the step size of a volume raymarcher can be adjusted to the LOD, which requires opacity
 *                correction" (L269): Delta = step_voxels s_ref 2^lambda (0.5-voxel steps at full
 *                resolution, L414); alpha' = 1 - (1 - alpha)^(Delta / (ref_step_voxels s_ref)).
 *  R5 march      t from the entry of the volume's box; lambda and Delta from the interval start t, the
 *                last interval is clipped to the exit, the sample sits at the interval's mid-point;
 *                front-to-back: C += (1 - A) alpha' rgb, A += (1 - A) alpha'; stop at A >= alpha_cutoff.
 *  R6 ESS        (L271) the opacity hierarchy is the A channel of the palette on the coarser mip levels.
 *                A ray is in "empty mode" when it enters the volume and after every sample that was skipped or
 *                whose interpolated opacity fell below the threshold; it leaves it with the first sample at or
 *                above the threshold ("uses the hierarchy for skipping longer segments": the hierarchy is only
 *                consulted where the ray is in empty space).  In empty mode, before a sample is fetched: from
 *                level l1 + 1 upwards, "as long as the opacity value in parent voxels falls below a certain
 *                threshold" climb; the largest such block [lo, hi) is remembered and every sample whose
 *                16-voxel footprint lies inside it is skipped: trilinear at level l reads voxels
 *                floor(p / 2^l - 1/2) and the next one, both inside the block iff
 *                lo + 2^l / 2 <= p < hi - 2^l / 2; l = l1 is the binding level (no shrinking at faces
 *                on the volume's boundary, where the fetch clamps to the edge).
 * Output: [H][W][4] = (C_r, C_g, C_b, A), associated colour over a transparent background. */

typedef struct mgo_view {
    const uint32_t *node_idx;      /* all levels concatenated */
    const uint64_t *level_offset;  /* [n_levels] first voxel of each level */
    const uint32_t *level_dim;     /* [n_levels][3] = X_l, Y_l, Z_l */
    uint32_t n_levels;
    const double *palette;         /* [n_nodes][4] */
} mgo_view;

static const double *mgo_voxel_colour(const mgo_view *v, uint32_t l, int64_t i, int64_t j, int64_t k)
{
    const uint32_t *d = v->level_dim + 3 * l;
    if (i < 0) i = 0;
    if (j < 0) j = 0;
    if (k < 0) k = 0;
    if (i > (int64_t)d[0] - 1) i = (int64_t)d[0] - 1;
    if (j > (int64_t)d[1] - 1) j = (int64_t)d[1] - 1;
    if (k > (int64_t)d[2] - 1) k = (int64_t)d[2] - 1;
    uint64_t lin = ((uint64_t)k * d[1] + (uint64_t)j) * d[0] + (uint64_t)i;
    return v->palette + 4 * (uint64_t)v->node_idx[v->level_offset[l] + lin];
}

/* R3, one level: trilinear interpolation at p (level-0 voxel coordinates). */
static void mgo_trilinear(const mgo_view *v, uint32_t l, const double p[3], double out[4])
{
    double scale = ldexp(1.0, -(int)l);
    double u[3], fr[3];
    int64_t i0[3];
    for (int a = 0; a < 3; a++) {
        u[a] = p[a] * scale - 0.5;
        double fl = floor(u[a]);
        i0[a] = (int64_t)fl;
        fr[a] = u[a] - fl;
    }
    for (int ch = 0; ch < 4; ch++)
        out[ch] = 0.0;
    for (int dz = 0; dz < 2; dz++)
        for (int dy = 0; dy < 2; dy++)
            for (int dx = 0; dx < 2; dx++) {
                double wgt = (dx ? fr[0] : 1.0 - fr[0]) * (dy ? fr[1] : 1.0 - fr[1]) * (dz ? fr[2] : 1.0 - fr[2]);
                const double *c = mgo_voxel_colour(v, l, i0[0] + dx, i0[1] + dy, i0[2] + dz);
                for (int ch = 0; ch < 4; ch++)
                    out[ch] += wgt * c[ch];
            }
}

/* R3: colour at p for a fractional level lambda in [0, l_max]. */
void mgo_sample_lod(const uint32_t *node_idx, const uint64_t *level_offset, const uint32_t *level_dim,
                    uint32_t n_levels, const double *palette, const double *p_vox, double lambda,
                    double *out)
{
    mgo_view v = {node_idx, level_offset, level_dim, n_levels, palette};
    uint32_t l_max = n_levels - 1;
    if (lambda < 0.0) lambda = 0.0;
    if (lambda > (double)l_max) lambda = (double)l_max;
    uint32_t l0 = (uint32_t)floor(lambda);
    uint32_t l1 = l0 + 1 > l_max ? l_max : l0 + 1;
    double f = lambda - (double)l0;
    double c0[4], c1[4];
    mgo_trilinear(&v, l0, p_vox, c0);
    mgo_trilinear(&v, l1, p_vox, c1);
    for (int ch = 0; ch < 4; ch++)
        out[ch] = (1.0 - f) * c0[ch] + f * c1[ch];
}

/* R1: direction of pixel (i, j).  cam = eye[3], right[3], up[3], forward[3]. */
void mgo_pixel_ray(const double *cam, double tan_half_fov, uint32_t W, uint32_t H, uint32_t i, uint32_t j,
                   double *dir)
{
    double u = (2.0 * ((double)i + 0.5) / (double)W - 1.0) * tan_half_fov * (double)W / (double)H;
    double v = (1.0 - 2.0 * ((double)j + 0.5) / (double)H) * tan_half_fov;
    double n = 0.0;
    for (int a = 0; a < 3; a++) {
        dir[a] = cam[9 + a] + u * cam[3 + a] + v * cam[6 + a];
        n += dir[a] * dir[a];
    }
    n = sqrt(n);
    for (int a = 0; a < 3; a++)
        dir[a] /= n;
}

/* Slab test of the ray eye + t dir against the box [0, ext].  Returns 0 on a miss. */
static int mgo_ray_box(const double *eye, const double *dir, const double *ext, double *t_near, double *t_far)
{
    double tn = 0.0, tf = INFINITY;
    for (int a = 0; a < 3; a++) {
        if (dir[a] == 0.0) {
            if (eye[a] < 0.0 || eye[a] > ext[a])
                return 0;
        } else {
            double t1 = (0.0 - eye[a]) / dir[a], t2 = (ext[a] - eye[a]) / dir[a];
            double lo = t1 < t2 ? t1 : t2, hi = t1 < t2 ? t2 : t1;
            if (lo > tn) tn = lo;
            if (hi < tf) tf = hi;
        }
    }
    if (!(tn < tf))
        return 0;
    *t_near = tn;
    *t_far = tf;
    return 1;
}

/* R2-R6 for one ray.  par = tan_half_fov, sx, sy, sz, step_voxels, ref_step_voxels, lod_bias,
 * ess_threshold (< 0: no empty-space skipping), alpha_cutoff.  stats[0] += samples evaluated,
 * stats[1] += samples skipped. */
static void mgo_march(const mgo_view *v, const double *cam, const double *par, uint32_t H, const double *dir,
                      double *rgba, uint64_t *stats)
{
    const double tanh_ = par[0], *s = par + 1, step = par[4], ref = par[5], bias = par[6], thr = par[7], cutoff = par[8];
    const uint32_t l_max = v->n_levels - 1;
    const double s_ref = fmin(s[0], fmin(s[1], s[2]));
    double ext[3];
    for (int a = 0; a < 3; a++)
        ext[a] = (double)v->level_dim[a] * s[a];
    double C[3] = {0, 0, 0}, A = 0.0;
    rgba[0] = rgba[1] = rgba[2] = rgba[3] = 0.0;
    double t_near, t_far;
    if (!mgo_ray_box(cam, dir, ext, &t_near, &t_far))
        return;
    double cos_view = dir[0] * cam[9] + dir[1] * cam[10] + dir[2] * cam[11];
    int box_valid = 0;
    double box_lo[3] = {0, 0, 0}, box_hi[3] = {0, 0, 0};
    int box_open_lo[3] = {0, 0, 0}, box_open_hi[3] = {0, 0, 0};     /* face on the volume's boundary */
    int empty_mode = 1;                                             /* R6: a ray enters the volume in empty mode */
    double t = t_near;
    while (t < t_far && A < cutoff) {
        double rho = t * cos_view * (2.0 * tanh_ / (double)H) / s_ref;              /* R2 */
        double lambda = rho > 0.0 ? log2(rho) + bias : 0.0;
        if (lambda < 0.0) lambda = 0.0;
        if (lambda > (double)l_max) lambda = (double)l_max;
        double delta = step * s_ref * exp2(lambda);                                 /* R4 */
        double de = delta < t_far - t ? delta : t_far - t;                          /* R5 */
        double ts = t + 0.5 * de;
        double p[3];
        for (int a = 0; a < 3; a++)
            p[a] = (cam[a] + ts * dir[a]) / s[a];
        uint32_t l0 = (uint32_t)floor(lambda);
        uint32_t l1 = l0 + 1 > l_max ? l_max : l0 + 1;
        double f = lambda - (double)l0;
        t += delta;
        if (thr >= 0.0 && empty_mode) {                                             /* R6 */
            double m = 0.5 * ldexp(1.0, (int)l1);
            int inside = 0;
            if (box_valid) {
                inside = 1;
                for (int a = 0; a < 3; a++)
                    if ((!box_open_lo[a] && p[a] < box_lo[a] + m) || (!box_open_hi[a] && p[a] >= box_hi[a] - m))
                        inside = 0;
            }
            if (!inside) {
                box_valid = 0;
                for (uint32_t L = l1 + 1; L <= l_max; L++) {
                    const uint32_t *d = v->level_dim + 3 * L;
                    int64_t q[3];
                    for (int a = 0; a < 3; a++) {
                        q[a] = (int64_t)floor(ldexp(p[a], -(int)L));
                        if (q[a] < 0) q[a] = 0;
                        if (q[a] > (int64_t)d[a] - 1) q[a] = (int64_t)d[a] - 1;
                    }
                    if (!(mgo_voxel_colour(v, L, q[0], q[1], q[2])[3] < thr))
                        break;
                    box_valid = 1;
                    for (int a = 0; a < 3; a++) {
                        box_lo[a] = ldexp((double)q[a], (int)L);
                        box_hi[a] = ldexp((double)(q[a] + 1), (int)L);
                        box_open_lo[a] = q[a] == 0;
                        box_open_hi[a] = q[a] == (int64_t)d[a] - 1;
                    }
                }
                if (box_valid) {
                    inside = 1;
                    for (int a = 0; a < 3; a++)
                        if ((!box_open_lo[a] && p[a] < box_lo[a] + m) || (!box_open_hi[a] && p[a] >= box_hi[a] - m))
                            inside = 0;
                }
            }
            if (inside) {
                if (stats) stats[1]++;
                continue;
            }
        }
        double c0[4], c1[4], c[4];
        mgo_trilinear(v, l0, p, c0);
        mgo_trilinear(v, l1, p, c1);
        for (int ch = 0; ch < 4; ch++)
            c[ch] = (1.0 - f) * c0[ch] + f * c1[ch];
        double alpha = c[3] < 0.0 ? 0.0 : (c[3] > 1.0 ? 1.0 : c[3]);
        empty_mode = alpha < thr;                                                   /* R6 */
        double ac = 1.0 - pow(1.0 - alpha, de / (ref * s_ref));                      /* R4 */
        for (int ch = 0; ch < 3; ch++)
            C[ch] += (1.0 - A) * ac * c[ch];
        A += (1.0 - A) * ac;
        if (stats) stats[0]++;
    }
    rgba[0] = C[0]; rgba[1] = C[1]; rgba[2] = C[2]; rgba[3] = A;
}

/* The image: every pixel (i, j), j = row from the top.  out = [H][W][4] doubles. */
void mgo_render(const uint32_t *node_idx, const uint64_t *level_offset, const uint32_t *level_dim,
                uint32_t n_levels, const double *palette, const double *cam, const double *par,
                uint32_t W, uint32_t H, double *out, uint64_t *stats)
{
    mgo_view v = {node_idx, level_offset, level_dim, n_levels, palette};
    uint64_t st[2] = {0, 0};
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : st[:2])
    for (int64_t j = 0; j < (int64_t)H; j++)
        for (uint32_t i = 0; i < W; i++) {
            double dir[3];
            uint64_t loc[2] = {0, 0};
            mgo_pixel_ray(cam, par[0], W, H, i, (uint32_t)j, dir);
            mgo_march(&v, cam, par, H, dir, out + 4 * ((uint64_t)j * W + i), loc);
            st[0] += loc[0];
            st[1] += loc[1];
        }
    if (stats) { stats[0] = st[0]; stats[1] = st[1]; }
}

/* Selected pixels of the same image (full-size parity on sampled outputs): pixel q = (ij[2q], ij[2q+1])
 * = (column i, row j) of the W x H image; out = [n_pix][4].  Same per-ray code as mgo_render. */
void mgo_render_pixels(const uint32_t *node_idx, const uint64_t *level_offset, const uint32_t *level_dim,
                       uint32_t n_levels, const double *palette, const double *cam, const double *par,
                       uint32_t W, uint32_t H, const uint32_t *ij, uint64_t n_pix, double *out, uint64_t *stats)
{
    mgo_view v = {node_idx, level_offset, level_dim, n_levels, palette};
    uint64_t st[2] = {0, 0};
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : st[:2])
    for (int64_t q = 0; q < (int64_t)n_pix; q++) {
        double dir[3];
        uint64_t loc[2] = {0, 0};
        mgo_pixel_ray(cam, par[0], W, H, ij[2 * q], ij[2 * q + 1], dir);
        mgo_march(&v, cam, par, H, dir, out + 4 * q, loc);
        st[0] += loc[0];
        st[1] += loc[1];
    }
    if (stats) { stats[0] = st[0]; stats[1] = st[1]; }
}

/* ==== NEXT-4: mixture lookup table with error propagation, and sub-volume (range) queries ====
 * PAPER.md section 3.5 (Eq. 17-18), section 3.6 (L243-L253), L375-L377, Table 4.
 *
 * Mixture lookup table (L375): "assigning a mixture e_i with variance 0 to each leaf node i ... we
 * propagate this information through the DAG, including the error described in Eq. (18).  Each node
 * thus stores ... the expected value mu and its variance delta mu."  Dense here: mu, dmu = [n_nodes][n_leaves].
 *   mu_i  = (1 - w) a_i + w b_i
 *   dmu_i = sqrt( mu_i^2 ( (da_i / a_i)^2 + (db_i / b_i)^2 + 2 (dw / w)^2 ) )            (Eq. 18, as printed)
 * dw = the standard deviation stored with the weight's quantiser bin (L176).  Reading Q19: a ratio
 * whose denominator is 0 (the component is absent from that child, so its uncertainty is 0 too) is
 * dropped from the sum. */
void mgo_mixture_lut(const uint32_t *child_a, const uint32_t *child_b, const double *weight, const double *weight_sigma,
                     uint64_t n_nodes, uint64_t n_leaves, double *mu, double *dmu)
{
    memset(mu, 0, (size_t)n_nodes * n_leaves * sizeof(double));
    memset(dmu, 0, (size_t)n_nodes * n_leaves * sizeof(double));
    for (uint64_t n = 0; n < n_leaves; n++)
        mu[n * n_leaves + n] = 1.0;
    for (uint64_t n = n_leaves; n < n_nodes; n++) {
        double w = weight[n], rw = weight_sigma[n] / w;
        const double *ma = mu + (uint64_t)child_a[n] * n_leaves, *da = dmu + (uint64_t)child_a[n] * n_leaves;
        const double *mb = mu + (uint64_t)child_b[n] * n_leaves, *db = dmu + (uint64_t)child_b[n] * n_leaves;
        for (uint64_t i = 0; i < n_leaves; i++) {
            double m = (1.0 - w) * ma[i] + w * mb[i];
            double rel2 = 2.0 * rw * rw;
            if (ma[i] != 0.0) rel2 += (da[i] / ma[i]) * (da[i] / ma[i]);
            if (mb[i] != 0.0) rel2 += (db[i] / mb[i]) * (db[i] / mb[i]);
            mu[n * n_leaves + i] = m;
            dmu[n * n_leaves + i] = sqrt(m * m * rel2);
        }
    }
}

/* Section 3.6: "we decompose the 1D ranges along x, y and z according to their alignment with the mip
 * levels".  [lo, hi) is cut, left to right, into the largest aligned power-of-two pieces: a piece
 * starts at x, has length 2^l, x is a multiple of 2^l, and l <= max_level.  Returns the number of pieces. */
uint32_t mgo_fa_axis(uint64_t lo, uint64_t hi, uint32_t max_level, uint64_t *start, uint32_t *level)
{
    uint32_t n = 0;
    uint64_t x = lo;
    while (x < hi) {
        uint32_t l = 0;
        while (l + 1 <= max_level && x % ((uint64_t)1 << (l + 1)) == 0 && x + ((uint64_t)1 << (l + 1)) <= hi)
            l++;
        start[n] = x;
        level[n] = l;
        n++;
        x += (uint64_t)1 << l;
    }
    return n;
}

/* Footprint assembly (L245-L247): "the tensor product of these ranges is comprised of rectangular boxes
 * ... Each of these boxes is tesselated by cubes of a side length l equal to the shortest of the three
 * box extents.  Each cube represents a single sample from H at level log2(l).  The contribution of each
 * sample ... is denormalized (multiplication by l^3) before being accumulated."  Errors add in quadrature
 * (Eq. 17).  box = x0, y0, z0, x1, y1, z1 (half-open, inside the volume).  expect / err = [n_leaves].
 * Returns the number of samples fetched. */
uint64_t mgo_range_query_fa(const uint32_t *node_idx, const uint64_t *level_offset, const uint32_t *level_dim,
                            uint32_t n_levels, const double *mu, const double *dmu, uint64_t n_leaves,
                            const uint64_t *box, double *expect, double *err)
{
    uint64_t sx[130], sy[130], sz[130], fetches = 0;
    uint32_t lx[130], ly[130], lz[130];
    uint32_t nx = mgo_fa_axis(box[0], box[3], n_levels - 1, sx, lx);
    uint32_t ny = mgo_fa_axis(box[1], box[4], n_levels - 1, sy, ly);
    uint32_t nz = mgo_fa_axis(box[2], box[5], n_levels - 1, sz, lz);
    for (uint64_t i = 0; i < n_leaves; i++)
        expect[i] = err[i] = 0.0;
    for (uint32_t c = 0; c < nz; c++)
        for (uint32_t b = 0; b < ny; b++)
            for (uint32_t a = 0; a < nx; a++) {
                uint32_t l = lx[a] < ly[b] ? lx[a] : ly[b];
                if (lz[c] < l) l = lz[c];
                double scale = ldexp(1.0, 3 * (int)l);                       /* l^3 voxels per cube */
                const uint32_t *d = level_dim + 3 * l;
                for (uint64_t z = sz[c] >> l; z < (sz[c] + ((uint64_t)1 << lz[c])) >> l; z++)
                    for (uint64_t y = sy[b] >> l; y < (sy[b] + ((uint64_t)1 << ly[b])) >> l; y++)
                        for (uint64_t x = sx[a] >> l; x < (sx[a] + ((uint64_t)1 << lx[a])) >> l; x++) {
                            uint64_t node = node_idx[level_offset[l] + (z * d[1] + y) * d[0] + x];
                            const double *m = mu + node * n_leaves, *dm = dmu + node * n_leaves;
                            for (uint64_t i = 0; i < n_leaves; i++) {
                                expect[i] += scale * m[i];
                                err[i] += (scale * dm[i]) * (scale * dm[i]);
                            }
                            fetches++;
                        }
            }
    for (uint64_t i = 0; i < n_leaves; i++)
        err[i] = sqrt(err[i]);
    return fetches;
}

/* The naive approach of L377: "adds the contributions of each voxel at the finest level". */
uint64_t mgo_range_query_naive(const uint32_t *node_idx0, const uint32_t *dim0, const double *mu, uint64_t n_leaves,
                               const uint64_t *box, double *expect)
{
    uint64_t fetches = 0;
    for (uint64_t i = 0; i < n_leaves; i++)
        expect[i] = 0.0;
    for (uint64_t z = box[2]; z < box[5]; z++)
        for (uint64_t y = box[1]; y < box[4]; y++)
            for (uint64_t x = box[0]; x < box[3]; x++) {
                const double *m = mu + (uint64_t)node_idx0[(z * dim0[1] + y) * dim0[0] + x] * n_leaves;
                for (uint64_t i = 0; i < n_leaves; i++)
                    expect[i] += m[i];
                fetches++;
            }
    return fetches;
}
