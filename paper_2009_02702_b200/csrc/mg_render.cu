// mg_render.cu -- NEXT-2: headless ray-marcher over the paletted histogram mipmap.
//
// PAPER.md section 4 (L265-L271, L414): the renderer treats the histogram mipmap as a paletted
// texture (L267): a sample fetches node IDs and looks their colours up in the palette that
// mg_propagate wrote; "the computation of the mip level as well as the interpolation" are done by
// hand (L269), the step grows with the LOD and opacities are corrected for it (L269), and the A
// channel of the coarser levels drives hierarchical empty-space skipping (L271).  Readings R1-R6:
// include/mg.h, DESIGN.md section 3.
//
// Mapping: one thread per ray; a CTA is an 8 x 8 pixel tile (each warp an 8 x 4 tile, so the 32
// rays of a warp walk through neighbouring voxels and their gathers share sectors).  Per sample at
// most 2 x (8 index gathers + 8 palette gathers): the index volume streams through L2 from HBM, the
// palette (16 B per node, tens of MB) stays L2-resident.  Three data-dependent shortcuts that do
// not change the value beyond rounding: the second level is not fetched when frac(lambda) == 0; a
// footprint whose 8 voxels name the same node costs one palette gather; skipped samples (R6) cost
// no memory access at all.  Two more: the parent voxel at which the last climb of R6 stopped is
// remembered (consecutive samples share it, so most samples climb without a gather), and with
// MG_VIEW_HISTOGRAM_MIPMAP the COARSE level is fetched first -- its 8 voxels cover the children
// holding the fine level's 8 voxels, and a leaf node in a histogram mipmap is a pure voxel, so if
// the 8 coarse voxels name one leaf all 16 taps are that leaf: segment interiors cost 8 index
// gathers + 1 palette gather instead of 16 + 2.  The block tests of R6 run on floor(2 p) in
// integers (exactly the oracle's comparisons, see Block).
// Arithmetic: t, the step and the sample position in fp64 (the B200's fp64 pipe is half the fp32 rate); the position
// is then held in 32.32 fixed point, from which the voxel indices, the trilinear fractions (to 2^-32 voxel) and the
// block tests of every level follow by integer shifts; the fractional LOD, the weights, colours and opacity correction
// in fp32; the compositing sums C and A in fp64 (thousands of samples per ray would otherwise add their fp32
// rounding errors).
#include <math.h>

#include <algorithm>
#include <cstring>

#include "mg_internal.h"

namespace {

constexpr int kTileX = 8, kTileY = 8;

struct RenderParams {
    const uint32_t* idx;
    const float4* pal;
    float4* out;
    unsigned long long* stats;
    unsigned long long off[MG_MAX_MIP_LEVELS];
    int dim[MG_MAX_MIP_LEVELS][3];
    int n_levels;
    unsigned W, H;
    double eye[3], right[3], up[3], fwd[3];
    double inv_s[3], ext[3];
    double tan_half_fov, pix;       // pix = 2^lod_bias (2 tan_half_fov / H) / s_ref
    double pow_lmax;                // 2^l_max
    double thr;                     // ess threshold (< 0: off)
    double step_ref;                // step_voxels * s_ref
    double cutoff;
    float inv_ref;                  // 1 / (ref_step_voxels * s_ref)
    uint32_t n_leaves;              // > 0: MG_VIEW_HISTOGRAM_MIPMAP (nodes below it are pure voxels)
    const uint16_t* ess_mask;       // per voxel of level 2: bit k = its ancestor on level 2 + k is empty (mg_ess_mask_build), or NULL
};

__device__ __forceinline__ int clampi(int v, int hi) { return v < 0 ? 0 : (v > hi ? hi : v); }

// The 2 x 2 x 2 voxels around p on level l (R3: voxel i of level l is centred at (i + 1/2) 2^l, indices
// clamped to the level) and the interpolation fractions.
struct Cell {
    uint32_t n[8];          // node of voxel (dz, dy, dx) at n[4 dz + 2 dy + dx]
    float fx, fy, fz;
};

// q = floor(p 2^32): the sample position in 32.32 fixed point.  u = p / 2^l - 1/2 becomes U = (q >> l) - 2^31, whose
// integer part is the voxel index and whose low 32 bits are the interpolation fraction (to 2^-32 of a voxel) -- integer
// shifts instead of fp64 multiplies, floors and subtractions per level.  SMALL: every level has < 2^32 voxels, so the
// row offsets are computed in 32 bits.
template <bool SMALL>
__device__ __forceinline__ void fetch_cell(const RenderParams& P, int l, long long qx, long long qy, long long qz, Cell& c)
{
    const long long Ux = (qx >> l) - (1ll << 31), Uy = (qy >> l) - (1ll << 31), Uz = (qz >> l) - (1ll << 31);
    c.fx = __uint2float_rn((unsigned)Ux) * 2.3283064365386963e-10f;
    c.fy = __uint2float_rn((unsigned)Uy) * 2.3283064365386963e-10f;
    c.fz = __uint2float_rn((unsigned)Uz) * 2.3283064365386963e-10f;
    const int X = P.dim[l][0], Y = P.dim[l][1], Z = P.dim[l][2];
    const int ix = (int)(Ux >> 32), iy = (int)(Uy >> 32), iz = (int)(Uz >> 32);
    const int x0 = clampi(ix, X - 1), x1 = clampi(ix + 1, X - 1);
    const int y0 = clampi(iy, Y - 1), y1 = clampi(iy + 1, Y - 1);
    const int z0 = clampi(iz, Z - 1), z1 = clampi(iz + 1, Z - 1);
    const uint32_t* base = P.idx + P.off[l];
    if (SMALL) {
        const unsigned r00 = ((unsigned)z0 * Y + y0) * X, r01 = ((unsigned)z0 * Y + y1) * X;
        const unsigned r10 = ((unsigned)z1 * Y + y0) * X, r11 = ((unsigned)z1 * Y + y1) * X;
        c.n[0] = __ldg(base + (r00 + x0)); c.n[1] = __ldg(base + (r00 + x1)); c.n[2] = __ldg(base + (r01 + x0)); c.n[3] = __ldg(base + (r01 + x1));
        c.n[4] = __ldg(base + (r10 + x0)); c.n[5] = __ldg(base + (r10 + x1)); c.n[6] = __ldg(base + (r11 + x0)); c.n[7] = __ldg(base + (r11 + x1));
    } else {
        const uint32_t* r00 = base + ((size_t)z0 * Y + y0) * X;
        const uint32_t* r01 = base + ((size_t)z0 * Y + y1) * X;
        const uint32_t* r10 = base + ((size_t)z1 * Y + y0) * X;
        const uint32_t* r11 = base + ((size_t)z1 * Y + y1) * X;
        c.n[0] = __ldg(r00 + x0); c.n[1] = __ldg(r00 + x1); c.n[2] = __ldg(r01 + x0); c.n[3] = __ldg(r01 + x1);
        c.n[4] = __ldg(r10 + x0); c.n[5] = __ldg(r10 + x1); c.n[6] = __ldg(r11 + x0); c.n[7] = __ldg(r11 + x1);
    }
}

__device__ __forceinline__ bool one_node(const Cell& c)
{
    return ((c.n[0] ^ c.n[1]) | (c.n[0] ^ c.n[2]) | (c.n[0] ^ c.n[3]) | (c.n[0] ^ c.n[4]) | (c.n[0] ^ c.n[5]) |
            (c.n[0] ^ c.n[6]) | (c.n[0] ^ c.n[7])) == 0;
}

__device__ __forceinline__ void tap(float4& acc, const float4* __restrict__ pal, uint32_t n, float wgt)
{
    const float4 c = __ldg(pal + n);
    acc.x = fmaf(wgt, c.x, acc.x); acc.y = fmaf(wgt, c.y, acc.y);
    acc.z = fmaf(wgt, c.z, acc.z); acc.w = fmaf(wgt, c.w, acc.w);
}

// Trilinear interpolation of the palette over a fetched cell; a cell naming one node costs one gather.
__device__ __forceinline__ float4 shade_cell(const RenderParams& P, const Cell& c)
{
    if (one_node(c)) return __ldg(P.pal + c.n[0]);
    const float fx = c.fx, fy = c.fy, fz = c.fz, gx = 1.f - fx, gy = 1.f - fy, gz = 1.f - fz;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    tap(acc, P.pal, c.n[0], gx * gy * gz); tap(acc, P.pal, c.n[1], fx * gy * gz);
    tap(acc, P.pal, c.n[2], gx * fy * gz); tap(acc, P.pal, c.n[3], fx * fy * gz);
    tap(acc, P.pal, c.n[4], gx * gy * fz); tap(acc, P.pal, c.n[5], fx * gy * fz);
    tap(acc, P.pal, c.n[6], gx * fy * fz); tap(acc, P.pal, c.n[7], fx * fy * fz);
    return acc;
}

// R4: alpha' = 1 - (1 - alpha)^e = -expm1(e log1p(-alpha)), accurate to ~1e-7 relative like the libm pair, but the
// common case of a translucent sample (alpha <= 1/16, |e log1p(-alpha)| < 1/8) costs two short polynomials instead of
// two libm calls: log1p(-a) = -a (1 + a/2 + ... + a^6/7) (truncation < a^7/8) and expm1(y) = y (1 + y/2 + ... + y^5/720)
// (truncation < y^7/5040).
__device__ __forceinline__ float opacity_correct(float alpha, float e)
{
    if (alpha <= 0.f) return 0.f;
    float y;                                                             // e log1p(-alpha) <= 0
    if (alpha <= 0.0625f) {
        float p = fmaf(alpha, 1.f / 7.f, 1.f / 6.f);
        p = fmaf(alpha, p, 0.2f); p = fmaf(alpha, p, 0.25f); p = fmaf(alpha, p, 1.f / 3.f); p = fmaf(alpha, p, 0.5f);
        p = fmaf(alpha, p, 1.f);
        y = -e * (alpha * p);
    } else {
        y = e * log1pf(-alpha);                                          // alpha = 1: -inf, and the result is 1
    }
    if (y > -0.125f) {
        float p = fmaf(y, 1.f / 720.f, 1.f / 120.f);
        p = fmaf(y, p, 1.f / 24.f); p = fmaf(y, p, 1.f / 6.f); p = fmaf(y, p, 0.5f); p = fmaf(y, p, 1.f);
        return -y * p;
    }
    return -expm1f(y);
}

// R6 block: voxel-aligned box in level-0 coordinates, kept in HALF-voxel integers so that the oracle's
// tests on p become integer tests on h = floor(2 p):  p < lo + m  <=>  h < 2 lo + 2 m  and
// p >= hi - m  <=>  h >= 2 hi - 2 m  (2 lo, 2 hi, 2 m = 2^l1 are integers).  A face on the volume's
// boundary needs no margin (the fetch clamps there): its bound is pushed out of reach instead.
struct Block {
    int lo2[3], hi2[3];     // 2 lo, 2 hi
    unsigned open;          // bit a: lo face of axis a is open; bit 3 + a: hi face
    bool valid;
};

__device__ __forceinline__ void set_block(Block& B, int qx, int qy, int qz, int L, const int* dim)
{
    B.valid = true;
    B.lo2[0] = qx << (L + 1); B.lo2[1] = qy << (L + 1); B.lo2[2] = qz << (L + 1);
    B.hi2[0] = (qx + 1) << (L + 1); B.hi2[1] = (qy + 1) << (L + 1); B.hi2[2] = (qz + 1) << (L + 1);
    B.open = (qx == 0) | ((qy == 0) << 1) | ((qz == 0) << 2) | ((qx == dim[0] - 1) << 3) | ((qy == dim[1] - 1) << 4) |
             ((qz == dim[2] - 1) << 5);
}

__device__ __forceinline__ bool inside_block(const Block& B, int m2, int hx, int hy, int hz)
{
    const int h[3] = {hx, hy, hz};
    bool in = B.valid;
#pragma unroll
    for (int a = 0; a < 3; a++) {
        if (!((B.open >> a) & 1u) && h[a] < B.lo2[a] + m2) in = false;
        if (!((B.open >> (3 + a)) & 1u) && h[a] >= B.hi2[a] - m2) in = false;
    }
    return in;
}

// One thread per voxel of level 2: which of its ancestors (itself included) are empty, i.e. have a palette opacity
// below the threshold -- the comparisons the climb of R6 makes, made once per TF update instead of once per probe.
struct EssMaskParams {
    const uint32_t* idx;
    const float4* pal;
    uint16_t* mask;
    unsigned long long off[MG_MAX_MIP_LEVELS];
    int dim[MG_MAX_MIP_LEVELS][3];
    int n_levels;
    double thr;
};

__global__ void __launch_bounds__(256) k_ess_mask(const __grid_constant__ EssMaskParams P)
{
    const int X2 = P.dim[2][0], Y2 = P.dim[2][1], Z2 = P.dim[2][2];
    const uint64_t n2 = (uint64_t)X2 * Y2 * Z2;
    for (uint64_t v = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; v < n2; v += (uint64_t)gridDim.x * blockDim.x) {
        const int x = (int)(v % X2), y = (int)((v / X2) % Y2), z = (int)(v / ((uint64_t)X2 * Y2));
        unsigned m = 0;
        for (int L = 2; L < P.n_levels; L++) {
            const int k = L - 2;
            const uint32_t n = __ldg(P.idx + P.off[L] + ((size_t)(z >> k) * P.dim[L][1] + (y >> k)) * P.dim[L][0] + (x >> k));
            const float alpha = __ldg(reinterpret_cast<const float*>(P.pal + n) + 3);
            if ((double)alpha < P.thr) m |= 1u << k;
        }
        P.mask[v] = (uint16_t)m;
    }
}

// ESS: 0 = no empty-space skipping (R6 compiled out), 1 = the climb of R6 per probe, 2 = the largest empty block above a
// probe comes from P.ess_mask (one 2-byte load) instead of the climb.
//
// One thread per ray, one sample per loop iteration: the 32 rays of a warp stay in step (neighbouring voxels, shared
// sectors).  A skipped sample therefore saves its fetch but not its iteration, and it saves nothing at all while
// another ray of the warp fetches in the same iteration.  Three ways of letting a ray run ahead through a proven
// block were measured on B200 and are NOT in the kernel (1600 x 1200, config 3 with 95 % of the segments transparent,
// 78 % of the samples skipped; this loop: 39.8 ms, no skipping: 48.5 ms): a per-ray fast-forward through the part of
// the ray that lies inside the block shrunk by R6's margin (exact: the window is conservative, samples outside it take
// the ordinary test) 51.8 ms with 98 % of the skipped samples fast-forwarded -- the rays of a warp drift apart and
// every iteration pays for the longest run; the same as a warp vote (__all_sync: every live ray inside its window)
// in a warp-uniform loop 47.3 ms; an inner skip loop per ray 140 ms; compaction of the rays that need a fetch into full
// warps through a shared-memory request list (CTAs of 16 x 16 rays, three barriers per round) 62.6 ms.
template <bool SMALL, int ESS>
__global__ void __launch_bounds__(kTileX * kTileY)
k_render(const __grid_constant__ RenderParams P)
{
    constexpr unsigned kFull = 0xffffffffu;
    constexpr bool ess = ESS != 0;
    constexpr bool MASK = ESS == 2;
    const unsigned i = blockIdx.x * kTileX + (threadIdx.x & (kTileX - 1));
    const unsigned j = blockIdx.y * kTileY + threadIdx.x / kTileX;
    const bool live = i < P.W && j < P.H;
    unsigned n_eval = 0, n_skip = 0, n_uni = 0;
    double Cr = 0.0, Cg = 0.0, Cb = 0.0, A = 0.0;
    double d[3] = {0.0, 0.0, 1.0};
    double tn = 0.0, tf = INFINITY, rho_t = 0.0;
    bool hit = live;
    if (live) {
        // R1: pixel ray
        const double u = (2.0 * ((double)i + 0.5) / (double)P.W - 1.0) * P.tan_half_fov * (double)P.W / (double)P.H;
        const double v = (1.0 - 2.0 * ((double)j + 0.5) / (double)P.H) * P.tan_half_fov;
        double nrm = 0.0;
#pragma unroll
        for (int a = 0; a < 3; a++) {
            d[a] = P.fwd[a] + u * P.right[a] + v * P.up[a];
            nrm += d[a] * d[a];
        }
        nrm = sqrt(nrm);
#pragma unroll
        for (int a = 0; a < 3; a++) d[a] /= nrm;
        // slab test against [0, ext]
#pragma unroll
        for (int a = 0; a < 3; a++) {
            if (d[a] == 0.0) {
                if (P.eye[a] < 0.0 || P.eye[a] > P.ext[a]) hit = false;
            } else {
                const double t1 = (0.0 - P.eye[a]) / d[a], t2 = (P.ext[a] - P.eye[a]) / d[a];
                tn = fmax(tn, fmin(t1, t2));
                tf = fmin(tf, fmax(t1, t2));
            }
        }
        if (!(tn < tf)) hit = false;
        const double cos_view = d[0] * P.fwd[0] + d[1] * P.fwd[1] + d[2] * P.fwd[2];
        rho_t = cos_view * P.pix;                                            // rho 2^bias = t * rho_t (R2)
    }
    const int l_max = P.n_levels - 1;
    const bool uni = P.n_leaves != 0;                                        // MG_VIEW_HISTOGRAM_MIPMAP
    Block E;                                                                 // the empty block of R6
    E.valid = false;
    E.open = 0;
#pragma unroll
    for (int a = 0; a < 3; a++) E.lo2[a] = E.hi2[a] = 0;
    int miss_L = -1, miss_x = 0, miss_y = 0, miss_z = 0;                     // last parent voxel found not empty (climb only)
    bool empty_mode = true;                                                  // R6: a ray enters the volume in empty mode
    double t = tn;
    while (hit && t < tf && A < P.cutoff) {
        // ---- one sample.  R2 + R4 without transcendentals on the ray parameter: 2^lambda = clamp(rho 2^bias, 1, 2^l_max),
        // so Delta = step s_ref 2^lambda is a product in fp64 and t follows the oracle's to rounding.
        const double pow_lambda = fmin(fmax(t * rho_t, 1.0), P.pow_lmax);
        const float lambda = fminf(log2f((float)pow_lambda), (float)l_max);
        const double delta = P.step_ref * pow_lambda;                        // R4
        const double de = fmin(delta, tf - t);                               // R5
        const double ts = fma(0.5, de, t);
        const double px = fma(ts, d[0], P.eye[0]) * P.inv_s[0];
        const double py = fma(ts, d[1], P.eye[1]) * P.inv_s[1];
        const double pz = fma(ts, d[2], P.eye[2]) * P.inv_s[2];
        const long long qx = __double2ll_rd(px * 4294967296.0), qy = __double2ll_rd(py * 4294967296.0),
                        qz = __double2ll_rd(pz * 4294967296.0);              // 32.32 fixed point (see fetch_cell)
        const float fl = floorf(lambda);
        const int l0 = (int)fl;
        const int l1 = min(l0 + 1, l_max);
        const float f = lambda - fl;
        t += delta;
        if (ess && empty_mode) {                                             // R6: probe only where the ray is in empty space
            const int m2 = 1 << l1;                                          // 2 m, m = 2^l1 / 2
            const int hx = (int)(qx >> 31), hy = (int)(qy >> 31), hz = (int)(qz >> 31);   // floor(2 p): half-voxel integers
            bool inside = inside_block(E, m2, hx, hy, hz);
            if (!inside) {
                // Not inside the remembered block: the oracle forgets it and climbs again from level l1 + 1 while the
                // parent voxel is empty; the largest such block is remembered.
                E.valid = false;
                if (MASK) {
                    if (l1 + 1 <= l_max) {
                        const int x2 = clampi(hx >> 3, P.dim[2][0] - 1), y2 = clampi(hy >> 3, P.dim[2][1] - 1),
                                  z2 = clampi(hz >> 3, P.dim[2][2] - 1);
                        const unsigned m = (unsigned)__ldg(P.ess_mask + ((size_t)z2 * P.dim[2][1] + y2) * P.dim[2][0] + x2) >> (l1 - 1);
                        const int run = __ffs(~m) - 1;                       // consecutive empty ancestors from level l1 + 1 on
                        if (run > 0) {
                            const int L = l1 + run;
                            set_block(E, clampi(hx >> (L + 1), P.dim[L][0] - 1), clampi(hy >> (L + 1), P.dim[L][1] - 1),
                                      clampi(hz >> (L + 1), P.dim[L][2] - 1), L, P.dim[L]);
                        }
                    }
                } else {
                    // The climb is a pure function of the parent voxels, so a parent already found not empty is not
                    // fetched again (consecutive samples share it).
                    for (int L = l1 + 1; L <= l_max; L++) {
                        const int cx = clampi(hx >> (L + 1), P.dim[L][0] - 1);
                        const int cy = clampi(hy >> (L + 1), P.dim[L][1] - 1);
                        const int cz = clampi(hz >> (L + 1), P.dim[L][2] - 1);
                        if (L == miss_L && cx == miss_x && cy == miss_y && cz == miss_z) break;
                        const uint32_t n = __ldg(P.idx + P.off[L] + ((size_t)cz * P.dim[L][1] + cy) * P.dim[L][0] + cx);
                        const float alpha_parent = __ldg(reinterpret_cast<const float*>(P.pal + n) + 3);
                        if (!((double)alpha_parent < P.thr)) {
                            miss_L = L; miss_x = cx; miss_y = cy; miss_z = cz;
                            break;
                        }
                        set_block(E, cx, cy, cz, L, P.dim[L]);
                    }
                }
                inside = inside_block(E, m2, hx, hy, hz);
            }
            if (inside) {
                n_skip++;
                continue;
            }
        }
        // The level needed first: with MG_VIEW_HISTOGRAM_MIPMAP the COARSE one -- its 8 voxels cover the children that
        // hold the fine level's 8 voxels, so if they all name ONE LEAF (a pure voxel of a histogram mipmap) every tap of
        // both levels is that leaf.
        Cell cell;
        const bool coarse_first = uni && f != 0.f;                            // frac(lambda) = 0: only level l0 is needed
        fetch_cell<SMALL>(P, coarse_first ? l1 : l0, qx, qy, qz, cell);
        float4 c;                                                            // R3
        if (coarse_first && one_node(cell) && cell.n[0] < P.n_leaves) {
            c = __ldg(P.pal + cell.n[0]);
            n_uni++;
        } else {
            float4 c1 = make_float4(0.f, 0.f, 0.f, 0.f);
            if (coarse_first) {                                              // cell = coarse level (f != 0, l0 < l1)
                c1 = shade_cell(P, cell);
                fetch_cell<SMALL>(P, l0, qx, qy, qz, cell);
                c = shade_cell(P, cell);
            } else {                                                         // cell = fine level
                c = shade_cell(P, cell);
                if (f != 0.f) {
                    fetch_cell<SMALL>(P, l1, qx, qy, qz, cell);
                    c1 = shade_cell(P, cell);
                }
            }
            if (f != 0.f) {
                const float g = 1.f - f;
                c.x = fmaf(f, c1.x, g * c.x); c.y = fmaf(f, c1.y, g * c.y);
                c.z = fmaf(f, c1.z, g * c.z); c.w = fmaf(f, c1.w, g * c.w);
            }
        }
        const float alpha = fminf(fmaxf(c.w, 0.f), 1.f);
        empty_mode = (double)alpha < P.thr;                                   // R6
        const float e = (float)de * P.inv_ref;
        const float ac = opacity_correct(alpha, e);                           // 1 - (1 - alpha)^e
        const double wgt = (1.0 - A) * (double)ac;                            // R5, accumulated in fp64
        Cr = fma(wgt, (double)c.x, Cr); Cg = fma(wgt, (double)c.y, Cg); Cb = fma(wgt, (double)c.z, Cb);
        A += wgt;
        n_eval++;
    }
    if (live) P.out[(size_t)j * P.W + i] = make_float4((float)Cr, (float)Cg, (float)Cb, (float)A);
    if (P.stats) {
        const unsigned e = __reduce_add_sync(kFull, n_eval);
        const unsigned s = __reduce_add_sync(kFull, n_skip);
        const unsigned u = __reduce_add_sync(kFull, n_uni);
        if ((threadIdx.x & 31) == 0) {
            if (e) atomicAdd(P.stats, (unsigned long long)e);
            if (s) atomicAdd(P.stats + 1, (unsigned long long)s);
            if (u) atomicAdd(P.stats + 2, (unsigned long long)u);
        }
    }
}

}  // namespace

// Checks `mip` (the ceil-halving chain of L80, levels not overlapping) and copies it into off / dim.
static int check_mipmap(const mg_mipmap_desc* mip, unsigned long long* off, int (*dim)[3], const char* who)
{
    if (mip->n_levels == 0 || mip->n_levels > MG_MAX_MIP_LEVELS) {
        mg::set_error("%s: n_levels = %u not in 1..%d", who, mip->n_levels, MG_MAX_MIP_LEVELS);
        return MG_ERR_INVALID_ARG;
    }
    for (uint32_t l = 0; l < mip->n_levels; l++) {
        for (int a = 0; a < 3; a++) {
            const uint32_t dl = mip->level_dim[l][a];
            if (dl == 0 || dl > (1u << 20) || (l > 0 && dl != (mip->level_dim[l - 1][a] + 1) / 2)) {
                mg::set_error("%s: level %u axis %d has %u voxels: not the ceil-halving chain of L80", who, l, a, dl);
                return MG_ERR_INVALID_ARG;
            }
            dim[l][a] = (int)dl;
        }
        if (l > 0) {
            const uint64_t prev = (uint64_t)mip->level_dim[l - 1][0] * mip->level_dim[l - 1][1] * mip->level_dim[l - 1][2];
            if (mip->level_offset[l] < mip->level_offset[l - 1] + prev) {
                mg::set_error("%s: level %u starts inside level %u", who, l, l - 1);
                return MG_ERR_INVALID_ARG;
            }
        }
        off[l] = mip->level_offset[l];
    }
    return MG_OK;
}

extern "C" int mg_ess_mask_build(mg_graph* g, const uint32_t* node_idx_mipmap, const mg_mipmap_desc* mip, const float* node_rgba,
                                 double ess_threshold, uint16_t* ess_mask, void* stream)
{
    if (!g || !node_idx_mipmap || !mip || !node_rgba || !ess_mask) { mg::set_error("mg_ess_mask_build: NULL argument"); return MG_ERR_INVALID_ARG; }
    if (((uintptr_t)node_rgba & 15) || ((uintptr_t)node_idx_mipmap & 3) || ((uintptr_t)ess_mask & 1)) {
        mg::set_error("mg_ess_mask_build: misaligned buffer");
        return MG_ERR_INVALID_ARG;
    }
    if (isnan(ess_threshold)) { mg::set_error("mg_ess_mask_build: ess_threshold is NaN"); return MG_ERR_INVALID_ARG; }
    EssMaskParams P;
    memset(&P, 0, sizeof(P));
    int rc = check_mipmap(mip, P.off, P.dim, "mg_ess_mask_build");
    if (rc != MG_OK) return rc;
    if (mip->n_levels < 3 || mip->n_levels > 18) {
        mg::set_error("mg_ess_mask_build: needs 3 .. 18 mip levels (one bit per level from level 2 on), got %u", mip->n_levels);
        return MG_ERR_INVALID_ARG;
    }
    rc = mg::check_device(g, "mg_ess_mask_build");
    if (rc != MG_OK) return rc;
    P.idx = node_idx_mipmap;
    P.pal = reinterpret_cast<const float4*>(node_rgba);
    P.mask = ess_mask;
    P.n_levels = (int)mip->n_levels;
    P.thr = ess_threshold;
    const uint64_t n2 = (uint64_t)P.dim[2][0] * P.dim[2][1] * P.dim[2][2];
    const unsigned blocks = (unsigned)std::min<uint64_t>((n2 + 255) / 256, 148ull * 32);
    k_ess_mask<<<blocks, 256, 0, (cudaStream_t)stream>>>(P);
    MG_CUDA(cudaGetLastError());
    mg::count_launch();
    return MG_OK;
}

extern "C" int mg_render(mg_graph* g, const uint32_t* node_idx_mipmap, const mg_mipmap_desc* mip,
                         const float* node_rgba, const mg_view* view, float* out_rgba, uint64_t* stats_device,
                         void* stream)
{
    return mg_render_ex(g, node_idx_mipmap, mip, node_rgba, view, nullptr, out_rgba, stats_device, stream);
}

extern "C" int mg_render_ex(mg_graph* g, const uint32_t* node_idx_mipmap, const mg_mipmap_desc* mip,
                            const float* node_rgba, const mg_view* view, const mg_render_aux* aux, float* out_rgba,
                            uint64_t* stats_device, void* stream)
{
    if (!g || !node_idx_mipmap || !mip || !node_rgba || !view || !out_rgba) {
        mg::set_error("mg_render: NULL argument");
        return MG_ERR_INVALID_ARG;
    }
    if (((uintptr_t)node_rgba & 15) || ((uintptr_t)out_rgba & 15) || ((uintptr_t)node_idx_mipmap & 3) ||
        ((uintptr_t)stats_device & 7)) {
        mg::set_error("mg_render: node_rgba / out_rgba must be 16-byte aligned (stats 8, indices 4)");
        return MG_ERR_INVALID_ARG;
    }
    if (mip->n_levels == 0 || mip->n_levels > MG_MAX_MIP_LEVELS) {
        mg::set_error("mg_render: n_levels = %u not in 1..%d", mip->n_levels, MG_MAX_MIP_LEVELS);
        return MG_ERR_INVALID_ARG;
    }
    if (view->flags & ~(uint32_t)MG_VIEW_HISTOGRAM_MIPMAP) {
        mg::set_error("mg_render: unknown view flags 0x%x", view->flags);
        return MG_ERR_INVALID_ARG;
    }
    if (view->width == 0 || view->height == 0 || view->width > 65536u || view->height > 65536u) {
        mg::set_error("mg_render: image size %u x %u out of range", view->width, view->height);
        return MG_ERR_INVALID_ARG;
    }
    const double* s = view->spacing;
    if (!(s[0] > 0.0) || !(s[1] > 0.0) || !(s[2] > 0.0) || !(view->step_voxels > 0.0) || !(view->ref_step_voxels > 0.0) ||
        !(view->tan_half_fov > 0.0) || !isfinite(view->lod_bias) || !isfinite(view->step_voxels) ||
        !isfinite(view->tan_half_fov) || isnan(view->ess_threshold) || isnan(view->alpha_cutoff)) {
        mg::set_error("mg_render: spacing, step_voxels, ref_step_voxels and tan_half_fov must be positive and finite");
        return MG_ERR_INVALID_ARG;
    }
    {
        const int rc = mg::check_device(g, "mg_render");
        if (rc != MG_OK) return rc;
    }
    RenderParams P;
    memset(&P, 0, sizeof(P));
    {
        const int rc = check_mipmap(mip, P.off, P.dim, "mg_render");
        if (rc != MG_OK) return rc;
    }
    if (aux && aux->ess_mask && view->ess_threshold >= 0.0) {
        if (mip->n_levels < 3 || mip->n_levels > 18 || ((uintptr_t)aux->ess_mask & 1)) {
            mg::set_error("mg_render: aux->ess_mask needs 3 .. 18 mip levels and 2-byte alignment");
            return MG_ERR_INVALID_ARG;
        }
        P.ess_mask = aux->ess_mask;
    }
    P.idx = node_idx_mipmap;
    P.pal = reinterpret_cast<const float4*>(node_rgba);
    P.out = reinterpret_cast<float4*>(out_rgba);
    P.stats = reinterpret_cast<unsigned long long*>(stats_device);
    P.n_levels = (int)mip->n_levels;
    P.W = view->width;
    P.H = view->height;
    const double s_ref = fmin(s[0], fmin(s[1], s[2]));
    {   // a ray takes at most diagonal / (step_voxels s_ref) steps: refuse views that would march (almost) forever
        double diag2 = 0.0;
        for (int a = 0; a < 3; a++) diag2 += (double)mip->level_dim[0][a] * s[a] * (double)mip->level_dim[0][a] * s[a];
        if (sqrt(diag2) / (view->step_voxels * s_ref) > 16777216.0) {
            mg::set_error("mg_render: step_voxels = %g needs more than 2^24 steps per ray", view->step_voxels);
            return MG_ERR_INVALID_ARG;
        }
    }
    for (int a = 0; a < 3; a++) {
        P.eye[a] = view->eye[a]; P.right[a] = view->right[a]; P.up[a] = view->up[a]; P.fwd[a] = view->forward[a];
        P.inv_s[a] = 1.0 / s[a];
        P.ext[a] = (double)mip->level_dim[0][a] * s[a];
    }
    P.tan_half_fov = view->tan_half_fov;
    P.pix = exp2(view->lod_bias) * (2.0 * view->tan_half_fov / (double)view->height) / s_ref;
    P.pow_lmax = ldexp(1.0, (int)mip->n_levels - 1);
    P.thr = view->ess_threshold;
    P.step_ref = view->step_voxels * s_ref;
    P.inv_ref = (float)(1.0 / (view->ref_step_voxels * s_ref));
    P.cutoff = view->alpha_cutoff;
    P.n_leaves = (view->flags & MG_VIEW_HISTOGRAM_MIPMAP) ? g->n_leaves : 0u;
    const dim3 grid((P.W + kTileX - 1) / kTileX, (P.H + kTileY - 1) / kTileY);
    bool small = true;
    for (uint32_t l = 0; l < mip->n_levels; l++)
        small = small && (uint64_t)mip->level_dim[l][0] * mip->level_dim[l][1] * mip->level_dim[l][2] < (1ull << 32);
    cudaStream_t st = (cudaStream_t)stream;
    const int mode = !(P.thr >= 0.0) ? 0 : (P.ess_mask ? 2 : 1);
    if (small) {
        if (mode == 0) k_render<true, 0><<<grid, kTileX * kTileY, 0, st>>>(P);
        else if (mode == 1) k_render<true, 1><<<grid, kTileX * kTileY, 0, st>>>(P);
        else k_render<true, 2><<<grid, kTileX * kTileY, 0, st>>>(P);
    } else {
        if (mode == 0) k_render<false, 0><<<grid, kTileX * kTileY, 0, st>>>(P);
        else if (mode == 1) k_render<false, 1><<<grid, kTileX * kTileY, 0, st>>>(P);
        else k_render<false, 2><<<grid, kTileX * kTileY, 0, st>>>(P);
    }
    MG_CUDA(cudaGetLastError());
    mg::count_launch();
    return MG_OK;
}
