// mg_query.cu -- NEXT-4: mixture lookup table (Eq. 17-18) and sub-volume (range) queries.
//
// PAPER.md section 3.5 (L225-L241), section 3.6 (L243-L253), L375-L377, Table 4.  The paper builds
// the table on the CPU and calls range queries "not well suited for the GPU, since the number of
// non-zero entries in the sparse mixtures is hard to predict" (L253).  Here both run on the device:
//   * the table is a CSR (leaf, mu, dmu) per node whose row CAPACITIES are known before any value is:
//     cap(n) = min(n_leaves, cap(a) + cap(b)) -- exact for graphs made by the factorisation (the two
//     children of a node carry disjoint parts of a mixture), an upper bound for any other DAG -- so one
//     allocation and one merge kernel per topological level suffice (no count/scan/fill passes);
//   * a query is spread over several CTAs; each warp takes boxes of the footprint's tensor product,
//     its lanes take the cubes of the box, every cube is one mipmap sample whose sparse row is added
//     into the dense per-query result with fp64 atomics in L2.  Samples that are pure voxels (row =
//     one leaf, the bulk of every query) are pre-aggregated per warp with __match_any_sync so that a
//     homogeneous region costs one atomic per warp instead of 32 on the same address.
// fp64 throughout (the B200's fp64 pipe is half the fp32 rate; the work is gather/atomic-bound).
#include <math.h>

#include <algorithm>
#include <cstring>
#include <new>
#include <vector>

#include "mg_internal.h"

struct mg_mixture_lut {
    int device = 0;
    uint64_t n_nodes = 0;
    uint32_t n_leaves = 0;
    uint64_t capacity = 0, nnz = 0;
    uint32_t max_row = 0;
    uint64_t* d_row_ptr = nullptr;    // [n_nodes + 1] row starts (capacity layout)
    uint32_t* d_row_len = nullptr;    // [n_nodes] entries in use
    uint32_t* d_col = nullptr;        // [capacity] leaf index, ascending inside a row
    double* d_mu = nullptr;           // [capacity]
    double* d_dmu = nullptr;          // [capacity]
    uint64_t* d_boxes = nullptr;      // staging for mg_range_query (batches of more than kInlineQueries boxes)
    uint32_t* d_done = nullptr;       // [boxes_cap] per-query completion counters
    uint32_t boxes_cap = 0;
    uint64_t device_bytes = 0;
};

namespace {

constexpr int kBuildThreads = 128;
constexpr int kQueryThreads = 256;
constexpr int kNaiveUnroll = 4;
constexpr int kMaxPieces = 2 * MG_MAX_MIP_LEVELS + 2;     // pieces of one axis: at most 2 per level
constexpr int kInlineQueries = 64;                        // batches up to this size carry their boxes in the kernel parameters

__global__ void k_lut_leaves(uint32_t n_leaves, const uint64_t* __restrict__ row_ptr, uint32_t* row_len, uint32_t* col,
                             double* mu, double* dmu)
{
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_leaves) return;
    const uint64_t r = row_ptr[n];
    row_len[n] = 1;
    col[r] = n;
    mu[r] = 1.0;          // e_i ...
    dmu[r] = 0.0;         // ... "with variance 0" (L375)
}

// Row capacities on the device, one topological level at a time: cap(n) = min(n_leaves, cap(a) + cap(b)), leaves 1.
__global__ void __launch_bounds__(256)
k_lut_cap_level(const uint32_t* __restrict__ ga, const uint32_t* __restrict__ gb, uint32_t lo, uint32_t hi, uint32_t n_leaves, uint32_t* cap)
{
    const uint32_t n = lo + blockIdx.x * 256 + threadIdx.x;
    if (n >= hi) return;
    if (n < n_leaves) { cap[n] = 1; return; }
    const uint64_t c = (uint64_t)cap[ga[n]] + cap[gb[n]];
    cap[n] = (uint32_t)(c < n_leaves ? c : n_leaves);
}

// Exclusive prefix sum of n uint32 values into uint64 (row starts), two levels: tiles of kScanTile values per CTA.
constexpr int kScanTile = 2048;     // 256 threads x 8 values

__global__ void __launch_bounds__(256) k_scan_tile_sums(const uint32_t* __restrict__ v, uint64_t n, uint64_t* __restrict__ tile_sum)
{
    __shared__ unsigned long long warp_sum[8];
    const uint64_t base = (uint64_t)blockIdx.x * kScanTile;
    unsigned long long s = 0;
    for (int k = 0; k < 8; k++) {
        const uint64_t i = base + (uint64_t)k * 256 + threadIdx.x;
        if (i < n) s += v[i];
    }
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
        for (int w = 0; w < 8; w++) t += warp_sum[w];
        tile_sum[blockIdx.x] = t;
    }
}

// one CTA: exclusive scan of the tile sums in place; total to tile_sum[n_tiles]
__global__ void __launch_bounds__(1024) k_scan_tiles(uint64_t* tile_sum, uint32_t n_tiles)
{
    __shared__ unsigned long long part[1024];
    const uint32_t per = (n_tiles + 1023) / 1024;
    const uint32_t t0 = min(threadIdx.x * per, n_tiles), t1 = min(t0 + per, n_tiles);
    unsigned long long s = 0;
    for (uint32_t t = t0; t < t1; t++) s += tile_sum[t];
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long acc = 0;
        for (int i = 0; i < 1024; i++) { const unsigned long long x = part[i]; part[i] = acc; acc += x; }
        tile_sum[n_tiles] = acc;
    }
    __syncthreads();
    unsigned long long acc = part[threadIdx.x];
    for (uint32_t t = t0; t < t1; t++) { const unsigned long long x = tile_sum[t]; tile_sum[t] = acc; acc += x; }
}

__global__ void __launch_bounds__(256)
k_scan_finish(const uint32_t* __restrict__ v, uint64_t n, const uint64_t* __restrict__ tile_sum, uint64_t* __restrict__ out)
{
    __shared__ unsigned long long warp_sum[8];
    // thread t owns the 8 consecutive values base + 8 t .. base + 8 t + 7
    const uint64_t i0 = (uint64_t)blockIdx.x * kScanTile + 8ull * threadIdx.x;
    uint32_t x[8];
    unsigned long long s = 0;
    for (int k = 0; k < 8; k++) { x[k] = (i0 + k < n) ? v[i0 + k] : 0u; s += x[k]; }
    unsigned long long incl = s;
    const unsigned lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int d = 1; d < 32; d <<= 1) { const unsigned long long up = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += up; }
    if (lane == 31) warp_sum[w] = incl;
    __syncthreads();
    unsigned long long before = tile_sum[blockIdx.x];
    for (unsigned q = 0; q < w; q++) before += warp_sum[q];
    unsigned long long acc = before + incl - s;
    for (int k = 0; k < 8; k++) { if (i0 + k < n) out[i0 + k] = acc; acc += x[k]; }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 255) out[n] = tile_sum[gridDim.x];   // (tile_sum[n_tiles] = the total)
}

// nnz and the longest row of the finished table: stats[0] += sum, stats[1] = max
__global__ void __launch_bounds__(256) k_lut_stats(const uint32_t* __restrict__ row_len, uint64_t n, unsigned long long* stats)
{
    unsigned long long s = 0;
    unsigned m = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (uint64_t)gridDim.x * 256) { const uint32_t l = row_len[i]; s += l; m = max(m, l); }
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0) { atomicAdd(stats, s); atomicMax(stats + 1, (unsigned long long)m); }
}

// One topological level [lo, hi): thread per node, a two-way merge of the children's sorted rows.
__global__ void __launch_bounds__(kBuildThreads)
k_lut_level(const uint32_t* __restrict__ ga, const uint32_t* __restrict__ gb, const float* __restrict__ gw,
            const float* __restrict__ gsig, uint32_t lo, uint32_t hi, const uint64_t* __restrict__ row_ptr,
            uint32_t* row_len, uint32_t* col, double* mu, double* dmu)
{
    const uint32_t n = lo + blockIdx.x * kBuildThreads + threadIdx.x;
    if (n >= hi) return;
    const uint32_t a = ga[n], b = gb[n];
    const double w = (double)gw[n];
    const double rw = gsig ? (double)gsig[n] / w : 0.0;
    const double rw2 = 2.0 * rw * rw;                                    // 2 (dw / w)^2
    uint64_t pa = row_ptr[a], pb = row_ptr[b];
    const uint64_t ea = pa + row_len[a], eb = pb + row_len[b];
    uint64_t o = row_ptr[n];
    const uint64_t o0 = o;
    while (pa < ea || pb < eb) {
        const uint32_t ca = pa < ea ? col[pa] : 0xFFFFFFFFu, cb = pb < eb ? col[pb] : 0xFFFFFFFFu;
        const uint32_t c = ca < cb ? ca : cb;
        double va = 0.0, da = 0.0, vb = 0.0, db = 0.0;
        if (ca == c) { va = mu[pa]; da = dmu[pa]; pa++; }
        if (cb == c) { vb = mu[pb]; db = dmu[pb]; pb++; }
        const double m = (1.0 - w) * va + w * vb;
        double rel2 = rw2;                                               // Eq. 18; absent component: no ratio (Q19)
        if (va != 0.0) rel2 += (da / va) * (da / va);
        if (vb != 0.0) rel2 += (db / vb) * (db / vb);
        col[o] = c;
        mu[o] = m;
        dmu[o] = sqrt(m * m * rel2);
        o++;
    }
    row_len[n] = (uint32_t)(o - o0);
}

}  // namespace

extern "C" void mg_mixture_lut_free(mg_mixture_lut* lut)
{
    if (!lut) return;
    cudaFree(lut->d_row_ptr); cudaFree(lut->d_row_len); cudaFree(lut->d_col);
    cudaFree(lut->d_mu); cudaFree(lut->d_dmu); cudaFree(lut->d_boxes); cudaFree(lut->d_done);
    delete lut;
}

extern "C" int mg_mixture_lut_build(mg_graph* g, const float* weight_sigma, mg_mixture_lut** out, void* stream)
{
    if (!g || !out) { mg::set_error("mg_mixture_lut_build: NULL argument"); return MG_ERR_INVALID_ARG; }
    *out = nullptr;
    {
        const int rc = mg::check_device(g, "mg_mixture_lut_build");
        if (rc != MG_OK) return rc;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const uint64_t n = g->n_nodes;
    const uint32_t nl = g->n_leaves;
    // Row capacities cap(n) = min(n_leaves, cap(a) + cap(b)) and the row starts (their exclusive prefix sum) on the
    // device: one small kernel per topological level + a two-level scan.  (Round 1 did this pass on the host: 14 MB of
    // graph down, 14 MB of row starts up, 7 MB of row lengths down -- 10 of the 10.7 ms of a build on cfg 3.)
    uint32_t* d_cap = nullptr;
    uint64_t* d_row_ptr = nullptr;
    uint64_t* d_tiles = nullptr;
    unsigned long long* d_stats = nullptr;
    const uint32_t n_tiles = (uint32_t)((n + kScanTile - 1) / kScanTile);
    auto fail0 = [&](int rc) { cudaFree(d_cap); cudaFree(d_row_ptr); cudaFree(d_tiles); cudaFree(d_stats); return rc; };
#define LUT0_CUDA(call)                                                             \
    do {                                                                            \
        cudaError_t e__ = (call);                                                   \
        if (e__ != cudaSuccess) return fail0(mg::cuda_fail(e__, #call));            \
    } while (0)
    LUT0_CUDA(cudaMalloc(&d_cap, n * sizeof(uint32_t)));
    LUT0_CUDA(cudaMalloc(&d_row_ptr, (n + 1) * sizeof(uint64_t)));
    LUT0_CUDA(cudaMalloc(&d_tiles, ((size_t)n_tiles + 1) * sizeof(uint64_t)));
    LUT0_CUDA(cudaMalloc(&d_stats, 2 * sizeof(unsigned long long)));
    LUT0_CUDA(cudaMemsetAsync(d_stats, 0, 2 * sizeof(unsigned long long), st));
    for (uint32_t L = 0; L < g->n_levels; L++) {
        const uint32_t lo = (uint32_t)g->level_off[L], hi = (uint32_t)g->level_off[L + 1];
        if (hi == lo) continue;
        k_lut_cap_level<<<(hi - lo + 255) / 256, 256, 0, st>>>(g->d_a, g->d_b, lo, hi, nl, d_cap);
        mg::count_launch();
    }
    k_scan_tile_sums<<<n_tiles, 256, 0, st>>>(d_cap, n, d_tiles);
    k_scan_tiles<<<1, 1024, 0, st>>>(d_tiles, n_tiles);
    k_scan_finish<<<n_tiles, 256, 0, st>>>(d_cap, n, d_tiles, d_row_ptr);
    mg::count_launch(3);
    LUT0_CUDA(cudaGetLastError());
    uint64_t total = 0;
    LUT0_CUDA(cudaMemcpyAsync(&total, d_row_ptr + n, sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
    LUT0_CUDA(cudaStreamSynchronize(st));
    cudaFree(d_cap);
    cudaFree(d_tiles);
    d_cap = nullptr; d_tiles = nullptr;
    size_t free_b = 0, total_b = 0;
    LUT0_CUDA(cudaMemGetInfo(&free_b, &total_b));
    const uint64_t need = total * 20 + n * 4 + (weight_sigma ? n * 4 : 0);
    if (need > free_b) {
        mg::set_error("mg_mixture_lut_build: the table needs %llu entries (%.1f GB), %.1f GB are free",
                      (unsigned long long)total, need / 1e9, free_b / 1e9);
        return fail0(MG_ERR_OOM);
    }
#undef LUT0_CUDA
    mg_mixture_lut* lut = new (std::nothrow) mg_mixture_lut;
    if (!lut) { mg::set_error("mg_mixture_lut_build: out of host memory"); return fail0(MG_ERR_OOM); }
    lut->d_row_ptr = d_row_ptr;                                          // owned by the table from here on
    lut->device = g->device;
    lut->n_nodes = n;
    lut->n_leaves = nl;
    lut->capacity = total;
    float* d_sig = nullptr;
    auto fail = [&](int rc) { cudaFree(d_sig); cudaFree(d_stats); mg_mixture_lut_free(lut); return rc; };
#define LUT_CUDA(call)                                                              \
    do {                                                                            \
        cudaError_t e__ = (call);                                                   \
        if (e__ != cudaSuccess) return fail(mg::cuda_fail(e__, #call));             \
    } while (0)
    LUT_CUDA(cudaMalloc(&lut->d_row_len, n * sizeof(uint32_t)));
    LUT_CUDA(cudaMalloc(&lut->d_col, std::max<uint64_t>(total, 1) * sizeof(uint32_t)));
    LUT_CUDA(cudaMalloc(&lut->d_mu, std::max<uint64_t>(total, 1) * sizeof(double)));
    LUT_CUDA(cudaMalloc(&lut->d_dmu, std::max<uint64_t>(total, 1) * sizeof(double)));
    lut->device_bytes = (n + 1) * 8 + n * 4 + total * 20;
    if (weight_sigma) {
        LUT_CUDA(cudaMalloc(&d_sig, n * sizeof(float)));
        LUT_CUDA(cudaMemcpyAsync(d_sig, weight_sigma, n * sizeof(float), cudaMemcpyHostToDevice, st));
    }
    k_lut_leaves<<<(nl + 255) / 256, 256, 0, st>>>(nl, lut->d_row_ptr, lut->d_row_len, lut->d_col, lut->d_mu, lut->d_dmu);
    LUT_CUDA(cudaGetLastError());
    mg::count_launch();
    for (uint32_t L = 1; L < g->n_levels; L++) {
        const uint32_t lo = (uint32_t)g->level_off[L], hi = (uint32_t)g->level_off[L + 1];
        if (hi == lo) continue;
        k_lut_level<<<(hi - lo + kBuildThreads - 1) / kBuildThreads, kBuildThreads, 0, st>>>(
            g->d_a, g->d_b, g->d_w, d_sig, lo, hi, lut->d_row_ptr, lut->d_row_len, lut->d_col, lut->d_mu, lut->d_dmu);
        LUT_CUDA(cudaGetLastError());
        mg::count_launch();
    }
    k_lut_stats<<<(unsigned)std::min<uint64_t>((n + 255) / 256, 148 * 8), 256, 0, st>>>(lut->d_row_len, n, d_stats);
    LUT_CUDA(cudaGetLastError());
    mg::count_launch();
    unsigned long long stats[2] = {0, 0};
    LUT_CUDA(cudaMemcpyAsync(stats, d_stats, sizeof(stats), cudaMemcpyDeviceToHost, st));
    LUT_CUDA(cudaStreamSynchronize(st));
#undef LUT_CUDA
    cudaFree(d_sig);
    cudaFree(d_stats);
    lut->nnz = stats[0];
    lut->max_row = (uint32_t)stats[1];
    *out = lut;
    return MG_OK;
}

extern "C" int mg_mixture_lut_info(const mg_mixture_lut* lut, mg_lut_info* info)
{
    if (!lut || !info) { mg::set_error("mg_mixture_lut_info: NULL argument"); return MG_ERR_INVALID_ARG; }
    info->n_nodes = lut->n_nodes;
    info->nnz = lut->nnz;
    info->capacity = lut->capacity;
    info->device_bytes = lut->device_bytes;
    info->n_leaves = lut->n_leaves;
    info->max_row_nnz = lut->max_row;
    return MG_OK;
}

extern "C" int mg_mixture_lut_export(const mg_mixture_lut* lut, uint64_t* row_ptr, uint32_t* leaf, double* mu, double* dmu)
{
    if (!lut) { mg::set_error("mg_mixture_lut_export: NULL table"); return MG_ERR_INVALID_ARG; }
    const uint64_t n = lut->n_nodes;
    std::vector<uint64_t> cap_ptr(n + 1);
    std::vector<uint32_t> len(n);
    MG_CUDA(cudaMemcpy(cap_ptr.data(), lut->d_row_ptr, (n + 1) * sizeof(uint64_t), cudaMemcpyDeviceToHost));
    MG_CUDA(cudaMemcpy(len.data(), lut->d_row_len, n * sizeof(uint32_t), cudaMemcpyDeviceToHost));
    std::vector<uint32_t> c;
    std::vector<double> m, d;
    if (leaf) { c.resize(lut->capacity); MG_CUDA(cudaMemcpy(c.data(), lut->d_col, lut->capacity * sizeof(uint32_t), cudaMemcpyDeviceToHost)); }
    if (mu) { m.resize(lut->capacity); MG_CUDA(cudaMemcpy(m.data(), lut->d_mu, lut->capacity * sizeof(double), cudaMemcpyDeviceToHost)); }
    if (dmu) { d.resize(lut->capacity); MG_CUDA(cudaMemcpy(d.data(), lut->d_dmu, lut->capacity * sizeof(double), cudaMemcpyDeviceToHost)); }
    uint64_t o = 0;
    for (uint64_t i = 0; i < n; i++) {                                   // compact: capacity layout -> exact CSR
        if (row_ptr) row_ptr[i] = o;
        const uint64_t s = cap_ptr[i];
        if (leaf) memcpy(leaf + o, c.data() + s, len[i] * sizeof(uint32_t));
        if (mu) memcpy(mu + o, m.data() + s, len[i] * sizeof(double));
        if (dmu) memcpy(dmu + o, d.data() + s, len[i] * sizeof(double));
        o += len[i];
    }
    if (row_ptr) row_ptr[n] = o;
    return MG_OK;
}

namespace {

struct QueryParams {
    const uint32_t* idx;
    unsigned long long off[MG_MAX_MIP_LEVELS];
    int dim[MG_MAX_MIP_LEVELS][3];
    int n_levels;
    uint32_t n_leaves;
    const uint64_t* row_ptr;
    const uint32_t* row_len;
    const uint32_t* col;
    const double* mu;
    const double* dmu;
    const uint64_t* boxes;           // [n_queries][6] staged on the device, or NULL: the boxes travel in `inline_box`
    uint32_t inline_box[kInlineQueries][6];
    uint32_t* done;                  // [n_queries] CTAs of the query that have finished (zeroed by k_query_prologue)
    double* expect;
    double* var;                     // may be NULL
    unsigned long long* fetches;     // may be NULL
    int force_walk;                  // MG_QUERY_FA_WALK
};

// Add one mipmap sample (node, denormalised by `scale` voxels) to query q's dense result.  Called by all
// 32 lanes of a warp (`active` says which hold a sample).  Leaves (pure voxels: mu = e_node, dmu = 0) are
// grouped by node across the warp first, so a homogeneous region costs one atomic per warp.
__device__ __forceinline__ void add_sample(const QueryParams& P, double* expect, double* var, bool active, uint32_t node,
                                           double scale)
{
    const unsigned lane = threadIdx.x & 31;
    const bool pure = active && node < P.n_leaves;
    const unsigned pm = __ballot_sync(0xffffffffu, pure);
    if (pure) {
        const unsigned grp = __match_any_sync(pm, node);
        if (lane == (unsigned)(__ffs(grp) - 1)) atomicAdd(expect + node, scale * (double)__popc(grp));
    } else if (active) {
        const uint64_t r = P.row_ptr[node];
        const uint32_t len = P.row_len[node];
        for (uint32_t k = 0; k < len; k++) {
            const uint32_t c = P.col[r + k];
            atomicAdd(expect + c, scale * P.mu[r + k]);
            if (var) {
                const double d = scale * P.dmu[r + k];
                if (d != 0.0) atomicAdd(var + c, d * d);
            }
        }
    }
}

__device__ __forceinline__ void load_box(const QueryParams& P, uint32_t q, uint32_t* b)
{
#pragma unroll
    for (int a = 0; a < 6; a++) b[a] = P.boxes ? (uint32_t)P.boxes[6ull * q + a] : P.inline_box[q][a];
}

__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// One launch instead of three memsets: the dense results, the fetch counters and the per-query completion counters.
__global__ void __launch_bounds__(256)
k_query_prologue(double* expect, double* var, unsigned long long* fetches, uint32_t* done, uint64_t n_out, uint32_t n_queries)
{
    griddep_launch_dependents();                                          // the query kernel may set up while this one zeroes
    const uint64_t stride = (uint64_t)gridDim.x * 256;
    for (uint64_t i = (uint64_t)blockIdx.x * 256 + threadIdx.x; i < n_out; i += stride) {
        expect[i] = 0.0;
        if (var) var[i] = 0.0;
    }
    for (uint64_t i = (uint64_t)blockIdx.x * 256 + threadIdx.x; i < n_queries; i += stride) {
        if (fetches) fetches[i] = 0ull;
        done[i] = 0u;
    }
}

// Eq. 17: errors add in quadrature -- the LAST CTA of a query to finish takes the square roots of its variances
// (every CTA fences its atomics, then counts itself done; no separate finishing kernel).
__device__ __forceinline__ void finish_query(const QueryParams& P, uint32_t q, double* var)
{
    __shared__ bool s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(P.done + q, 1u) == gridDim.y - 1;
    __syncthreads();
    if (!s_last || !var) return;
    __threadfence();
    for (uint32_t i = threadIdx.x; i < P.n_leaves; i += blockDim.x) var[i] = sqrt(__ldcg(var + i));
}

// Section 3.6, one axis: [lo, hi) cut left to right into the largest aligned power-of-two pieces.
__device__ int fa_axis(uint32_t lo, uint32_t hi, int max_level, uint32_t* start, int* level)
{
    int n = 0;
    uint32_t x = lo;
    while (x < hi) {
        int l = 0;
        while (l + 1 <= max_level && (x & ((2u << l) - 1u)) == 0 && x + (2u << l) <= hi) l++;
        start[n] = x;
        level[n] = l;
        n++;
        x += 1u << l;
    }
    return n;
}

// The box t = a + nx (b + ny c) of the footprint's tensor product: its cube level and grid of cubes.
struct FaBox {
    int l, ex, ey, ez;                  // cube level; cubes per axis = 2^e
    uint32_t bx, by, bz;                // first cube, in level-l voxel coordinates
    unsigned long long n_cubes;
};

__device__ __forceinline__ FaBox fa_box(const uint32_t (*s_start)[kMaxPieces], const int (*s_level)[kMaxPieces], int a, int b, int c)
{
    FaBox B;
    const int lx = s_level[0][a], ly = s_level[1][b], lz = s_level[2][c];
    B.l = min(lx, min(ly, lz));                                          // cube side = the shortest extent
    B.ex = lx - B.l; B.ey = ly - B.l; B.ez = lz - B.l;
    B.n_cubes = 1ull << (B.ex + B.ey + B.ez);
    B.bx = s_start[0][a] >> B.l; B.by = s_start[1][b] >> B.l; B.bz = s_start[2][c] >> B.l;
    return B;
}

// Chunk ch (32 cubes, one per lane) of a box: one mipmap sample per cube, denormalised by side^3 = 8^l.
__device__ __forceinline__ unsigned fa_chunk(const QueryParams& P, double* expect, double* var, const FaBox& B, unsigned long long ch)
{
    const unsigned lane = threadIdx.x & 31;
    const unsigned long long k = (ch << 5) + lane;
    const bool active = k < B.n_cubes;
    uint32_t node = 0;
    if (active) {
        const uint32_t ix = (uint32_t)(k & ((1ull << B.ex) - 1)), iy = (uint32_t)((k >> B.ex) & ((1ull << B.ey) - 1)),
                       iz = (uint32_t)(k >> (B.ex + B.ey));
        node = __ldg(P.idx + P.off[B.l] + ((size_t)(B.bz + iz) * P.dim[B.l][1] + (B.by + iy)) * P.dim[B.l][0] + (B.bx + ix));
    }
    add_sample(P, expect, var, active, node, __hiloint2double((1023 + 3 * B.l) << 20, 0));
    return (unsigned)min(32ull, B.n_cubes - (ch << 5));
}

constexpr int kMaxBoxes = 4096;         // boxes whose chunk prefix fits the CTA's shared memory

// grid = (n_queries, splits); the warps of all CTAs of a query share its chunks (32 cubes of one box).  Every
// CTA builds the prefix sum of the chunks per box in shared memory (threads over boxes, then a scan), and warp w of
// the query takes the chunks g = w, w + n_warps, ...: a binary search finds the box.  Queries with more than
// kMaxBoxes boxes fall back to every warp walking all boxes (chunk c of box t goes to warp (t + c) mod n_warps).
__global__ void __launch_bounds__(kQueryThreads)
k_range_query_fa(const __grid_constant__ QueryParams P)
{
    __shared__ uint32_t s_start[3][kMaxPieces];
    __shared__ int s_level[3][kMaxPieces];
    __shared__ int s_n[3];
    __shared__ unsigned long long s_pref[kMaxBoxes + 1];
    __shared__ unsigned long long s_part[kQueryThreads];
    const uint32_t q = blockIdx.x;
    uint32_t box[6];
    load_box(P, q, box);
    if (threadIdx.x < 3)
        s_n[threadIdx.x] = fa_axis(box[threadIdx.x], box[3 + threadIdx.x], P.n_levels - 1,
                                   s_start[threadIdx.x], s_level[threadIdx.x]);
    __syncthreads();
    griddep_wait();                                                       // k_query_prologue has zeroed the results
    const int nx = s_n[0], ny = s_n[1], nz = s_n[2];
    const unsigned lane = threadIdx.x & 31;
    const unsigned n_warps = gridDim.y * (kQueryThreads / 32), warp = blockIdx.y * (kQueryThreads / 32) + threadIdx.x / 32;
    double* expect = P.expect + (uint64_t)q * P.n_leaves;
    double* var = P.var ? P.var + (uint64_t)q * P.n_leaves : nullptr;
    unsigned long long n_fetch = 0;
    const unsigned n_boxes = (unsigned)(nx * ny * nz);
    if (n_boxes <= (unsigned)kMaxBoxes && !P.force_walk) {
        // chunks per box -> inclusive prefix: each thread a run of boxes, then the runs' totals are scanned
        const unsigned per = (n_boxes + kQueryThreads - 1) / kQueryThreads;
        const unsigned t0 = min(threadIdx.x * per, n_boxes), t1 = min(t0 + per, n_boxes);
        unsigned long long run = 0;
        for (unsigned t = t0; t < t1; t++) {
            const FaBox B = fa_box(s_start, s_level, (int)(t % nx), (int)((t / nx) % ny), (int)(t / (nx * ny)));
            run += (B.n_cubes + 31) >> 5;
            s_pref[t + 1] = run;
        }
        s_part[threadIdx.x] = run;
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned long long acc = 0;
            for (int i = 0; i < kQueryThreads; i++) { const unsigned long long v = s_part[i]; s_part[i] = acc; acc += v; }
            s_pref[0] = 0;
        }
        __syncthreads();
        const unsigned long long base = s_part[threadIdx.x];
        for (unsigned t = t0; t < t1; t++) s_pref[t + 1] += base;
        __syncthreads();
        const unsigned long long total = s_pref[n_boxes];
        for (unsigned long long g = warp; g < total; g += n_warps) {
            unsigned lo = 0, hi = n_boxes;                               // largest t with s_pref[t] <= g
            while (hi - lo > 1) {
                const unsigned mid = (lo + hi) >> 1;
                if (s_pref[mid] <= g) lo = mid; else hi = mid;
            }
            const FaBox B = fa_box(s_start, s_level, (int)(lo % nx), (int)((lo / nx) % ny), (int)(lo / (nx * ny)));
            const unsigned f = fa_chunk(P, expect, var, B, g - s_pref[lo]);
            if (lane == 0) n_fetch += f;
        }
    } else {
        // (a, b, c) and t mod n_warps are carried along incrementally: no divisions in the walk
        int a = -1, b = 0, c = 0;
        unsigned tm = n_warps - 1;                                       // (t - 1) mod n_warps
        for (unsigned t = 0; t < n_boxes; t++) {
            if (++a == nx) { a = 0; if (++b == ny) { b = 0; ++c; } }
            if (++tm == n_warps) tm = 0;
            const FaBox B = fa_box(s_start, s_level, a, b, c);
            const unsigned long long n_chunks = (B.n_cubes + 31) >> 5;
            for (unsigned long long ch = warp >= tm ? warp - tm : warp + n_warps - tm; ch < n_chunks; ch += n_warps) {
                const unsigned f = fa_chunk(P, expect, var, B, ch);
                if (lane == 0) n_fetch += f;
            }
        }
    }
    if (P.fetches && lane == 0 && n_fetch) atomicAdd(P.fetches + q, n_fetch);
    finish_query(P, q, var);
}

// The naive approach (L377): every level-0 voxel of the box is one sample.  Warps take rows of the box (lanes
// along x: coalesced, no divisions in the inner loop).  Level-0 voxels are leaves (L223), so with SMEM their counts
// go to a per-CTA histogram in shared memory (uint32[n_leaves], grouped per warp by __match_any_sync first) that is
// flushed once with one fp64 atomic per non-zero bin; any other node, or a table too large for shared memory
// (SMEM = false), takes the general path of add_sample.
template <bool SMEM>
__global__ void __launch_bounds__(kQueryThreads)
k_range_query_naive(const __grid_constant__ QueryParams P)
{
    extern __shared__ uint32_t s_cnt[];
    const uint32_t q = blockIdx.x;
    uint32_t box[6];
    load_box(P, q, box);
    const uint32_t x0 = box[0], y0 = box[1], z0 = box[2];
    const uint32_t dx = box[3] - x0, dy = box[4] - y0, dz = box[5] - z0;
    griddep_wait();                                                       // k_query_prologue has zeroed the results
    const int X = P.dim[0][0], Y = P.dim[0][1];
    double* expect = P.expect + (uint64_t)q * P.n_leaves;
    double* var = P.var ? P.var + (uint64_t)q * P.n_leaves : nullptr;
    if (SMEM) {
        for (uint32_t i = threadIdx.x; i < P.n_leaves; i += kQueryThreads) s_cnt[i] = 0;
        __syncthreads();
    }
    const unsigned lane = threadIdx.x & 31;
    const unsigned n_warps = gridDim.y * (kQueryThreads / 32), warp = blockIdx.y * (kQueryThreads / 32) + threadIdx.x / 32;
    const uint64_t n_rows = (uint64_t)dy * dz;                             // up to 2^40 (2^20 voxels per axis)
    for (uint64_t r = warp; r < n_rows; r += n_warps) {
        const uint32_t iy = (uint32_t)(r % dy), iz = (uint32_t)(r / dy);
        const uint32_t* row = P.idx + P.off[0] + ((size_t)(z0 + iz) * Y + (y0 + iy)) * X + x0;
        for (uint32_t bx = 0; bx < dx; bx += 32 * kNaiveUnroll) {          // warp-uniform trip count
            uint32_t node[kNaiveUnroll];
            bool active[kNaiveUnroll];
#pragma unroll
            for (int u = 0; u < kNaiveUnroll; u++) {                       // the loads of the whole group first
                active[u] = bx + 32 * u + lane < dx;
                node[u] = active[u] ? __ldg(row + bx + 32 * u + lane) : 0u;
            }
#pragma unroll
            for (int u = 0; u < kNaiveUnroll; u++) {
                if (bx + 32 * u >= dx) break;                              // (uniform)
                if (SMEM) {
                    const bool pure = active[u] && node[u] < P.n_leaves;
                    const unsigned pm = __ballot_sync(0xffffffffu, pure);
                    const uint32_t first = __shfl_sync(0xffffffffu, node[u], 0);
                    if (pm == 0xffffffffu && __all_sync(0xffffffffu, node[u] == first)) {
                        if (lane == 0) atomicAdd(&s_cnt[first], 32u);      // a run of one segment: the common case
                    } else {
                        if (pure) {
                            const unsigned grp = __match_any_sync(pm, node[u]);
                            if (lane == (unsigned)(__ffs(grp) - 1)) atomicAdd(&s_cnt[node[u]], (uint32_t)__popc(grp));
                        }
                        add_sample(P, expect, var, active[u] && !pure, node[u], 1.0);   // not a leaf: its table row
                    }
                } else {
                    add_sample(P, expect, var, active[u], node[u], 1.0);
                }
            }
        }
    }
    if (SMEM) {
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < P.n_leaves; i += kQueryThreads)
            if (s_cnt[i]) atomicAdd(expect + i, (double)s_cnt[i]);
    }
    if (P.fetches && blockIdx.y == 0 && threadIdx.x == 0) atomicAdd(P.fetches + q, (unsigned long long)dx * dy * dz);
    finish_query(P, q, var);
}

}  // namespace

extern "C" int mg_range_query(mg_mixture_lut* lut, const uint32_t* node_idx_mipmap, const mg_mipmap_desc* mip,
                              const uint64_t* boxes, uint32_t n_queries, double* expect, double* err, uint64_t* fetches,
                              uint32_t mode, void* stream)
{
    if (!lut || !node_idx_mipmap || !mip || !expect || (n_queries && !boxes)) {
        mg::set_error("mg_range_query: NULL argument");
        return MG_ERR_INVALID_ARG;
    }
    if (mode != MG_QUERY_FA && mode != MG_QUERY_NAIVE && mode != MG_QUERY_FA_WALK) { mg::set_error("mg_range_query: unknown mode %u", mode); return MG_ERR_INVALID_ARG; }
    if (((uintptr_t)expect & 7) || ((uintptr_t)err & 7) || ((uintptr_t)fetches & 7) || ((uintptr_t)node_idx_mipmap & 3)) {
        mg::set_error("mg_range_query: misaligned buffer");
        return MG_ERR_INVALID_ARG;
    }
    if (mip->n_levels == 0 || mip->n_levels > MG_MAX_MIP_LEVELS) {
        mg::set_error("mg_range_query: n_levels = %u not in 1..%d", mip->n_levels, MG_MAX_MIP_LEVELS);
        return MG_ERR_INVALID_ARG;
    }
    QueryParams P;
    memset(&P, 0, sizeof(P));
    for (uint32_t l = 0; l < mip->n_levels; l++) {
        for (int a = 0; a < 3; a++) {
            const uint32_t dl = mip->level_dim[l][a];
            if (dl == 0 || dl > (1u << 20) || (l > 0 && dl != (mip->level_dim[l - 1][a] + 1) / 2)) {
                mg::set_error("mg_range_query: level %u axis %d has %u voxels: not the ceil-halving chain of L80", l, a, dl);
                return MG_ERR_INVALID_ARG;
            }
            P.dim[l][a] = (int)dl;
        }
        P.off[l] = mip->level_offset[l];
    }
    const uint32_t* top = mip->level_dim[mip->n_levels - 1];
    if (top[0] != 1 || top[1] != 1 || top[2] != 1) {
        mg::set_error("mg_range_query: the mipmap must run up to its 1 x 1 x 1 level");
        return MG_ERR_INVALID_ARG;
    }
    for (uint32_t q = 0; q < n_queries; q++) {
        const uint64_t* b = boxes + 6ull * q;
        for (int a = 0; a < 3; a++)
            if (!(b[a] < b[3 + a]) || b[3 + a] > mip->level_dim[0][a]) {
                mg::set_error("mg_range_query: box %u is empty or leaves the volume along axis %d", q, a);
                return MG_ERR_INVALID_ARG;
            }
    }
    if (n_queries == 0) return MG_OK;
    {
        int dev = -1;
        MG_CUDA(cudaGetDevice(&dev));
        if (dev != lut->device) { mg::set_error("mg_range_query: the table lives on CUDA device %d but device %d is current", lut->device, dev); return MG_ERR_INVALID_ARG; }
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (n_queries > lut->boxes_cap) {
        MG_CUDA(cudaStreamSynchronize(st));                              // earlier queries may still read the old buffers
        cudaFree(lut->d_boxes);
        cudaFree(lut->d_done);
        lut->d_boxes = nullptr;
        lut->d_done = nullptr;
        lut->boxes_cap = 0;
        const uint32_t cap = std::max<uint32_t>(n_queries, kInlineQueries);
        MG_CUDA(cudaMalloc(&lut->d_boxes, (size_t)cap * 6 * sizeof(uint64_t)));
        MG_CUDA(cudaMalloc(&lut->d_done, (size_t)cap * sizeof(uint32_t)));
        lut->boxes_cap = cap;
    }
    const uint64_t n_out = (uint64_t)n_queries * lut->n_leaves;
    if (n_queries <= (uint32_t)kInlineQueries) {                          // small batch: the boxes ride in the kernel parameters
        P.boxes = nullptr;
        for (uint32_t q = 0; q < n_queries; q++)
            for (int a = 0; a < 6; a++) P.inline_box[q][a] = (uint32_t)boxes[6ull * q + a];
    } else {
        MG_CUDA(cudaMemcpyAsync(lut->d_boxes, boxes, (size_t)n_queries * 6 * sizeof(uint64_t), cudaMemcpyHostToDevice, st));
        P.boxes = lut->d_boxes;
    }
    P.done = lut->d_done;
    {
        const unsigned blocks = (unsigned)std::min<uint64_t>((std::max<uint64_t>(n_out, n_queries) + 255) / 256, 148ull * 8);
        k_query_prologue<<<blocks, 256, 0, st>>>(expect, err, reinterpret_cast<unsigned long long*>(fetches), lut->d_done, n_out, n_queries);
        MG_CUDA(cudaGetLastError());
        mg::count_launch();
    }
    P.idx = node_idx_mipmap;
    P.n_levels = (int)mip->n_levels;
    P.n_leaves = lut->n_leaves;
    P.row_ptr = lut->d_row_ptr; P.row_len = lut->d_row_len; P.col = lut->d_col; P.mu = lut->d_mu; P.dmu = lut->d_dmu;
    P.expect = expect;
    P.var = err;
    P.fetches = reinterpret_cast<unsigned long long*>(fetches);
    // spread a query over enough CTAs to fill the machine when there are few queries (148 SMs x 8 CTAs)
    uint32_t splits = std::max<uint32_t>(1, std::min<uint32_t>(64, (148 * 8 + n_queries - 1) / n_queries));
    if (mode == MG_QUERY_NAIVE) {
        // the per-CTA leaf histogram counts in uint32: a CTA takes rows round-robin, at most vol / splits + 8 rows'
        // worth of voxels, so keep vol / splits <= 2^31 (dx <= 2^20 leaves the margin)
        uint64_t max_vol = 0;
        for (uint32_t q = 0; q < n_queries; q++) {
            const uint64_t* b = boxes + 6ull * q;
            max_vol = std::max(max_vol, (b[3] - b[0]) * (b[4] - b[1]) * (b[5] - b[2]));
        }
        const uint64_t need = (max_vol >> 31) + 1;
        if (need > 65535) { mg::set_error("mg_range_query: MG_QUERY_NAIVE supports boxes of up to 2^46 voxels"); return MG_ERR_INVALID_ARG; }
        splits = std::max<uint32_t>(splits, (uint32_t)need);
    }
    const dim3 grid(n_queries, splits);
    P.force_walk = (mode == MG_QUERY_FA_WALK);
    // launched with programmatic stream serialisation: the decomposition of the boxes overlaps the prologue's zeroing; every
    // kernel executes griddepcontrol.wait before its first atomic
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(kQueryThreads);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (mode != MG_QUERY_NAIVE) {
        MG_CUDA(cudaLaunchKernelEx(&cfg, k_range_query_fa, P));
    } else {
        const size_t smem = (size_t)lut->n_leaves * sizeof(uint32_t);
        if (smem <= 200 * 1024) {                                          // per-CTA leaf histogram in shared memory
            static mg::SmemAttrOnce once;                                  // per (function, device)
            const int rc = once.ensure((const void*)k_range_query_naive<true>, 200 * 1024, lut->device);
            if (rc != MG_OK) return rc;
            cfg.dynamicSmemBytes = smem;
            MG_CUDA(cudaLaunchKernelEx(&cfg, k_range_query_naive<true>, P));
        } else {
            MG_CUDA(cudaLaunchKernelEx(&cfg, k_range_query_naive<false>, P));
        }
    }
    mg::count_launch();
    return MG_OK;
}
