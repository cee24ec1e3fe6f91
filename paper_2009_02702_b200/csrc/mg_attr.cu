// mg_attr.cu -- NEXT-1: propagation of ANY numeric segment attribute with C channels per node.
//
//   x[n][ch] = (1 - w[n]) x[a[n]][ch] + w[n] x[b[n]][ch]
//
// "the Mixture Graph allows the efficient computation of any kind of numeric segmentation
// attribute" (L269).  The paper's own uses besides RGBA: opacity alone for empty-space skipping
// (L271 (i)-(ii)) and diffuse / specular light contributions (L277); K transfer functions batched as
// 4 K channels share ONE pass over the graph arrays (12 B per node read once instead of K times).
//
// Layout: [node][C], channel fastest, so a gather of one child is C*4 contiguous bytes.
// Mapping: one thread = one (node, vector chunk) item, V = float4 / float2 / float chosen from the
// divisibility of C (and the pointers' alignment); the threads of one node are neighbours, so the
// stores of a warp are fully contiguous, the a/b/w loads are broadcasts and each child's gather is
// one contiguous segment.  Level 1 gathers straight from the caller's leaf array and the threads
// past its items copy the leaves (a4), exactly like k_level<true> of mg_propagate.cu.
// The small top levels run in ONE CTA (k_tail_attr) with __syncthreads() between levels; it works
// through L2 (ld.cg / st) rather than shared memory because C is a run-time quantity.
// Same PDL rule as mg_propagate.cu: data written by an earlier kernel is read with ld.cg only.
#include "mg_internal.h"

namespace {

constexpr int kThreads = 256;
constexpr int kTailThreads = 1024;

__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ float lerp1(float ca, float cb, float w) { return fmaf(w, cb, fmaf(-w, ca, ca)); }
__device__ __forceinline__ float lerpv(float ca, float cb, float w) { return lerp1(ca, cb, w); }
__device__ __forceinline__ float2 lerpv(float2 ca, float2 cb, float w) { return make_float2(lerp1(ca.x, cb.x, w), lerp1(ca.y, cb.y, w)); }
__device__ __forceinline__ float4 lerpv(float4 ca, float4 cb, float w)
{
    return make_float4(lerp1(ca.x, cb.x, w), lerp1(ca.y, cb.y, w), lerp1(ca.z, cb.z, w), lerp1(ca.w, cb.w, w));
}

// One level [lo, hi): item i = (node lo + i / chunks, chunk i % chunks).  `src` is the leaf array for
// FIRST (level 1: every child is a leaf) and the node array otherwise.
template <typename V, bool FIRST>
__global__ void __launch_bounds__(kThreads)
k_level_attr(const uint32_t* __restrict__ ga, const uint32_t* __restrict__ gb, const float* __restrict__ gw,
             const V* __restrict__ src, V* x, uint32_t lo, uint32_t chunks, uint64_t n_items, uint64_t n_leaf_items)
{
    griddep_launch_dependents();
    const uint64_t i = (uint64_t)blockIdx.x * kThreads + threadIdx.x;
    uint32_t a = 0, b = 0, q = 0, n = 0;
    float w = 0.f;
    const bool live = i < n_items;
    if (live) {                                    // static operands: before the dependency wait
        n = lo + (uint32_t)(i / chunks);
        q = (uint32_t)(i % chunks);
        a = __ldg(ga + n); b = __ldg(gb + n); w = __ldg(gw + n);
    }
    griddep_wait();
    if (live) {
        const V ca = FIRST ? __ldg(src + (uint64_t)a * chunks + q) : __ldcg(src + (uint64_t)a * chunks + q);
        const V cb = FIRST ? __ldg(src + (uint64_t)b * chunks + q) : __ldcg(src + (uint64_t)b * chunks + q);
        x[(uint64_t)n * chunks + q] = lerpv(ca, cb, w);
    } else if (FIRST) {
        const uint64_t k = i - n_items;            // leaf assignment x[k] = attr[k], bit-exact
        if (k < n_leaf_items) x[k] = __ldg(src + k);
    }
}

// Levels [first_level, n_levels) in one CTA.  Reads of x go through L2 (ld.cg): entries written by
// this CTA before the preceding __syncthreads(), or by earlier kernels of the update.
template <typename V>
__global__ void __launch_bounds__(kTailThreads, 1)
k_tail_attr(const uint32_t* __restrict__ ga, const uint32_t* __restrict__ gb, const float* __restrict__ gw,
            const V* __restrict__ leaf, V* x, const uint32_t* __restrict__ off, uint32_t first_level, uint32_t n_levels,
            uint32_t chunks, uint64_t n_leaf_items, int copy_leaves)
{
    griddep_launch_dependents();
    griddep_wait();
    if (copy_leaves) {
        for (uint64_t k = threadIdx.x; k < n_leaf_items; k += kTailThreads) x[k] = __ldcg(leaf + k);
        __threadfence_block();
        __syncthreads();
    }
    for (uint32_t L = first_level; L < n_levels; L++) {
        const uint32_t lo = __ldg(off + L), hi = __ldg(off + L + 1);
        const uint64_t items = (uint64_t)(hi - lo) * chunks;
        for (uint64_t i = threadIdx.x; i < items; i += kTailThreads) {
            const uint32_t n = lo + (uint32_t)(i / chunks), q = (uint32_t)(i % chunks);
            const uint32_t a = __ldg(ga + n), b = __ldg(gb + n);
            const float w = __ldg(gw + n);
            x[(uint64_t)n * chunks + q] = lerpv(__ldcg(x + (uint64_t)a * chunks + q), __ldcg(x + (uint64_t)b * chunks + q), w);
        }
        __threadfence_block();
        __syncthreads();                           // the level barrier
    }
}

template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(bool pdl, void (*kernel)(KArgs...), unsigned grid, unsigned block, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// Levels with fewer items than this (and every later level) go to the single-CTA tail.
constexpr uint64_t kTailMaxLevelNodes = 4096;

template <typename V>
int propagate_attr(mg_graph* g, const float* leaf_attr, float* node_attr, uint32_t chunks, cudaStream_t st)
{
    const V* leaf = reinterpret_cast<const V*>(leaf_attr);
    V* x = reinterpret_cast<V*>(node_attr);
    const uint32_t n_levels = g->n_levels;
    const uint64_t n_leaf_items = (uint64_t)g->n_leaves * chunks;
    // tail = longest suffix of levels that are all small
    uint32_t first_tail = n_levels;
    while (first_tail > 1 && g->level_off[first_tail] - g->level_off[first_tail - 1] <= kTailMaxLevelNodes &&
           n_levels - first_tail < MG_TAIL_MAX_LEVELS) first_tail--;
    bool first = true;
    for (uint32_t L = 1; L < first_tail; L++) {
        const uint32_t lo = (uint32_t)g->level_off[L], hi = (uint32_t)g->level_off[L + 1];
        const uint64_t n_items = (uint64_t)(hi - lo) * chunks;
        const uint64_t total = n_items + (L == 1 ? n_leaf_items : 0);
        const uint64_t blocks = (total + kThreads - 1) / kThreads;
        if (blocks > 0x7fffffffull) { mg::set_error("mg_propagate_attr: level %u too large for one launch", L); return MG_ERR_INVALID_ARG; }
        if (L == 1)
            MG_CUDA(launch_pdl(false, k_level_attr<V, true>, (unsigned)blocks, kThreads, st, g->d_a, g->d_b, g->d_w, leaf, x, lo, chunks,
                               n_items, n_leaf_items));
        else
            MG_CUDA(launch_pdl(true, k_level_attr<V, false>, (unsigned)blocks, kThreads, st, g->d_a, g->d_b, g->d_w, (const V*)x, x, lo,
                               chunks, n_items, (uint64_t)0));
        mg::count_launch();
        first = false;
    }
    if (first_tail < n_levels || first) {
        MG_CUDA(launch_pdl(!first, k_tail_attr<V>, 1u, (unsigned)kTailThreads, st, g->d_a, g->d_b, g->d_w, leaf, x, g->d_level_off,
                           first_tail, n_levels, chunks, n_leaf_items, first ? 1 : 0));
        mg::count_launch();
    }
    return MG_OK;
}

}  // namespace

extern "C" int mg_propagate_attr(mg_graph* g, const float* leaf_attr, float* node_attr, uint32_t n_channels, void* stream)
{
    if (!g || !leaf_attr || !node_attr) { mg::set_error("mg_propagate_attr: NULL argument"); return MG_ERR_INVALID_ARG; }
    if (n_channels == 0 || n_channels > MG_MAX_ATTR_CHANNELS) {
        mg::set_error("mg_propagate_attr: n_channels must be 1 .. %d", MG_MAX_ATTR_CHANNELS); return MG_ERR_INVALID_ARG;
    }
    if (((uintptr_t)leaf_attr | (uintptr_t)node_attr) & 3) { mg::set_error("mg_propagate_attr: buffers must be 4-byte aligned"); return MG_ERR_INVALID_ARG; }
    if (leaf_attr == node_attr) { mg::set_error("mg_propagate_attr: leaf_attr and node_attr must not alias"); return MG_ERR_INVALID_ARG; }
    const int rc = mg::check_device(g, "mg_propagate_attr");
    if (rc != MG_OK) return rc;
    // node_attr may be (part of) the node_rgba the 8/16-bit palettes mirror: they stop mirroring it here
    mg::invalidate_palettes_if_written(g, node_attr, g->n_nodes * (uint64_t)n_channels * 4);
    const uintptr_t al = (uintptr_t)leaf_attr | (uintptr_t)node_attr;
    cudaStream_t st = (cudaStream_t)stream;
    if (n_channels % 4 == 0 && (al & 15) == 0) return propagate_attr<float4>(g, leaf_attr, node_attr, n_channels / 4, st);
    if (n_channels % 2 == 0 && (al & 7) == 0) return propagate_attr<float2>(g, leaf_attr, node_attr, n_channels / 2, st);
    return propagate_attr<float>(g, leaf_attr, node_attr, n_channels, st);
}
