// mg_propagate.cu -- leaf assignment (a4) and level-synchronous propagation (a5) for sm_100a.
//
//   c[n] = (1 - w[n]) c[a[n]] + w[n] c[b[n]]
//
// computed per channel in fp32 as fma(w, cb, fma(-w, ca, ca)) (reading Q12).  The graph is stored
// level-contiguously, so a topological level (L211) is an index range and "nodes with identical
// values can be processed without synchronization" (L213) becomes one launch per large level.
// This is a gather/lerp stream bound by HBM/L2, not a contraction: no tensor cores.
//
// Kernels
//   k_level<FIRST>   one thread = 4 consecutive nodes: three 16-byte streaming loads (child_a,
//                    child_b, weight), eight 16-byte palette gathers, four 16-byte colour stores and
//                    the 8-bit / 16-bit palette entries of those nodes.  FIRST: level 1, whose
//                    children are all leaves -- gathers come straight from the TF and the spare
//                    threads perform the leaf copy, so the update needs no separate copy kernel.
//   k_tail           ONE persistent CTA runs all the small top levels, __syncthreads() between
//                    levels instead of kernel boundaries, ENTIRELY in shared memory: a/b/w of
//                    the whole tail are staged up front (static data: before the grid-dependency
//                    wait), the distinct children below the tail are gathered once, and every
//                    level is then shared-memory gathers + one barrier (~0.2 us instead of two
//                    DRAM/L2 round trips per level).
//
// Every kernel but the first of an update is launched with programmatic dependent launch (PDL): it
// signals `griddepcontrol.launch_dependents` at once, loads its static operands (graph arrays), and
// only then executes `griddepcontrol.wait` (= the previous kernel on the stream has completed and
// its writes are visible) before touching colours.  The launch latency and the a/b/w stream of
// level L+1 overlap level L.  Rule: inside a PDL-launched kernel, data written by an earlier kernel
// (colours, and the TF, which the caller may rewrite between updates) is read through L2 (ld.cg);
// the non-coherent path (ld.global.nc) is used only for the immutable graph arrays and, in the
// normally-launched first kernel, for the TF.
#include <cuda_fp16.h>

#include "mg_internal.h"

namespace {

constexpr int kLevelThreads = 256;
constexpr int kTailThreads = 1024;
constexpr int kTailMaxLevels = MG_TAIL_MAX_LEVELS;   // levels the tail kernel can hold offsets for

__device__ __forceinline__ uint4 ld_stream_u4(const void* p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

// Colours written by an earlier kernel of the same update: read through L2 (.cg), never through the
// non-coherent path -- with PDL this kernel's CTAs may be resident before the producer has finished.
__device__ __forceinline__ float4 ld_colour(const float4* p) { return __ldcg(p); }

__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ float4 lerp4(float4 ca, float4 cb, float w)
{
    float4 r;
    r.x = fmaf(w, cb.x, fmaf(-w, ca.x, ca.x));
    r.y = fmaf(w, cb.y, fmaf(-w, ca.y, ca.y));
    r.z = fmaf(w, cb.z, fmaf(-w, ca.z, ca.z));
    r.w = fmaf(w, cb.w, fmaf(-w, ca.w, ca.w));
    return r;
}

// RGBA8: clamp to [0,1] (NaN -> 0), times 255, round half to even, R in byte 0 (reading Q13).
__device__ __forceinline__ uint32_t to_rgba8(float4 c)
{
    uint32_t r = __float2uint_rn(__saturatef(c.x) * 255.0f);
    uint32_t g = __float2uint_rn(__saturatef(c.y) * 255.0f);
    uint32_t b = __float2uint_rn(__saturatef(c.z) * 255.0f);
    uint32_t a = __float2uint_rn(__saturatef(c.w) * 255.0f);
    return r | (g << 8) | (b << 16) | (a << 24);
}

__device__ __forceinline__ uint2 to_rgba16f(float4 c)
{
    __half2 lo = __floats2half2_rn(c.x, c.y);
    __half2 hi = __floats2half2_rn(c.z, c.w);
    uint2 r;
    r.x = *reinterpret_cast<uint32_t*>(&lo);
    r.y = *reinterpret_cast<uint32_t*>(&hi);
    return r;
}

// PAL: also derive the node's 8-bit / 16-bit palette entries (off for graphs loaded with MG_NO_PALETTES).
template <bool PAL>
__device__ __forceinline__ void store_node(float4* c, uint32_t* __restrict__ pal8,
                                           uint2* __restrict__ pal16, uint32_t n, float4 v)
{
    c[n] = v;
    if (PAL) {
        pal8[n] = to_rgba8(v);
        pal16[n] = to_rgba16f(v);
    }
}

// FIRST: the source is the caller's TF (read-only input: non-coherent path); else node colours.
template <bool FIRST>
__device__ __forceinline__ float4 ld_src(const float4* p) { return FIRST ? __ldg(p) : ld_colour(p); }

// One level [lo, hi).  Work is cut into groups of 4 nodes aligned to absolute index 4g, so the
// 16-byte loads of a/b/w are aligned whatever lo is; edge groups fall back to scalar accesses.
template <bool FIRST, bool PAL>
__global__ void __launch_bounds__(kLevelThreads)
k_level(const uint32_t* __restrict__ ga, const uint32_t* __restrict__ gb, const float* __restrict__ gw,
        const float4* __restrict__ src,   // FIRST: the TF; else: node colours of the lower levels
        float4* c, uint32_t* __restrict__ pal8, uint2* __restrict__ pal16,
        uint32_t lo, uint32_t hi, uint32_t n_leaves, uint32_t n_groups)
{
    griddep_launch_dependents();
    const uint32_t t = blockIdx.x * kLevelThreads + threadIdx.x;
    const uint32_t n0 = (lo & ~3u) + 4u * t;
    const bool live = t < n_groups;
    const bool full = live && n0 >= lo && n0 + 4u <= hi;
    uint4 a = make_uint4(0, 0, 0, 0), b = a, wu = a;
    if (full) {                                   // static operands: before the dependency wait
        a = ld_stream_u4(ga + n0);
        b = ld_stream_u4(gb + n0);
        wu = ld_stream_u4(gw + n0);
    }
    griddep_wait();                               // lower levels complete; previous readers of c / pal done
    if (full) {
        const float4 ca0 = ld_src<FIRST>(src + a.x), cb0 = ld_src<FIRST>(src + b.x);
        const float4 ca1 = ld_src<FIRST>(src + a.y), cb1 = ld_src<FIRST>(src + b.y);
        const float4 ca2 = ld_src<FIRST>(src + a.z), cb2 = ld_src<FIRST>(src + b.z);
        const float4 ca3 = ld_src<FIRST>(src + a.w), cb3 = ld_src<FIRST>(src + b.w);
        const float4 r0 = lerp4(ca0, cb0, __uint_as_float(wu.x));
        const float4 r1 = lerp4(ca1, cb1, __uint_as_float(wu.y));
        const float4 r2 = lerp4(ca2, cb2, __uint_as_float(wu.z));
        const float4 r3 = lerp4(ca3, cb3, __uint_as_float(wu.w));
        c[n0] = r0; c[n0 + 1] = r1; c[n0 + 2] = r2; c[n0 + 3] = r3;
        if (PAL) {
            *reinterpret_cast<uint4*>(pal8 + n0) = make_uint4(to_rgba8(r0), to_rgba8(r1), to_rgba8(r2), to_rgba8(r3));
            const uint2 h0 = to_rgba16f(r0), h1 = to_rgba16f(r1), h2 = to_rgba16f(r2), h3 = to_rgba16f(r3);
            *reinterpret_cast<uint4*>(pal16 + n0) = make_uint4(h0.x, h0.y, h1.x, h1.y);
            *reinterpret_cast<uint4*>(pal16 + n0 + 2) = make_uint4(h2.x, h2.y, h3.x, h3.y);
        }
    } else if (live) {
#pragma unroll
        for (uint32_t k = 0; k < 4; k++) {
            const uint32_t n = n0 + k;
            if (n >= lo && n < hi)
                store_node<PAL>(c, pal8, pal16, n, lerp4(ld_src<FIRST>(src + ga[n]), ld_src<FIRST>(src + gb[n]), gw[n]));
        }
    }
    if (FIRST) {
        // leaf assignment c[k] = TF[k], bit-exact (L371), by the threads past the node groups
        const uint32_t total = gridDim.x * kLevelThreads;
        const uint32_t spare0 = n_groups;
        const uint32_t n_spare = total - spare0;
        if (t >= spare0)
            for (uint32_t k = t - spare0; k < n_leaves; k += n_spare) store_node<PAL>(c, pal8, pal16, k, __ldg(src + k));
    }
}

// All levels L in [first_level, n_levels) in one CTA, in shared memory on LOCAL indices:
//   s_c[0, n_ext)            colours of the distinct children below the tail (gathered once)
//   s_c[n_ext, n_ext + T)    colours of the tail's nodes, in index order
// ta/tb are the tail's children in local indices, gw_tail its weights; off[] the level offsets.
template <bool PAL>
__global__ void __launch_bounds__(kTailThreads, 1)
k_tail(const uint32_t* __restrict__ ta, const uint32_t* __restrict__ tb, const float* __restrict__ gw_tail,
       const uint32_t* __restrict__ ext, const float4* __restrict__ tf, float4* c,
       uint32_t* __restrict__ pal8, uint2* __restrict__ pal16, const uint32_t* __restrict__ off,
       uint32_t first_level, uint32_t n_levels, uint32_t n_leaves, uint32_t base, uint32_t T, uint32_t n_ext,
       int copy_leaves)
{
    extern __shared__ float4 s_c[];
    __shared__ uint32_t s_off[kTailMaxLevels + 1];
    uint32_t* s_a = reinterpret_cast<uint32_t*>(s_c + n_ext + T);
    uint32_t* s_b = s_a + T;
    float* s_w = reinterpret_cast<float*>(s_b + T);
    griddep_launch_dependents();
    const uint32_t tid = threadIdx.x;
    // static operands first (they do not depend on the previous kernel)
    for (uint32_t t = tid; t < T; t += kTailThreads) { s_a[t] = ta[t]; s_b[t] = tb[t]; s_w[t] = gw_tail[t]; }
    if (tid <= n_levels - first_level) s_off[tid] = off[first_level + tid] - base;
    uint32_t my_ext[4];                            // up to 4096 external children prefetched in registers
#pragma unroll
    for (int k = 0; k < 4; k++) { const uint32_t e = tid + k * kTailThreads; my_ext[k] = (e < n_ext) ? ext[e] : 0u; }
    griddep_wait();
    if (copy_leaves)
        for (uint32_t k = tid; k < n_leaves; k += kTailThreads) store_node<PAL>(c, pal8, pal16, k, ld_colour(tf + k));
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const uint32_t e = tid + k * kTailThreads;
        if (e < n_ext) s_c[e] = ld_colour((my_ext[k] < n_leaves) ? tf + my_ext[k] : c + my_ext[k]);
    }
    for (uint32_t e = tid + 4 * kTailThreads; e < n_ext; e += kTailThreads) {
        const uint32_t g = ext[e];
        s_c[e] = ld_colour((g < n_leaves) ? tf + g : c + g);
    }
    __syncthreads();
    for (uint32_t L = first_level; L < n_levels; L++) {
        const uint32_t lo = s_off[L - first_level], hi = s_off[L - first_level + 1];
        for (uint32_t t = lo + tid; t < hi; t += kTailThreads) {
            const float4 r = lerp4(s_c[s_a[t]], s_c[s_b[t]], s_w[t]);
            s_c[n_ext + t] = r;
            store_node<PAL>(c, pal8, pal16, base + t, r);
        }
        __syncthreads();   // the level barrier
    }
}

}  // namespace

using namespace mg;

// Launch with programmatic stream serialization (PDL): the kernel may become resident while its
// predecessor on the stream is still running; it orders itself with griddepcontrol.wait.
template <typename... KArgs, typename... Args>
static cudaError_t launch_pdl(bool pdl, void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t st,
                              Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;          // the first kernel of an update is a normal launch (full kernel boundary)
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

template <bool PAL>
static int propagate_impl(mg_graph* g, const float* tf_dev, float* node_rgba, cudaStream_t st)
{
    const float4* tf4 = reinterpret_cast<const float4*>(tf_dev);
    float4* c4 = reinterpret_cast<float4*>(node_rgba);
    const uint32_t n_levels = g->n_levels;
    const uint32_t fused = g->first_fused_level;                       // 0 = no tail
    const uint32_t last_big = (fused ? fused : n_levels) - 1;          // big levels are 1 .. last_big
    for (uint32_t L = 1; L <= last_big; L++) {
        const uint32_t lo = (uint32_t)g->level_off[L], hi = (uint32_t)g->level_off[L + 1];
        const uint32_t n_groups = ((hi + 3) >> 2) - (lo >> 2);
        if (L == 1) {
            // spare threads copy the leaves: make sure there are some, about one per 4 leaves
            uint32_t want = n_groups + (g->n_leaves + 3) / 4;
            uint32_t blocks = (want + kLevelThreads - 1) / kLevelThreads;
            if ((uint64_t)blocks * kLevelThreads == n_groups) blocks++;
            MG_CUDA(launch_pdl(false, k_level<true, PAL>, blocks, kLevelThreads, 0, st, g->d_a, g->d_b, g->d_w, tf4, c4, g->d_pal8,
                               g->d_pal16, lo, hi, g->n_leaves, n_groups));
        } else {
            uint32_t blocks = (n_groups + kLevelThreads - 1) / kLevelThreads;
            MG_CUDA(launch_pdl(true, k_level<false, PAL>, blocks, kLevelThreads, 0, st, g->d_a, g->d_b, g->d_w, (const float4*)c4, c4,
                               g->d_pal8, g->d_pal16, lo, hi, g->n_leaves, n_groups));
        }
        count_launch();
    }
    if (fused || last_big == 0) {
        // tail kernel; also the only kernel when every level is small (then it copies the leaves)
        const uint32_t first = fused ? fused : n_levels;               // n_levels: no internal level at all
        const int copy_leaves = (last_big == 0);
        const size_t smem = (size_t)(g->tail_n_ext + g->tail_n) * sizeof(float4) + (size_t)g->tail_n * 12;
        MG_CUDA(launch_pdl(last_big != 0, k_tail<PAL>, 1u, (unsigned)kTailThreads, smem, st, g->d_tail_a, g->d_tail_b,
                           g->d_w + g->tail_base, g->d_tail_ext, tf4, c4, g->d_pal8, g->d_pal16, g->d_level_off, first,
                           n_levels, g->n_leaves, g->tail_base, g->tail_n, g->tail_n_ext, copy_leaves));
        count_launch();
    }
    // the palettes now mirror node_rgba: what MG_PALETTE_FROM_LAST_PROPAGATE refers to (mg_colorize)
    g->pal_src = PAL ? node_rgba : nullptr;
    return MG_OK;
}

static int check_args(mg_graph* g, const float* tf, float* node_rgba, const char* who)
{
    if (!g || !tf || !node_rgba) { set_error("%s: NULL argument", who); return MG_ERR_INVALID_ARG; }
    if (((uintptr_t)node_rgba & 15) != 0) { set_error("%s: node_rgba must be 16-byte aligned", who); return MG_ERR_INVALID_ARG; }
    int rc = check_device(g, who);
    if (rc != MG_OK) return rc;
    // the tail kernel's dynamic shared memory limit: once per (function, device)
    static SmemAttrOnce once_pal, once_nopal;
    return g->no_palettes ? once_nopal.ensure((const void*)k_tail<false>, MG_TAIL_SMEM_BYTES, g->device)
                          : once_pal.ensure((const void*)k_tail<true>, MG_TAIL_SMEM_BYTES, g->device);
}

static int propagate_any(mg_graph* g, const float* tf_dev, float* node_rgba, cudaStream_t st)
{
    return g->no_palettes ? propagate_impl<false>(g, tf_dev, node_rgba, st) : propagate_impl<true>(g, tf_dev, node_rgba, st);
}

extern "C" int mg_propagate(mg_graph* g, const float* tf_rgba, float* node_rgba, void* stream)
{
    int rc = check_args(g, tf_rgba, node_rgba, "mg_propagate");
    if (rc != MG_OK) return rc;
    if (((uintptr_t)tf_rgba & 15) != 0) { set_error("mg_propagate: tf_rgba must be 16-byte aligned"); return MG_ERR_INVALID_ARG; }
    return propagate_any(g, tf_rgba, node_rgba, (cudaStream_t)stream);
}

extern "C" int mg_propagate_host(mg_graph* g, const float* tf_rgba_host, float* node_rgba, void* stream)
{
    int rc = check_args(g, tf_rgba_host, node_rgba, "mg_propagate_host");
    if (rc != MG_OK) return rc;
    MG_CUDA(cudaMemcpyAsync(g->d_tf_stage, tf_rgba_host, (size_t)g->n_leaves * 16, cudaMemcpyHostToDevice, (cudaStream_t)stream));
    return propagate_any(g, g->d_tf_stage, node_rgba, (cudaStream_t)stream);
}
