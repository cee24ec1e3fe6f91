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
//                    levels instead of kernel boundaries; the colours it produces are kept in
//                    shared memory (as far as they fit) so later levels gather on-chip.
#include <cuda_fp16.h>

#include "mg_internal.h"

namespace {

constexpr int kLevelThreads = 256;
constexpr int kTailThreads = 1024;

__device__ __forceinline__ uint4 ld_stream_u4(const void* p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

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

__device__ __forceinline__ void store_node(float4* c, uint32_t* __restrict__ pal8,
                                           uint2* __restrict__ pal16, uint32_t n, float4 v)
{
    c[n] = v;
    pal8[n] = to_rgba8(v);
    pal16[n] = to_rgba16f(v);
}

// One level [lo, hi).  Work is cut into groups of 4 nodes aligned to absolute index 4g, so the
// 16-byte loads of a/b/w are aligned whatever lo is; edge groups fall back to scalar accesses.
template <bool FIRST>
__global__ void __launch_bounds__(kLevelThreads)
k_level(const uint32_t* __restrict__ ga, const uint32_t* __restrict__ gb, const float* __restrict__ gw,
        const float4* __restrict__ src,   // FIRST: the TF; else: node colours of the lower levels
        float4* c, uint32_t* __restrict__ pal8, uint2* __restrict__ pal16,
        uint32_t lo, uint32_t hi, uint32_t n_leaves, uint32_t n_groups)
{
    const uint32_t t = blockIdx.x * kLevelThreads + threadIdx.x;
    if (t < n_groups) {
        const uint32_t n0 = (lo & ~3u) + 4u * t;
        if (n0 >= lo && n0 + 4u <= hi) {
            const uint4 a = ld_stream_u4(ga + n0);
            const uint4 b = ld_stream_u4(gb + n0);
            const uint4 wu = ld_stream_u4(gw + n0);
            const float4 ca0 = __ldg(src + a.x), cb0 = __ldg(src + b.x);
            const float4 ca1 = __ldg(src + a.y), cb1 = __ldg(src + b.y);
            const float4 ca2 = __ldg(src + a.z), cb2 = __ldg(src + b.z);
            const float4 ca3 = __ldg(src + a.w), cb3 = __ldg(src + b.w);
            const float4 r0 = lerp4(ca0, cb0, __uint_as_float(wu.x));
            const float4 r1 = lerp4(ca1, cb1, __uint_as_float(wu.y));
            const float4 r2 = lerp4(ca2, cb2, __uint_as_float(wu.z));
            const float4 r3 = lerp4(ca3, cb3, __uint_as_float(wu.w));
            c[n0] = r0; c[n0 + 1] = r1; c[n0 + 2] = r2; c[n0 + 3] = r3;
            *reinterpret_cast<uint4*>(pal8 + n0) = make_uint4(to_rgba8(r0), to_rgba8(r1), to_rgba8(r2), to_rgba8(r3));
            const uint2 h0 = to_rgba16f(r0), h1 = to_rgba16f(r1), h2 = to_rgba16f(r2), h3 = to_rgba16f(r3);
            *reinterpret_cast<uint4*>(pal16 + n0) = make_uint4(h0.x, h0.y, h1.x, h1.y);
            *reinterpret_cast<uint4*>(pal16 + n0 + 2) = make_uint4(h2.x, h2.y, h3.x, h3.y);
        } else {
#pragma unroll
            for (uint32_t k = 0; k < 4; k++) {
                const uint32_t n = n0 + k;
                if (n >= lo && n < hi)
                    store_node(c, pal8, pal16, n, lerp4(__ldg(src + ga[n]), __ldg(src + gb[n]), gw[n]));
            }
        }
    }
    if (FIRST) {
        // leaf assignment c[k] = TF[k], bit-exact (L371), by the threads past the node groups
        const uint32_t total = gridDim.x * kLevelThreads;
        const uint32_t spare0 = n_groups;
        const uint32_t n_spare = total - spare0;
        if (t >= spare0)
            for (uint32_t k = t - spare0; k < n_leaves; k += n_spare) store_node(c, pal8, pal16, k, __ldg(src + k));
    }
}

// All levels L in [first_level, n_levels) in one CTA.  off[] are the level offsets.  Nodes
// [smem_base, smem_base + smem_nodes) are mirrored in shared memory.
__global__ void __launch_bounds__(kTailThreads, 1)
k_tail(const uint32_t* __restrict__ ga, const uint32_t* __restrict__ gb, const float* __restrict__ gw,
       const float4* __restrict__ tf, float4* c, uint32_t* __restrict__ pal8, uint2* __restrict__ pal16,
       const uint32_t* __restrict__ off, uint32_t first_level, uint32_t n_levels, uint32_t n_leaves,
       uint32_t smem_base, uint32_t smem_nodes, int copy_leaves)
{
    extern __shared__ float4 s_c[];
    const uint32_t tid = threadIdx.x;
    if (copy_leaves) {
        for (uint32_t k = tid; k < n_leaves; k += kTailThreads) {
            const float4 v = __ldg(tf + k);
            store_node(c, pal8, pal16, k, v);
            if (k - smem_base < smem_nodes) s_c[k - smem_base] = v;   // unsigned wrap: k >= smem_base
        }
        __syncthreads();
    }
    for (uint32_t L = first_level; L < n_levels; L++) {
        const uint32_t lo = off[L], hi = off[L + 1];
        for (uint32_t n = lo + tid; n < hi; n += kTailThreads) {
            const uint32_t a = ga[n], b = gb[n];
            const float w = gw[n];
            const uint32_t sa = a - smem_base, sb = b - smem_base;
            const float4 ca = (sa < smem_nodes) ? s_c[sa] : c[a];
            const float4 cb = (sb < smem_nodes) ? s_c[sb] : c[b];
            const float4 r = lerp4(ca, cb, w);
            store_node(c, pal8, pal16, n, r);
            if (n - smem_base < smem_nodes) s_c[n - smem_base] = r;
        }
        __syncthreads();   // the level barrier: every store above is visible to the CTA after it
    }
}

}  // namespace

using namespace mg;

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
            k_level<true><<<blocks, kLevelThreads, 0, st>>>(g->d_a, g->d_b, g->d_w, tf4, c4, g->d_pal8, g->d_pal16,
                                                            lo, hi, g->n_leaves, n_groups);
        } else {
            uint32_t blocks = (n_groups + kLevelThreads - 1) / kLevelThreads;
            k_level<false><<<blocks, kLevelThreads, 0, st>>>(g->d_a, g->d_b, g->d_w, c4, c4, g->d_pal8, g->d_pal16,
                                                             lo, hi, g->n_leaves, n_groups);
        }
        count_launch();
    }
    if (fused || last_big == 0) {
        // tail kernel; also the only kernel when every level is small (then it copies the leaves)
        const uint32_t first = fused ? fused : n_levels;               // n_levels: no internal level at all
        const int copy_leaves = (last_big == 0);
        const uint32_t smem_base = copy_leaves ? 0u : (uint32_t)g->level_off[first];
        uint32_t smem_nodes = g->tail_smem_nodes;
        if (copy_leaves) {
            uint64_t all = g->n_nodes;
            smem_nodes = (uint32_t)(all < 12288 ? all : 12288);
        }
        const size_t smem = (size_t)smem_nodes * sizeof(float4);
        k_tail<<<1, kTailThreads, smem, st>>>(g->d_a, g->d_b, g->d_w, tf4, c4, g->d_pal8, g->d_pal16,
                                              g->d_level_off, first, n_levels, g->n_leaves, smem_base, smem_nodes,
                                              copy_leaves);
        count_launch();
    }
    MG_CUDA(cudaGetLastError());
    g->pal_src = node_rgba;
    return MG_OK;
}

static int check_args(mg_graph* g, const float* tf, float* node_rgba, const char* who)
{
    if (!g || !tf || !node_rgba) { set_error("%s: NULL argument", who); return MG_ERR_INVALID_ARG; }
    if (((uintptr_t)node_rgba & 15) != 0) { set_error("%s: node_rgba must be 16-byte aligned", who); return MG_ERR_INVALID_ARG; }
    return MG_OK;
}

static int ensure_tail_smem()
{
    static bool done = false;   // per process; the attribute is per function (all devices share the setting call)
    if (!done) {
        MG_CUDA(cudaFuncSetAttribute(k_tail, cudaFuncAttributeMaxDynamicSharedMemorySize, 12288 * (int)sizeof(float4)));
        done = true;
    }
    return MG_OK;
}

extern "C" int mg_propagate(mg_graph* g, const float* tf_rgba, float* node_rgba, void* stream)
{
    int rc = check_args(g, tf_rgba, node_rgba, "mg_propagate");
    if (rc != MG_OK) return rc;
    if (((uintptr_t)tf_rgba & 15) != 0) { set_error("mg_propagate: tf_rgba must be 16-byte aligned"); return MG_ERR_INVALID_ARG; }
    rc = ensure_tail_smem();
    if (rc != MG_OK) return rc;
    return propagate_impl(g, tf_rgba, node_rgba, (cudaStream_t)stream);
}

extern "C" int mg_propagate_host(mg_graph* g, const float* tf_rgba_host, float* node_rgba, void* stream)
{
    int rc = check_args(g, tf_rgba_host, node_rgba, "mg_propagate_host");
    if (rc != MG_OK) return rc;
    rc = ensure_tail_smem();
    if (rc != MG_OK) return rc;
    MG_CUDA(cudaMemcpyAsync(g->d_tf_stage, tf_rgba_host, (size_t)g->n_leaves * 16, cudaMemcpyHostToDevice, (cudaStream_t)stream));
    return propagate_impl(g, g->d_tf_stage, node_rgba, (cudaStream_t)stream);
}
