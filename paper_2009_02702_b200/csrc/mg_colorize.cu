// mg_colorize.cu -- colourise (a6): out[v] = convert(c[node_idx[v]]).
//
// "The mipmap itself is essentially a paletted texture" (L221): the conversion fp32 -> RGBA8 / fp16
// is done ONCE PER NODE (by the propagation kernels, or by k_convert_palette for a foreign
// node_rgba), so the per-voxel work is a pure 4-byte (8-byte) gather from a palette that fits L1/L2
// plus a coalesced 16-byte store.  HBM-bound: 4 B index read + 4 B (8 B) write per voxel.
//
// k_colorize: one thread = VPT voxels as VPT/4 16-byte index vectors, block-strided so that every
// load/store instruction of a warp covers 512 contiguous bytes.  Index loads and output stores use
// streaming cache operators (the 11.5 GB stream must not evict the palette from L2).
#include <cuda_fp16.h>

#include <algorithm>
#include <cstdlib>

#include "mg_internal.h"

namespace {

constexpr int kThreads = 256;
// 16-byte index vectors per thread, all loaded before the first gather.  Measured on B200, cfg 3, RGBA8:
// 1 -> 1.820 ms, 2 -> 1.748, 3 -> 1.669, 4 -> 1.676, 8 -> 1.689; fp16 output (two stores per vector): 2 -> 2.685, 4 -> 2.715.
template <bool W16> struct VecPerThread { static constexpr int value = W16 ? 2 : 4; };

__device__ __forceinline__ uint4 ld_cs_u4(const uint4* p)
{
    uint4 r;
    asm volatile("ld.global.cs.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_cs_u4(uint4* p, uint4 v)
{
    asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

__device__ __forceinline__ uint32_t cvt8(float4 c)
{
    uint32_t r = __float2uint_rn(__saturatef(c.x) * 255.0f);
    uint32_t g = __float2uint_rn(__saturatef(c.y) * 255.0f);
    uint32_t b = __float2uint_rn(__saturatef(c.z) * 255.0f);
    uint32_t a = __float2uint_rn(__saturatef(c.w) * 255.0f);
    return r | (g << 8) | (b << 16) | (a << 24);
}
__device__ __forceinline__ uint2 cvt16(float4 c)
{
    __half2 lo = __floats2half2_rn(c.x, c.y);
    __half2 hi = __floats2half2_rn(c.z, c.w);
    uint2 r;
    r.x = *reinterpret_cast<uint32_t*>(&lo);
    r.y = *reinterpret_cast<uint32_t*>(&hi);
    return r;
}

// Derive the palette(s) a colourise call gathers from out of node_rgba (the default of mg_colorize; skipped
// only under MG_PALETTE_FROM_LAST_PROPAGATE).  A normal launch: node_rgba may have been written by anything.
template <bool W8, bool W16>
__global__ void __launch_bounds__(256)
k_convert_palette(const float4* __restrict__ c, uint32_t n, uint32_t* __restrict__ pal8, uint2* __restrict__ pal16)
{
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float4 v = __ldg(c + i);
        if (W8) pal8[i] = cvt8(v);
        if (W16) pal16[i] = cvt16(v);
    }
}

// Vector body.  idx4/out point at the 16-byte aligned start; n_vec = number of 4-voxel vectors.
template <bool W8, bool W16>
__global__ void __launch_bounds__(kThreads)
k_colorize(const uint4* __restrict__ idx4, uint64_t n_vec, const uint32_t* __restrict__ pal8,
           const uint2* __restrict__ pal16, uint4* __restrict__ out8, uint4* __restrict__ out16)
{
    constexpr int kVec = VecPerThread<W16>::value;
    const uint64_t base = (uint64_t)blockIdx.x * (kThreads * kVec) + threadIdx.x;
    uint4 id[kVec];
#pragma unroll
    for (int k = 0; k < kVec; k++) {
        const uint64_t v = base + (uint64_t)k * kThreads;
        if (v < n_vec) id[k] = ld_cs_u4(idx4 + v);
    }
#pragma unroll
    for (int k = 0; k < kVec; k++) {
        const uint64_t v = base + (uint64_t)k * kThreads;
        if (v < n_vec) {
            if (W8) {
                uint4 o;
                o.x = __ldg(pal8 + id[k].x); o.y = __ldg(pal8 + id[k].y);
                o.z = __ldg(pal8 + id[k].z); o.w = __ldg(pal8 + id[k].w);
                st_cs_u4(out8 + v, o);
            }
            if (W16) {
                const uint2 h0 = __ldg(pal16 + id[k].x), h1 = __ldg(pal16 + id[k].y);
                const uint2 h2 = __ldg(pal16 + id[k].z), h3 = __ldg(pal16 + id[k].w);
                st_cs_u4(out16 + 2 * v, make_uint4(h0.x, h0.y, h1.x, h1.y));
                st_cs_u4(out16 + 2 * v + 1, make_uint4(h2.x, h2.y, h3.x, h3.y));
            }
        }
    }
}

// RGBA8 palette larger than the L2 can hold for random gathers.  Measured on B200 (profiles/r02_cfg5_ncu.txt): a
// randomly gathered table is served from L2 up to ~64 MB -- half the 126 MB: the two dies mirror read-shared lines --
// and from DRAM at ~90 B per 4-byte gather beyond that.  The palette is then cut into T tiles of <= kTileBytes and the
// volume is swept T times: sweep t gathers only the voxels whose node lies in tile t and merges them into the output
// vectors the earlier sweeps wrote.  Streams stay coalesced: 4 B index read per sweep, plus a 16-B read-modify-write
// of the vectors that hold a voxel of the tile (no read on the first sweep).  Each sweep costs about one streaming
// pass (0.25 ms per 134 M voxels), so few, larger tiles win although they are only partly L2-resident: config 5
// (256 MB) 1 sweep 2.06 ms, 2 -> 1.60, 3 -> 1.43, 4 -> 1.53, 8 -> 2.14.  L2 eviction-priority hints (evict_last on the
// gathers, evict_first on the streams) changed nothing.  The fp16 palette (8 B per node, twice the sweeps, 16-B output
// per voxel) never gained: it always takes the single sweep.
// The tile size is a property of the graph object (mg_graph::pal_tile_bytes = MG_DEFAULT_PAL_TILE_BYTES, 88 MB, unless
// MG_COLORIZE_TILE_BYTES was set in the environment when mg_load_graph ran): nothing is looked up per call.
constexpr uint32_t kMaxTiles = 4;                     // beyond that the T streaming sweeps cost more than the DRAM gathers

__device__ __forceinline__ uint4 ld_cg_u4(const uint4* p)
{
    uint4 r;
    asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

template <bool FIRST>
__global__ void __launch_bounds__(kThreads)
k_colorize_tile(const uint4* __restrict__ idx4, uint64_t n_vec, const uint32_t* __restrict__ pal8, uint32_t lo, uint32_t n_tile,
                uint4* out)                                           // out: read (by the later sweeps) and written
{
    constexpr int kVec = VecPerThread<false>::value;
    const uint64_t base = (uint64_t)blockIdx.x * (kThreads * kVec) + threadIdx.x;
    uint4 id[kVec];
#pragma unroll
    for (int k = 0; k < kVec; k++) {
        const uint64_t v = base + (uint64_t)k * kThreads;
        if (v < n_vec) id[k] = ld_cs_u4(idx4 + v);
    }
#pragma unroll
    for (int k = 0; k < kVec; k++) {
        const uint64_t v = base + (uint64_t)k * kThreads;
        if (v >= n_vec) continue;
        const bool in0 = id[k].x - lo < n_tile, in1 = id[k].y - lo < n_tile, in2 = id[k].z - lo < n_tile, in3 = id[k].w - lo < n_tile;
        if (!(in0 | in1 | in2 | in3)) continue;                       // other sweeps own all four voxels
        uint4 o = make_uint4(0, 0, 0, 0);
        if (!FIRST && !(in0 & in1 & in2 & in3)) o = ld_cg_u4(out + v);   // (.cg measured 5 % faster than .cs here)
        if (in0) o.x = __ldg(pal8 + id[k].x);
        if (in1) o.y = __ldg(pal8 + id[k].y);
        if (in2) o.z = __ldg(pal8 + id[k].z);
        if (in3) o.w = __ldg(pal8 + id[k].w);
        st_cs_u4(out + v, o);
    }
}

// Number of RGBA8 palette tiles: 1 = the palette fits (or is too large to gain), plain single-sweep kernel.
inline uint32_t palette_tiles(uint64_t tb, uint64_t n_nodes, uint64_t n_vec)
{
    const uint64_t t = (n_nodes * 4 + tb - 1) / tb;
    if (t < 2 || t > kMaxTiles) return 1;
    if (n_vec * 4 < n_nodes / 4) return 1;           // few voxels: they touch a small part of the palette once
    return (uint32_t)t;
}

// Scalar path: ragged head/tail around the vector body, or whole calls whose pointers are not
// mutually alignable.  Voxels [0, n).
template <bool W8, bool W16>
__global__ void __launch_bounds__(256)
k_colorize_scalar(const uint32_t* __restrict__ idx, uint64_t n, const uint32_t* __restrict__ pal8,
                  const uint2* __restrict__ pal16, uint32_t* __restrict__ out8, uint2* __restrict__ out16)
{
    for (uint64_t v = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t i = idx[v];
        if (W8) out8[v] = __ldg(pal8 + i);
        if (W16) out16[v] = __ldg(pal16 + i);
    }
}

template <bool W8, bool W16>
int launch_colorize(const mg_graph* g, const uint32_t* idx, uint64_t n, uint32_t* out8, uint2* out16, cudaStream_t st)
{
    // head: voxels until idx is 16-byte aligned; the outputs must become 16-byte aligned at the same voxel
    uint64_t head = ((16 - ((uintptr_t)idx & 15)) & 15) / 4;
    if (head > n) head = n;
    bool vec_ok = true;
    if (W8 && (((uintptr_t)(out8 + head)) & 15)) vec_ok = false;
    if (W16 && (((uintptr_t)(out16 + head)) & 15)) vec_ok = false;
    if (!vec_ok) {
        uint64_t blocks = (n + 255) / 256;
        if (blocks > 148ull * 32) blocks = 148ull * 32;
        k_colorize_scalar<W8, W16><<<(unsigned)blocks, 256, 0, st>>>(idx, n, g->d_pal8, g->d_pal16, out8, out16);
        mg::count_launch();
        return MG_OK;
    }
    const uint64_t n_vec = (n - head) / 4;
    const uint64_t tail0 = head + 4 * n_vec;
    if (n_vec) {
        constexpr int kVec = VecPerThread<W16>::value;
        const uint64_t blocks = (n_vec + (uint64_t)kThreads * kVec - 1) / ((uint64_t)kThreads * kVec);
        if (blocks > 0x7fffffffull) { mg::set_error("mg_colorize: too many voxels for one launch"); return MG_ERR_INVALID_ARG; }
        // NORMAL launches (no programmatic dependent launch): the palette gathers use the non-coherent
        // path (ld.global.nc, L1-cached), which is only safe behind a full kernel boundary -- measured: with
        // PDL a back-to-back update read stale palette lines (tests/test_gpu_parity.py::test_back_to_back...).
        const uint4* idx4 = reinterpret_cast<const uint4*>(idx + head);
        const uint32_t t8 = W8 ? palette_tiles(g->pal_tile_bytes, g->n_nodes, n_vec) : 1;
        if (t8 == 1) {
            k_colorize<W8, W16><<<(unsigned)blocks, kThreads, 0, st>>>(
                idx4, n_vec, g->d_pal8, g->d_pal16,
                reinterpret_cast<uint4*>(W8 ? out8 + head : nullptr), reinterpret_cast<uint4*>(W16 ? out16 + head : nullptr));
            mg::count_launch();
        } else {
            // RGBA8 tile by tile; the fp16 output of MG_BOTH takes its own single sweep
            uint4* o = reinterpret_cast<uint4*>(out8 + head);
            const uint64_t bl = (n_vec + (uint64_t)kThreads * VecPerThread<false>::value - 1) / ((uint64_t)kThreads * VecPerThread<false>::value);
            const uint32_t per = (uint32_t)((g->n_nodes + t8 - 1) / t8);
            for (uint32_t t = 0; t < t8; t++) {
                const uint32_t lo = t * per, nt = (uint32_t)std::min<uint64_t>(per, g->n_nodes - lo);
                if (t == 0) k_colorize_tile<true><<<(unsigned)bl, kThreads, 0, st>>>(idx4, n_vec, g->d_pal8, lo, nt, o);
                else k_colorize_tile<false><<<(unsigned)bl, kThreads, 0, st>>>(idx4, n_vec, g->d_pal8, lo, nt, o);
                mg::count_launch();
            }
            if (W16) {
                const uint64_t b16 = (n_vec + (uint64_t)kThreads * VecPerThread<true>::value - 1) / ((uint64_t)kThreads * VecPerThread<true>::value);
                k_colorize<false, true><<<(unsigned)b16, kThreads, 0, st>>>(idx4, n_vec, g->d_pal8, g->d_pal16, nullptr,
                                                                            reinterpret_cast<uint4*>(out16 + head));
                mg::count_launch();
            }
        }
    }
    if (head) {
        k_colorize_scalar<W8, W16><<<1, 32, 0, st>>>(idx, head, g->d_pal8, g->d_pal16, out8, out16);
        mg::count_launch();
    }
    if (tail0 < n) {
        k_colorize_scalar<W8, W16><<<1, 32, 0, st>>>(idx + tail0, n - tail0, g->d_pal8, g->d_pal16,
                                                      W8 ? out8 + tail0 : nullptr, W16 ? out16 + tail0 : nullptr);
        mg::count_launch();
    }
    return MG_OK;
}

}  // namespace

using namespace mg;

// The palette contract of mg_colorize / mg_colorize_packed (include/mg.h): by default the palettes of the
// requested format are derived from node_rgba here, on `st`, so the gather sees exactly the caller's buffer;
// with MG_PALETTE_FROM_LAST_PROPAGATE the caller states that node_rgba is what the last mg_propagate on this
// graph filled (and nothing wrote it since) and the palettes that call derived are gathered as they are.
int mg::prepare_palettes(mg_graph* g, const float* node_rgba, uint32_t format, cudaStream_t st, const char* who)
{
    const uint32_t fmt = format & 3u;
    if (format & MG_PALETTE_FROM_LAST_PROPAGATE) {
        if (format & MG_FORCE_CONVERT) { set_error("%s: MG_FORCE_CONVERT and MG_PALETTE_FROM_LAST_PROPAGATE exclude each other", who); return MG_ERR_INVALID_ARG; }
        if (g->no_palettes) { set_error("%s: MG_PALETTE_FROM_LAST_PROPAGATE on a graph loaded with MG_NO_PALETTES", who); return MG_ERR_INVALID_ARG; }
        if (!g->pal_src || g->pal_src != node_rgba) {
            set_error("%s: MG_PALETTE_FROM_LAST_PROPAGATE, but node_rgba is not the buffer the last mg_propagate on this graph "
                      "filled (or a library call wrote it / re-derived the palettes since)", who);
            return MG_ERR_INVALID_ARG;
        }
        return MG_OK;
    }
    const uint32_t n = (uint32_t)g->n_nodes;
    uint32_t blocks = (n + 255) / 256;
    if (blocks > 148u * 16) blocks = 148u * 16;
    const float4* c = reinterpret_cast<const float4*>(node_rgba);
    if (fmt == MG_RGBA8) k_convert_palette<true, false><<<blocks, 256, 0, st>>>(c, n, g->d_pal8, g->d_pal16);
    else if (fmt == MG_RGBA16F) k_convert_palette<false, true><<<blocks, 256, 0, st>>>(c, n, g->d_pal8, g->d_pal16);
    else k_convert_palette<true, true><<<blocks, 256, 0, st>>>(c, n, g->d_pal8, g->d_pal16);
    count_launch();
    g->pal_src = nullptr;          // the palettes now mirror a buffer the library knows nothing about
    return MG_OK;
}

extern "C" int mg_colorize(mg_graph* g, uint32_t mip_level, const uint32_t* node_idx_volume, uint64_t n_voxels,
                           const float* node_rgba, void* out_rgba, void* out_rgba_aux, uint32_t format, void* stream)
{
    (void)mip_level;
    if (!g || !node_rgba) { set_error("mg_colorize: NULL argument"); return MG_ERR_INVALID_ARG; }
    const uint32_t fmt = format & 3u;
    if (fmt == 0 || (format & ~(3u | MG_FORCE_CONVERT | MG_PALETTE_FROM_LAST_PROPAGATE))) { set_error("mg_colorize: bad format 0x%x", format); return MG_ERR_INVALID_ARG; }
    if (n_voxels && (!node_idx_volume || !out_rgba)) { set_error("mg_colorize: NULL buffer"); return MG_ERR_INVALID_ARG; }
    if (fmt == MG_BOTH && n_voxels && !out_rgba_aux) { set_error("mg_colorize: MG_BOTH needs out_rgba_aux"); return MG_ERR_INVALID_ARG; }
    if (((uintptr_t)node_idx_volume & 3) || ((uintptr_t)out_rgba & 3) || (fmt == MG_RGBA16F && ((uintptr_t)out_rgba & 7)) ||
        (fmt == MG_BOTH && ((uintptr_t)out_rgba_aux & 7)) || ((uintptr_t)node_rgba & 15)) {
        set_error("mg_colorize: misaligned buffer"); return MG_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    int rc = check_device(g, "mg_colorize");
    if (rc != MG_OK) return rc;
    rc = prepare_palettes(g, node_rgba, format, st, "mg_colorize");
    if (rc != MG_OK) return rc;
    if (n_voxels) {
        if (fmt == MG_RGBA8) rc = launch_colorize<true, false>(g, node_idx_volume, n_voxels, (uint32_t*)out_rgba, nullptr, st);
        else if (fmt == MG_RGBA16F) rc = launch_colorize<false, true>(g, node_idx_volume, n_voxels, nullptr, (uint2*)out_rgba, st);
        else rc = launch_colorize<true, true>(g, node_idx_volume, n_voxels, (uint32_t*)out_rgba, (uint2*)out_rgba_aux, st);
    }
    if (rc != MG_OK) return rc;
    MG_CUDA(cudaGetLastError());
    return MG_OK;
}

extern "C" int mg_tf_update_host(mg_graph* g, const float* tf_rgba_host, float* node_rgba, const uint32_t* node_idx_volume,
                                 uint64_t n_voxels, void* out_device, void* out_host, uint32_t format, void* stream)
{
    if ((format & 3u) == MG_BOTH || (format & ~3u)) { set_error("mg_tf_update_host: format must be MG_RGBA8 or MG_RGBA16F"); return MG_ERR_INVALID_ARG; }
    int rc = mg_propagate_host(g, tf_rgba_host, node_rgba, stream);
    if (rc != MG_OK) return rc;
    // this call has just enqueued the propagation that filled node_rgba on this very stream
    const uint32_t reuse = g->no_palettes ? 0u : (uint32_t)MG_PALETTE_FROM_LAST_PROPAGATE;
    rc = mg_colorize(g, 0xFFFFFFFFu, node_idx_volume, n_voxels, node_rgba, out_device, nullptr, (format & 3u) | reuse, stream);
    if (rc != MG_OK) return rc;
    if (out_host && n_voxels) {
        const size_t bytes = (size_t)n_voxels * (((format & 3u) == MG_RGBA8) ? 4 : 8);
        MG_CUDA(cudaMemcpyAsync(out_host, out_device, bytes, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    }
    return MG_OK;
}
