// mg_packed.cu -- NEXT-3: bit-packed node-ID volumes as colourise input.
//
// The paper stores, per mip level l, i_min(l) and for every voxel (node ID - i_min(l)) at a fixed
// bitrate r(l) = ceil(log2(i_max(l) - i_min(l) + 1)) (Table 1 rows (8), (9), (A); Eq. 15-16,
// L199-L207) and addresses the stream by bit address in the shader (L267).  Reading Q18:
// voxel v occupies bits [v r, (v+1) r) of its level's stream, LSB first, little endian.
// This cuts the colourise input from 32 bits per voxel to r(l) (11 bits on level 0 of config 3).
//
//   k_index_range      min / max of a node-index volume (i_min, i_max of Eq. 15)
//   k_pack_bits<R>     one thread = 32 voxels = R words of the stream, staged through shared memory (no atomics)
//   k_colorize_packed  one CTA = one tile of 4096 voxels of ONE level (uniform switch on the level's
//                      bitrate into a compile-time-R body, see colorize_tile).  All levels of a mipmap
//                      go in ONE launch: the per-level table travels as a __grid_constant__ parameter.
#include <cuda_fp16.h>

#include <cstring>

#include "mg_internal.h"

namespace {

constexpr int kThreads = 256;
constexpr int kTileVox = 4096;                 // voxels per CTA: 4 groups of 4 per thread, their words all loaded before the
                                               // first gather (measured, cfg 3: 2048 -> 1.291 ms, 3072 -> 1.247, 4096 -> 1.248, 8192 -> 1.245)
constexpr int kMaxLevels = MG_MAX_PACKED_LEVELS;

struct PackedLevel {
    const uint32_t* words;   // level stream (16-byte aligned)
    uint64_t n_vox;
    uint64_t out_off;        // first voxel of the level in the outputs (multiple of 4)
    uint32_t bits;
    uint32_t i_min;
    uint32_t tile_begin;     // first CTA of the level
    uint32_t pad;
};
struct PackedParams {
    PackedLevel lv[kMaxLevels];
    uint32_t n_levels;
};

__device__ __forceinline__ void st_cs_u4(uint4* p, uint4 v)
{
    asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// 16-byte streaming loads, two per thread in flight; one atomic pair per warp at the end (grid-stride: few warps).
__global__ void __launch_bounds__(256) k_index_range(const uint32_t* __restrict__ idx, uint64_t n, uint32_t* __restrict__ mm)
{
    const mg::Span sp = mg::span_of(idx, n);
    const uint4* v4 = reinterpret_cast<const uint4*>(idx + sp.head);
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint32_t lo = 0xFFFFFFFFu, hi = 0u;
    auto take = [&](const uint4 a) {
        lo = min(lo, min(min(a.x, a.y), min(a.z, a.w)));
        hi = max(hi, max(max(a.x, a.y), max(a.z, a.w)));
    };
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + stride < sp.nv; i += 2 * stride) {
        const uint4 a = __ldcs(v4 + i), b = __ldcs(v4 + i + stride);
        take(a);
        take(b);
    }
    if (i < sp.nv) take(__ldcs(v4 + i));
    if (blockIdx.x == 0 && threadIdx.x < sp.head + (n - sp.tail)) {
        const uint32_t v = idx[mg::ragged(sp, threadIdx.x)];
        lo = min(lo, v); hi = max(hi, v);
    }
    lo = __reduce_min_sync(0xFFFFFFFFu, lo);
    hi = __reduce_max_sync(0xFFFFFFFFu, hi);
    if ((threadIdx.x & 31) == 0 && lo <= hi) { atomicMin(mm, lo); atomicMax(mm + 1, hi); }
}

// The encoder, at the compile-time bitrate R: 32 consecutive voxels fill exactly R words, so a thread that owns 32
// voxels packs them with shifts known at compile time and touches nobody else's words (no atomics, no division).
// A CTA takes kPackTile = 256 x 32 voxels: coalesced 16-byte loads into shared memory (row stride 33 words: the 32
// threads of a warp then read 32 different banks), R words per thread packed in registers, written back to shared
// memory and stored with coalesced 4-byte stores -- the kernel is a stream (round 1's one-thread-per-word encoder ran
// a variable-length loop per word and was issue-bound: 78 % issue slots at 43 % DRAM throughput, 1.59 ms on level 0 of
// config 3 against 1.04 ms at the copy peak).  Words past the data (the stream's zero padding) are written as zeros.
constexpr int kPackThreads = 256;
constexpr int kPackTile = kPackThreads * 32;

template <int R>
__device__ __forceinline__ void pack_tile(const uint32_t* __restrict__ idx, uint64_t n, uint32_t i_min, uint32_t* __restrict__ words,
                                          uint64_t n_words, uint32_t* smem)
{
    constexpr uint32_t vmask = R >= 32 ? 0xFFFFFFFFu : ((1u << R) - 1u);  // a value outside [i_min, i_min + 2^R) must not spill
    const uint64_t v0 = (uint64_t)blockIdx.x * kPackTile;                 // first voxel of the tile
    const uint32_t t = threadIdx.x;
    // ---- load: voxel v0 + e lands at smem[e + e / 32]
    const uint64_t left = v0 < n ? n - v0 : 0;
    const uint32_t nv = (uint32_t)(left < (uint64_t)kPackTile ? left : (uint64_t)kPackTile);
    if ((((uintptr_t)(idx + v0)) & 15) == 0) {
        const uint4* src = reinterpret_cast<const uint4*>(idx + v0);
#pragma unroll
        for (int k = 0; k < 8; k++) {
            const uint32_t e = 4u * (t + k * kPackThreads);
            uint4 x = make_uint4(i_min, i_min, i_min, i_min);
            if (e + 4 <= nv) x = __ldcs(src + (e >> 2));
            else if (e < nv) { x.x = idx[v0 + e]; if (e + 1 < nv) x.y = idx[v0 + e + 1]; if (e + 2 < nv) x.z = idx[v0 + e + 2]; }
            uint32_t* d = smem + e + (e >> 5);                            // 4 consecutive elements never cross a row of 32
            d[0] = x.x; d[1] = x.y; d[2] = x.z; d[3] = x.w;
        }
    } else {
#pragma unroll 8
        for (int k = 0; k < 32; k++) {
            const uint32_t e = t + k * kPackThreads;
            smem[e + (e >> 5)] = e < nv ? __ldcs(idx + v0 + e) : i_min;
        }
    }
    __syncthreads();
    // ---- pack the thread's 32 voxels (row t) into R words
    uint32_t out[R > 0 ? R : 1];
#pragma unroll
    for (int q = 0; q < (R > 0 ? R : 1); q++) out[q] = 0u;
#pragma unroll
    for (int i = 0; i < 32; i++) {
        const uint32_t val = (smem[t * 33 + i] - i_min) & vmask;
        constexpr int dummy = 0; (void)dummy;
        const int bit = i * R, wq = bit >> 5, sh = bit & 31;              // compile-time after unrolling
        out[wq] |= val << sh;
        if (sh + R > 32) out[wq + 1] |= val >> (32 - sh);
    }
    __syncthreads();
    constexpr bool kSkew = (R % 2) == 0;                                   // word i of the tile at smem[i] for odd R (stride R: 32 banks),
#pragma unroll
    for (int q = 0; q < R; q++) {                                          // at smem[i + i / 32] for even R (the skew restores 32 banks)
        const uint32_t wi = t * R + q;
        smem[kSkew ? wi + (wi >> 5) : wi] = out[q];
    }
    __syncthreads();
    // ---- store: the tile's kPackThreads * R words are contiguous in the stream
    const uint64_t w0 = (uint64_t)blockIdx.x * (kPackThreads * R);
#pragma unroll 4
    for (int q = 0; q < R; q++) {
        const uint32_t wl = t + q * kPackThreads;
        if (w0 + wl < n_words) words[w0 + wl] = smem[kSkew ? wl + (wl >> 5) : wl];
    }
}

template <int R>
__global__ void __launch_bounds__(kPackThreads)
k_pack_bits(const uint32_t* __restrict__ idx, uint64_t n, uint32_t i_min, uint32_t* __restrict__ words, uint64_t n_words)
{
    __shared__ uint32_t smem[kPackThreads * 33];
    pack_tile<R>(idx, n, i_min, words, n_words, smem);
}

// One tile (kTileVox voxels of one level) at the compile-time bitrate R.  A lane handles groups of 4
// consecutive voxels (4 R bits, one 16-byte RGBA8 store): it loads the NW aligned 32-bit words that
// cover the group (neighbouring lanes overlap: the same sectors, served by L1), realigns them by the
// group's bit offset (a runtime funnel shift) and extracts the four values at COMPILE-TIME positions
// j R -- no shared memory, no barrier, word selection never depends on runtime data.
template <int R, bool W8, bool W16>
__device__ __forceinline__ void colorize_tile(const uint32_t* __restrict__ words, uint32_t i_min, uint32_t id_max, uint32_t nv, uint64_t o0,
                                              const uint32_t* __restrict__ pal8, const uint2* __restrict__ pal16,
                                              uint32_t* __restrict__ out8, uint2* __restrict__ out16)
{
    constexpr int NW = (R == 0) ? 0 : (4 * R + 62) / 32;               // words that can hold 4 R bits at any bit offset
    constexpr int NG = kTileVox / (4 * kThreads);                       // groups per thread
    constexpr uint32_t mask = R >= 32 ? 0xFFFFFFFFu : ((1u << R) - 1u);
    uint32_t a[NG][NW + 1];
#pragma unroll
    for (int k = 0; k < NG; k++) {
        const uint32_t vb = (threadIdx.x + k * kThreads) * 4;
        const uint32_t i0 = (vb * R) >> 5;
#pragma unroll
        for (int q = 0; q < NW; q++) a[k][q] = (vb < nv) ? __ldg(words + i0 + q) : 0u;
        a[k][NW] = 0u;
    }
#pragma unroll
    for (int k = 0; k < NG; k++) {
        const uint32_t vb = (threadIdx.x + k * kThreads) * 4;
        if (vb >= nv) continue;
        const uint32_t sh = (vb * R) & 31;
        uint32_t w[NW + 1];                                             // the group's bits, realigned to bit 0
#pragma unroll
        for (int q = 0; q < NW; q++) w[q] = __funnelshift_r(a[k][q], a[k][q + 1], sh);
        w[NW] = 0u;
        uint32_t id[4];
#pragma unroll
        for (int j = 0; j < 4; j++) {
            constexpr int dummy = 0; (void)dummy;
            const int p = j * R;                                        // compile-time after unrolling
            uint32_t v = 0;
            if (R > 0) v = (p & 31) ? __funnelshift_r(w[p >> 5], w[(p >> 5) + 1 <= NW ? (p >> 5) + 1 : NW], p & 31) : w[p >> 5];
            id[j] = min(i_min + (v & mask), id_max);                   // a stale (i_min, r) pair must not gather out of bounds
        }
        const uint64_t o = o0 + vb;
        if (vb + 4 <= nv) {
            if (W8) st_cs_u4(reinterpret_cast<uint4*>(out8 + o),
                             make_uint4(__ldg(pal8 + id[0]), __ldg(pal8 + id[1]), __ldg(pal8 + id[2]), __ldg(pal8 + id[3])));
            if (W16) {
                const uint2 h0 = __ldg(pal16 + id[0]), h1 = __ldg(pal16 + id[1]), h2 = __ldg(pal16 + id[2]), h3 = __ldg(pal16 + id[3]);
                st_cs_u4(reinterpret_cast<uint4*>(out16 + o), make_uint4(h0.x, h0.y, h1.x, h1.y));
                st_cs_u4(reinterpret_cast<uint4*>(out16 + o) + 1, make_uint4(h2.x, h2.y, h3.x, h3.y));
            }
        } else {
#pragma unroll
            for (int j = 0; j < 4; j++)
                if (vb + j < nv) {
                    if (W8) out8[o + j] = __ldg(pal8 + id[j]);
                    if (W16) out16[o + j] = __ldg(pal16 + id[j]);
                }
        }
    }
}

template <bool W8, bool W16>
__global__ void __launch_bounds__(kThreads)
k_colorize_packed(const __grid_constant__ PackedParams P, const uint32_t* __restrict__ pal8, const uint2* __restrict__ pal16,
                  uint32_t id_max, uint32_t* __restrict__ out8, uint2* __restrict__ out16)
{
    uint32_t l = 0;
    while (l + 1 < P.n_levels && blockIdx.x >= P.lv[l + 1].tile_begin) l++;
    const PackedLevel& L = P.lv[l];
    const uint64_t tile = blockIdx.x - L.tile_begin;
    const uint64_t v0 = tile * kTileVox;
    const uint32_t nv = (uint32_t)min((uint64_t)kTileVox, L.n_vox - v0);
    const uint32_t* words = L.words + tile * (uint64_t)(kTileVox / 32) * L.bits;   // a tile starts on a word boundary
    const uint64_t o0 = L.out_off + v0;
#define MG_CASE(R) case R: colorize_tile<R, W8, W16>(words, L.i_min, id_max, nv, o0, pal8, pal16, out8, out16); break;
    switch (L.bits) {                                                    // uniform per CTA
        MG_CASE(0) MG_CASE(1) MG_CASE(2) MG_CASE(3) MG_CASE(4) MG_CASE(5) MG_CASE(6) MG_CASE(7) MG_CASE(8)
        MG_CASE(9) MG_CASE(10) MG_CASE(11) MG_CASE(12) MG_CASE(13) MG_CASE(14) MG_CASE(15) MG_CASE(16)
        MG_CASE(17) MG_CASE(18) MG_CASE(19) MG_CASE(20) MG_CASE(21) MG_CASE(22) MG_CASE(23) MG_CASE(24)
        MG_CASE(25) MG_CASE(26) MG_CASE(27) MG_CASE(28) MG_CASE(29) MG_CASE(30) MG_CASE(31) MG_CASE(32)
        default: break;
    }
#undef MG_CASE
}

}  // namespace

using namespace mg;

extern "C" uint64_t mg_packed_stream_bytes(uint64_t n_voxels, uint32_t bits)
{
    const uint64_t payload = (n_voxels * (uint64_t)bits + 7) / 8;
    return ((payload + 15) & ~(uint64_t)15) + 16;
}

extern "C" uint32_t mg_bits_per_voxel(uint32_t i_min, uint32_t i_max)
{
    if (i_max < i_min) return 0;
    const uint64_t range = (uint64_t)i_max - i_min + 1;
    uint32_t r = 0;
    while ((1ull << r) < range) r++;
    return r;
}

extern "C" int mg_index_range(const uint32_t* idx_device, uint64_t n, uint32_t* i_min, uint32_t* i_max, void* stream)
{
    if (!idx_device || !i_min || !i_max || n == 0) { set_error("mg_index_range: NULL argument or n = 0"); return MG_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    uint32_t* d_mm = nullptr;
    MG_CUDA(cudaMalloc((void**)&d_mm, 8));
    const uint32_t init[2] = {0xFFFFFFFFu, 0u};
    cudaError_t e = cudaMemcpyAsync(d_mm, init, 8, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) {
        uint64_t blocks = (n / 4 + 256) / 256;
        if (blocks > 148ull * 8) blocks = 148ull * 8;
        k_index_range<<<(unsigned)blocks, 256, 0, st>>>(idx_device, n, d_mm);
        count_launch();
        uint32_t out[2] = {0, 0};
        e = cudaMemcpyAsync(out, d_mm, 8, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        *i_min = out[0]; *i_max = out[1];
    }
    cudaFree(d_mm);
    if (e != cudaSuccess) return cuda_fail(e, "mg_index_range");
    return MG_OK;
}

extern "C" int mg_pack_indices(const uint32_t* idx_device, uint64_t n, uint32_t i_min, uint32_t bits, void* packed_device, void* stream)
{
    if ((!idx_device && n) || !packed_device) { set_error("mg_pack_indices: NULL argument"); return MG_ERR_INVALID_ARG; }
    if (bits > 32) { set_error("mg_pack_indices: bits must be <= 32"); return MG_ERR_INVALID_ARG; }
    if ((uintptr_t)packed_device & 15) { set_error("mg_pack_indices: the stream must be 16-byte aligned"); return MG_ERR_INVALID_ARG; }
    const uint64_t n_words = mg_packed_stream_bytes(n, bits) / 4;
    cudaStream_t st = (cudaStream_t)stream;
    if (bits == 0) {                                                      // every voxel is node i_min: the stream is its padding
        MG_CUDA(cudaMemsetAsync(packed_device, 0, n_words * 4, st));
        return MG_OK;
    }
    // tiles of 8192 voxels = 256 R words; enough of them to cover the padding words behind the data too
    const uint64_t blocks = (n_words + (uint64_t)kPackThreads * bits - 1) / ((uint64_t)kPackThreads * bits);
    if (blocks > 0x7fffffffull) { set_error("mg_pack_indices: too many voxels for one launch"); return MG_ERR_INVALID_ARG; }
    uint32_t* words = (uint32_t*)packed_device;
#define MG_CASE(R) case R: k_pack_bits<R><<<(unsigned)blocks, kPackThreads, 0, st>>>(idx_device, n, i_min, words, n_words); break;
    switch (bits) {
        MG_CASE(1) MG_CASE(2) MG_CASE(3) MG_CASE(4) MG_CASE(5) MG_CASE(6) MG_CASE(7) MG_CASE(8)
        MG_CASE(9) MG_CASE(10) MG_CASE(11) MG_CASE(12) MG_CASE(13) MG_CASE(14) MG_CASE(15) MG_CASE(16)
        MG_CASE(17) MG_CASE(18) MG_CASE(19) MG_CASE(20) MG_CASE(21) MG_CASE(22) MG_CASE(23) MG_CASE(24)
        MG_CASE(25) MG_CASE(26) MG_CASE(27) MG_CASE(28) MG_CASE(29) MG_CASE(30) MG_CASE(31) MG_CASE(32)
        default: break;
    }
#undef MG_CASE
    count_launch();
    MG_CUDA(cudaGetLastError());
    return MG_OK;
}

extern "C" int mg_colorize_packed(mg_graph* g, const void* packed_device, const mg_packed_level* levels, uint32_t n_levels,
                                  const float* node_rgba, void* out_rgba, void* out_rgba_aux, uint32_t format, void* stream)
{
    if (!g || !node_rgba || !levels || !packed_device || !out_rgba) { set_error("mg_colorize_packed: NULL argument"); return MG_ERR_INVALID_ARG; }
    const uint32_t fmt = format & 3u;
    if (fmt == 0 || (format & ~(3u | MG_FORCE_CONVERT | MG_PALETTE_FROM_LAST_PROPAGATE))) { set_error("mg_colorize_packed: bad format 0x%x", format); return MG_ERR_INVALID_ARG; }
    if (fmt == MG_BOTH && !out_rgba_aux) { set_error("mg_colorize_packed: MG_BOTH needs out_rgba_aux"); return MG_ERR_INVALID_ARG; }
    if (n_levels == 0 || n_levels > (uint32_t)kMaxLevels) { set_error("mg_colorize_packed: n_levels must be 1..%d", kMaxLevels); return MG_ERR_INVALID_ARG; }
    if (((uintptr_t)packed_device & 15) || ((uintptr_t)out_rgba & 15) || (fmt == MG_BOTH && ((uintptr_t)out_rgba_aux & 15)) || ((uintptr_t)node_rgba & 15)) {
        set_error("mg_colorize_packed: buffers must be 16-byte aligned"); return MG_ERR_INVALID_ARG;
    }
    int rc = check_device(g, "mg_colorize_packed");
    if (rc != MG_OK) return rc;
    PackedParams P;
    memset(&P, 0, sizeof(P));
    uint64_t tiles = 0;
    uint32_t m = 0;
    for (uint32_t l = 0; l < n_levels; l++) {
        const mg_packed_level& s = levels[l];
        if (s.bits > 32 || (s.out_offset & 3) || (s.byte_offset & 15)) {
            set_error("mg_colorize_packed: level %u: bits <= 32, out_offset %% 4 == 0 and byte_offset %% 16 == 0 are required", l);
            return MG_ERR_INVALID_ARG;
        }
        if (s.n_voxels == 0) continue;
        if (s.i_min >= g->n_nodes) { set_error("mg_colorize_packed: level %u: i_min = %u is not a node of this graph", l, s.i_min); return MG_ERR_INVALID_ARG; }
        PackedLevel& d = P.lv[m++];
        d.words = reinterpret_cast<const uint32_t*>(static_cast<const char*>(packed_device) + s.byte_offset);
        d.n_vox = s.n_voxels; d.out_off = s.out_offset; d.bits = s.bits; d.i_min = s.i_min;
        d.tile_begin = (uint32_t)tiles;
        tiles += (s.n_voxels + kTileVox - 1) / kTileVox;
        if (tiles > 0x7fffffffull) { set_error("mg_colorize_packed: too many voxels for one launch"); return MG_ERR_INVALID_ARG; }
    }
    P.n_levels = m;
    cudaStream_t st = (cudaStream_t)stream;
    rc = prepare_palettes(g, node_rgba, format, st, "mg_colorize_packed");
    if (rc != MG_OK) return rc;
    if (m == 0) return MG_OK;
    const uint32_t id_max = (uint32_t)g->n_nodes - 1;
    // normal launches: the palette gathers use the non-coherent path (see mg_colorize.cu)
    if (fmt == MG_RGBA8) k_colorize_packed<true, false><<<(unsigned)tiles, kThreads, 0, st>>>(P, g->d_pal8, g->d_pal16, id_max, (uint32_t*)out_rgba, nullptr);
    else if (fmt == MG_RGBA16F) k_colorize_packed<false, true><<<(unsigned)tiles, kThreads, 0, st>>>(P, g->d_pal8, g->d_pal16, id_max, nullptr, (uint2*)out_rgba);
    else k_colorize_packed<true, true><<<(unsigned)tiles, kThreads, 0, st>>>(P, g->d_pal8, g->d_pal16, id_max, (uint32_t*)out_rgba, (uint2*)out_rgba_aux);
    count_launch();
    MG_CUDA(cudaGetLastError());
    return MG_OK;
}

// ------------------------------------------------------------------------------------------------
// mg_index_ranges_static -- Eq. 15's (i_min, i_max) of EVERY level of a mipmap without allocating.
//
// mg_index_range above takes its 8 bytes of scratch (the two words the warps' atomicMin / atomicMax
// meet in) from cudaMalloc and gives them back with cudaFree on every call.  Some callers cannot do
// that: a renderer or a training process whose own arena already owns all of the device's memory (the
// driver then has nothing left to hand out, or hands it out from the fragments the arena wanted
// back), and a frame loop that cannot afford cudaFree's wait for every stream of the device between
// a TF update and the next frame.  For them the scratch lives in the library image: one
// (min, max) pair per level in a file-scope __device__ array, MG_INDEX_RANGES_STATIC_MAX_LEVELS
// pairs = 256 bytes, resident on every GPU that loads libmg.so until the process exits.
//
// In host code `g_range_scratch` is only the symbol's host-side shadow, not a device address, so the
// address the range kernel gets comes from cudaGetSymbolAddress, looked up once per device with that
// device current (range_scratch_of_current_device).  The reset kernel is device code of this file and
// names the array directly.  The array is shared by every call and keeps the previous call's pairs:
// each call resets the pairs it will use before it reduces into them, and two calls whose kernels
// overlap on one GPU (different host threads, different streams) would reduce into the same pairs.
// ------------------------------------------------------------------------------------------------
namespace {

constexpr uint32_t kStaticLevels = MG_INDEX_RANGES_STATIC_MAX_LEVELS;
constexpr int kStaticMaxDevices = 64;

static __device__ __align__(256) uint32_t g_range_scratch[2 * kStaticLevels];

struct RangeLevels {
    uint64_t off[kStaticLevels + 1];   // level l = elements [off[l], off[l + 1]) of the index buffer
    uint32_t n_levels;
};

// pair l starts at (UINT32_MAX, 0): the neutral elements of min and max
__global__ void k_range_scratch_reset(uint32_t n_levels)
{
    const uint32_t l = threadIdx.x;
    if (l < n_levels) { g_range_scratch[2 * l] = 0xFFFFFFFFu; g_range_scratch[2 * l + 1] = 0u; }
}

// k_index_range over several levels in one launch: every CTA walks the levels in turn and takes its grid-stride
// share of each (16-byte streaming loads between the level's 16-byte boundaries, the ragged ends by CTA 0), then
// one atomic pair per warp into the level's pair of `mm`.
__global__ void __launch_bounds__(256) k_index_range_levels(const uint32_t* __restrict__ idx, const __grid_constant__ RangeLevels L,
                                                            uint32_t* __restrict__ mm)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint32_t l = 0; l < L.n_levels; l++) {
        const uint64_t n = L.off[l + 1] - L.off[l];
        if (n == 0) continue;                                             // uniform over the grid
        const uint32_t* p = idx + L.off[l];
        const mg::Span sp = mg::span_of(p, n);
        const uint4* v4 = reinterpret_cast<const uint4*>(p + sp.head);
        uint32_t lo = 0xFFFFFFFFu, hi = 0u;
        for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < sp.nv; i += stride) {
            const uint4 a = __ldcs(v4 + i);
            lo = min(lo, min(min(a.x, a.y), min(a.z, a.w)));
            hi = max(hi, max(max(a.x, a.y), max(a.z, a.w)));
        }
        if (blockIdx.x == 0 && threadIdx.x < sp.head + (n - sp.tail)) {
            const uint32_t v = p[mg::ragged(sp, threadIdx.x)];
            lo = min(lo, v); hi = max(hi, v);
        }
        lo = __reduce_min_sync(0xFFFFFFFFu, lo);
        hi = __reduce_max_sync(0xFFFFFFFFu, hi);
        if ((threadIdx.x & 31) == 0 && lo <= hi) { atomicMin(mm + 2 * l, lo); atomicMax(mm + 2 * l + 1, hi); }
    }
}

std::atomic<uint32_t*> g_range_scratch_addr[kStaticMaxDevices];           // device address of g_range_scratch, per device

// Set-up, once per device: ask the runtime where this device's instance of the array lives.
int range_scratch_of_current_device(uint32_t** out)
{
    int dev = -1;
    MG_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) {
        mg::set_error("mg_index_ranges_static: device ordinal %d is beyond the %d this entry point keeps an address for", dev, kStaticMaxDevices);
        return MG_ERR_INVALID_ARG;
    }
    uint32_t* p = g_range_scratch_addr[dev].load(std::memory_order_acquire);
    if (!p) {
        MG_CUDA(cudaGetSymbolAddress((void**)&p, g_range_scratch));      // the same answer from every thread: no lock needed
        g_range_scratch_addr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return MG_OK;
}

}  // namespace

extern "C" int mg_index_ranges_static(const uint32_t* idx_device, const uint64_t* level_offsets_host, uint32_t n_levels,
                                      uint32_t* i_min_host, uint32_t* i_max_host, void* stream)
{
    if (!idx_device || !level_offsets_host || !i_min_host || !i_max_host) { set_error("mg_index_ranges_static: NULL argument"); return MG_ERR_INVALID_ARG; }
    if (n_levels == 0 || n_levels > kStaticLevels) {
        set_error("mg_index_ranges_static: n_levels = %u, but the built-in scratch holds 1..%u levels (MG_INDEX_RANGES_STATIC_MAX_LEVELS); "
                  "use mg_index_range per level beyond that", n_levels, kStaticLevels);
        return MG_ERR_INVALID_ARG;
    }
    RangeLevels L;
    memset(&L, 0, sizeof(L));
    uint64_t longest = 0;
    for (uint32_t l = 0; l <= n_levels; l++) {
        L.off[l] = level_offsets_host[l];
        if (l && L.off[l] < L.off[l - 1]) { set_error("mg_index_ranges_static: level_offsets must not decrease (level %u)", l - 1); return MG_ERR_INVALID_ARG; }
        if (l && L.off[l] - L.off[l - 1] > longest) longest = L.off[l] - L.off[l - 1];
    }
    L.n_levels = n_levels;
    uint32_t* d_mm = nullptr;
    const int rc = range_scratch_of_current_device(&d_mm);
    if (rc != MG_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    k_range_scratch_reset<<<1, kStaticLevels, 0, st>>>(n_levels);
    uint64_t blocks = (longest / 4 + 256) / 256;
    if (blocks > 148ull * 8) blocks = 148ull * 8;
    k_index_range_levels<<<(unsigned)blocks, 256, 0, st>>>(idx_device, L, d_mm);
    count_launch(2);
    MG_CUDA(cudaGetLastError());
    uint32_t out[2 * kStaticLevels];
    MG_CUDA(cudaMemcpyAsync(out, d_mm, 2 * sizeof(uint32_t) * n_levels, cudaMemcpyDeviceToHost, st));
    MG_CUDA(cudaStreamSynchronize(st));
    for (uint32_t l = 0; l < n_levels; l++) { i_min_host[l] = out[2 * l]; i_max_host[l] = out[2 * l + 1]; }
    return MG_OK;
}
