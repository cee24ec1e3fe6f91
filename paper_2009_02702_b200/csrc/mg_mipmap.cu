// mg_mipmap.cu -- NEXT-4 (second half): device front end of the histogram mipmap (a0, Eq. 4).
//
// Level 0 of the mipmap is 87 % of its voxels and, on the paper's data, > 97 % of all voxels are pure
// (Table 2: 1.006-1.025 non-zeros per voxel).  Everything the builder does with those is a stream:
//   mg_mipmap_leaf_index     S -> leaf number (sorted distinct IDs present become the leaves, Q14)
//   mg_mipmap_front_level1   each level-1 parent = average of its existing children (Eq. 4): if they are one
//                            segment the parent is that leaf; otherwise the parent goes on a list with its children
// and runs here at HBM speed with the volume where the generator left it (on the device).  The host builder
// (mgb_build_from_level1) then only merges / hash-conses the listed parents and the levels >= 2 -- 12 % of the
// voxels -- and level 0's node index never leaves the device.
#include <algorithm>
#include <vector>

#include "mg_internal.h"

namespace {

constexpr int kThreads = 256;
constexpr uint32_t kNone = 0xFFFFFFFFu;

// The three leaf-index passes stream the 4-byte volume once each: 16-byte loads, two per thread in flight, the
// 0-3 elements before the first 16-byte boundary and after the last whole vector taken one by one by block 0.
using mg::Span;
using mg::span_of;
using mg::ragged;

__global__ void __launch_bounds__(kThreads) k_max_id(const uint32_t* __restrict__ seg, uint64_t n, uint32_t* out)
{
    const Span sp = span_of(seg, n);
    const uint4* v4 = reinterpret_cast<const uint4*>(seg + sp.head);
    const uint64_t stride = (uint64_t)gridDim.x * kThreads;
    uint32_t m = 0;
    uint64_t i = (uint64_t)blockIdx.x * kThreads + threadIdx.x;
    for (; i + stride < sp.nv; i += 2 * stride) {
        const uint4 a = __ldcs(v4 + i), b = __ldcs(v4 + i + stride);
        m = max(max(max(a.x, a.y), max(a.z, a.w)), max(m, max(max(b.x, b.y), max(b.z, b.w))));
    }
    if (i < sp.nv) {
        const uint4 a = __ldcs(v4 + i);
        m = max(m, max(max(a.x, a.y), max(a.z, a.w)));
    }
    if (blockIdx.x == 0 && threadIdx.x < sp.head + (n - sp.tail)) m = max(m, seg[ragged(sp, threadIdx.x)]);
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}

// test first: a handful of hot bytes, mostly already set (racing stores of the same value)
__device__ __forceinline__ void mark(uint8_t* present, uint32_t s, uint32_t& last)
{
    if (s != last) {
        if (!present[s]) present[s] = 1;
        last = s;
    }
}

__global__ void __launch_bounds__(kThreads) k_mark_ids(const uint32_t* __restrict__ seg, uint64_t n, uint8_t* present)
{
    const Span sp = span_of(seg, n);
    const uint4* v4 = reinterpret_cast<const uint4*>(seg + sp.head);
    const uint64_t stride = (uint64_t)gridDim.x * kThreads;
    uint32_t last = kNone;
    uint64_t i = (uint64_t)blockIdx.x * kThreads + threadIdx.x;
    for (; i + stride < sp.nv; i += 2 * stride) {
        const uint4 a = __ldcs(v4 + i), b = __ldcs(v4 + i + stride);
        mark(present, a.x, last); mark(present, a.y, last); mark(present, a.z, last); mark(present, a.w, last);
        mark(present, b.x, last); mark(present, b.y, last); mark(present, b.z, last); mark(present, b.w, last);
    }
    if (i < sp.nv) {
        const uint4 a = __ldcs(v4 + i);
        mark(present, a.x, last); mark(present, a.y, last); mark(present, a.z, last); mark(present, a.w, last);
    }
    if (blockIdx.x == 0 && threadIdx.x < sp.head + (n - sp.tail)) mark(present, seg[ragged(sp, threadIdx.x)], last);
}

// level0[v] = leaf_of[S(v)]; seg and level0 may be the same buffer (element-wise: every thread reads its elements
// before it writes them, and nobody else touches them).  VEC needs seg and level0 congruent modulo 16 bytes.
template <bool VEC>
__global__ void __launch_bounds__(kThreads) k_map_ids(const uint32_t* seg, uint64_t n, const uint32_t* __restrict__ leaf_of, uint32_t* level0)
{
    const uint64_t stride = (uint64_t)gridDim.x * kThreads;
    uint64_t i = (uint64_t)blockIdx.x * kThreads + threadIdx.x;
    if (!VEC) {
        for (; i < n; i += stride) level0[i] = __ldg(leaf_of + seg[i]);
        return;
    }
    const Span sp = span_of(seg, n);
    const uint4* v4 = reinterpret_cast<const uint4*>(seg + sp.head);
    uint4* o4 = reinterpret_cast<uint4*>(level0 + sp.head);
    auto map4 = [&](const uint4 a) { return make_uint4(__ldg(leaf_of + a.x), __ldg(leaf_of + a.y), __ldg(leaf_of + a.z), __ldg(leaf_of + a.w)); };
    for (; i + stride < sp.nv; i += 2 * stride) {
        const uint4 a = __ldcs(v4 + i), b = __ldcs(v4 + i + stride);
        const uint4 ra = map4(a), rb = map4(b);
        o4[i] = ra;
        o4[i + stride] = rb;
    }
    if (i < sp.nv) o4[i] = map4(__ldcs(v4 + i));
    if (blockIdx.x == 0 && threadIdx.x < sp.head + (n - sp.tail)) {
        const uint64_t r = ragged(sp, threadIdx.x);
        level0[r] = __ldg(leaf_of + seg[r]);
    }
}

// kPar level-1 parents per thread (x fastest; n1 < 2^32), kThreads * kPar consecutive parents per CTA.  Children
// t = 4 dz + 2 dy + dx; kNone outside the volume.  PAIR (cx even, l0 8-byte aligned): the two x-children of a row
// always both exist and come as one 8-byte load.  The list slots of a CTA's mixed parents come from ONE atomic on the
// global counter: on the paper-shaped volumes a quarter of all warps hold a mixed parent, and that many value-returning
// atomics on one address serialise in L2 to longer than the whole stream takes.
constexpr int kPar = 4;

template <bool PAIR>
__global__ void __launch_bounds__(kThreads)
k_front_level1(const uint32_t* __restrict__ l0, uint32_t cx, uint32_t cy, uint32_t cz, uint32_t px, uint32_t py, uint64_t n1,
               uint32_t* __restrict__ level1, uint32_t* __restrict__ mixed_voxel, uint32_t* __restrict__ mixed_children,
               unsigned long long capacity, unsigned long long* counter)
{
    __shared__ unsigned warp_total[kThreads / 32];
    __shared__ unsigned long long cta_base;
    const uint64_t v0 = (uint64_t)blockIdx.x * (kThreads * kPar) + threadIdx.x;
    uint32_t ch[kPar][8];
    unsigned mixed = 0;                                               // bit p: parent p of this thread is mixed
#pragma unroll
    for (int p = 0; p < kPar; p++) {
        const uint64_t v = v0 + (uint64_t)p * kThreads;
        if (v >= n1) continue;
        const uint32_t v32 = (uint32_t)v, row = v32 / px, i = v32 - row * px, k = row / py, j = row - k * py;
#pragma unroll
        for (int t = 0; t < 8; t += PAIR ? 2 : 1) {
            const uint32_t x = 2 * i + (t & 1), y = 2 * j + ((t >> 1) & 1), z = 2 * k + (t >> 2);
            const uint64_t at = ((uint64_t)z * cy + y) * cx + x;
            if (PAIR) {
                const uint2 c = (y < cy && z < cz) ? __ldcs(reinterpret_cast<const uint2*>(l0 + at)) : make_uint2(kNone, kNone);
                ch[p][t] = c.x;
                ch[p][t + 1] = c.y;
            } else {
                ch[p][t] = (x < cx && y < cy && z < cz) ? __ldg(l0 + at) : kNone;
            }
        }
    }
#pragma unroll
    for (int p = 0; p < kPar; p++) {
        const uint64_t v = v0 + (uint64_t)p * kThreads;
        if (v >= n1) continue;
        bool pure = true;
#pragma unroll
        for (int t = 1; t < 8; t++) pure = pure && (ch[p][t] == ch[p][0] || ch[p][t] == kNone);   // child 0 always exists
        level1[v] = pure ? ch[p][0] : kNone;
        if (!pure) mixed |= 1u << p;
    }
    // exclusive prefix of the mixed counts over the CTA: shuffles inside a warp, shared memory across the warps
    const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5, cnt = __popc(mixed);
    unsigned incl = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned up = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += up;
    }
    if (lane == 31) warp_total[warp] = incl;
    __syncthreads();
    unsigned before = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kThreads / 32; w++) {
        const unsigned c = warp_total[w];
        if (w < (int)warp) before += c;
        total += c;
    }
    if (total == 0) return;                                           // uniform over the CTA
    if (threadIdx.x == 0) cta_base = atomicAdd(counter, (unsigned long long)total);
    __syncthreads();
    unsigned long long slot = cta_base + before + (incl - cnt);
#pragma unroll
    for (int p = 0; p < kPar; p++) {
        if (!(mixed & (1u << p))) continue;
        if (slot < capacity) {
            mixed_voxel[slot] = (uint32_t)(v0 + (uint64_t)p * kThreads);
            uint4* dst = reinterpret_cast<uint4*>(mixed_children + 8 * slot);
            dst[0] = make_uint4(ch[p][0], ch[p][1], ch[p][2], ch[p][3]);
            dst[1] = make_uint4(ch[p][4], ch[p][5], ch[p][6], ch[p][7]);
        }
        slot++;
    }
}

}  // namespace

extern "C" int mg_mipmap_leaf_index(const uint32_t* seg_device, uint64_t n_voxels, uint32_t* level0_device,
                                    uint32_t* leaf_segment_id, uint32_t capacity, uint32_t* n_leaves, void* stream)
{
    if (!seg_device || !level0_device || !leaf_segment_id || !n_leaves || n_voxels == 0) {
        mg::set_error("mg_mipmap_leaf_index: NULL argument or empty volume");
        return MG_ERR_INVALID_ARG;
    }
    *n_leaves = 0;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned grid = (unsigned)std::min<uint64_t>((n_voxels / 4 + kThreads) / kThreads, 148ull * 8);   // 2048 threads per SM
    uint32_t* d_max = nullptr;
    uint8_t* d_present = nullptr;
    uint32_t* d_leaf_of = nullptr;
    auto fail = [&](int rc) { cudaFree(d_max); cudaFree(d_present); cudaFree(d_leaf_of); return rc; };
#define MM_CUDA(call)                                                              \
    do {                                                                           \
        cudaError_t e__ = (call);                                                  \
        if (e__ != cudaSuccess) return fail(mg::cuda_fail(e__, #call));            \
    } while (0)
    MM_CUDA(cudaMalloc(&d_max, sizeof(uint32_t)));
    MM_CUDA(cudaMemsetAsync(d_max, 0, sizeof(uint32_t), st));
    k_max_id<<<grid, kThreads, 0, st>>>(seg_device, n_voxels, d_max);
    MM_CUDA(cudaGetLastError());
    mg::count_launch();
    uint32_t mx = 0;
    MM_CUDA(cudaMemcpyAsync(&mx, d_max, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    MM_CUDA(cudaStreamSynchronize(st));
    if (mx >= (1u << 28)) {
        mg::set_error("mg_mipmap_leaf_index: segment IDs up to %u need a presence table beyond 2^28 entries; use mgb_build", mx);
        return fail(MG_ERR_INVALID_ARG);
    }
    const size_t n_ids = (size_t)mx + 1;
    MM_CUDA(cudaMalloc(&d_present, n_ids));
    MM_CUDA(cudaMemsetAsync(d_present, 0, n_ids, st));
    k_mark_ids<<<grid, kThreads, 0, st>>>(seg_device, n_voxels, d_present);
    MM_CUDA(cudaGetLastError());
    mg::count_launch();
    std::vector<uint8_t> present(n_ids);
    MM_CUDA(cudaMemcpyAsync(present.data(), d_present, n_ids, cudaMemcpyDeviceToHost, st));
    MM_CUDA(cudaStreamSynchronize(st));
    std::vector<uint32_t> leaf_of(n_ids, 0);
    uint64_t count = 0;
    for (size_t i = 0; i < n_ids; i++)
        if (present[i]) {
            if (count < capacity) leaf_segment_id[count] = (uint32_t)i;
            leaf_of[i] = (uint32_t)count++;
        }
    *n_leaves = (uint32_t)count;
    if (count > capacity) {
        mg::set_error("mg_mipmap_leaf_index: %llu distinct segment IDs, capacity %u", (unsigned long long)count, capacity);
        return fail(MG_ERR_INVALID_ARG);
    }
    MM_CUDA(cudaMalloc(&d_leaf_of, n_ids * sizeof(uint32_t)));
    MM_CUDA(cudaMemcpyAsync(d_leaf_of, leaf_of.data(), n_ids * sizeof(uint32_t), cudaMemcpyHostToDevice, st));
    if ((((uintptr_t)seg_device ^ (uintptr_t)level0_device) & 15) == 0)
        k_map_ids<true><<<grid, kThreads, 0, st>>>(seg_device, n_voxels, d_leaf_of, level0_device);
    else
        k_map_ids<false><<<grid, kThreads, 0, st>>>(seg_device, n_voxels, d_leaf_of, level0_device);
    MM_CUDA(cudaGetLastError());
    mg::count_launch();
    MM_CUDA(cudaStreamSynchronize(st));                                // leaf_of (host) and the temporaries die here
#undef MM_CUDA
    return fail(MG_OK);
}

extern "C" int mg_mipmap_front_level1(const uint32_t* level0_device, uint64_t X, uint64_t Y, uint64_t Z, uint32_t* level1_device,
                                      uint32_t* mixed_voxel_device, uint32_t* mixed_children_device, uint64_t capacity,
                                      uint64_t* n_mixed, void* stream)
{
    if (!level0_device || !level1_device || !n_mixed || (capacity && (!mixed_voxel_device || !mixed_children_device))) {
        mg::set_error("mg_mipmap_front_level1: NULL argument");
        return MG_ERR_INVALID_ARG;
    }
    *n_mixed = 0;
    if (X == 0 || Y == 0 || Z == 0 || X > 0x7fffffffull || Y > 0x7fffffffull || Z > 0x7fffffffull) {
        mg::set_error("mg_mipmap_front_level1: bad dimensions");
        return MG_ERR_INVALID_ARG;
    }
    if ((uintptr_t)mixed_children_device & 15) { mg::set_error("mg_mipmap_front_level1: mixed_children must be 16-byte aligned"); return MG_ERR_INVALID_ARG; }
    const uint64_t px = (X + 1) / 2, py = (Y + 1) / 2, pz = (Z + 1) / 2, n1 = px * py * pz;
    if (n1 >= (1ull << 32)) { mg::set_error("mg_mipmap_front_level1: level 1 has 2^32 voxels or more"); return MG_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* d_counter = nullptr;
    MG_CUDA(cudaMalloc(&d_counter, sizeof(unsigned long long)));
    cudaError_t e = cudaMemsetAsync(d_counter, 0, sizeof(unsigned long long), st);
    if (e == cudaSuccess) {
        const unsigned grid = (unsigned)((n1 + kThreads * kPar - 1) / (kThreads * kPar));
        if (X % 2 == 0 && ((uintptr_t)level0_device & 7) == 0)
            k_front_level1<true><<<grid, kThreads, 0, st>>>(level0_device, (uint32_t)X, (uint32_t)Y, (uint32_t)Z, (uint32_t)px, (uint32_t)py,
                                                            n1, level1_device, mixed_voxel_device, mixed_children_device, capacity, d_counter);
        else
            k_front_level1<false><<<grid, kThreads, 0, st>>>(level0_device, (uint32_t)X, (uint32_t)Y, (uint32_t)Z, (uint32_t)px, (uint32_t)py,
                                                             n1, level1_device, mixed_voxel_device, mixed_children_device, capacity, d_counter);
        e = cudaGetLastError();
        mg::count_launch();
    }
    unsigned long long c = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&c, d_counter, sizeof(c), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d_counter);
    if (e != cudaSuccess) return mg::cuda_fail(e, "mg_mipmap_front_level1");
    *n_mixed = c;
    return MG_OK;
}
