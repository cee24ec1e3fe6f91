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

__global__ void k_max_id(const uint32_t* __restrict__ seg, uint64_t n, uint32_t* out)
{
    uint32_t m = 0;
    for (uint64_t v = (uint64_t)blockIdx.x * kThreads + threadIdx.x; v < n; v += (uint64_t)gridDim.x * kThreads) m = max(m, __ldg(seg + v));
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0) atomicMax(out, m);
}

__global__ void k_mark_ids(const uint32_t* __restrict__ seg, uint64_t n, uint8_t* present)
{
    uint32_t last = kNone;
    for (uint64_t v = (uint64_t)blockIdx.x * kThreads + threadIdx.x; v < n; v += (uint64_t)gridDim.x * kThreads) {
        const uint32_t s = __ldg(seg + v);
        if (s != last) {                                              // test first: a handful of hot bytes, mostly already set
            if (!present[s]) present[s] = 1;                          // (racing stores of the same value)
            last = s;
        }
    }
}

// level0[v] = leaf_of[S(v)]; seg and level0 may be the same buffer (element-wise).
__global__ void k_map_ids(const uint32_t* seg, uint64_t n, const uint32_t* __restrict__ leaf_of, uint32_t* level0)
{
    for (uint64_t v = (uint64_t)blockIdx.x * kThreads + threadIdx.x; v < n; v += (uint64_t)gridDim.x * kThreads)
        level0[v] = __ldg(leaf_of + seg[v]);
}

// One thread per level-1 parent (x fastest).  Children t = 4 dz + 2 dy + dx; kNone outside the volume.
__global__ void __launch_bounds__(kThreads)
k_front_level1(const uint32_t* __restrict__ l0, uint32_t cx, uint32_t cy, uint32_t cz, uint32_t px, uint32_t py, uint64_t n1,
               uint32_t* __restrict__ level1, uint32_t* __restrict__ mixed_voxel, uint32_t* __restrict__ mixed_children,
               unsigned long long capacity, unsigned long long* counter)
{
    const uint64_t v = (uint64_t)blockIdx.x * kThreads + threadIdx.x;
    const bool live = v < n1;
    uint32_t ch[8];
    bool pure = true;
    if (live) {
        const uint32_t i = (uint32_t)(v % px), j = (uint32_t)((v / px) % py), k = (uint32_t)(v / ((uint64_t)px * py));
#pragma unroll
        for (int t = 0; t < 8; t++) {
            const uint32_t x = 2 * i + (t & 1), y = 2 * j + ((t >> 1) & 1), z = 2 * k + (t >> 2);
            ch[t] = (x < cx && y < cy && z < cz) ? __ldg(l0 + ((uint64_t)z * cy + y) * cx + x) : kNone;
        }
#pragma unroll
        for (int t = 1; t < 8; t++) pure = pure && (ch[t] == ch[0] || ch[t] == kNone);   // child 0 always exists
        level1[v] = pure ? ch[0] : kNone;
    }
    // one atomic per warp for the list slots
    const unsigned m = __ballot_sync(0xffffffffu, live && !pure);
    if (m == 0) return;
    const unsigned lane = threadIdx.x & 31, leader = __ffs(m) - 1;
    unsigned long long base = 0;
    if (lane == leader) base = atomicAdd(counter, (unsigned long long)__popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (live && !pure) {
        const unsigned long long slot = base + __popc(m & ((1u << lane) - 1));
        if (slot < capacity) {
            mixed_voxel[slot] = (uint32_t)v;
            uint4* dst = reinterpret_cast<uint4*>(mixed_children + 8 * slot);
            dst[0] = make_uint4(ch[0], ch[1], ch[2], ch[3]);
            dst[1] = make_uint4(ch[4], ch[5], ch[6], ch[7]);
        }
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
    const unsigned grid = (unsigned)std::min<uint64_t>((n_voxels + kThreads - 1) / kThreads, 148ull * 16);
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
    k_map_ids<<<grid, kThreads, 0, st>>>(seg_device, n_voxels, d_leaf_of, level0_device);
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
        k_front_level1<<<(unsigned)((n1 + kThreads - 1) / kThreads), kThreads, 0, st>>>(
            level0_device, (uint32_t)X, (uint32_t)Y, (uint32_t)Z, (uint32_t)px, (uint32_t)py, n1, level1_device, mixed_voxel_device,
            mixed_children_device, capacity, d_counter);
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
