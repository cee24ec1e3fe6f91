// Internal declarations shared by the translation units of libmg.so (NOT part of the C ABI,
// not used by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <string>
#include <vector>

#include "../../include/mg.h"

// Single-CTA tail kernel limits (mg_api.cu plans against them, mg_propagate.cu sizes its buffers with them).
#define MG_TAIL_SMEM_BYTES (224 * 1024)
#define MG_TAIL_MAX_LEVELS 128
// RGBA8 palette tile of the tiled colourise (mg_colorize.cu): what the L2 serves for random gathers
#define MG_DEFAULT_PAL_TILE_BYTES (88ull << 20)

namespace mg {

void set_error(const char* fmt, ...);
int cuda_fail(cudaError_t e, const char* what);   // records the message, returns MG_ERR_CUDA / MG_ERR_OOM
void count_launch(unsigned n = 1);

#define MG_CUDA(call)                                         \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return mg::cuda_fail(e__, #call); \
    } while (0)

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) belongs to the function instance in the CURRENT device's
// context, so it is set once per (function, device): a bit per device id, devices >= 64 set it every time.
struct SmemAttrOnce {
    std::atomic<uint64_t> mask{0};
    int ensure(const void* func, int bytes, int device);
};

// Host-side relabelling (csrc/relabel.cpp, also linked into the builder library).
// Input: any children-before-parents graph.  Output: level-contiguous numbering.
//   new_of_old[n]  new index of node n (leaves keep their index)
//   level_off      [depth + 2] offsets of the levels in the new numbering
// Returns 0, or -1 if a child does not precede its parent / equals its sibling.
int relabel_by_level(const uint32_t* child_a, const uint32_t* child_b, uint64_t n_nodes,
                     uint32_t n_leaves, std::vector<uint32_t>& new_of_old,
                     std::vector<uint64_t>& level_off);

#ifdef __CUDACC__
// A stream of n 4-byte elements at p, split for 16-byte loads: [0, head) one by one | nv uint4 from p + head |
// [tail, n) one by one.  head + (n - tail) <= 6.
struct Span { uint64_t head, nv, tail; };
__device__ __forceinline__ Span span_of(const void* p, uint64_t n)
{
    uint64_t head = ((16 - ((uintptr_t)p & 15)) & 15) / 4;
    if (head > n) head = n;
    const uint64_t nv = (n - head) / 4;
    return {head, nv, head + 4 * nv};
}
// index of the i-th ragged element (i < head + n - tail)
__device__ __forceinline__ uint64_t ragged(const Span& s, uint64_t i) { return i < s.head ? i : s.tail + (i - s.head); }
#endif

}  // namespace mg

struct mg_graph;
namespace mg {
// API entry guard: g's device must be the current one (include/mg.h, Conventions).
int check_device(const mg_graph* g, const char* who);
// A library call is about to write [p, p + bytes): if that overlaps the buffer the palettes mirror, they no
// longer do.
void invalidate_palettes_if_written(mg_graph* g, const void* p, uint64_t bytes);
// mg_colorize.cu: derive the palettes `format` needs from node_rgba on `st`, or check MG_PALETTE_FROM_LAST_PROPAGATE.
int prepare_palettes(mg_graph* g, const float* node_rgba, uint32_t format, cudaStream_t st, const char* who);
}  // namespace mg

struct mg_graph {
    int device = 0;
    uint64_t n_nodes = 0;
    uint32_t n_leaves = 0;
    uint32_t n_levels = 0;                 // depth + 1
    std::vector<uint64_t> level_off;       // [n_levels + 1], library numbering
    std::vector<uint32_t> leaf_segment_id; // may be empty
    std::vector<uint32_t> new_of_old;      // empty = identity
    // device SoA (library numbering); leaves' entries are zero
    uint32_t* d_a = nullptr;
    uint32_t* d_b = nullptr;
    float* d_w = nullptr;
    uint32_t* d_level_off = nullptr;       // [n_levels + 1] as uint32 (n_nodes < 2^32)
    uint32_t* d_new_of_old = nullptr;      // only if relabelled
    // per-graph scratch
    float* d_tf_stage = nullptr;           // [n_leaves][4]
    uint32_t* d_pal8 = nullptr;            // [n_nodes] RGBA8
    uint2* d_pal16 = nullptr;              // [n_nodes] 4 x fp16
    // node_rgba that mg_propagate last filled TOGETHER WITH both palettes, and that no library call has written
    // since; nullptr otherwise.  Only consulted to reject a wrong MG_PALETTE_FROM_LAST_PROPAGATE (mg_colorize).
    const float* pal_src = nullptr;
    bool no_palettes = false;              // MG_NO_PALETTES: mg_propagate does not derive the palettes
    uint64_t pal_tile_bytes = MG_DEFAULT_PAL_TILE_BYTES;   // fixed at mg_load_graph (MG_COLORIZE_TILE_BYTES in its environment)
    // launch plan: levels >= first_fused_level run in the single-CTA tail kernel (0 = none).  The tail
    // works entirely in shared memory on LOCAL indices: [0, tail_n_ext) = the distinct children that lie
    // below the tail ("external": gathered once), [tail_n_ext, tail_n_ext + tail_n) = the tail's nodes.
    uint32_t first_fused_level = 0;
    uint32_t tail_base = 0;                // library index of the first tail node (= level_off[first_fused_level])
    uint32_t tail_n = 0;                   // nodes in the tail
    uint32_t tail_n_ext = 0;               // distinct external children
    uint32_t* d_tail_ext = nullptr;        // [tail_n_ext] library indices of the external children
    uint32_t* d_tail_a = nullptr;          // [tail_n] children in local indices
    uint32_t* d_tail_b = nullptr;
    uint64_t device_bytes = 0;
};
