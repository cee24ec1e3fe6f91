// Internal declarations of libmg_builder.so (host-only; NOT part of the C ABI, not used by oracle/).
#pragma once
#include <stdint.h>

#include <string>
#include <vector>

#include "../../../include/mg_builder.h"

namespace mg {
// csrc/relabel.cpp (also part of libmg.so): topological levels (L211) + level-contiguous numbering.
int relabel_by_level(const uint32_t* child_a, const uint32_t* child_b, uint64_t n_nodes, uint32_t n_leaves,
                     std::vector<uint32_t>& new_of_old, std::vector<uint64_t>& level_off);
}

namespace mgb {

void set_error(const char* fmt, ...);

// A set of DISTINCT mixtures with >= 2 non-zeros, in canonical ("scanline", L257) order: mixture q has
// entries [off[q], off[q+1]) of (leaf, count), leaves strictly increasing, counts > 0 and reduced
// (their gcd is 1; by Eq. 4 every total is a power of two, but nothing below relies on that).
struct MixtureSet {
    uint32_t n_leaves = 0;
    std::vector<uint64_t> off{0};
    std::vector<uint32_t> leaf;
    std::vector<uint64_t> count;
    uint64_t size() const { return off.size() - 1; }
};

// Result of the factorisation (a1), creation-order numbering: leaves 0..n_leaves-1, then internal
// nodes with children preceding parents (Eq. 8).
struct Factorised {
    std::vector<uint32_t> a, b;          // children; a < b in creation numbering ("canonical orientation")
    std::vector<uint32_t> bin;           // weight bin of the node (quantised builds)
    std::vector<double> w_sum;           // sum of the exact ratios m_b / (m_a + m_b) merged into the node
    std::vector<double> w_sq;            // sum of their squares (per-bin sigma, L176)
    std::vector<uint32_t> w_cnt;         // how many factorisation steps produced / re-used the node
    std::vector<uint32_t> node_of_mix;   // [n mixtures] node that represents the mixture
    uint64_t n_stage1 = 0, n_stage2 = 0, n_big = 0;
    bool phi2_exact = true;
};

int factorise(const MixtureSet& ms, const mgb_params& p, Factorised& out);

// Histogram mipmap (a0).  level_ids[l][v] = leaf number (pure voxel) or n_leaves + canonical mixture
// number.  level_ids[0] is the leaf-index volume.
struct Mipmap {
    std::vector<uint64_t> dims;                    // X_l, Y_l, Z_l per level
    std::vector<std::vector<uint32_t>> level_ids;  // per level
    std::vector<uint32_t> leaf_segment_id;         // sorted distinct IDs present (Q14)
    uint64_t nnz_total = 0;
    MixtureSet mixtures;
    std::vector<uint32_t> front_mixture;           // LevelsFront only: canonical number of every listed mixture
};

// Levels 0 and 1 classified outside the host builder (mgb_build_from_level1): level 0 is not passed at all.
struct Level1Front {
    const uint32_t* leaf_segment_id;   // [n_leaves] sorted distinct segment IDs
    uint32_t n_leaves;
    const uint32_t* level1;            // [X_1 Y_1 Z_1] leaf number of a pure parent, 0xFFFFFFFF otherwise
    const uint32_t* mixed_voxel;       // [n_mixed] level-1 voxel index of every non-pure parent (any order)
    const uint32_t* mixed_children;    // [n_mixed][8] leaf numbers of its existing children, 0xFFFFFFFF = missing
    uint64_t n_mixed;
};

// Levels 1 .. level_done built outside the host builder (mg_mipmap_levels_build of include/mg.h): the distinct mixtures
// found so far with their first occurrence, and the handles of the last finished level.
struct LevelsFront {
    const uint32_t* leaf_segment_id;   // [n_leaves] sorted distinct segment IDs
    uint32_t n_leaves;
    uint32_t level_done;               // >= 1
    const uint32_t* handles;           // [voxels of level_done] leaf number, or 0x80000000 | number of a listed mixture
    uint64_t n_mix;
    const uint64_t* mix_offset;        // [n_mix] first entry
    const uint32_t* mix_k;             // [n_mix] non-zeros (>= 2)
    const uint32_t* mix_tlog;          // [n_mix] the counts sum to 2^tlog
    const uint64_t* mix_first_pos;     // [n_mix] level << 40 | voxel of the first occurrence
    const uint32_t* leaf;              // entries: leaves ascending inside a mixture
    const uint64_t* count;
    uint64_t n_entries;
    uint64_t nnz_levels;               // non-zeros summed over every voxel of the levels 1 .. level_done
};

// With `front`, seg is not read and out.level_ids[0] stays empty.  With `levels`, neither are the levels
// 1 .. level_done - 1, and out.front_mixture[q] = canonical number of the q-th listed mixture.
int build_mipmap(const uint32_t* seg, uint64_t X, uint64_t Y, uint64_t Z, int n_threads, Mipmap& out,
                 const Level1Front* front = nullptr, const LevelsFront* levels = nullptr);

}  // namespace mgb

struct mgb_result {
    mgb_info info{};
    std::vector<uint64_t> dims;
    std::vector<uint32_t> child_a, child_b;
    std::vector<float> weight;
    std::vector<double> weight_exact;
    std::vector<float> weight_sigma;     // per node: sigma of its weight's quantiser bin (0 when unquantised)
    std::vector<uint64_t> level_off;
    std::vector<uint32_t> leaf_segment_id;
    std::vector<std::vector<uint32_t>> node_idx;   // per mip level, final numbering
    std::vector<float> codeword, sigma;
    std::vector<uint64_t> bin_count;
    std::vector<uint32_t> front_mixture_node;      // mgb_build_from_levels: node of every mixture the caller listed
};
