// Topological levels + level-contiguous relabelling.
//
// level(source) = 0, level(node) = max(level(a), level(b)) + 1 -- a linear scan, valid because
// children precede parents (Eq. 8).  The new numbering keeps the leaves, makes every level
// contiguous (so one level = one index range = one launch) and, inside a level, orders nodes by
// (higher child, lower child) in the NEW numbering so that neighbouring threads gather
// neighbouring palette entries (L2 / L1 sector locality): on config 5 the higher child becomes a
// sequential sweep over the previous level (2.02 -> 1.72 ms).  Ordering by (lower child, higher child)
// instead -- the far gathers monotone, the near ones left to L2 -- was measured at 1.74 ms: no better.
// Values are untouched: relabelling never changes a node's (a, b, w), only where it lives.
#include <algorithm>
#include <cstdint>
#include <vector>
#if defined(_OPENMP)
#include <parallel/algorithm>
#define MG_SORT __gnu_parallel::sort
#else
#define MG_SORT std::sort
#endif

namespace mg {

int relabel_by_level(const uint32_t* child_a, const uint32_t* child_b, uint64_t n_nodes,
                     uint32_t n_leaves, std::vector<uint32_t>& new_of_old,
                     std::vector<uint64_t>& level_off)
{
    std::vector<uint32_t> level(n_nodes, 0);
    uint32_t depth = 0;
    for (uint64_t n = n_leaves; n < n_nodes; n++) {
        uint32_t a = child_a[n], b = child_b[n];
        if (a >= n || b >= n || a == b) return -1;
        uint32_t l = std::max(level[a], level[b]) + 1;
        level[n] = l;
        depth = std::max(depth, l);
    }
    level_off.assign(depth + 2, 0);
    for (uint64_t n = 0; n < n_nodes; n++) level_off[level[n] + 1]++;
    for (uint32_t l = 0; l <= depth; l++) level_off[l + 1] += level_off[l];

    // bucket the nodes by level, in old-index order
    std::vector<uint32_t> by_level(n_nodes);
    {
        std::vector<uint64_t> cur(level_off.begin(), level_off.end() - 1);
        for (uint64_t n = 0; n < n_nodes; n++) by_level[cur[level[n]]++] = (uint32_t)n;
    }
    new_of_old.resize(n_nodes);
    for (uint32_t n = 0; n < n_leaves; n++) new_of_old[n] = n;   // level 0 = leaves, order kept

    struct Key { uint64_t k; uint32_t old; };
    std::vector<Key> keys;
    for (uint32_t l = 1; l <= depth; l++) {
        uint64_t lo = level_off[l], hi = level_off[l + 1];
        keys.resize(hi - lo);
#pragma omp parallel for schedule(static)
        for (int64_t q = 0; q < (int64_t)(hi - lo); q++) {
            uint32_t n = by_level[lo + q];
            uint32_t na = new_of_old[child_a[n]], nb = new_of_old[child_b[n]];
            keys[q] = Key{((uint64_t)std::max(na, nb) << 32) | std::min(na, nb), n};
        }
        MG_SORT(keys.begin(), keys.end(), [](const Key& x, const Key& y) {
            return x.k != y.k ? x.k < y.k : x.old < y.old;
        });
#pragma omp parallel for schedule(static)
        for (int64_t q = 0; q < (int64_t)(hi - lo); q++) new_of_old[keys[q].old] = (uint32_t)(lo + q);
    }
    return 0;
}

}  // namespace mg
