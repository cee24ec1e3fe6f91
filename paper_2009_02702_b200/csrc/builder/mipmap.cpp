// mipmap.cpp -- a0: the normalised histogram mipmap of a segment-ID volume (Eq. 4).
//
//   H(i,j,k,0) = e_{S(i,j,k)};   H(i,j,k,l) = (1/N) sum over the EXISTING children (2i..2i+1, 2j..2j+1,
//   2k..2k+1) of H(.,.,.,l-1),   N = number of existing children (reading Q2), dims ceil-halved (L80).
//
// Host design (nothing here is the paper's: its encoder is serial C++ "without the STL", L261):
//   * N is 1, 2, 4 or 8, so every entry is a dyadic rational: a mixture is kept as EXACT integer counts
//     whose total is a power of two, divided by their common power of two.  The reduced form does not
//     depend on the level, so equal mixtures of different levels are one object.
//   * > 97 % of the voxels are pure (Table 2: 1.006-1.025 non-zeros per voxel): a parent whose
//     existing children all carry the same mixture inherits it without touching the table.
//   * every other parent merges its children's sparse vectors (sorted (index, value) pairs, L261) and
//     hash-conses the result in a sharded table, so only DISTINCT mixtures reach the factoriser.
//   * per-voxel state is one uint32: the leaf number (pure) or a mixture handle.
//   * threads race for handles, so mixtures are renumbered afterwards by their first occurrence in
//     (level, z, y, x) order -- the "scanline order" of L257 -- which makes the output deterministic.
#include <omp.h>

#include <algorithm>
#include <atomic>
#include <cstring>
#include <memory>
#include <unordered_set>

#include "builder_internal.h"

namespace mgb {
namespace {

struct Entry {
    uint32_t leaf;
    uint32_t pad;
    uint64_t count;
};

struct Rec {
    Entry* data;
    uint32_t k;       // non-zeros
    uint32_t hash;
    uint32_t tlog;    // the reduced counts sum to 2^tlog
    std::atomic<uint64_t> first_pos;
};

constexpr uint32_t kShardBits = 9, kShards = 1u << kShardBits, kLocalBits = 22;
constexpr uint32_t kMixed = 0x80000000u;
constexpr uint32_t kRecChunk = 4096, kMaxRecChunks = (1u << kLocalBits) / kRecChunk;
constexpr size_t kArenaChunk = 1u << 16;

struct Shard {
    std::atomic_flag lock = ATOMIC_FLAG_INIT;
    Rec* rec_chunks[kMaxRecChunks] = {};
    uint32_t n_recs = 0;
    std::vector<Entry*> arena;
    size_t arena_used = kArenaChunk;
    std::vector<uint32_t> slot_local, slot_hash;   // open addressing; slot_local = local + 1, 0 = empty
    uint32_t mask = 0;

    ~Shard()
    {
        for (uint32_t c = 0; c < kMaxRecChunks; c++) delete[] rec_chunks[c];
        for (Entry* p : arena) free(p);
    }
    Rec& rec(uint32_t local) const { return rec_chunks[local / kRecChunk][local % kRecChunk]; }

    Entry* alloc(uint32_t k)
    {
        if (k > kArenaChunk) {   // oversize mixture: its own block
            Entry* p = (Entry*)malloc((size_t)k * sizeof(Entry));
            if (p) arena.insert(arena.begin(), p);   // keep the current chunk last
            return p;
        }
        if (arena_used + k > kArenaChunk) {
            Entry* p = (Entry*)malloc(kArenaChunk * sizeof(Entry));
            if (!p) return nullptr;
            arena.push_back(p);
            arena_used = 0;
        }
        Entry* r = arena.back() + arena_used;
        arena_used += k;
        return r;
    }
    void grow()
    {
        uint32_t cap = mask ? 2 * (mask + 1) : 1024;
        std::vector<uint32_t> nl(cap, 0), nh(cap, 0);
        for (uint32_t s = 0; s <= mask && mask; s++)
            if (slot_local[s]) {
                uint32_t i = slot_hash[s] & (cap - 1);
                while (nl[i]) i = (i + 1) & (cap - 1);
                nl[i] = slot_local[s];
                nh[i] = slot_hash[s];
            }
        slot_local.swap(nl);
        slot_hash.swap(nh);
        mask = cap - 1;
    }
};

inline uint64_t mix64(uint64_t x)
{
    x ^= x >> 33; x *= 0xff51afd7ed558ccdull;
    x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ull;
    return x ^ (x >> 33);
}

inline uint64_t hash_entries(const Entry* e, uint32_t k)
{
    uint64_t h = 0x9E3779B97F4A7C15ull ^ k;
    for (uint32_t i = 0; i < k; i++) h = mix64(h ^ (((uint64_t)e[i].leaf << 40) + e[i].count)) + 0x632BE59BD9B4E019ull;
    return h;
}

struct Table {
    std::unique_ptr<Shard[]> shards{new Shard[kShards]};
    std::atomic<bool> failed{false};

    const Rec& rec(uint32_t handle) const
    {
        return shards[(handle >> kLocalBits) & (kShards - 1)].rec(handle & ((1u << kLocalBits) - 1));
    }

    // Returns the handle (kMixed | shard | local) of the mixture, inserting it if new; 0 on failure.
    uint32_t intern(const Entry* e, uint32_t k, uint32_t tlog, uint64_t pos)
    {
        const uint64_t h = hash_entries(e, k);
        const uint32_t sh = (uint32_t)(h & (kShards - 1));
        const uint32_t h32 = (uint32_t)(h >> 32);
        Shard& S = shards[sh];
        while (S.lock.test_and_set(std::memory_order_acquire)) { }
        if (S.mask == 0 || (uint64_t)(S.n_recs + 1) * 10 > (uint64_t)(S.mask + 1) * 6) S.grow();
        uint32_t i = h32 & S.mask, local = 0;
        bool found = false;
        while (S.slot_local[i]) {
            if (S.slot_hash[i] == h32) {
                const Rec& r = S.rec(S.slot_local[i] - 1);
                if (r.k == k) {
                    bool eq = true;
                    for (uint32_t q = 0; q < k; q++)
                        if (r.data[q].leaf != e[q].leaf || r.data[q].count != e[q].count) { eq = false; break; }
                    if (eq) { found = true; local = S.slot_local[i] - 1; break; }
                }
            }
            i = (i + 1) & S.mask;
        }
        if (!found) {
            if (S.n_recs >= (1u << kLocalBits)) { S.lock.clear(std::memory_order_release); failed = true; return 0; }
            local = S.n_recs;
            if (!S.rec_chunks[local / kRecChunk]) S.rec_chunks[local / kRecChunk] = new (std::nothrow) Rec[kRecChunk];
            Entry* d = S.rec_chunks[local / kRecChunk] ? S.alloc(k) : nullptr;
            if (!d) { S.lock.clear(std::memory_order_release); failed = true; return 0; }
            memcpy(d, e, (size_t)k * sizeof(Entry));
            Rec& r = S.rec(local);
            r.data = d; r.k = k; r.hash = h32; r.tlog = tlog;
            r.first_pos.store(pos, std::memory_order_relaxed);
            S.slot_local[i] = local + 1;
            S.slot_hash[i] = h32;
            S.n_recs++;
        }
        S.lock.clear(std::memory_order_release);
        if (found) {
            std::atomic<uint64_t>& fp = S.rec(local).first_pos;
            uint64_t cur = fp.load(std::memory_order_relaxed);
            while (pos < cur && !fp.compare_exchange_weak(cur, pos, std::memory_order_relaxed)) { }
        }
        return kMixed | (sh << kLocalBits) | local;
    }
};

// The mixture of a parent whose n existing children (handles ch[]) are not all equal: merge them with weight
// 1/N each (Eq. 4), reduce, hash-cons.  Returns the parent's handle (a leaf number if the merge is pure, else a
// table handle; 0 with table.failed set on failure) and adds the mixture's non-zeros to nnz.
uint32_t merge_children(Table& table, const uint32_t* ch, int n, uint32_t l, uint64_t voxel, std::vector<Entry>& buf,
                        std::vector<Entry>& merged, uint64_t& nnz)
{
    // common scale 2^tmax, each child weighs 1/N
    uint32_t tmax = 0;
    for (int q = 0; q < n; q++)
        if (ch[q] & kMixed) tmax = std::max(tmax, table.rec(ch[q]).tlog);
    buf.clear();
    for (int q = 0; q < n; q++) {
        if (ch[q] & kMixed) {
            const Rec& rc = table.rec(ch[q]);
            for (uint32_t t = 0; t < rc.k; t++)
                buf.push_back(Entry{rc.data[t].leaf, 0, rc.data[t].count << (tmax - rc.tlog)});
        } else {
            buf.push_back(Entry{ch[q], 0, 1ull << tmax});
        }
    }
    if (buf.size() <= 24) {
        for (size_t a = 1; a < buf.size(); a++) {
            Entry e = buf[a];
            size_t b = a;
            while (b > 0 && buf[b - 1].leaf > e.leaf) { buf[b] = buf[b - 1]; b--; }
            buf[b] = e;
        }
    } else {
        std::sort(buf.begin(), buf.end(), [](const Entry& a, const Entry& b) { return a.leaf < b.leaf; });
    }
    merged.clear();
    for (const Entry& e : buf) {
        if (!merged.empty() && merged.back().leaf == e.leaf) merged.back().count += e.count;
        else merged.push_back(e);
    }
    int tz = 64;
    for (const Entry& e : merged) tz = std::min(tz, __builtin_ctzll(e.count));
    for (Entry& e : merged) e.count >>= tz;
    const uint32_t nlog = (n == 8) ? 3 : (n == 4) ? 2 : (n == 2) ? 1 : 0;   // N is 1, 2, 4 or 8
    const uint32_t tlog = tmax + nlog - (uint32_t)tz;
    const uint64_t pos = ((uint64_t)l << 40) | voxel;
    nnz += merged.size();
    if (merged.size() == 1) return merged[0].leaf;
    return table.intern(merged.data(), (uint32_t)merged.size(), tlog, pos);
}

// Sorted distinct IDs present (every one becomes a leaf, background included: Q14) and ids0 = leaf number.
int index_leaves(const uint32_t* seg, uint64_t n, std::vector<uint32_t>& ids, std::vector<uint32_t>& ids0)
{
    uint32_t mx = 0;
#pragma omp parallel for reduction(max : mx) schedule(static)
    for (int64_t v = 0; v < (int64_t)n; v++) mx = std::max(mx, seg[v]);
    ids0.resize(n);
    if (mx < (1u << 28)) {
        std::vector<uint8_t> present((size_t)mx + 1, 0);
        uint8_t* pr = present.data();
#pragma omp parallel for schedule(static)
        for (int64_t v = 0; v < (int64_t)n; v++)
            if (!__atomic_load_n(&pr[seg[v]], __ATOMIC_RELAXED)) __atomic_store_n(&pr[seg[v]], (uint8_t)1, __ATOMIC_RELAXED);
        std::vector<uint32_t> leaf_of((size_t)mx + 1, 0);
        ids.clear();
        for (uint64_t i = 0; i <= mx; i++)
            if (present[i]) { leaf_of[i] = (uint32_t)ids.size(); ids.push_back((uint32_t)i); }
        const uint32_t* lo = leaf_of.data();
        uint32_t* o = ids0.data();
#pragma omp parallel for schedule(static)
        for (int64_t v = 0; v < (int64_t)n; v++) o[v] = lo[seg[v]];
    } else {   // sparse, huge IDs: collect per thread, merge, binary search
        std::vector<std::unordered_set<uint32_t>> sets(omp_get_max_threads());
#pragma omp parallel
        {
            std::unordered_set<uint32_t>& s = sets[omp_get_thread_num()];
            uint32_t last = ~seg[0];
#pragma omp for schedule(static)
            for (int64_t v = 0; v < (int64_t)n; v++)
                if (seg[v] != last) { last = seg[v]; s.insert(last); }
        }
        std::unordered_set<uint32_t> all;
        for (auto& s : sets) all.insert(s.begin(), s.end());
        ids.assign(all.begin(), all.end());
        std::sort(ids.begin(), ids.end());
        uint32_t* o = ids0.data();
#pragma omp parallel for schedule(static)
        for (int64_t v = 0; v < (int64_t)n; v++)
            o[v] = (uint32_t)(std::lower_bound(ids.begin(), ids.end(), seg[v]) - ids.begin());
    }
    return 0;
}

}  // namespace

int build_mipmap(const uint32_t* seg, uint64_t X, uint64_t Y, uint64_t Z, int n_threads, Mipmap& out, const Level1Front* front,
                 const LevelsFront* levels)
{
    if (n_threads > 0) omp_set_num_threads(n_threads);
    // ---- O-1 / L80: dims, ceil-halved down to 1^3
    out.dims.clear();
    for (uint64_t x = X, y = Y, z = Z;;) {
        out.dims.push_back(x); out.dims.push_back(y); out.dims.push_back(z);
        if (x == 1 && y == 1 && z == 1) break;
        x = (x + 1) / 2; y = (y + 1) / 2; z = (z + 1) / 2;
    }
    const uint32_t n_levels = (uint32_t)(out.dims.size() / 3);
    out.level_ids.assign(n_levels, {});
    if (levels) out.leaf_segment_id.assign(levels->leaf_segment_id, levels->leaf_segment_id + levels->n_leaves);
    else if (!front) index_leaves(seg, X * Y * Z, out.leaf_segment_id, out.level_ids[0]);   // level 0: H = e_S (Eq. 4, first line)
    else out.leaf_segment_id.assign(front->leaf_segment_id, front->leaf_segment_id + front->n_leaves);
    const uint32_t n_leaves = (uint32_t)out.leaf_segment_id.size();
    uint64_t nnz_total = X * Y * Z;

    Table table;
    uint32_t first_level = 1;
    if (front && n_levels > 1) {
        // Levels 0 and 1 were classified elsewhere (the device front end): level 0 stays with the caller, the pure
        // parents of level 1 already hold their leaf, the others come as a list of (voxel, existing children).
        const uint64_t n1 = out.dims[3] * out.dims[4] * out.dims[5];
        out.level_ids[1].assign(front->level1, front->level1 + n1);
        uint32_t* P = out.level_ids[1].data();
        uint64_t nnz_level = n1 - front->n_mixed, n_marked = 0;
#pragma omp parallel for reduction(+ : n_marked) schedule(static)
        for (int64_t v = 0; v < (int64_t)n1; v++) n_marked += (P[v] == 0xFFFFFFFFu);
        if (n_marked != front->n_mixed) {
            set_error("histogram mipmap: level 1 marks %llu parents as not pure, the list has %llu", (unsigned long long)n_marked,
                      (unsigned long long)front->n_mixed);
            return MGB_ERR_INVALID_ARG;
        }
        bool bad = false;
#pragma omp parallel reduction(+ : nnz_level) reduction(|| : bad)
        {
            std::vector<Entry> buf, merged;
#pragma omp for schedule(dynamic, 1024)
            for (int64_t q = 0; q < (int64_t)front->n_mixed; q++) {
                const uint64_t v = front->mixed_voxel[q];
                uint32_t ch[8];
                int n = 0;
                for (int t = 0; t < 8; t++) {
                    const uint32_t c = front->mixed_children[8 * q + t];
                    if (c != 0xFFFFFFFFu) ch[n++] = c;
                }
                bool ok = v < n1 && P[v] == 0xFFFFFFFFu && (n == 2 || n == 4 || n == 8);
                for (int t = 0; t < n; t++) ok = ok && ch[t] < n_leaves;
                if (!ok) { bad = true; continue; }
                P[v] = merge_children(table, ch, n, 1, v, buf, merged, nnz_level);
            }
        }
        if (bad) { set_error("histogram mipmap: inconsistent level-1 front end (voxel, child count or leaf out of range)"); return MGB_ERR_INVALID_ARG; }
        if (table.failed) { set_error("histogram mipmap: mixture table full or out of memory at level 1"); return MGB_ERR_LIMIT; }
        int64_t first_bad = -1;
#pragma omp parallel for schedule(static)
        for (int64_t v = 0; v < (int64_t)n1; v++)
            if (P[v] == 0xFFFFFFFFu || (!(P[v] & kMixed) && P[v] >= n_leaves)) {
#pragma omp critical
                if (first_bad < 0 || v < first_bad) first_bad = v;
            }
        if (first_bad >= 0) {
            set_error("histogram mipmap: level-1 voxel %lld is neither a leaf nor in the mixed list", (long long)first_bad);
            return MGB_ERR_INVALID_ARG;
        }
        nnz_total += nnz_level;
        first_level = 2;
    }
    std::vector<uint32_t> front_handle;                // LevelsFront: table handle of every listed mixture
    if (levels) {
        // Levels 1 .. level_done were built elsewhere (the device): take over the distinct mixtures found there, each
        // with its first occurrence, and the handles of the last finished level; continue above it.
        const uint32_t Ld = levels->level_done;
        if (Ld == 0 || Ld >= n_levels) { set_error("histogram mipmap: level_done = %u is not a level 1 .. %u", Ld, n_levels - 1); return MGB_ERR_INVALID_ARG; }
        front_handle.assign(levels->n_mix, 0);
        bool bad = false;
#pragma omp parallel reduction(|| : bad)
        {
            std::vector<Entry> e;
#pragma omp for schedule(dynamic, 1024)
            for (int64_t q = 0; q < (int64_t)levels->n_mix; q++) {
                const uint64_t o = levels->mix_offset[q];
                const uint32_t k = levels->mix_k[q];
                // the caller's arrays are checked before anything is sized or shifted by them
                bool ok = k >= 2 && k <= levels->n_entries && o <= levels->n_entries - k && levels->mix_tlog[q] < 64 &&
                          (levels->mix_first_pos[q] >> 40) >= 1 && (levels->mix_first_pos[q] >> 40) <= Ld;
                if (!ok) { bad = true; continue; }
                uint64_t total = 0;
                e.resize(k);
                for (uint32_t t = 0; ok && t < k; t++) {
                    e[t] = Entry{levels->leaf[o + t], 0, levels->count[o + t]};
                    ok = e[t].leaf < n_leaves && e[t].count > 0 && (t == 0 || e[t].leaf > e[t - 1].leaf) && total + e[t].count >= total;
                    total += e[t].count;
                }
                ok = ok && total == (1ull << levels->mix_tlog[q]);
                if (!ok) { bad = true; continue; }
                front_handle[q] = table.intern(e.data(), k, levels->mix_tlog[q], levels->mix_first_pos[q]);
            }
        }
        if (bad) { set_error("histogram mipmap: a listed mixture is malformed (entries, total or first occurrence)"); return MGB_ERR_INVALID_ARG; }
        if (table.failed) { set_error("histogram mipmap: mixture table full or out of memory while taking over the listed mixtures"); return MGB_ERR_LIMIT; }
        const uint64_t nd = out.dims[3 * Ld] * out.dims[3 * Ld + 1] * out.dims[3 * Ld + 2];
        out.level_ids[Ld].resize(nd);
        uint32_t* P = out.level_ids[Ld].data();
        bool bad_handle = false;
#pragma omp parallel for schedule(static) reduction(|| : bad_handle)
        for (int64_t v = 0; v < (int64_t)nd; v++) {
            const uint32_t h = levels->handles[v];
            if (h & kMixed) {
                const uint32_t q = h & ~kMixed;
                if (q >= levels->n_mix) { bad_handle = true; continue; }
                P[v] = front_handle[q];
            } else {
                if (h >= n_leaves) { bad_handle = true; continue; }
                P[v] = h;
            }
        }
        if (bad_handle) { set_error("histogram mipmap: a handle of level %u names no leaf and no listed mixture", Ld); return MGB_ERR_INVALID_ARG; }
        nnz_total += levels->nnz_levels;
        first_level = Ld + 1;
    }
    for (uint32_t l = first_level; l < n_levels; l++) {
        const uint64_t cx = out.dims[3 * l - 3], cy = out.dims[3 * l - 2], cz = out.dims[3 * l - 1];
        const uint64_t px = out.dims[3 * l], py = out.dims[3 * l + 1], pz = out.dims[3 * l + 2];
        out.level_ids[l].resize(px * py * pz);
        const uint32_t* C = out.level_ids[l - 1].data();
        uint32_t* P = out.level_ids[l].data();
        uint64_t nnz_level = 0;
#pragma omp parallel reduction(+ : nnz_level)
        {
            std::vector<Entry> buf, merged;
#pragma omp for schedule(dynamic, 8)
            for (int64_t r = 0; r < (int64_t)(pz * py); r++) {
                const uint64_t k = (uint64_t)r / py, j = (uint64_t)r % py;
                const uint32_t* rows[4];
                int n_rows = 0;
                for (uint64_t w = 2 * k; w <= 2 * k + 1 && w < cz; w++)
                    for (uint64_t v = 2 * j; v <= 2 * j + 1 && v < cy; v++) rows[n_rows++] = C + (w * cy + v) * cx;
                for (uint64_t i = 0; i < px; i++) {
                    const uint64_t x0 = 2 * i;
                    const int nx = (x0 + 1 < cx) ? 2 : 1;
                    uint32_t ch[8] = {0, 0, 0, 0, 0, 0, 0, 0};
                    int n = 0;
                    for (int q = 0; q < n_rows; q++) {
                        ch[n++] = rows[q][x0];
                        if (nx == 2) ch[n++] = rows[q][x0 + 1];
                    }
                    bool same = true;
                    for (int q = 1; q < n; q++) same &= (ch[q] == ch[0]);
                    if (same) {   // the average of identical mixtures is that mixture
                        P[(uint64_t)r * px + i] = ch[0];
                        nnz_level += (ch[0] & kMixed) ? table.rec(ch[0]).k : 1;
                        continue;
                    }
                    P[(uint64_t)r * px + i] = merge_children(table, ch, n, l, (uint64_t)r * px + i, buf, merged, nnz_level);
                }
            }
        }
        if (table.failed) { set_error("histogram mipmap: mixture table full or out of memory at level %u", l); return MGB_ERR_LIMIT; }
        nnz_total += nnz_level;
    }
    out.nnz_total = nnz_total;

    // ---- canonical numbering: by first occurrence in (level, z, y, x) order
    struct Key { uint64_t pos; uint32_t handle; };
    std::vector<Key> keys;
    for (uint32_t s = 0; s < kShards; s++)
        for (uint32_t q = 0; q < table.shards[s].n_recs; q++)
            keys.push_back(Key{table.shards[s].rec(q).first_pos.load(), kMixed | (s << kLocalBits) | q});
    std::sort(keys.begin(), keys.end(), [](const Key& a, const Key& b) { return a.pos < b.pos; });
    const uint64_t M = keys.size();
    if ((uint64_t)n_leaves + M >= kMixed) { set_error("too many distinct mixtures (%llu)", (unsigned long long)M); return MGB_ERR_LIMIT; }
    std::vector<std::vector<uint32_t>> canon(kShards);
    for (uint32_t s = 0; s < kShards; s++) canon[s].resize(table.shards[s].n_recs);
    MixtureSet& ms = out.mixtures;
    ms.n_leaves = n_leaves;
    ms.off.assign(M + 1, 0);
    for (uint64_t q = 0; q < M; q++) {
        const uint32_t h = keys[q].handle;
        canon[(h >> kLocalBits) & (kShards - 1)][h & ((1u << kLocalBits) - 1)] = (uint32_t)q;
        ms.off[q + 1] = ms.off[q] + table.rec(h).k;
    }
    ms.leaf.resize(ms.off[M]);
    ms.count.resize(ms.off[M]);
#pragma omp parallel for schedule(dynamic, 1024)
    for (int64_t q = 0; q < (int64_t)M; q++) {
        const Rec& rc = table.rec(keys[q].handle);
        for (uint32_t t = 0; t < rc.k; t++) {
            ms.leaf[ms.off[q] + t] = rc.data[t].leaf;
            ms.count[ms.off[q] + t] = rc.data[t].count;
        }
    }
    if (levels) {
        out.front_mixture.resize(levels->n_mix);
        for (uint64_t q = 0; q < levels->n_mix; q++) {
            const uint32_t h = front_handle[q];
            out.front_mixture[q] = canon[(h >> kLocalBits) & (kShards - 1)][h & ((1u << kLocalBits) - 1)];
        }
    }
    for (uint32_t l = 1; l < n_levels; l++) {
        uint32_t* P = out.level_ids[l].data();
        const int64_t nv = (int64_t)out.level_ids[l].size();
#pragma omp parallel for schedule(static)
        for (int64_t v = 0; v < nv; v++) {
            const uint32_t h = P[v];
            if (h & kMixed) P[v] = n_leaves + canon[(h >> kLocalBits) & (kShards - 1)][h & ((1u << kLocalBits) - 1)];
        }
    }
    return MGB_OK;
}

}  // namespace mgb
