// factorise.cpp -- a1: factorisation of the distinct mixtures into binary lerps with node re-use.
//
//   lambda = (m_i e_i + m_j e_j) / (m_i + m_j)   and   m <- m - m_i e_i - m_j e_j + (m_i + m_j) e_lambda
//   (Eq. 5-7; Eq. 5's denominator read as m_i + m_j, Q3; worked example Fig. 2).
//   A node is the triple (i, j, w) = (1 - w) s_i + w s_j (L259); identical triples are ONE node
//   ("prune-and-recycle", L29, L130, L144, Fig. 4).  Canonical orientation here: i < j and
//   w = m_j / (m_i + m_j), so the node key is (i, j, bin(w)) (quantised, L176) or (i, j, m_i : m_j reduced)
//   (unquantised: only exactly equal ratios merge).
//
// Schedule (L257): stage 1 = greedy max-reduction phi_2 (Eq. 13-14) over the mixtures with
// tau < ||m||_0 <= big_cutoff: score(i,j) = sum over pool mixtures containing i and j of (||m||_0 - 1),
// take the arg max (ties: lexicographically smallest (i,j), Q6), factor ALL its occurrences, repeat until
// every pool mixture has dropped to <= tau non-zeros.  Stage 2 = every mixture in scanline order, finished
// by pairing in rounds (smallest node numbers first: a balanced tournament, depth ceil(log2 k)) or, with
// MGB_PICK_SMALLEST_MASS, the two smallest masses (the order Fig. 2 shows).
// Relaxations (L319 anticipates "faster heuristics"; any factorisation is valid, L144): mixtures above
// big_cutoff skip stage 1, and when the exact score maintenance would cost more than phi2_exact_budget
// updates the norms in phi_2 are frozen at their initial values (updates drop from O(k^2) to O(k)).
#include <algorithm>
#include <cmath>
#include <numeric>
#include <queue>

#include "builder_internal.h"

namespace mgb {
namespace {

struct WE {
    uint32_t node;
    uint64_t mass;
};

inline uint64_t hash3(uint64_t a, uint64_t b, uint64_t c)
{
    uint64_t h = a * 0x9E3779B97F4A7C15ull;
    h ^= h >> 32;
    h = (h + b) * 0xff51afd7ed558ccdull;
    h ^= h >> 29;
    h = (h + c) * 0xc4ceb9fe1a85ec53ull;
    return h ^ (h >> 32);
}

// (child lo, child hi, ratio key) -> node
struct NodeTable {
    Factorised& F;
    const uint32_t n_leaves;
    const uint32_t qbits;                 // 0 = unquantised
    std::vector<uint64_t> r1, r2;         // ratio key per internal node: (bin, 0) or reduced (m_lo, m_hi)
    std::vector<uint32_t> slot;           // node - n_leaves + 1, 0 = empty
    uint64_t mask;

    NodeTable(Factorised& f, uint32_t nl, uint32_t qb) : F(f), n_leaves(nl), qbits(qb), slot(1u << 16, 0), mask((1u << 16) - 1) {}

    void grow()
    {
        std::vector<uint32_t> ns((mask + 1) * 2, 0);
        const uint64_t nm = ns.size() - 1;
        for (uint32_t s : slot)
            if (s) {
                const uint32_t q = s - 1;
                uint64_t i = hash3(((uint64_t)F.a[q] << 32) | F.b[q], r1[q], r2[q]) & nm;
                while (ns[i]) i = (i + 1) & nm;
                ns[i] = s;
            }
        slot.swap(ns);
        mask = nm;
    }

    // Combine entries (i, mi) and (j, mj) of one mixture: returns the node (1 - w) s_lo + w s_hi.
    uint32_t combine(uint32_t i, uint64_t mi, uint32_t j, uint64_t mj)
    {
        const uint32_t lo = std::min(i, j), hi = std::max(i, j);
        const uint64_t mlo = (i < j) ? mi : mj, mhi = (i < j) ? mj : mi;
        uint64_t k1, k2;
        if (qbits) { k1 = (mhi << qbits) / (mlo + mhi); k2 = 0; }   // floor(w 2^b), exact; w < 1 so k1 < 2^b
        else { const uint64_t g = std::gcd(mlo, mhi); k1 = mlo / g; k2 = mhi / g; }
        const double w = (double)mhi / (double)(mlo + mhi);
        const uint64_t pk = ((uint64_t)lo << 32) | hi;
        uint64_t s = hash3(pk, k1, k2) & mask;
        while (slot[s]) {
            const uint32_t q = slot[s] - 1;
            if (F.a[q] == lo && F.b[q] == hi && r1[q] == k1 && r2[q] == k2) {
                F.w_sum[q] += w;
                F.w_sq[q] += w * w;
                F.w_cnt[q]++;
                return n_leaves + q;
            }
            s = (s + 1) & mask;
        }
        const uint32_t q = (uint32_t)F.a.size();
        F.a.push_back(lo); F.b.push_back(hi); F.bin.push_back((uint32_t)(qbits ? k1 : 0));
        F.w_sum.push_back(w); F.w_sq.push_back(w * w); F.w_cnt.push_back(1);
        r1.push_back(k1); r2.push_back(k2);
        slot[s] = q + 1;
        if ((uint64_t)F.a.size() * 10 > (mask + 1) * 6) grow();
        return n_leaves + q;
    }
};

// e is sorted by node; insert (node, mass), merging with an equal node.
inline void insert_sorted(std::vector<WE>& e, uint32_t node, uint64_t mass)
{
    size_t p = 0;
    while (p < e.size() && e[p].node < node) p++;
    if (p < e.size() && e[p].node == node) e[p].mass += mass;
    else e.insert(e.begin() + p, WE{node, mass});
}

// Stage 2: finish one mixture.  Returns the node that represents it.
uint32_t finish(std::vector<WE>& e, NodeTable& T, uint32_t pick_order, std::vector<WE>& next)
{
    if (pick_order == MGB_PICK_SMALLEST_MASS) {
        while (e.size() > 1) {
            size_t x = 0, y = 1;
            if (e[y].mass < e[x].mass) std::swap(x, y);                // x = smallest, y = second smallest
            for (size_t q = 2; q < e.size(); q++) {
                if (e[q].mass < e[x].mass) { y = x; x = q; }
                else if (e[q].mass < e[y].mass) y = q;
            }
            const WE ex = e[x], ey = e[y];
            const uint32_t n = T.combine(ex.node, ex.mass, ey.node, ey.mass);
            e.erase(e.begin() + std::max(x, y));
            e.erase(e.begin() + std::min(x, y));
            insert_sorted(e, n, ex.mass + ey.mass);
        }
        return e[0].node;
    }
    // rounds: (e0,e1), (e2,e3), ...; an odd last entry is carried to the front of the next round
    while (e.size() > 1) {
        next.clear();
        if (e.size() & 1) next.push_back(e.back());
        for (size_t q = 0; q + 1 < e.size(); q += 2) {
            const uint32_t n = T.combine(e[q].node, e[q].mass, e[q + 1].node, e[q + 1].mass);
            const uint64_t m = e[q].mass + e[q + 1].mass;
            bool dup = false;
            for (WE& w : next)
                if (w.node == n) { w.mass += m; dup = true; break; }     // a re-used node may already be there
            if (!dup) next.push_back(WE{n, m});
        }
        e.swap(next);
    }
    return e[0].node;
}

struct PairMap {   // pair key (i << 32 | j, i < j, never 0) -> score
    std::vector<uint64_t> key;
    std::vector<int64_t> val;
    uint64_t mask, n = 0;
    PairMap() : key(1u << 16, 0), val(1u << 16, 0), mask((1u << 16) - 1) {}
    static uint64_t h(uint64_t k) { k *= 0x9E3779B97F4A7C15ull; return k ^ (k >> 29); }
    int64_t& ref(uint64_t k)
    {
        if ((n + 1) * 10 > (mask + 1) * 6) {
            std::vector<uint64_t> nk((mask + 1) * 2, 0);
            std::vector<int64_t> nv((mask + 1) * 2, 0);
            const uint64_t nm = nk.size() - 1;
            for (uint64_t s = 0; s <= mask; s++)
                if (key[s]) {
                    uint64_t i = h(key[s]) & nm;
                    while (nk[i]) i = (i + 1) & nm;
                    nk[i] = key[s]; nv[i] = val[s];
                }
            key.swap(nk); val.swap(nv); mask = nm;
        }
        uint64_t i = h(k) & mask;
        while (key[i] && key[i] != k) i = (i + 1) & mask;
        if (!key[i]) { key[i] = k; n++; }
        return val[i];
    }
    int64_t get(uint64_t k) const
    {
        uint64_t i = h(k) & mask;
        while (key[i] && key[i] != k) i = (i + 1) & mask;
        return key[i] ? val[i] : 0;
    }
};

// Eq. 13 (L164): a mixture with ||h||_0 non-zeros contributes ||h||_0 - 1 to phi_2, "or 2 when ||h||_0 = 2".
inline int64_t norm_gain(uint64_t k) { return k == 2 ? 2 : (int64_t)k - 1; }

inline uint64_t pkey(uint32_t x, uint32_t y) { return x < y ? ((uint64_t)x << 32) | y : ((uint64_t)y << 32) | x; }

}  // namespace

int factorise(const MixtureSet& ms, const mgb_params& p, Factorised& F)
{
    const uint64_t M = ms.size();
    const uint32_t n_leaves = ms.n_leaves;
    const uint32_t tau = std::max(p.tau, 1u);   // a mixture with one non-zero is finished
    F = Factorised();
    F.node_of_mix.assign(M, 0);
    NodeTable T(F, n_leaves, p.quant_bits);

    // ---- stage 1 pool: tau < k <= big_cutoff
    struct PM {
        std::vector<WE> e;   // sorted by node
        uint32_t mix;
        int64_t g;           // the weight of this mixture in phi_2: ||m||_0 - 1 (frozen at the initial value if !exact)
        bool active;
    };
    std::vector<PM> pool;
    std::vector<int64_t> pool_of_mix;   // -1 = not in the pool
    double cost = 0;
    for (uint64_t q = 0; q < M; q++) {
        const uint64_t k = ms.off[q + 1] - ms.off[q];
        if (k > tau && (p.big_cutoff == 0 || k <= p.big_cutoff)) cost += (double)k * k * k / 6.0 + (double)k * k;
        else if (k > tau) F.n_big++;
    }
    const bool exact = cost <= (double)p.phi2_exact_budget;
    F.phi2_exact = exact;
    pool_of_mix.assign(M, -1);
    for (uint64_t q = 0; q < M; q++) {
        const uint64_t k = ms.off[q + 1] - ms.off[q];
        if (k > tau && (p.big_cutoff == 0 || k <= p.big_cutoff)) {
            PM m;
            m.mix = (uint32_t)q; m.g = norm_gain(k); m.active = true;
            for (uint64_t t = ms.off[q]; t < ms.off[q + 1]; t++) m.e.push_back(WE{ms.leaf[t], ms.count[t]});
            pool_of_mix[q] = (int64_t)pool.size();
            pool.push_back(std::move(m));
        }
    }
    F.n_stage1 = pool.size();
    F.n_stage2 = M - F.n_stage1 - F.n_big;

    if (!pool.empty()) {
        PairMap S;
        std::vector<std::vector<uint32_t>> occ(n_leaves);       // node -> pool mixtures it entered
        using HE = std::pair<int64_t, uint64_t>;                // (score, ~key): max score, then smallest key
        std::priority_queue<HE> heap;
        for (uint32_t m = 0; m < pool.size(); m++) {
            const std::vector<WE>& e = pool[m].e;
            for (size_t x = 0; x < e.size(); x++) {
                occ[e[x].node].push_back(m);
                for (size_t y = x + 1; y < e.size(); y++) S.ref(pkey(e[x].node, e[y].node)) += pool[m].g;
            }
        }
        for (uint64_t s = 0; s <= S.mask; s++)
            if (S.key[s]) heap.push(HE{S.val[s], ~S.key[s]});
        uint64_t n_active = pool.size();
        while (n_active && !heap.empty()) {
            const HE top = heap.top();
            heap.pop();
            const uint64_t key = ~top.second;
            const int64_t cur = S.get(key);
            if (cur != top.first) {            // stale entry: scores only ever drop lazily
                if (cur > 0) heap.push(HE{cur, top.second});
                continue;
            }
            if (cur <= 0) continue;
            const uint32_t i = (uint32_t)(key >> 32), j = (uint32_t)key;
            const uint32_t src = occ[i].size() <= occ[j].size() ? i : j;
            for (size_t oq = 0; oq < occ[src].size(); oq++) {      // factor ALL occurrences (Eq. 14)
                const uint32_t m = occ[src][oq];
                PM& pm = pool[m];
                if (!pm.active) continue;
                std::vector<WE>& e = pm.e;
                size_t xi = e.size(), xj = e.size();
                for (size_t x = 0; x < e.size(); x++) {
                    if (e[x].node == i) xi = x;
                    else if (e[x].node == j) xj = x;
                }
                if (xi == e.size() || xj == e.size()) continue;
                const int64_t g_old = pm.g;
                if (exact) {
                    for (size_t x = 0; x < e.size(); x++)
                        for (size_t y = x + 1; y < e.size(); y++) S.ref(pkey(e[x].node, e[y].node)) -= g_old;
                } else {
                    for (size_t x = 0; x < e.size(); x++)
                        if (x != xi && x != xj) { S.ref(pkey(i, e[x].node)) -= g_old; S.ref(pkey(j, e[x].node)) -= g_old; }
                    S.ref(key) -= g_old;
                }
                const uint64_t mi = e[xi].mass, mj = e[xj].mass;
                const uint32_t nn = T.combine(i, mi, j, mj);
                e.erase(e.begin() + std::max(xi, xj));
                e.erase(e.begin() + std::min(xi, xj));
                const size_t before = e.size();
                insert_sorted(e, nn, mi + mj);
                const bool fresh = e.size() > before;              // false: nn was already an entry, masses merged
                if (e.size() > tau) {
                    const int64_t g_new = exact ? norm_gain(e.size()) : g_old;
                    pm.g = g_new;
                    if (exact) {
                        for (size_t x = 0; x < e.size(); x++)
                            for (size_t y = x + 1; y < e.size(); y++) {
                                const uint64_t k2 = pkey(e[x].node, e[y].node);
                                int64_t& v = S.ref(k2);
                                v += g_new;
                                if (e[x].node == nn || e[y].node == nn) heap.push(HE{v, ~k2});
                            }
                    } else if (fresh) {
                        for (size_t x = 0; x < e.size(); x++)
                            if (e[x].node != nn) {
                                const uint64_t k2 = pkey(nn, e[x].node);
                                int64_t& v = S.ref(k2);
                                v += g_new;
                                heap.push(HE{v, ~k2});
                            }
                    }
                    if (fresh) {
                        if (occ.size() <= nn) occ.resize((size_t)nn + 1);
                        occ[nn].push_back(m);
                    }
                } else {                                           // leaves the pool; stage 2 finishes it
                    if (!exact)   // frozen norms: withdraw the pairs this mixture still contributes (a fresh nn never did)
                        for (size_t x = 0; x < e.size(); x++)
                            for (size_t y = x + 1; y < e.size(); y++)
                                if (!(fresh && (e[x].node == nn || e[y].node == nn))) S.ref(pkey(e[x].node, e[y].node)) -= g_old;
                    pm.active = false;
                    n_active--;
                }
            }
        }
        if (n_active) { set_error("factorise: stage 1 stalled with %llu active mixtures", (unsigned long long)n_active); return MGB_ERR_LIMIT; }
    }

    // ---- stage 2: every mixture, scanline order
    std::vector<WE> e, next;
    for (uint64_t q = 0; q < M; q++) {
        if (pool_of_mix[q] >= 0) {
            e = pool[pool_of_mix[q]].e;
        } else {
            e.clear();
            for (uint64_t t = ms.off[q]; t < ms.off[q + 1]; t++) e.push_back(WE{ms.leaf[t], ms.count[t]});
        }
        F.node_of_mix[q] = finish(e, T, p.pick_order, next);
        if ((uint64_t)n_leaves + F.a.size() >= 0xFFFFFFF0ull) { set_error("factorise: more than 2^32 nodes"); return MGB_ERR_LIMIT; }
    }
    return MGB_OK;
}

}  // namespace mgb
