// mg_mixtures.cu -- NEXT-4 (second half, continued): the levels >= 1 of the histogram mipmap on the device.
//
//   H(i,j,k,l) = (1/N) sum over the EXISTING children of H(.,.,.,l-1)            (Eq. 4; reading Q2)
//
// What the host builder does per level (csrc/builder/mipmap.cpp) restated for the GPU: a parent whose existing
// children carry one and the same mixture inherits it; every other parent MERGES its children's sparse integer
// mixtures (sorted (leaf, count) lists on a common power-of-two scale, each child weighing 1/N), divides by the common
// power of two and HASH-CONSES the result, so that only distinct mixtures reach the factoriser (L88-L98).  Per level:
//   k_classify   one thread per parent: gather the <= 8 child handles; all equal -> inherit, else append to a list
//                (level 1, 98 % of the parents: the streaming classifier of mg_mipmap_front_level1, which lists the
//                parents together with their <= 8 leaves, and k_merge_leaves, one THREAD per listed parent)
//   k_merge      one warp per listed parent: rank-merge the children's sorted lists in shared memory, combine equal
//                leaves, reduce, hash (64 bit), park the result in a per-level scratch arena
//   k_claim      find-or-claim the hash in an open-addressing table; atomicMin of the parent's position
//                (level << 40 | voxel) on the slot: the minimum is the mixture's first occurrence in scanline order
//                (L257), which is what the host's canonical numbering sorts by -- and it elects ONE writer per new mixture
//   k_publish    the elected parent appends its entries to the mixture store and publishes the mixture's number
//   k_resolve    every listed parent compares its entries with the stored ones (a 64-bit collision is reported, not
//                ignored) and writes its handle
// A handle is a leaf number (< 2^31) or 0x80000000 | mixture number.  A level with a parent whose children total more
// than kMaxMerge entries is left to the host (mgb_build_from_levels continues from the last finished level): those are
// the few thousand voxels of the top levels, where one mixture holds hundreds of segments.
#include <algorithm>
#include <new>
#include <vector>

#include "mg_internal.h"

struct mg_mixture_table {
    int device = 0;
    uint32_t n_leaves = 0;
    uint64_t cap_m = 0, cap_e = 0, cap_h = 0;
    uint64_t* d_off = nullptr;     // [cap_m] first entry of the mixture
    uint32_t* d_k = nullptr;       // [cap_m] non-zeros
    uint32_t* d_tlog = nullptr;    // [cap_m] the reduced counts sum to 2^tlog
    uint64_t* d_first = nullptr;   // [cap_m] first occurrence (level << 40 | voxel)
    uint32_t* d_leaf = nullptr;    // [cap_e]
    uint64_t* d_cnt = nullptr;     // [cap_e]
    uint64_t* d_hash = nullptr;    // [cap_h] 0 = empty
    uint64_t* d_hfirst = nullptr;  // [cap_h]
    uint32_t* d_hid = nullptr;     // [cap_h] mixture number, kNoId until published
    unsigned long long* d_ctr = nullptr;   // see Ctr
    uint64_t n_mix = 0, n_ent = 0;
    uint32_t levels_done = 0;
    uint64_t nnz_levels = 0;       // non-zeros summed over all voxels of the finished levels 1 .. levels_done
    uint64_t device_bytes = 0;
};

namespace {

constexpr int kThreads = 256;
constexpr int kMergeWarps = 4;               // warps per k_merge CTA
constexpr int kMaxMerge = 256;               // entries of all children of one parent that a warp merges in shared memory
constexpr uint32_t kNone = 0xFFFFFFFFu, kMixed = 0x80000000u, kNoId = 0xFFFFFFFFu;
enum Ctr { kNMix = 0, kNEnt, kNPending, kScratch, kFlags, kNnz, kNCtr };
enum Flag : unsigned long long { kTooBig = 1, kScratchFull = 2, kStoreFull = 4, kTableFull = 8, kCollision = 16 };

struct LevelGeom {
    uint32_t cx, cy, cz;     // children's level
    uint32_t px, py, pz;     // parents' level
    uint32_t level;
};

__device__ __forceinline__ uint64_t mix64(uint64_t x)
{
    x ^= x >> 33; x *= 0xff51afd7ed558ccdull;
    x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ull;
    return x ^ (x >> 33);
}

// The <= 8 existing children of parent v, kNone for a missing one; returns their number N (1, 2, 4 or 8).
__device__ __forceinline__ int load_children(const uint32_t* __restrict__ C, const LevelGeom& G, uint32_t v, uint32_t* ch)
{
    const uint32_t row = v / G.px, i = v - row * G.px, k = row / G.py, j = row - k * G.py;
    int n = 0;
#pragma unroll
    for (int t = 0; t < 8; t++) {
        const uint32_t x = 2 * i + (t & 1), y = 2 * j + ((t >> 1) & 1), z = 2 * k + (t >> 2);
        const bool ex = x < G.cx && y < G.cy && z < G.cz;
        ch[t] = ex ? __ldg(C + ((uint64_t)z * G.cy + y) * G.cx + x) : kNone;
        n += ex;
    }
    return n;
}

__global__ void __launch_bounds__(kThreads)
k_classify(const uint32_t* __restrict__ C, const LevelGeom G, uint32_t n_par, uint32_t* __restrict__ P, uint32_t* __restrict__ list,
           uint32_t list_cap, const uint32_t* __restrict__ mix_k, unsigned long long* ctr)
{
    const uint32_t v = blockIdx.x * kThreads + threadIdx.x;
    bool pend = false;
    unsigned nnz = 0;
    if (v < n_par) {
        uint32_t ch[8];
        load_children(C, G, v, ch);
        bool same = true;
#pragma unroll
        for (int t = 1; t < 8; t++) same = same && (ch[t] == ch[0] || ch[t] == kNone);   // child 0 always exists
        P[v] = same ? ch[0] : kNone;                                  // the average of identical mixtures is that mixture
        pend = !same;
        if (same) nnz = (ch[0] & kMixed) ? __ldg(mix_k + (ch[0] & ~kMixed)) : 1u;
    }
    const unsigned m = __ballot_sync(0xffffffffu, pend);
    const unsigned lane = threadIdx.x & 31;
    const unsigned tot = __reduce_add_sync(0xffffffffu, nnz);
    unsigned long long base = 0;
    if (lane == 0) {
        if (m) base = atomicAdd(ctr + kNPending, (unsigned long long)__popc(m));
        if (tot) atomicAdd(ctr + kNnz, (unsigned long long)tot);
    }
    base = __shfl_sync(0xffffffffu, base, 0);
    if (pend) {
        const unsigned long long at = base + __popc(m & ((1u << lane) - 1u));
        if (at < list_cap) list[at] = v;
    }
}

// Per listed parent after the merge: where its entries are parked and what they hash to.
struct Pending {
    uint32_t* voxel;       // [n] (the list of k_classify)
    uint64_t* off;         // [n] first entry in the scratch arena
    uint32_t* k;           // [n] non-zeros (0: nothing to intern -- the level is abandoned, or the merge came out pure)
    uint32_t* tlog;        // [n]
    uint64_t* hash;        // [n]
    uint64_t* slot;        // [n] slot of the hash table (k_claim)
};

// One warp per listed parent.  Shared memory per warp: the children's entries in child order (A), then sorted by leaf (B),
// then the combined entries (A again).
__global__ void __launch_bounds__(kMergeWarps * 32)
k_merge(const uint32_t* __restrict__ C, const LevelGeom G, uint32_t* __restrict__ P, const Pending Q, uint32_t n_pending,
        const uint64_t* __restrict__ mix_off, const uint32_t* __restrict__ mix_k, const uint32_t* __restrict__ mix_tlog,
        const uint32_t* __restrict__ ent_leaf, const uint64_t* __restrict__ ent_cnt, uint32_t* __restrict__ s_leaf,
        uint64_t* __restrict__ s_cnt, uint64_t scratch_cap, unsigned long long* ctr)
{
    __shared__ uint32_t leafA[kMergeWarps][kMaxMerge], leafB[kMergeWarps][kMaxMerge];
    __shared__ uint64_t cntA[kMergeWarps][kMaxMerge], cntB[kMergeWarps][kMaxMerge];
    const unsigned lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t q = blockIdx.x * kMergeWarps + w;
    if (q >= n_pending) return;                                       // (whole warps leave together)
    const uint32_t v = Q.voxel[q];
    // lane t < 8 looks at child t
    uint32_t ch[8];
    const int n_ch = load_children(C, G, v, ch);
    uint32_t my = kNone;
#pragma unroll
    for (int t = 0; t < 8; t++)
        if (lane == (unsigned)t) my = ch[t];
    uint32_t my_k = 0, my_tlog = 0;
    uint64_t my_off = 0;
    if (my != kNone) {
        if (my & kMixed) { const uint32_t id = my & ~kMixed; my_k = __ldg(mix_k + id); my_tlog = __ldg(mix_tlog + id); my_off = __ldg(mix_off + id); }
        else my_k = 1;
    }
    const uint32_t tmax = __reduce_max_sync(0xffffffffu, my_tlog);
    const uint32_t total = __reduce_add_sync(0xffffffffu, my_k);
    if (total > (uint32_t)kMaxMerge) {                                 // left to the host: the level is abandoned
        if (lane == 0) { atomicOr(ctr + kFlags, (unsigned long long)kTooBig); Q.k[q] = 0; }
        return;
    }
    uint32_t cbase[8], ck[8];                                         // every lane knows every child's range
    {
        uint32_t run = 0;
#pragma unroll
        for (int t = 0; t < 8; t++) {
            ck[t] = __shfl_sync(0xffffffffu, my_k, t);
            cbase[t] = run;
            run += ck[t];
        }
    }
    // gather the children's entries on the common scale 2^tmax (each child weighs 1/N)
#pragma unroll
    for (int t = 0; t < 8; t++) {
        const uint32_t h = __shfl_sync(0xffffffffu, my, t), tl = __shfl_sync(0xffffffffu, my_tlog, t);
        const uint64_t off = __shfl_sync(0xffffffffu, my_off, t);
        if (ck[t] == 0) continue;
        if (!(h & kMixed)) {
            if (lane == 0) { leafA[w][cbase[t]] = h; cntA[w][cbase[t]] = 1ull << tmax; }
        } else {
            for (uint32_t e = lane; e < ck[t]; e += 32) {
                leafA[w][cbase[t] + e] = __ldg(ent_leaf + off + e);
                cntA[w][cbase[t] + e] = __ldg(ent_cnt + off + e) << (tmax - tl);
            }
        }
    }
    __syncwarp();
    // rank merge: element e of child c goes to (its index in c) + (elements of the other children before it)
    for (uint32_t e = lane; e < total; e += 32) {
        int c = 0;
#pragma unroll
        for (int t = 1; t < 8; t++)
            if (ck[t] && e >= cbase[t]) c = t;
        const uint32_t lf = leafA[w][e];
        uint32_t rank = e - cbase[c];
#pragma unroll
        for (int t = 0; t < 8; t++) {
            if (t == c || ck[t] == 0) continue;
            uint32_t lo = 0, hi = ck[t];                              // number of elements of child t that sort before lf
            while (lo < hi) {
                const uint32_t mid = (lo + hi) >> 1;
                const uint32_t x = leafA[w][cbase[t] + mid];
                if (x < lf || (x == lf && t < c)) lo = mid + 1; else hi = mid;
            }
            rank += lo;
        }
        leafB[w][rank] = lf;
        cntB[w][rank] = cntA[w][e];
    }
    __syncwarp();
    // combine equal leaves (at most one per child, adjacent after the sort)
    uint32_t kk = 0;
    for (uint32_t j0 = 0; j0 < total; j0 += 32) {
        const uint32_t j = j0 + lane;
        const bool head = j < total && (j == 0 || leafB[w][j] != leafB[w][j - 1]);
        uint64_t sum = 0;
        if (head)
            for (uint32_t r = j; r < total && leafB[w][r] == leafB[w][j]; r++) sum += cntB[w][r];
        const unsigned hm = __ballot_sync(0xffffffffu, head);
        if (head) {
            const uint32_t o = kk + __popc(hm & ((1u << lane) - 1u));
            leafA[w][o] = leafB[w][j];
            cntA[w][o] = sum;
        }
        kk += __popc(hm);
    }
    __syncwarp();
    // reduce by the common power of two, hash
    int tz = 64;
    for (uint32_t j = lane; j < kk; j += 32) tz = min(tz, __ffsll((long long)cntA[w][j]) - 1);
    tz = __reduce_min_sync(0xffffffffu, tz);
    uint64_t h = 0;
    for (uint32_t j = lane; j < kk; j += 32) {
        const uint64_t c = cntA[w][j] >> tz;
        cntA[w][j] = c;
        h += mix64((((uint64_t)leafA[w][j] << 32) | (j + 1)) * 0x9E3779B97F4A7C15ull + c);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) h += __shfl_xor_sync(0xffffffffu, h, d);
    h = mix64(h ^ kk);
    if (h == 0) h = 1;
    const uint32_t nlog = (n_ch == 8) ? 3u : (n_ch == 4) ? 2u : (n_ch == 2) ? 1u : 0u;
    __syncwarp();
    if (kk == 1) {                                                     // (cannot happen for hash-consed children; kept exact anyway)
        if (lane == 0) { P[v] = leafA[w][0]; Q.k[q] = 0; atomicAdd(ctr + kNnz, 1ull); }
        return;
    }
    unsigned long long so = 0;
    if (lane == 0) {
        so = atomicAdd(ctr + kScratch, (unsigned long long)kk);
        atomicAdd(ctr + kNnz, (unsigned long long)kk);
    }
    so = __shfl_sync(0xffffffffu, so, 0);
    if (so + kk > scratch_cap) {
        if (lane == 0) { atomicOr(ctr + kFlags, (unsigned long long)kScratchFull); Q.k[q] = 0; }
        return;
    }
    for (uint32_t j = lane; j < kk; j += 32) { s_leaf[so + j] = leafA[w][j]; s_cnt[so + j] = cntA[w][j]; }
    if (lane == 0) { Q.off[q] = so; Q.k[q] = kk; Q.tlog[q] = tmax + nlog - (uint32_t)tz; Q.hash[q] = h; }
}

// Level 1: the children are leaves, at most 8 of them -- one THREAD per listed parent sorts them in registers, run-length
// encodes, reduces and hashes (same hash as k_merge); scratch space comes from one warp-aggregated atomic.
// children: [n][8] leaf numbers, kNone for a child outside the volume (the list of mg_mipmap_front_level1).
__global__ void __launch_bounds__(kThreads)
k_merge_leaves(const uint32_t* __restrict__ children, const Pending Q, uint32_t n_pending, uint32_t* __restrict__ s_leaf,
               uint64_t* __restrict__ s_cnt, unsigned long long* ctr)
{
    const uint32_t q = blockIdx.x * kThreads + threadIdx.x;
    const bool live = q < n_pending;
    uint32_t c[8];
    uint32_t kk = 0, n = 0;
    uint32_t lf[8], cn[8];
    if (live) {
        const uint4 lo = __ldg(reinterpret_cast<const uint4*>(children + 8ull * q)), hi = __ldg(reinterpret_cast<const uint4*>(children + 8ull * q) + 1);
        c[0] = lo.x; c[1] = lo.y; c[2] = lo.z; c[3] = lo.w; c[4] = hi.x; c[5] = hi.y; c[6] = hi.z; c[7] = hi.w;
        // sorting network for 8 keys (19 compare-exchanges); kNone sorts last
#define MG_CX(i, j) { const uint32_t a_ = min(c[i], c[j]), b_ = max(c[i], c[j]); c[i] = a_; c[j] = b_; }
        MG_CX(0, 1) MG_CX(2, 3) MG_CX(4, 5) MG_CX(6, 7)
        MG_CX(0, 2) MG_CX(1, 3) MG_CX(4, 6) MG_CX(5, 7)
        MG_CX(1, 2) MG_CX(5, 6) MG_CX(0, 4) MG_CX(3, 7)
        MG_CX(1, 5) MG_CX(2, 6)
        MG_CX(1, 4) MG_CX(3, 6)
        MG_CX(2, 4) MG_CX(3, 5)
        MG_CX(3, 4)
#undef MG_CX
#pragma unroll
        for (int t = 0; t < 8; t++) {
            if (c[t] == kNone) continue;
            n++;
            if (kk && lf[kk - 1] == c[t]) cn[kk - 1]++;
            else { lf[kk] = c[t]; cn[kk] = 1; kk++; }
        }
    }
    // scratch: one atomic per warp
    const unsigned lane = threadIdx.x & 31;
    uint32_t incl = kk;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t up = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= (unsigned)d) incl += up; }
    const uint32_t tot = __shfl_sync(0xffffffffu, incl, 31);
    unsigned long long base = 0;
    if (lane == 0 && tot) { base = atomicAdd(ctr + kScratch, (unsigned long long)tot); atomicAdd(ctr + kNnz, (unsigned long long)tot); }
    base = __shfl_sync(0xffffffffu, base, 0);
    if (!live) return;
    int tz = 32;
#pragma unroll
    for (int j = 0; j < 8; j++)
        if ((uint32_t)j < kk) tz = min(tz, __ffs((int)cn[j]) - 1);
    uint64_t h = 0;
    const uint64_t so = base + (incl - kk);
#pragma unroll
    for (int j = 0; j < 8; j++) {
        if ((uint32_t)j >= kk) continue;
        const uint64_t cnt = cn[j] >> tz;
        h += mix64((((uint64_t)lf[j] << 32) | (uint32_t)(j + 1)) * 0x9E3779B97F4A7C15ull + cnt);
        s_leaf[so + j] = lf[j];
        s_cnt[so + j] = cnt;
    }
    h = mix64(h ^ kk);
    if (h == 0) h = 1;
    const uint32_t nlog = (n == 8) ? 3u : (n == 4) ? 2u : (n == 2) ? 1u : 0u;
    Q.off[q] = so; Q.k[q] = kk; Q.tlog[q] = nlog - (uint32_t)tz; Q.hash[q] = h;     // (kk >= 2: the list holds non-pure parents only)
}

__global__ void __launch_bounds__(kThreads)
k_claim(const Pending Q, uint32_t n_pending, uint32_t level, uint64_t* hash, uint64_t* hfirst, uint64_t mask, unsigned long long* ctr)
{
    const uint32_t q = blockIdx.x * kThreads + threadIdx.x;
    if (q >= n_pending || Q.k[q] == 0) return;
    const unsigned long long h = Q.hash[q];
    const unsigned long long pos = ((unsigned long long)level << 40) | Q.voxel[q];
    uint64_t s = h & mask;
    for (uint64_t probes = 0;; probes++) {
        const unsigned long long old = atomicCAS(reinterpret_cast<unsigned long long*>(hash + s), 0ull, h);
        if (old == 0ull || old == h) break;
        s = (s + 1) & mask;
        if (probes > mask) { atomicOr(ctr + kFlags, (unsigned long long)kTableFull); Q.slot[q] = ~0ull; return; }
    }
    atomicMin(reinterpret_cast<unsigned long long*>(hfirst + s), pos);
    Q.slot[q] = s;
}

__global__ void __launch_bounds__(kThreads)
k_publish(const Pending Q, uint32_t n_pending, uint32_t level, const uint32_t* __restrict__ s_leaf, const uint64_t* __restrict__ s_cnt,
          const uint64_t* __restrict__ hfirst, uint32_t* hid, uint64_t* mix_off, uint32_t* mix_k, uint32_t* mix_tlog, uint64_t* mix_first,
          uint32_t* ent_leaf, uint64_t* ent_cnt, uint64_t cap_m, uint64_t cap_e, unsigned long long* ctr)
{
    const uint32_t q = blockIdx.x * kThreads + threadIdx.x;
    if (q >= n_pending || Q.k[q] == 0 || Q.slot[q] == ~0ull) return;
    const uint64_t s = Q.slot[q];
    const unsigned long long pos = ((unsigned long long)level << 40) | Q.voxel[q];
    if (hfirst[s] != pos || hid[s] != kNoId) return;                   // not the first occurrence, or a mixture of an earlier level
    const uint32_t k = Q.k[q];
    const unsigned long long id = atomicAdd(ctr + kNMix, 1ull), eo = atomicAdd(ctr + kNEnt, (unsigned long long)k);
    if (id >= cap_m || eo + k > cap_e) { atomicOr(ctr + kFlags, (unsigned long long)kStoreFull); return; }
    const uint64_t so = Q.off[q];
    for (uint32_t j = 0; j < k; j++) { ent_leaf[eo + j] = s_leaf[so + j]; ent_cnt[eo + j] = s_cnt[so + j]; }
    mix_off[id] = eo; mix_k[id] = k; mix_tlog[id] = Q.tlog[q]; mix_first[id] = pos;
    hid[s] = (uint32_t)id;
}

__global__ void __launch_bounds__(kThreads)
k_resolve(const Pending Q, uint32_t n_pending, const uint32_t* __restrict__ s_leaf, const uint64_t* __restrict__ s_cnt,
          const uint32_t* __restrict__ hid, const uint64_t* __restrict__ mix_off, const uint32_t* __restrict__ mix_k,
          const uint32_t* __restrict__ ent_leaf, const uint64_t* __restrict__ ent_cnt, uint32_t* __restrict__ P, unsigned long long* ctr)
{
    const uint32_t q = blockIdx.x * kThreads + threadIdx.x;
    if (q >= n_pending || Q.k[q] == 0 || Q.slot[q] == ~0ull) return;
    const uint32_t id = hid[Q.slot[q]];
    if (id == kNoId) { atomicOr(ctr + kFlags, (unsigned long long)kStoreFull); return; }
    const uint32_t k = Q.k[q];
    bool eq = mix_k[id] == k;
    const uint64_t so = Q.off[q], eo = mix_off[id];
    for (uint32_t j = 0; eq && j < k; j++) eq = s_leaf[so + j] == ent_leaf[eo + j] && s_cnt[so + j] == ent_cnt[eo + j];
    if (!eq) { atomicOr(ctr + kFlags, (unsigned long long)kCollision); return; }
    P[Q.voxel[q]] = kMixed | id;
}

__global__ void __launch_bounds__(kThreads)
k_remap_handles(uint32_t* __restrict__ h, uint64_t n, const uint32_t* __restrict__ node_of_mixture, uint32_t n_mix)
{
    for (uint64_t i = (uint64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (uint64_t)gridDim.x * kThreads) {
        const uint32_t x = h[i];
        if (x & kMixed) {
            const uint32_t id = x & ~kMixed;
            h[i] = id < n_mix ? __ldg(node_of_mixture + id) : kNone;
        }
    }
}

template <typename T>
cudaError_t dalloc(mg_mixture_table* t, T** p, uint64_t n)
{
    const size_t bytes = (size_t)std::max<uint64_t>(n, 1) * sizeof(T);
    const cudaError_t e = cudaMalloc((void**)p, bytes);
    if (e == cudaSuccess) t->device_bytes += bytes;
    return e;
}

}  // namespace

extern "C" void mg_mixture_table_free(mg_mixture_table* t)
{
    if (!t) return;
    cudaFree(t->d_off); cudaFree(t->d_k); cudaFree(t->d_tlog); cudaFree(t->d_first); cudaFree(t->d_leaf); cudaFree(t->d_cnt);
    cudaFree(t->d_hash); cudaFree(t->d_hfirst); cudaFree(t->d_hid); cudaFree(t->d_ctr);
    cudaGetLastError();
    delete t;
}

extern "C" int mg_mipmap_levels_build_ex(const uint32_t* level0_device, uint64_t X, uint64_t Y, uint64_t Z, uint32_t n_leaves,
                                         uint32_t* levels_device, const uint64_t* level_offset, uint32_t n_levels,
                                         uint64_t cap_mixtures, uint64_t cap_entries, mg_mixture_table** out, void* stream)
{
    if (!out) { mg::set_error("mg_mipmap_levels_build: out is NULL"); return MG_ERR_INVALID_ARG; }
    *out = nullptr;
    if (!level0_device || !levels_device || !level_offset || X == 0 || Y == 0 || Z == 0 || n_leaves == 0 || n_leaves >= kMixed) {
        mg::set_error("mg_mipmap_levels_build: NULL argument, empty volume or n_leaves not in 1 .. 2^31 - 1");
        return MG_ERR_INVALID_ARG;
    }
    // the ceil-halving chain (L80)
    std::vector<uint64_t> dims;
    for (uint64_t x = X, y = Y, z = Z;;) {
        dims.push_back(x); dims.push_back(y); dims.push_back(z);
        if (x == 1 && y == 1 && z == 1) break;
        x = (x + 1) / 2; y = (y + 1) / 2; z = (z + 1) / 2;
    }
    if (n_levels != dims.size() / 3) {
        mg::set_error("mg_mipmap_levels_build: %llu x %llu x %llu has %zu mip levels, not %u", (unsigned long long)X, (unsigned long long)Y,
                      (unsigned long long)Z, dims.size() / 3, n_levels);
        return MG_ERR_INVALID_ARG;
    }
    if (n_levels > 1 && dims[3] * dims[4] * dims[5] >= (1ull << 32)) { mg::set_error("mg_mipmap_levels_build: level 1 must have < 2^32 voxels"); return MG_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    mg_mixture_table* T = new (std::nothrow) mg_mixture_table;
    if (!T) { mg::set_error("mg_mipmap_levels_build: out of host memory"); return MG_ERR_OOM; }
    T->n_leaves = n_leaves;
    uint32_t* d_list = nullptr;
    Pending Q = {};
    uint32_t* d_sleaf = nullptr;
    uint64_t* d_scnt = nullptr;
    uint32_t* d_children = nullptr;                                       // level 1 only: the <= 8 leaves of every listed parent
    auto drop_level = [&]() {
        cudaFree(d_children);
        d_children = nullptr;
        cudaFree(d_list); cudaFree(Q.off); cudaFree(Q.k); cudaFree(Q.tlog); cudaFree(Q.hash); cudaFree(Q.slot); cudaFree(d_sleaf); cudaFree(d_scnt);
        d_list = nullptr; Q = Pending{}; d_sleaf = nullptr; d_scnt = nullptr;
    };
    auto fail = [&](int rc) { drop_level(); mg_mixture_table_free(T); return rc; };
#define MT_CUDA(call)                                                       \
    do {                                                                    \
        cudaError_t e__ = (call);                                           \
        if (e__ != cudaSuccess) return fail(mg::cuda_fail(e__, #call));     \
    } while (0)
    MT_CUDA(cudaGetDevice(&T->device));
    MT_CUDA(dalloc(T, &T->d_ctr, (uint64_t)kNCtr));
    MT_CUDA(cudaMemsetAsync(T->d_ctr, 0, kNCtr * sizeof(unsigned long long), st));
    unsigned long long ctr[kNCtr] = {};                                   // (level 1 fills only two of them on the host)
    for (uint32_t l = 1; l < n_levels; l++) {
        LevelGeom G;
        G.cx = (uint32_t)dims[3 * l - 3]; G.cy = (uint32_t)dims[3 * l - 2]; G.cz = (uint32_t)dims[3 * l - 1];
        G.px = (uint32_t)dims[3 * l]; G.py = (uint32_t)dims[3 * l + 1]; G.pz = (uint32_t)dims[3 * l + 2];
        G.level = l;
        const uint32_t n_par = G.px * G.py * G.pz;
        const uint32_t* C = l == 1 ? level0_device : levels_device + level_offset[l - 1];
        uint32_t* P = levels_device + level_offset[l];
        // ---- classify; the list is sized by a guess and the pass repeated if it was too small
        unsigned long long nnz_before = 0;
        {
            MT_CUDA(cudaMemcpyAsync(&nnz_before, T->d_ctr + kNnz, sizeof(nnz_before), cudaMemcpyDeviceToHost, st));
            MT_CUDA(cudaStreamSynchronize(st));
        }
        uint32_t list_cap = std::max<uint32_t>(1024, l == 1 ? n_par / 12 : n_par / 3);
        uint32_t n_pending = 0;
        for (;;) {
            MT_CUDA(cudaMalloc((void**)&d_list, (size_t)list_cap * 4));
            if (l == 1) {
                // level 1 is 98 % of the work and its children are leaves: the streaming classifier of the front end
                // (16-byte / 8-byte loads, four parents per thread, one list atomic per CTA) lists the parents WITH their children
                cudaError_t e = cudaMalloc((void**)&d_children, (size_t)list_cap * 32);
                if (e != cudaSuccess) return fail(mg::cuda_fail(e, "cudaMalloc(children list)"));
                uint64_t n_mixed = 0;
                const int rc = mg_mipmap_front_level1(level0_device, X, Y, Z, P, d_list, d_children, list_cap, &n_mixed, stream);
                if (rc != MG_OK) return fail(rc);
                ctr[kNPending] = n_mixed;
                ctr[kNnz] = nnz_before + (n_par - n_mixed);               // every other parent is one leaf
                MT_CUDA(cudaMemcpyAsync(T->d_ctr + kNnz, &ctr[kNnz], sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
                MT_CUDA(cudaStreamSynchronize(st));                       // (ctr is a stack array that is rewritten below)
                if (n_mixed <= list_cap) { n_pending = (uint32_t)n_mixed; break; }
                cudaFree(d_children);
                d_children = nullptr;
            } else {
                MT_CUDA(cudaMemsetAsync(T->d_ctr + kNPending, 0, sizeof(unsigned long long), st));
                MT_CUDA(cudaMemcpyAsync(T->d_ctr + kNnz, &nnz_before, sizeof(nnz_before), cudaMemcpyHostToDevice, st));
                k_classify<<<(n_par + kThreads - 1) / kThreads, kThreads, 0, st>>>(C, G, n_par, P, d_list, list_cap, T->d_k, T->d_ctr);
                mg::count_launch();
                MT_CUDA(cudaGetLastError());
                MT_CUDA(cudaMemcpyAsync(ctr, T->d_ctr, sizeof(ctr), cudaMemcpyDeviceToHost, st));
                MT_CUDA(cudaStreamSynchronize(st));
                if (ctr[kNPending] <= list_cap) { n_pending = (uint32_t)ctr[kNPending]; break; }
            }
            cudaFree(d_list);
            d_list = nullptr;
            list_cap = (uint32_t)ctr[kNPending];
        }
        if (l == 1) {
            // the stores are sized once: by the caller, or from the number of level-1 merges (on segmentations with coherent
            // regions later levels add little: 1/8 of the voxels each).  A level that does not fit is the host's (below).
            T->cap_m = cap_mixtures ? cap_mixtures : (uint64_t)n_pending + n_pending / 2 + (1u << 20);
            T->cap_e = cap_entries ? cap_entries : 12ull * n_pending + (1u << 22);
            T->cap_h = 1;
            while (T->cap_h < 2 * T->cap_m) T->cap_h <<= 1;
            MT_CUDA(dalloc(T, &T->d_off, T->cap_m)); MT_CUDA(dalloc(T, &T->d_k, T->cap_m)); MT_CUDA(dalloc(T, &T->d_tlog, T->cap_m));
            MT_CUDA(dalloc(T, &T->d_first, T->cap_m)); MT_CUDA(dalloc(T, &T->d_leaf, T->cap_e)); MT_CUDA(dalloc(T, &T->d_cnt, T->cap_e));
            MT_CUDA(dalloc(T, &T->d_hash, T->cap_h)); MT_CUDA(dalloc(T, &T->d_hfirst, T->cap_h)); MT_CUDA(dalloc(T, &T->d_hid, T->cap_h));
            MT_CUDA(cudaMemsetAsync(T->d_hash, 0, T->cap_h * 8, st));
            MT_CUDA(cudaMemsetAsync(T->d_hfirst, 0xFF, T->cap_h * 8, st));
            MT_CUDA(cudaMemsetAsync(T->d_hid, 0xFF, T->cap_h * 4, st));
            // (k_classify of level 1 saw only leaves: it never read d_k)
        }
        if (n_pending) {
            Q.voxel = d_list;
            MT_CUDA(cudaMalloc((void**)&Q.off, (size_t)n_pending * 8)); MT_CUDA(cudaMalloc((void**)&Q.k, (size_t)n_pending * 4));
            MT_CUDA(cudaMalloc((void**)&Q.tlog, (size_t)n_pending * 4)); MT_CUDA(cudaMalloc((void**)&Q.hash, (size_t)n_pending * 8));
            MT_CUDA(cudaMalloc((void**)&Q.slot, (size_t)n_pending * 8));
            uint64_t scratch_cap = (l == 1 ? 8ull : 32ull) * n_pending + 4096;
            const unsigned long long nnz_classified = ctr[kNnz];
            for (;;) {
                MT_CUDA(cudaMalloc((void**)&d_sleaf, scratch_cap * 4));
                MT_CUDA(cudaMalloc((void**)&d_scnt, scratch_cap * 8));
                MT_CUDA(cudaMemsetAsync(T->d_ctr + kScratch, 0, sizeof(unsigned long long), st));
                MT_CUDA(cudaMemsetAsync(T->d_ctr + kFlags, 0, sizeof(unsigned long long), st));
                MT_CUDA(cudaMemcpyAsync(T->d_ctr + kNnz, &nnz_classified, sizeof(nnz_classified), cudaMemcpyHostToDevice, st));
                if (l == 1)
                    k_merge_leaves<<<(n_pending + kThreads - 1) / kThreads, kThreads, 0, st>>>(d_children, Q, n_pending, d_sleaf, d_scnt, T->d_ctr);
                else
                    k_merge<<<(n_pending + kMergeWarps - 1) / kMergeWarps, kMergeWarps * 32, 0, st>>>(
                        C, G, P, Q, n_pending, T->d_off, T->d_k, T->d_tlog, T->d_leaf, T->d_cnt, d_sleaf, d_scnt, scratch_cap, T->d_ctr);
                mg::count_launch();
                MT_CUDA(cudaGetLastError());
                MT_CUDA(cudaMemcpyAsync(ctr, T->d_ctr, sizeof(ctr), cudaMemcpyDeviceToHost, st));
                MT_CUDA(cudaStreamSynchronize(st));
                if (!(ctr[kFlags] & kScratchFull) || (ctr[kFlags] & kTooBig)) break;
                cudaFree(d_sleaf); cudaFree(d_scnt);
                d_sleaf = nullptr; d_scnt = nullptr;
                scratch_cap = std::max<uint64_t>(ctr[kScratch], 4 * scratch_cap);
            }
            if (ctr[kFlags] & kTooBig) {                               // this level and the ones above are the host's
                MT_CUDA(cudaMemcpyAsync(T->d_ctr + kNnz, &nnz_before, sizeof(nnz_before), cudaMemcpyHostToDevice, st));
                drop_level();
                break;
            }
            const unsigned grid = (n_pending + kThreads - 1) / kThreads;
            k_claim<<<grid, kThreads, 0, st>>>(Q, n_pending, l, T->d_hash, T->d_hfirst, T->cap_h - 1, T->d_ctr);
            k_publish<<<grid, kThreads, 0, st>>>(Q, n_pending, l, d_sleaf, d_scnt, T->d_hfirst, T->d_hid, T->d_off, T->d_k, T->d_tlog, T->d_first,
                                                 T->d_leaf, T->d_cnt, T->cap_m, T->cap_e, T->d_ctr);
            k_resolve<<<grid, kThreads, 0, st>>>(Q, n_pending, d_sleaf, d_scnt, T->d_hid, T->d_off, T->d_k, T->d_leaf, T->d_cnt, P, T->d_ctr);
            mg::count_launch(3);
            MT_CUDA(cudaGetLastError());
            MT_CUDA(cudaMemcpyAsync(ctr, T->d_ctr, sizeof(ctr), cudaMemcpyDeviceToHost, st));
            MT_CUDA(cudaStreamSynchronize(st));
            if (ctr[kFlags] & (kStoreFull | kTableFull)) {
                // The level's mixtures do not fit the stores.  What it published sits beyond n_mix / n_ent of the finished
                // levels and is never exported; its handles are scratch.  Like a kTooBig level, it and the levels above it
                // go to the host (mgb_build_from_levels continues from levels_done = l - 1).
                MT_CUDA(cudaMemcpyAsync(T->d_ctr + kNnz, &nnz_before, sizeof(nnz_before), cudaMemcpyHostToDevice, st));
                MT_CUDA(cudaStreamSynchronize(st));                       // (nnz_before is a local of this iteration)
                drop_level();
                break;
            }
            if (ctr[kFlags] & kCollision) {
                mg::set_error("mg_mipmap_levels_build: two different mixtures share a 64-bit hash at level %u: use the host builder", l);
                return fail(MG_ERR_INVALID_ARG);
            }
        }
        drop_level();
        T->levels_done = l;
        T->n_mix = ctr[kNMix];
        T->n_ent = ctr[kNEnt];
        T->nnz_levels = ctr[kNnz];
    }
#undef MT_CUDA
    *out = T;
    return MG_OK;
}

extern "C" int mg_mipmap_levels_build(const uint32_t* level0_device, uint64_t X, uint64_t Y, uint64_t Z, uint32_t n_leaves,
                                      uint32_t* levels_device, const uint64_t* level_offset, uint32_t n_levels,
                                      mg_mixture_table** out, void* stream)
{
    return mg_mipmap_levels_build_ex(level0_device, X, Y, Z, n_leaves, levels_device, level_offset, n_levels, 0, 0, out, stream);
}

extern "C" int mg_mixture_table_info(const mg_mixture_table* t, mg_mixture_table_info_t* info)
{
    if (!t || !info) { mg::set_error("mg_mixture_table_info: NULL argument"); return MG_ERR_INVALID_ARG; }
    info->n_mixtures = t->n_mix;
    info->n_entries = t->n_ent;
    info->nnz_levels = t->nnz_levels;
    info->device_bytes = t->device_bytes;
    info->levels_done = t->levels_done;
    info->n_leaves = t->n_leaves;
    return MG_OK;
}

extern "C" int mg_mixture_table_export(const mg_mixture_table* t, uint64_t* offset, uint32_t* k, uint32_t* tlog, uint64_t* first_pos,
                                       uint32_t* leaf, uint64_t* count)
{
    if (!t) { mg::set_error("mg_mixture_table_export: NULL table"); return MG_ERR_INVALID_ARG; }
    if (t->n_mix) {
        if (offset) MG_CUDA(cudaMemcpy(offset, t->d_off, t->n_mix * 8, cudaMemcpyDeviceToHost));
        if (k) MG_CUDA(cudaMemcpy(k, t->d_k, t->n_mix * 4, cudaMemcpyDeviceToHost));
        if (tlog) MG_CUDA(cudaMemcpy(tlog, t->d_tlog, t->n_mix * 4, cudaMemcpyDeviceToHost));
        if (first_pos) MG_CUDA(cudaMemcpy(first_pos, t->d_first, t->n_mix * 8, cudaMemcpyDeviceToHost));
    }
    if (t->n_ent) {
        if (leaf) MG_CUDA(cudaMemcpy(leaf, t->d_leaf, t->n_ent * 4, cudaMemcpyDeviceToHost));
        if (count) MG_CUDA(cudaMemcpy(count, t->d_cnt, t->n_ent * 8, cudaMemcpyDeviceToHost));
    }
    return MG_OK;
}

extern "C" int mg_mipmap_remap_handles(uint32_t* handles_device, uint64_t n, const uint32_t* node_of_mixture_device, uint32_t n_mixtures,
                                       void* stream)
{
    if ((!handles_device && n) || (!node_of_mixture_device && n_mixtures)) { mg::set_error("mg_mipmap_remap_handles: NULL argument"); return MG_ERR_INVALID_ARG; }
    if (n == 0) return MG_OK;
    const unsigned grid = (unsigned)std::min<uint64_t>((n + kThreads - 1) / kThreads, 148ull * 32);
    k_remap_handles<<<grid, kThreads, 0, (cudaStream_t)stream>>>(handles_device, n, node_of_mixture_device, n_mixtures);
    mg::count_launch();
    MG_CUDA(cudaGetLastError());
    return MG_OK;
}
