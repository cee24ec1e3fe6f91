// builder_api.cpp -- C ABI of the host builder (include/mg_builder.h): a0 -> a1 -> quantiser -> a2.
//
// Finalisation after the factoriser (factorise.cpp):
//   * scalar quantiser: 2^b uniform bins of (0,1); the codeword of a bin is the mean of
//     the exact ratios merged into it ("best represents the weights in the bin", reading Q7; an empty bin
//     gets its mid-point), sigma its empirical rms deviation from the codeword.
//   * interpolation symmetry (L259): (i, j, w) == (j, i, 1 - w).  Each node keeps the side whose
//     codeword is closer to the node's own mean ratio: either (lo, hi, cw[bin(w)]) or
//     (hi, lo, cw[bin(1 - w)]).  Node identity (what was merged) is not affected.
//   * weights are emitted as fp32 strictly inside (0,1) (L176: "ratios cannot be 0 or 1").
//   * a2: topological levels (L211) + level-contiguous relabelling (relabel.cpp), applied to the graph
//     and to the per-voxel node indices of every mip level.
#include <omp.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <numeric>

#include "builder_internal.h"

namespace mgb {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

namespace {

double now_s()
{
    return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

inline float open_unit_fp32(double w)
{
    float f = (float)w;
    const float lo = 1.0f / 16777216.0f / 256.0f;        // 2^-32
    const float hi = 1.0f - 1.0f / 16777216.0f;          // largest fp32 below 1
    if (!(f > lo)) f = lo;
    if (!(f < hi)) f = hi;
    return f;
}

// Turn the factoriser's creation-order nodes into the output graph (weights, orientation, codebook).
int finalise_graph(const Factorised& F, uint32_t n_leaves, const mgb_params& p, mgb_result& R,
                   std::vector<uint32_t>& new_of_old)
{
    const uint64_t n_int = F.a.size();
    const uint64_t n_nodes = (uint64_t)n_leaves + n_int;
    std::vector<uint32_t> ca(n_nodes, 0), cb(n_nodes, 0);
    std::vector<float> w32(n_nodes, 0.0f);
    std::vector<double> wex(n_nodes, 0.0);
    std::vector<float> wsg(n_nodes, 0.0f);           // sigma of the bin the node's codeword came from (L176, Eq. 18)
    const uint32_t b = p.quant_bits;
    R.codeword.clear(); R.sigma.clear(); R.bin_count.clear();
    R.info.max_bin_sigma = 0.0;
    if (b) {
        const uint64_t nb = 1ull << b;
        std::vector<double> s1(nb, 0.0), s2(nb, 0.0);
        R.bin_count.assign(nb, 0);
        for (uint64_t q = 0; q < n_int; q++) {
            s1[F.bin[q]] += F.w_sum[q];
            s2[F.bin[q]] += F.w_sq[q];
            R.bin_count[F.bin[q]] += F.w_cnt[q];
        }
        R.codeword.resize(nb);
        R.sigma.resize(nb);
        std::vector<double> cw(nb);
        for (uint64_t k = 0; k < nb; k++) {
            const double lo = (double)k / (double)nb, hi = (double)(k + 1) / (double)nb;
            if (R.bin_count[k]) {
                const double n = (double)R.bin_count[k];
                double c = s1[k] / n;
                c = std::min(std::max(c, lo), hi);
                cw[k] = c;
                const double var = std::max(0.0, s2[k] / n - 2.0 * c * s1[k] / n + c * c);
                R.sigma[k] = (float)std::sqrt(var);
            } else {
                cw[k] = 0.5 * (lo + hi);
                R.sigma[k] = 0.0f;
            }
            R.codeword[k] = open_unit_fp32(cw[k]);
            R.info.max_bin_sigma = std::max(R.info.max_bin_sigma, (double)R.sigma[k]);
        }
#pragma omp parallel for schedule(static)
        for (int64_t q = 0; q < (int64_t)n_int; q++) {
            const uint64_t n = n_leaves + (uint64_t)q;
            const double wm = F.w_sum[q] / (double)F.w_cnt[q];            // mean exact ratio on child hi
            const uint32_t k1 = F.bin[q];
            uint64_t k2 = (uint64_t)std::floor((1.0 - wm) * (double)nb);   // bin of the mirrored weight
            if (k2 >= nb) k2 = nb - 1;
            const double e1 = std::fabs((double)R.codeword[k1] - wm);
            const double e2 = std::fabs((double)R.codeword[k2] - (1.0 - wm));
            if (e2 < e1) { ca[n] = F.b[q]; cb[n] = F.a[q]; w32[n] = R.codeword[k2]; wex[n] = 1.0 - wm; wsg[n] = R.sigma[k2]; }
            else { ca[n] = F.a[q]; cb[n] = F.b[q]; w32[n] = R.codeword[k1]; wex[n] = wm; wsg[n] = R.sigma[k1]; }
        }
    } else {
#pragma omp parallel for schedule(static)
        for (int64_t q = 0; q < (int64_t)n_int; q++) {
            const uint64_t n = n_leaves + (uint64_t)q;
            const double wm = F.w_sum[q] / (double)F.w_cnt[q];            // all merged ratios are equal
            ca[n] = F.a[q]; cb[n] = F.b[q]; w32[n] = open_unit_fp32(wm); wex[n] = wm;
        }
    }

    std::vector<uint64_t> level_off;
    if (mg::relabel_by_level(ca.data(), cb.data(), n_nodes, n_leaves, new_of_old, level_off) != 0) {
        set_error("internal error: factorised graph is not children-before-parents");
        return MGB_ERR_LIMIT;
    }
    R.level_off = level_off;
    R.info.depth = (uint32_t)level_off.size() - 2;
    if (p.relabel) {
        R.child_a.assign(n_nodes, 0); R.child_b.assign(n_nodes, 0);
        R.weight.assign(n_nodes, 0.0f); R.weight_exact.assign(n_nodes, 0.0); R.weight_sigma.assign(n_nodes, 0.0f);
#pragma omp parallel for schedule(static)
        for (int64_t n = n_leaves; n < (int64_t)n_nodes; n++) {
            const uint32_t q = new_of_old[n];
            R.child_a[q] = new_of_old[ca[n]]; R.child_b[q] = new_of_old[cb[n]];
            R.weight[q] = w32[n]; R.weight_exact[q] = wex[n]; R.weight_sigma[q] = wsg[n];
        }
    } else {
        R.child_a.swap(ca); R.child_b.swap(cb); R.weight.swap(w32); R.weight_exact.swap(wex); R.weight_sigma.swap(wsg);
        for (uint64_t n = 0; n < n_nodes; n++) new_of_old[n] = (uint32_t)n;
    }
    R.info.n_nodes = n_nodes;
    return MGB_OK;
}

int check_params(const mgb_params* params, mgb_params& p)
{
    if (params) p = *params; else mgb_default_params(&p);
    if (p.quant_bits > 16) { set_error("quant_bits must be 0 (unquantised) or in [1,16] (L189)"); return MGB_ERR_INVALID_ARG; }
    if (p.pick_order > MGB_PICK_SMALLEST_MASS) { set_error("unknown pick_order %u", p.pick_order); return MGB_ERR_INVALID_ARG; }
    if (p.n_threads) omp_set_num_threads((int)p.n_threads);
    return MGB_OK;
}

}  // namespace
}  // namespace mgb

using namespace mgb;

extern "C" const char* mgb_last_error(void) { return g_err; }

extern "C" void mgb_default_params(mgb_params* p)
{
    if (!p) return;
    p->quant_bits = 9;
    p->tau = 3;
    p->big_cutoff = 32;
    p->pick_order = MGB_PICK_SMALLEST_INDEX;
    p->n_threads = 0;
    p->relabel = 1;
    p->phi2_exact_budget = 2000000000ull;
}

extern "C" void mgb_free(mgb_result* r) { delete r; }

extern "C" uint32_t mgb_mip_chain(uint64_t X, uint64_t Y, uint64_t Z, uint64_t* dims_out, uint32_t max_levels)
{
    if (X == 0 || Y == 0 || Z == 0) return 0;
    uint32_t l = 0;
    for (uint64_t x = X, y = Y, z = Z;;) {
        if (dims_out && l < max_levels) { dims_out[3 * l] = x; dims_out[3 * l + 1] = y; dims_out[3 * l + 2] = z; }
        l++;
        if (x == 1 && y == 1 && z == 1) return l;
        x = (x + 1) / 2; y = (y + 1) / 2; z = (z + 1) / 2;
    }
}

// a0 - a2 for a volume: from the segment IDs (front == nullptr), or from levels 0 / 1 classified by a front end.
static int build_volume(const uint32_t* seg, uint64_t X, uint64_t Y, uint64_t Z, const Level1Front* front,
                        const mgb_params* params, mgb_result** out, const LevelsFront* levels = nullptr)
{
    g_err[0] = 0;
    if (!out) { set_error("mgb_build: out is NULL"); return MGB_ERR_INVALID_ARG; }
    *out = nullptr;
    if ((!seg && !front && !levels) || X == 0 || Y == 0 || Z == 0) { set_error("mgb_build: NULL volume or zero dimension"); return MGB_ERR_INVALID_ARG; }
    if (X > 0x7fffffffull || Y > 0x7fffffffull || Z > 0x7fffffffull || X * Y * Z >= (1ull << 40)) {
        set_error("mgb_build: volume too large"); return MGB_ERR_INVALID_ARG;
    }
    mgb_params p;
    int rc = check_params(params, p);
    if (rc != MGB_OK) return rc;
    mgb_result* R = nullptr;
    try {
        R = new mgb_result();
        const double t0 = now_s();
        Mipmap mm;
        rc = build_mipmap(seg, X, Y, Z, (int)p.n_threads, mm, front, levels);
        if (rc != MGB_OK) { delete R; return rc; }
        const double t1 = now_s();
        Factorised F;
        rc = factorise(mm.mixtures, p, F);
        if (rc != MGB_OK) { delete R; return rc; }
        const double t2 = now_s();
        const uint32_t n_leaves = (uint32_t)mm.leaf_segment_id.size();
        std::vector<uint32_t> new_of_old;
        rc = finalise_graph(F, n_leaves, p, *R, new_of_old);
        if (rc != MGB_OK) { delete R; return rc; }
        // per-voxel node index: leaf number, or the node of the voxel's mixture; then the relabelling
        const uint32_t n_mip = (uint32_t)(mm.dims.size() / 3);
        R->node_idx.resize(n_mip);
        uint64_t n_vox_total = 0;
        for (uint32_t l = 0; l < n_mip; l++) {
            std::vector<uint32_t>& ids = mm.level_ids[l];
            const int64_t nv = (int64_t)ids.size();
            // with a front end the levels it classified stay with the caller: count their voxels all the same
            n_vox_total += (ids.empty() && (front || levels)) ? mm.dims[3 * l] * mm.dims[3 * l + 1] * mm.dims[3 * l + 2] : (uint64_t)nv;
            uint32_t* P = ids.data();
            const uint32_t* nom = F.node_of_mix.data();
            const uint32_t* perm = new_of_old.data();
#pragma omp parallel for schedule(static)
            for (int64_t v = 0; v < nv; v++) {
                const uint32_t id = P[v];
                P[v] = perm[id < n_leaves ? id : nom[id - n_leaves]];
            }
            R->node_idx[l].swap(ids);
        }
        if (levels) {                                                  // node of every mixture the caller listed
            R->front_mixture_node.resize(mm.front_mixture.size());
            for (size_t q = 0; q < mm.front_mixture.size(); q++) R->front_mixture_node[q] = new_of_old[F.node_of_mix[mm.front_mixture[q]]];
        }
        R->dims = mm.dims;
        R->leaf_segment_id = mm.leaf_segment_id;
        mgb_info& I = R->info;
        I.dims[0] = X; I.dims[1] = Y; I.dims[2] = Z;
        I.n_mip_levels = n_mip;
        I.n_leaves = n_leaves;
        I.n_voxels_total = n_vox_total;
        I.quant_bits = p.quant_bits;
        I.n_distinct_mixtures = mm.mixtures.size();
        I.nnz_total = mm.nnz_total;
        I.n_stage1 = F.n_stage1; I.n_stage2 = F.n_stage2; I.n_big = F.n_big;
        I.phi2_exact = F.phi2_exact ? 1 : 0;
        I.seconds_mipmap = t1 - t0;
        I.seconds_factorise = t2 - t1;
        I.seconds_finalise = now_s() - t2;
    } catch (const std::bad_alloc&) {
        delete R;
        set_error("mgb_build: out of host memory");
        return MGB_ERR_OOM;
    }
    *out = R;
    return MGB_OK;
}

extern "C" int mgb_build(const uint32_t* seg, uint64_t X, uint64_t Y, uint64_t Z, const mgb_params* params,
                         mgb_result** out)
{
    return build_volume(seg, X, Y, Z, nullptr, params, out);
}

extern "C" int mgb_build_from_level1(uint64_t X, uint64_t Y, uint64_t Z, const uint32_t* leaf_segment_id, uint32_t n_leaves,
                                     const uint32_t* level1, const uint32_t* mixed_voxel, const uint32_t* mixed_children,
                                     uint64_t n_mixed, const mgb_params* params, mgb_result** out)
{
    if (!leaf_segment_id || n_leaves == 0 || (n_mixed && (!mixed_voxel || !mixed_children))) {
        g_err[0] = 0;
        set_error("mgb_build_from_level1: NULL argument or no leaves");
        if (out) *out = nullptr;
        return MGB_ERR_INVALID_ARG;
    }
    const bool has_level1 = !(X == 1 && Y == 1 && Z == 1);
    if (has_level1 && !level1) {
        g_err[0] = 0;
        set_error("mgb_build_from_level1: level1 is NULL");
        if (out) *out = nullptr;
        return MGB_ERR_INVALID_ARG;
    }
    for (uint32_t k = 1; k < n_leaves; k++)
        if (leaf_segment_id[k] <= leaf_segment_id[k - 1]) {
            g_err[0] = 0;
            set_error("mgb_build_from_level1: leaf_segment_id must be strictly increasing");
            if (out) *out = nullptr;
            return MGB_ERR_INVALID_ARG;
        }
    Level1Front front{leaf_segment_id, n_leaves, level1, mixed_voxel, mixed_children, n_mixed};
    return build_volume(nullptr, X, Y, Z, &front, params, out);
}

extern "C" int mgb_build_from_levels(uint64_t X, uint64_t Y, uint64_t Z, const uint32_t* leaf_segment_id, uint32_t n_leaves,
                                     uint32_t level_done, const uint32_t* handles, uint64_t n_mixtures, const uint64_t* mix_offset,
                                     const uint32_t* mix_k, const uint32_t* mix_tlog, const uint64_t* mix_first_pos, const uint32_t* leaf,
                                     const uint64_t* count, uint64_t n_entries, uint64_t nnz_levels, const mgb_params* params,
                                     mgb_result** out)
{
    g_err[0] = 0;
    if (out) *out = nullptr;
    if (!leaf_segment_id || n_leaves == 0 || !handles || (n_mixtures && (!mix_offset || !mix_k || !mix_tlog || !mix_first_pos || !leaf || !count))) {
        set_error("mgb_build_from_levels: NULL argument or no leaves");
        return MGB_ERR_INVALID_ARG;
    }
    for (uint32_t k = 1; k < n_leaves; k++)
        if (leaf_segment_id[k] <= leaf_segment_id[k - 1]) {
            set_error("mgb_build_from_levels: leaf_segment_id must be strictly increasing");
            return MGB_ERR_INVALID_ARG;
        }
    LevelsFront lf{leaf_segment_id, n_leaves, level_done, handles, n_mixtures, mix_offset, mix_k, mix_tlog, mix_first_pos, leaf, count,
                   n_entries, nnz_levels};
    return build_volume(nullptr, X, Y, Z, nullptr, params, out, &lf);
}

extern "C" int mgb_get_front_mixture_nodes(const mgb_result* r, uint32_t* node_of_mixture)
{
    if (!r || (!node_of_mixture && !r->front_mixture_node.empty())) { set_error("mgb_get_front_mixture_nodes: NULL argument"); return MGB_ERR_INVALID_ARG; }
    if (!r->front_mixture_node.empty()) memcpy(node_of_mixture, r->front_mixture_node.data(), r->front_mixture_node.size() * sizeof(uint32_t));
    return MGB_OK;
}

extern "C" int mgb_build_from_mixtures(uint32_t n_leaves, uint64_t n_mixtures, const uint64_t* offsets,
                                       const uint32_t* leaf, const uint64_t* count, const mgb_params* params,
                                       mgb_result** out)
{
    g_err[0] = 0;
    if (!out) { set_error("mgb_build_from_mixtures: out is NULL"); return MGB_ERR_INVALID_ARG; }
    *out = nullptr;
    if (n_leaves == 0 || (n_mixtures && (!offsets || !leaf || !count))) { set_error("mgb_build_from_mixtures: NULL argument or no leaves"); return MGB_ERR_INVALID_ARG; }
    mgb_params p;
    int rc = check_params(params, p);
    if (rc != MGB_OK) return rc;
    mgb_result* R = nullptr;
    try {
        R = new mgb_result();
        const double t0 = now_s();
        // reduce (divide by the gcd) and hash-cons in order of first occurrence
        MixtureSet ms;
        ms.n_leaves = n_leaves;
        std::map<std::vector<uint64_t>, uint32_t> seen;   // flattened (leaf, count, ...) -> mixture number
        std::vector<uint32_t> ids(n_mixtures);
        uint64_t nnz = 0;
        for (uint64_t m = 0; m < n_mixtures; m++) {
            const uint64_t lo = offsets[m], hi = offsets[m + 1];
            if (hi <= lo) { delete R; set_error("mixture %llu is empty", (unsigned long long)m); return MGB_ERR_INVALID_ARG; }
            uint64_t g = 0;
            for (uint64_t t = lo; t < hi; t++) {
                if (leaf[t] >= n_leaves || count[t] == 0 || (t > lo && leaf[t] <= leaf[t - 1])) {
                    delete R; set_error("mixture %llu: entries must have increasing leaves < n_leaves and positive counts", (unsigned long long)m);
                    return MGB_ERR_INVALID_ARG;
                }
                g = std::gcd(g, count[t]);
            }
            nnz += hi - lo;
            if (hi - lo == 1) { ids[m] = leaf[lo]; continue; }
            std::vector<uint64_t> key;
            for (uint64_t t = lo; t < hi; t++) { key.push_back(leaf[t]); key.push_back(count[t] / g); }
            auto it = seen.find(key);
            if (it == seen.end()) {
                const uint32_t q = (uint32_t)ms.size();
                for (uint64_t t = lo; t < hi; t++) { ms.leaf.push_back(leaf[t]); ms.count.push_back(count[t] / g); }
                ms.off.push_back(ms.leaf.size());
                it = seen.emplace(std::move(key), q).first;
            }
            ids[m] = n_leaves + it->second;
        }
        const double t1 = now_s();
        Factorised F;
        rc = factorise(ms, p, F);
        if (rc != MGB_OK) { delete R; return rc; }
        const double t2 = now_s();
        std::vector<uint32_t> new_of_old;
        rc = finalise_graph(F, n_leaves, p, *R, new_of_old);
        if (rc != MGB_OK) { delete R; return rc; }
        for (uint64_t m = 0; m < n_mixtures; m++)
            ids[m] = new_of_old[ids[m] < n_leaves ? ids[m] : F.node_of_mix[ids[m] - n_leaves]];
        R->node_idx.resize(1);
        R->node_idx[0].swap(ids);
        R->dims = {n_mixtures, 1, 1};
        R->leaf_segment_id.resize(n_leaves);
        std::iota(R->leaf_segment_id.begin(), R->leaf_segment_id.end(), 0u);
        mgb_info& I = R->info;
        I.dims[0] = n_mixtures; I.dims[1] = 1; I.dims[2] = 1;
        I.n_mip_levels = 1;
        I.n_leaves = n_leaves;
        I.n_voxels_total = n_mixtures;
        I.quant_bits = p.quant_bits;
        I.n_distinct_mixtures = ms.size();
        I.nnz_total = nnz;
        I.n_stage1 = F.n_stage1; I.n_stage2 = F.n_stage2; I.n_big = F.n_big;
        I.phi2_exact = F.phi2_exact ? 1 : 0;
        I.seconds_mipmap = t1 - t0;
        I.seconds_factorise = t2 - t1;
        I.seconds_finalise = now_s() - t2;
    } catch (const std::bad_alloc&) {
        delete R;
        set_error("mgb_build_from_mixtures: out of host memory");
        return MGB_ERR_OOM;
    }
    *out = R;
    return MGB_OK;
}

extern "C" int mgb_get_info(const mgb_result* r, mgb_info* info)
{
    if (!r || !info) { set_error("mgb_get_info: NULL argument"); return MGB_ERR_INVALID_ARG; }
    *info = r->info;
    return MGB_OK;
}

extern "C" int mgb_mip_dims(const mgb_result* r, uint64_t* dims_out)
{
    if (!r || !dims_out) { set_error("mgb_mip_dims: NULL argument"); return MGB_ERR_INVALID_ARG; }
    memcpy(dims_out, r->dims.data(), r->dims.size() * sizeof(uint64_t));
    return MGB_OK;
}

extern "C" int mgb_get_graph(const mgb_result* r, uint32_t* child_a, uint32_t* child_b, float* weight,
                             double* weight_exact, uint64_t* level_offsets, uint32_t* leaf_segment_id)
{
    if (!r) { set_error("mgb_get_graph: NULL result"); return MGB_ERR_INVALID_ARG; }
    const size_t n = r->child_a.size();
    if (child_a) memcpy(child_a, r->child_a.data(), n * sizeof(uint32_t));
    if (child_b) memcpy(child_b, r->child_b.data(), n * sizeof(uint32_t));
    if (weight) memcpy(weight, r->weight.data(), n * sizeof(float));
    if (weight_exact) memcpy(weight_exact, r->weight_exact.data(), n * sizeof(double));
    if (level_offsets) memcpy(level_offsets, r->level_off.data(), r->level_off.size() * sizeof(uint64_t));
    if (leaf_segment_id) memcpy(leaf_segment_id, r->leaf_segment_id.data(), r->leaf_segment_id.size() * sizeof(uint32_t));
    return MGB_OK;
}

extern "C" const uint32_t* mgb_node_idx_ptr(const mgb_result* r, uint32_t level)
{
    if (!r || level >= r->node_idx.size()) { set_error("mgb_node_idx_ptr: bad level"); return nullptr; }
    if (r->node_idx[level].empty()) { set_error("mgb_node_idx_ptr: level %u is not stored (it was classified by the caller's front end)", level); return nullptr; }
    return r->node_idx[level].data();
}

extern "C" int mgb_get_node_idx(const mgb_result* r, uint32_t level, uint32_t* out)
{
    if (!r || !out || level >= r->node_idx.size()) { set_error("mgb_get_node_idx: bad argument"); return MGB_ERR_INVALID_ARG; }
    if (r->node_idx[level].empty()) { set_error("mgb_get_node_idx: level %u is not stored (it was classified by the caller's front end)", level); return MGB_ERR_INVALID_ARG; }
    memcpy(out, r->node_idx[level].data(), r->node_idx[level].size() * sizeof(uint32_t));
    return MGB_OK;
}

extern "C" int mgb_get_weight_sigma(const mgb_result* r, float* weight_sigma)
{
    if (!r || !weight_sigma) { set_error("mgb_get_weight_sigma: NULL argument"); return MGB_ERR_INVALID_ARG; }
    memcpy(weight_sigma, r->weight_sigma.data(), r->weight_sigma.size() * sizeof(float));
    return MGB_OK;
}

extern "C" int mgb_get_codebook(const mgb_result* r, float* codeword, float* sigma, uint64_t* count)
{
    if (!r) { set_error("mgb_get_codebook: NULL result"); return MGB_ERR_INVALID_ARG; }
    if (r->codeword.empty()) { set_error("mgb_get_codebook: unquantised build has no codebook"); return MGB_ERR_INVALID_ARG; }
    if (codeword) memcpy(codeword, r->codeword.data(), r->codeword.size() * sizeof(float));
    if (sigma) memcpy(sigma, r->sigma.data(), r->sigma.size() * sizeof(float));
    if (count) memcpy(count, r->bin_count.data(), r->bin_count.size() * sizeof(uint64_t));
    return MGB_OK;
}
