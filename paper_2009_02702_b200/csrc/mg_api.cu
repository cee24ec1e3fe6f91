// mg_api.cu -- graph object: validation, relabelling, device upload, info (include/mg.h).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "mg_internal.h"

namespace mg {

static thread_local char g_err[512] = "";
static std::atomic<uint64_t> g_launches{0};

void set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int cuda_fail(cudaError_t e, const char* what)
{
    set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    cudaGetLastError();   // clear the sticky-less error state
    return e == cudaErrorMemoryAllocation ? MG_ERR_OOM : MG_ERR_CUDA;
}

void count_launch(unsigned n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

int SmemAttrOnce::ensure(const void* func, int bytes, int device)
{
    const uint64_t bit = (device >= 0 && device < 64) ? (1ull << device) : 0;
    if (bit && (mask.load(std::memory_order_acquire) & bit)) return MG_OK;
    MG_CUDA(cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    if (bit) mask.fetch_or(bit, std::memory_order_release);
    return MG_OK;
}

int check_device(const mg_graph* g, const char* who)
{
    int dev = -1;
    MG_CUDA(cudaGetDevice(&dev));
    if (dev != g->device) {
        set_error("%s: the graph lives on CUDA device %d but device %d is current", who, g->device, dev);
        return MG_ERR_INVALID_ARG;
    }
    return MG_OK;
}

void invalidate_palettes_if_written(mg_graph* g, const void* p, uint64_t bytes)
{
    if (!g->pal_src) return;
    const uintptr_t a0 = (uintptr_t)p, a1 = a0 + bytes;
    const uintptr_t b0 = (uintptr_t)g->pal_src, b1 = b0 + g->n_nodes * 16;
    if (a0 < b1 && b0 < a1) g->pal_src = nullptr;
}

// Levels >= first_fused_level run inside ONE persistent CTA (k_tail) that works entirely in shared
// memory: the distinct "external" children (below the tail) are gathered once, then every level is
// smem gathers + a __syncthreads().  The tail is the longest suffix of levels whose working set fits:
//   16 B x (external children + tail nodes)  +  12 B x tail nodes (a, b, w staged)  <=  kTailSmemBytes
// and whose levels have at most kTailMaxLevelNodes nodes each (a bigger level is worth a full-grid launch).
static const uint64_t kTailMaxLevelNodes = 8192;
static const uint64_t kTailSmemBytes = MG_TAIL_SMEM_BYTES;

// ha / hb: host child arrays in library numbering.  Fills the plan and the local-index arrays.
static void plan_launches(mg_graph* g, const std::vector<uint32_t>& ha, const std::vector<uint32_t>& hb,
                          std::vector<uint32_t>& ext, std::vector<uint32_t>& la, std::vector<uint32_t>& lb)
{
    g->first_fused_level = 0;
    g->tail_base = (uint32_t)g->n_nodes;
    g->tail_n = g->tail_n_ext = 0;
    ext.clear(); la.clear(); lb.clear();
    // grow the tail downwards one level at a time, tracking the set of external children
    std::vector<uint32_t> cur_ext;                       // sorted distinct children below the current tail start
    uint32_t first = g->n_levels;
    for (uint32_t L = g->n_levels; L-- > 1;) {
        const uint64_t lo = g->level_off[L], hi = g->level_off[L + 1];
        if (hi - lo > kTailMaxLevelNodes || g->n_levels - L > MG_TAIL_MAX_LEVELS) break;
        std::vector<uint32_t> cand;
        cand.reserve(cur_ext.size() + 2 * (hi - lo));
        for (uint32_t e : cur_ext)
            if (e < lo) cand.push_back(e);               // nodes of level L stop being external
        for (uint64_t n = lo; n < hi; n++) { cand.push_back(ha[n]); cand.push_back(hb[n]); }   // all below lo (validated)
        std::sort(cand.begin(), cand.end());
        cand.erase(std::unique(cand.begin(), cand.end()), cand.end());
        const uint64_t T = g->n_nodes - lo;
        if (16 * (cand.size() + T) + 12 * T > kTailSmemBytes) break;
        cur_ext.swap(cand);
        first = L;
    }
    if (first >= g->n_levels) return;                    // no tail
    g->first_fused_level = first;
    g->tail_base = (uint32_t)g->level_off[first];
    g->tail_n = (uint32_t)(g->n_nodes - g->tail_base);
    g->tail_n_ext = (uint32_t)cur_ext.size();
    ext = cur_ext;
    la.resize(g->tail_n); lb.resize(g->tail_n);
    auto local = [&](uint32_t c) -> uint32_t {
        if (c >= g->tail_base) return g->tail_n_ext + (c - g->tail_base);
        return (uint32_t)(std::lower_bound(ext.begin(), ext.end(), c) - ext.begin());
    };
    for (uint32_t t = 0; t < g->tail_n; t++) { la[t] = local(ha[g->tail_base + t]); lb[t] = local(hb[g->tail_base + t]); }
}

template <typename T>
static int dev_alloc(mg_graph* g, T** p, uint64_t count)
{
    size_t bytes = (size_t)(count ? count : 1) * sizeof(T);
    bytes = (bytes + 255) & ~(size_t)255;
    MG_CUDA(cudaMalloc((void**)p, bytes));
    g->device_bytes += bytes;
    return MG_OK;
}

}  // namespace mg

using namespace mg;

extern "C" const char* mg_last_error(void) { return g_err; }
extern "C" uint64_t mg_kernel_launch_count(void) { return g_launches.load(); }

extern "C" void mg_free_graph(mg_graph* g)
{
    if (!g) return;
    int prev = 0;
    bool have = cudaGetDevice(&prev) == cudaSuccess;
    if (have) cudaSetDevice(g->device);
    cudaFree(g->d_a); cudaFree(g->d_b); cudaFree(g->d_w); cudaFree(g->d_level_off);
    cudaFree(g->d_new_of_old); cudaFree(g->d_tf_stage); cudaFree(g->d_pal8); cudaFree(g->d_pal16);
    cudaFree(g->d_tail_ext); cudaFree(g->d_tail_a); cudaFree(g->d_tail_b);
    if (have) cudaSetDevice(prev);
    cudaGetLastError();
    delete g;
}

extern "C" int mg_load_graph(const uint32_t* child_a, const uint32_t* child_b, const float* weight,
                             uint64_t n_nodes, uint32_t n_leaves, const uint64_t* level_offsets,
                             uint32_t n_topo_levels, const uint32_t* leaf_segment_id, uint32_t flags,
                             mg_graph** out)
{
    g_err[0] = 0;
    if (!out) { set_error("mg_load_graph: out is NULL"); return MG_ERR_INVALID_ARG; }
    *out = nullptr;
    if (n_leaves == 0 || n_nodes < n_leaves) { set_error("mg_load_graph: need 0 < n_leaves <= n_nodes"); return MG_ERR_INVALID_ARG; }
    if (n_nodes >= (1ull << 32)) { set_error("mg_load_graph: n_nodes must be < 2^32"); return MG_ERR_INVALID_ARG; }
    if (flags & ~(uint32_t)(MG_RELABEL | MG_NO_PALETTES)) { set_error("mg_load_graph: unknown flags 0x%x", flags); return MG_ERR_INVALID_ARG; }
    if (n_nodes > n_leaves && (!child_a || !child_b || !weight)) { set_error("mg_load_graph: NULL graph array"); return MG_ERR_INVALID_ARG; }
    const bool relabel = (flags & MG_RELABEL) != 0;
    if (!relabel && !level_offsets) { set_error("mg_load_graph: level_offsets is NULL without MG_RELABEL"); return MG_ERR_INVALID_ARG; }

    // ---- validation that does not depend on the numbering (I2: a != b, children precede, 0 < w < 1)
    for (uint64_t n = n_leaves; n < n_nodes; n++) {
        uint32_t a = child_a[n], b = child_b[n];
        float w = weight[n];
        if (a >= n || b >= n) { set_error("node %llu: child (%u, %u) does not precede it (Eq. 8)", (unsigned long long)n, a, b); return MG_ERR_INVALID_GRAPH; }
        if (a == b) { set_error("node %llu: both children are node %u", (unsigned long long)n, a); return MG_ERR_INVALID_GRAPH; }
        if (!(w > 0.0f && w < 1.0f)) { set_error("node %llu: weight %g outside the open interval (0,1) (L176)", (unsigned long long)n, (double)w); return MG_ERR_INVALID_GRAPH; }
    }
    if (leaf_segment_id)
        for (uint32_t k = 1; k < n_leaves; k++)
            if (leaf_segment_id[k] <= leaf_segment_id[k - 1]) { set_error("leaf_segment_id not strictly increasing at %u", k); return MG_ERR_INVALID_GRAPH; }

    mg_graph* g = new (std::nothrow) mg_graph();
    if (!g) { set_error("mg_load_graph: host allocation failed"); return MG_ERR_OOM; }
    g->n_nodes = n_nodes;
    g->n_leaves = n_leaves;
    g->no_palettes = (flags & MG_NO_PALETTES) != 0;
    if (const char* e = getenv("MG_COLORIZE_TILE_BYTES")) {               // read here, once per graph: never on the update path
        const long long v = atoll(e);
        if (v > 0) g->pal_tile_bytes = (uint64_t)v;
    }
    if (leaf_segment_id) g->leaf_segment_id.assign(leaf_segment_id, leaf_segment_id + n_leaves);

    std::vector<uint32_t> ha, hb;
    std::vector<float> hw;
    try {
        if (relabel) {
            if (relabel_by_level(child_a, child_b, n_nodes, n_leaves, g->new_of_old, g->level_off) != 0) {
                set_error("mg_load_graph: relabel failed (graph not children-before-parents)");
                delete g; return MG_ERR_INVALID_GRAPH;
            }
            g->n_levels = (uint32_t)g->level_off.size() - 1;
            ha.assign(n_nodes, 0); hb.assign(n_nodes, 0); hw.assign(n_nodes, 0.0f);
            const std::vector<uint32_t>& p = g->new_of_old;
#pragma omp parallel for schedule(static)
            for (int64_t n = n_leaves; n < (int64_t)n_nodes; n++) {
                uint32_t q = p[n];
                ha[q] = p[child_a[n]]; hb[q] = p[child_b[n]]; hw[q] = weight[n];
            }
        } else {
            if (n_topo_levels == 0) { set_error("mg_load_graph: n_topo_levels is 0"); delete g; return MG_ERR_INVALID_ARG; }
            g->n_levels = n_topo_levels;
            g->level_off.assign(level_offsets, level_offsets + n_topo_levels + 1);
            if (g->level_off[0] != 0 || g->level_off[1] != n_leaves || g->level_off[n_topo_levels] != n_nodes) {
                set_error("level_offsets must start 0, n_leaves and end n_nodes"); delete g; return MG_ERR_INVALID_GRAPH;
            }
            for (uint32_t L = 0; L < n_topo_levels; L++)
                if (g->level_off[L + 1] <= g->level_off[L]) { set_error("level %u is empty or offsets decrease", L); delete g; return MG_ERR_INVALID_GRAPH; }
            // level = max(level(a), level(b)) + 1 (L211): both children below off[L], one at or above off[L-1]
            for (uint32_t L = 1; L < n_topo_levels; L++) {
                uint64_t lo = g->level_off[L], prev = g->level_off[L - 1];
                for (uint64_t n = lo; n < g->level_off[L + 1]; n++) {
                    uint32_t a = child_a[n], b = child_b[n];
                    uint32_t mx = a > b ? a : b;
                    if (mx >= lo || mx < prev) {
                        set_error("node %llu (level %u): children (%u, %u) violate level = max + 1 (L211)", (unsigned long long)n, L, a, b);
                        delete g; return MG_ERR_INVALID_GRAPH;
                    }
                }
            }
            ha.assign(child_a, child_a + n_nodes); hb.assign(child_b, child_b + n_nodes); hw.assign(weight, weight + n_nodes);
            for (uint32_t n = 0; n < n_leaves; n++) { ha[n] = 0; hb[n] = 0; hw[n] = 0.0f; }
        }
    } catch (const std::bad_alloc&) {
        set_error("mg_load_graph: host allocation failed"); delete g; return MG_ERR_OOM;
    }
    std::vector<uint32_t> t_ext, t_a, t_b;
    try {
        plan_launches(g, ha, hb, t_ext, t_a, t_b);
    } catch (const std::bad_alloc&) {
        set_error("mg_load_graph: host allocation failed"); delete g; return MG_ERR_OOM;
    }

    // ---- device upload
    int rc = MG_OK;
    cudaError_t e = cudaGetDevice(&g->device);
    if (e != cudaSuccess) { rc = cuda_fail(e, "cudaGetDevice"); delete g; return rc; }
    std::vector<uint32_t> off32(g->level_off.begin(), g->level_off.end());
#define MG_TRY(x) do { rc = (x); if (rc != MG_OK) { mg_free_graph(g); return rc; } } while (0)
#define MG_TRY_CUDA(x) do { cudaError_t e2 = (x); if (e2 != cudaSuccess) { rc = cuda_fail(e2, #x); mg_free_graph(g); return rc; } } while (0)
    MG_TRY(dev_alloc(g, &g->d_a, n_nodes + 4));       // +4: vector loads of the last partial group
    MG_TRY(dev_alloc(g, &g->d_b, n_nodes + 4));
    MG_TRY(dev_alloc(g, &g->d_w, n_nodes + 4));
    MG_TRY(dev_alloc(g, &g->d_level_off, off32.size()));
    MG_TRY(dev_alloc(g, &g->d_tf_stage, (uint64_t)n_leaves * 4));
    MG_TRY(dev_alloc(g, &g->d_pal8, n_nodes + 4));
    MG_TRY(dev_alloc(g, &g->d_pal16, n_nodes + 4));
    MG_TRY_CUDA(cudaMemset(g->d_a, 0, (n_nodes + 4) * 4));
    MG_TRY_CUDA(cudaMemset(g->d_b, 0, (n_nodes + 4) * 4));
    MG_TRY_CUDA(cudaMemset(g->d_w, 0, (n_nodes + 4) * 4));
    MG_TRY_CUDA(cudaMemcpy(g->d_a, ha.data(), n_nodes * 4, cudaMemcpyHostToDevice));
    MG_TRY_CUDA(cudaMemcpy(g->d_b, hb.data(), n_nodes * 4, cudaMemcpyHostToDevice));
    MG_TRY_CUDA(cudaMemcpy(g->d_w, hw.data(), n_nodes * 4, cudaMemcpyHostToDevice));
    MG_TRY_CUDA(cudaMemcpy(g->d_level_off, off32.data(), off32.size() * 4, cudaMemcpyHostToDevice));
    if (g->tail_n) {
        MG_TRY(dev_alloc(g, &g->d_tail_ext, t_ext.size()));
        MG_TRY(dev_alloc(g, &g->d_tail_a, t_a.size()));
        MG_TRY(dev_alloc(g, &g->d_tail_b, t_b.size()));
        if (!t_ext.empty()) MG_TRY_CUDA(cudaMemcpy(g->d_tail_ext, t_ext.data(), t_ext.size() * 4, cudaMemcpyHostToDevice));
        MG_TRY_CUDA(cudaMemcpy(g->d_tail_a, t_a.data(), t_a.size() * 4, cudaMemcpyHostToDevice));
        MG_TRY_CUDA(cudaMemcpy(g->d_tail_b, t_b.data(), t_b.size() * 4, cudaMemcpyHostToDevice));
    }
    if (relabel) {
        MG_TRY(dev_alloc(g, &g->d_new_of_old, n_nodes));
        MG_TRY_CUDA(cudaMemcpy(g->d_new_of_old, g->new_of_old.data(), n_nodes * 4, cudaMemcpyHostToDevice));
    }
#undef MG_TRY
#undef MG_TRY_CUDA
    *out = g;
    return MG_OK;
}

extern "C" int mg_graph_info(const mg_graph* g, mg_info* info)
{
    if (!g || !info) { set_error("mg_graph_info: NULL argument"); return MG_ERR_INVALID_ARG; }
    info->n_nodes = g->n_nodes;
    info->n_internal = g->n_nodes - g->n_leaves;
    info->n_leaves = g->n_leaves;
    info->depth = g->n_levels - 1;
    info->n_topo_levels = g->n_levels;
    info->first_fused_level = g->first_fused_level;
    uint32_t big = (g->first_fused_level ? g->first_fused_level : g->n_levels) - 1;   // levels 1 .. first_fused-1
    info->n_launches_propagate = (big ? big : 0) + (g->first_fused_level ? 1 : 0) + ((big == 0 && !g->first_fused_level) ? 1 : 0);
    info->relabelled = g->new_of_old.empty() ? 0 : 1;
    info->device_bytes = g->device_bytes;
    return MG_OK;
}

extern "C" int mg_level_offsets(const mg_graph* g, uint64_t* level_offsets_host)
{
    if (!g || !level_offsets_host) { set_error("mg_level_offsets: NULL argument"); return MG_ERR_INVALID_ARG; }
    memcpy(level_offsets_host, g->level_off.data(), g->level_off.size() * sizeof(uint64_t));
    return MG_OK;
}

extern "C" int mg_node_permutation(const mg_graph* g, uint32_t* new_of_old_host)
{
    if (!g || !new_of_old_host) { set_error("mg_node_permutation: NULL argument"); return MG_ERR_INVALID_ARG; }
    if (g->new_of_old.empty())
        for (uint64_t n = 0; n < g->n_nodes; n++) new_of_old_host[n] = (uint32_t)n;
    else
        memcpy(new_of_old_host, g->new_of_old.data(), g->n_nodes * sizeof(uint32_t));
    return MG_OK;
}

__global__ void __launch_bounds__(256) k_relabel_indices(uint32_t* __restrict__ idx, uint64_t n,
                                                          const uint32_t* __restrict__ new_of_old)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
        idx[i] = __ldg(new_of_old + idx[i]);
}

__global__ void __launch_bounds__(256) k_check_indices(const uint32_t* __restrict__ idx, uint64_t n, uint32_t n_nodes, unsigned long long* bad)
{
    unsigned c = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) c += __ldcs(idx + i) >= n_nodes;
    c = __reduce_add_sync(0xffffffffu, c);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(bad, (unsigned long long)c);
}

extern "C" int mg_check_indices(const mg_graph* g, const uint32_t* node_idx_device, uint64_t n, uint64_t* n_bad_host, void* stream)
{
    if (!g || !n_bad_host || (!node_idx_device && n)) { set_error("mg_check_indices: NULL argument"); return MG_ERR_INVALID_ARG; }
    *n_bad_host = 0;
    if (n == 0) return MG_OK;
    const int rc = check_device(g, "mg_check_indices");
    if (rc != MG_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* d_bad = nullptr;
    MG_CUDA(cudaMalloc((void**)&d_bad, sizeof(unsigned long long)));
    cudaError_t e = cudaMemsetAsync(d_bad, 0, sizeof(unsigned long long), st);
    unsigned long long bad = 0;
    if (e == cudaSuccess) {
        const unsigned blocks = (unsigned)std::min<uint64_t>((n + 255) / 256, 148ull * 16);
        k_check_indices<<<blocks, 256, 0, st>>>(node_idx_device, n, (uint32_t)g->n_nodes, d_bad);
        count_launch();
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, d_bad, sizeof(bad), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d_bad);
    if (e != cudaSuccess) return cuda_fail(e, "mg_check_indices");
    *n_bad_host = bad;
    return MG_OK;
}

extern "C" int mg_relabel_indices(mg_graph* g, uint32_t* idx_device, uint64_t n, void* stream)
{
    if (!g || (!idx_device && n)) { set_error("mg_relabel_indices: NULL argument"); return MG_ERR_INVALID_ARG; }
    if (!g->d_new_of_old || n == 0) return MG_OK;
    const int rc = check_device(g, "mg_relabel_indices");
    if (rc != MG_OK) return rc;
    uint64_t blocks = (n + 255) / 256;
    if (blocks > 148ull * 64) blocks = 148ull * 64;
    k_relabel_indices<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(idx_device, n, g->d_new_of_old);
    count_launch();
    MG_CUDA(cudaGetLastError());
    return MG_OK;
}
