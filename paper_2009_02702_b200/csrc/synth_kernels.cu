// synth_kernels.cu -- GPU versions of the seeded volume generators of synth.py (libmg_synth.so).
//
// Input generation only: NONE of the method's arithmetic lives here (no histogram, no lerp).  The
// full-size configs need ~10^12 exact integer distance evaluations, too slow for numpy; these
// kernels evaluate the SAME recipes (same counter-based generator, same exact integer predicates,
// same tie-breaks), so the result is bit-identical to synth.voronoi_volume / synth.cylinder_volume.
// tests/test_synth_gpu.py compares the two on crops.
//
// C ABI (all volume pointers DEVICE, [Z][Y][X] x fastest; returns 0 or a negative cudaError):
//   mgs_voronoi    label = argmin_k dx^2 + dy^2 + (zscale dz)^2, ties -> lowest k, optional jitter
//   mgs_cylinders  label = 1 + the LAST cylinder containing the voxel (later overwrite earlier), else 0
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__host__ __device__ __forceinline__ uint64_t splitmix64(uint64_t x)
{
    uint64_t z = x + 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

constexpr int kSeedChunk = 2048;   // seeds staged in shared memory per pass (int4 each = 32 KB)

// One thread = one voxel of the region.  Distances in int64 (exact for any dims < 2^20).
// JITTER: the query point of voxel p is clamp(p + j(p)), j from a hash of the GLOBAL linear index.
template <bool JITTER, typename D>
__global__ void __launch_bounds__(256)
k_voronoi(const int4* __restrict__ seeds, int n_seeds, int X, int Y, int Z, int zscale, int amp, uint64_t key,
          int x0, int y0, int z0, int rx, int ry, int rz, uint32_t* __restrict__ out)
{
    __shared__ int4 s_seed[kSeedChunk];
    const int64_t n_region = (int64_t)rx * ry * rz;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = t < n_region;
    int qx = 0, qy = 0, qz = 0;
    if (live) {
        const int lx = (int)(t % rx), ly = (int)((t / rx) % ry), lz = (int)(t / ((int64_t)rx * ry));
        qx = x0 + lx; qy = y0 + ly; qz = z0 + lz;
        if (JITTER) {
            const uint64_t lin = ((uint64_t)qz * Y + qy) * X + qx;
            const uint64_t h = splitmix64(key + lin);
            const uint64_t m = 2 * amp + 1;
            const int jx = (int)(h % m) - amp, jy = (int)((h >> 16) % m) - amp, jz = (int)((h >> 32) % m) - amp;
            qx = min(max(qx + jx, 0), X - 1);
            qy = min(max(qy + jy, 0), Y - 1);
            qz = min(max(qz + jz, 0), Z - 1);
        }
    }
    D best = 0;
    uint32_t best_k = 0;
    bool have = false;
    for (int base = 0; base < n_seeds; base += kSeedChunk) {
        const int cnt = min(kSeedChunk, n_seeds - base);
        __syncthreads();
        for (int i = threadIdx.x; i < cnt; i += blockDim.x) s_seed[i] = seeds[base + i];
        __syncthreads();
        if (live) {
            for (int i = 0; i < cnt; i++) {
                const int4 s = s_seed[i];
                const D dx = qx - s.x, dy = qy - s.y, dz = (D)zscale * (qz - s.z);
                const D d = dx * dx + dy * dy + dz * dz;
                if (!have || d < best) { best = d; best_k = base + i; have = true; }   // strict <: lowest index wins ties
            }
        }
    }
    if (live) out[t] = best_k;
}

// Cylinders: the host bins them into tiles of kTile^3 voxels (conservative bounding boxes, CSR
// lists with ascending cylinder numbers); one CTA = one tile; a voxel scans its tile's list from
// the back and stops at the first hit (= the last cylinder that contains it).
constexpr int kTile = 8;

struct Cyl { long long cx, cy, cz, ax, ay, az, r16, L; };

__global__ void __launch_bounds__(kTile * kTile * kTile)
k_cylinders(const Cyl* __restrict__ cyl, const uint32_t* __restrict__ tile_off, const uint32_t* __restrict__ tile_list,
            int tx_n, int ty_n, int x0, int y0, int z0, int rx, int ry, int rz, uint32_t* __restrict__ out)
{
    const int tile = blockIdx.x;
    const int tx = tile % tx_n, ty = (tile / tx_n) % ty_n, tz = tile / (tx_n * ty_n);
    const int lx = tx * kTile + threadIdx.x % kTile;
    const int ly = ty * kTile + (threadIdx.x / kTile) % kTile;
    const int lz = tz * kTile + threadIdx.x / (kTile * kTile);
    if (lx >= rx || ly >= ry || lz >= rz) return;
    const long long px = x0 + lx, py = y0 + ly, pz = z0 + lz;
    uint32_t label = 0;
    const uint32_t lo = tile_off[tile], hi = tile_off[tile + 1];
    for (uint32_t e = hi; e-- > lo;) {
        const uint32_t k = tile_list[e];
        const Cyl c = cyl[k];
        const long long dx = px - c.cx, dy = py - c.cy, dz = pz - c.cz;
        const long long a2 = c.ax * c.ax + c.ay * c.ay + c.az * c.az;
        const long long t = dx * c.ax + dy * c.ay + dz * c.az;
        const long long d2 = dx * dx + dy * dy + dz * dz;
        if (4 * t * t <= c.L * c.L * a2 && 256 * (d2 * a2 - t * t) <= c.r16 * c.r16 * a2) { label = k + 1; break; }
    }
    out[((int64_t)lz * ry + ly) * rx + lx] = label;
}

}  // namespace

extern "C" {

// seeds: DEVICE int32[n_seeds][4] (x, y, z, unused).  region = {z0, z1, y0, y1, x0, x1} (host).
// out: DEVICE uint32[(z1-z0)*(y1-y0)*(x1-x0)].  jitter_key = splitmix64-derived stream key (synth.stream_key(seed, 2)).
int mgs_voronoi(const int32_t* seeds, int32_t n_seeds, int32_t X, int32_t Y, int32_t Z, int32_t zscale, int32_t jitter,
                uint64_t jitter_key, const int32_t* region, uint32_t* out, void* stream)
{
    const int z0 = region[0], z1 = region[1], y0 = region[2], y1 = region[3], x0 = region[4], x1 = region[5];
    const int rx = x1 - x0, ry = y1 - y0, rz = z1 - z0;
    const int64_t n = (int64_t)rx * ry * rz;
    if (n <= 0) return 0;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    const int4* s4 = reinterpret_cast<const int4*>(seeds);
    cudaStream_t st = (cudaStream_t)stream;
    // 32-bit distances are exact when 3 * max(extent)^2 < 2^31
    const int64_t ext = (int64_t)(X > Y ? X : Y) > (int64_t)zscale * Z ? (X > Y ? X : Y) : (int64_t)zscale * Z;
    const bool small = 3 * ext * ext < (1ll << 31);
    if (jitter > 0) {
        if (small) k_voronoi<true, int><<<blocks, 256, 0, st>>>(s4, n_seeds, X, Y, Z, zscale, jitter, jitter_key, x0, y0, z0, rx, ry, rz, out);
        else k_voronoi<true, long long><<<blocks, 256, 0, st>>>(s4, n_seeds, X, Y, Z, zscale, jitter, jitter_key, x0, y0, z0, rx, ry, rz, out);
    } else {
        if (small) k_voronoi<false, int><<<blocks, 256, 0, st>>>(s4, n_seeds, X, Y, Z, zscale, 0, 0, x0, y0, z0, rx, ry, rz, out);
        else k_voronoi<false, long long><<<blocks, 256, 0, st>>>(s4, n_seeds, X, Y, Z, zscale, 0, 0, x0, y0, z0, rx, ry, rz, out);
    }
    return -(int)cudaGetLastError();
}

// cyl: DEVICE int64[n][8] (cx, cy, cz, ax, ay, az, r16, L); tile_off: DEVICE uint32[n_tiles + 1];
// tile_list: DEVICE uint32[tile_off[n_tiles]] ascending inside each tile.  Tiles are 8^3 voxels of the
// region, x fastest: n_tiles = ceil(rx/8) * ceil(ry/8) * ceil(rz/8).
int mgs_cylinders(const int64_t* cyl, const uint32_t* tile_off, const uint32_t* tile_list, const int32_t* region,
                  uint32_t* out, void* stream)
{
    const int z0 = region[0], z1 = region[1], y0 = region[2], y1 = region[3], x0 = region[4], x1 = region[5];
    const int rx = x1 - x0, ry = y1 - y0, rz = z1 - z0;
    if (rx <= 0 || ry <= 0 || rz <= 0) return 0;
    const int tx = (rx + kTile - 1) / kTile, ty = (ry + kTile - 1) / kTile, tz = (rz + kTile - 1) / kTile;
    k_cylinders<<<(unsigned)(tx * ty * tz), kTile * kTile * kTile, 0, (cudaStream_t)stream>>>(
        reinterpret_cast<const Cyl*>(cyl), tile_off, tile_list, tx, ty, x0, y0, z0, rx, ry, rz, out);
    return -(int)cudaGetLastError();
}

int mgs_tile_size(void) { return kTile; }

}  // extern "C"
