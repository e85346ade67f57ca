// The streaming skeleton shared by the two HBM-bound kernels of the hot path (a-1 warp.cu, a-4
// gradient.cu): both make one pass over the K+1 planar vector fields (Eq. 1:
// x = xbar + sum_k u_k w_k needs all of them per voxel) and then chase 8-tap gathers in f0.
//
// A persistent CTA per SM, made of consumer groups of 8 warps that take the CTA's tiles in turn.
// Field tiles come HBM -> shared memory by TMA (cp.async.bulk.tensor, one 4-D box
// {TX x, 1 y, TZ z, 3(K+1) planes} per tile, completion signalled on an mbarrier), issued by the
// group's leader one or two tiles ahead.  The stream is thereby decoupled from the dependent chain
// (fields -> displaced position -> f0 gathers -> interpolation), which is what kept the first,
// register-staged version of these kernels at 35 % of the DRAM bandwidth (profiles/r01a).
//
// Tile = TX = 32 voxels along x, TZ along z, at fixed y: loads are 128 B rows of each plane, and
// the warp kernel's transposed store (z fastest, ray layout) is one 128 B line per (x, y).
#pragma once

#include <cuda.h>
#include <cuda_fp16.h>

#include <string>

#include "common.cuh"

namespace pcamm {

constexpr int TX = 32;             // tile extent along x
constexpr int GROUP_WARPS = 8;     // warps of a consumer group
constexpr int GROUP_THREADS = 32 * GROUP_WARPS;

// Tile t of the volume (x tiles fastest, then y, then z tiles: the CTAs that run side by side
// read neighbouring rows of the same z slices).
struct TileCoord {
    int x0, y, z0;
};

__host__ __device__ __forceinline__ int tiles_x(const Geom& G) { return (G.nx + TX - 1) / TX; }
__host__ __device__ __forceinline__ int tiles_z(const Geom& G, int tz) { return (G.nz + tz - 1) / tz; }
__host__ __device__ __forceinline__ long long tile_count(const Geom& G, int tz) {
    return (long long)tiles_x(G) * G.ny * tiles_z(G, tz);
}
// (t < 2^31: pcamm_model_create bounds the volume.)  The two divisions are multiplications by
// M = ceil(2^32 / d), exact for every t with t d < 2^32 (t M / 2^32 = t / d + t r / (d 2^32) with
// r = M d - 2^32 < d); the host sets the multipliers to 0 where that does not hold (tile_multipliers).
__device__ __forceinline__ TileCoord tile_coord(const Geom& G, int tz, long long t64) {
    const unsigned t = (unsigned)t64, ntx = (unsigned)tiles_x(G);
    const unsigned row = G.tile_mx ? __umulhi(t, G.tile_mx) : t / ntx;                   // (y, z tile)
    const unsigned zt = G.tile_my ? __umulhi(row, G.tile_my) : row / (unsigned)G.ny;
    TileCoord c;
    c.x0 = (int)(t - row * ntx) * TX;
    c.y = (int)(row - zt * (unsigned)G.ny);
    c.z0 = (int)zt * tz;
    return c;
}
inline void tile_multipliers(Geom& G) {
    const unsigned long long n_max = (unsigned long long)tile_count(G, 16), ntx = (unsigned long long)tiles_x(G), ny = (unsigned long long)G.ny;
    G.tile_mx = (ntx >= 2 && n_max * ntx < (1ull << 32)) ? (unsigned)(((1ull << 32) + ntx - 1) / ntx) : 0u;
    G.tile_my = (ny >= 2 && n_max * ny < (1ull << 32)) ? (unsigned)(((1ull << 32) + ny - 1) / ny) : 0u;
}

// ---------------------------------------------------------------- mbarrier / TMA (PTX)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    const uint32_t addr = smem_u32(bar);
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(addr), "r"(parity)
            : "memory");
    } while (!done);
}

// One 4-D box of the field tensor {x, y, z, plane} -> shared memory, evict-first in L2 (the
// fields are streamed once per pass and must not push f0 and the trial volumes out of L2).
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2,
                                            int c3, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5, %6}], [%2], %7;"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(policy)
        : "memory");
}
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ float lds_f32(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ float lds_f16(uint32_t addr) {
    unsigned short h;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(h) : "r"(addr));
    return __half2float(__ushort_as_half(h));
}
__device__ __forceinline__ void group_barrier(int group) {
    asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "n"(GROUP_THREADS) : "memory");
}

// Shared-memory stages of a streaming kernel: NG consumer groups with SPG stages each, a stage
// being P planes x TZ x TX floats.  The CTA's i-th tile (tile blockIdx.x + i * gridDim.x of the
// volume) belongs to group i % NG and is that group's (i / NG)-th tile; it goes through stage
// (i / NG) % SPG of the group's own little ring.  Every stage is filled and drained by ONE group,
// strictly in order: the group's leader thread issues the TMA load of the group's tile j + SPG
// into a stage as soon as the group has read tile j's fields out of it (a group barrier), so no
// "empty" barrier and no producer warp are needed, and waiting on the phase parity of the "full"
// barrier is sound (a group sharing stages with others could be a whole ring cycle ahead of the
// barrier it polls and mistake the previous phase for its own).
//
// H (reduced-precision storage): the stage holds xbar's three planes in float and
// the 3K planes of u_1 .. u_K in half (each u_k scaled by a power of two, common.cuh FieldScale),
// filled by two TMA loads from two tensors that complete on the same barrier.
template <int P, int TZ, int NG, int SPG, bool H = false>
struct FieldRing {
    static constexpr int NS = NG * SPG;
    static constexpr uint32_t XBAR_BYTES = 3u * TZ * TX * 4u;
    static constexpr uint32_t STAGE_BYTES = H ? XBAR_BYTES + (uint32_t)(P - 3) * TZ * TX * 2u : (uint32_t)P * TZ * TX * 4u;
    static constexpr size_t BYTES = (size_t)NS * STAGE_BYTES + NS * sizeof(uint64_t);

    unsigned char* data;   // 128 B aligned
    uint64_t* full;        // [NS] TMA completion

    __device__ __forceinline__ void bind(unsigned char* smem) {
        data = smem;
        full = reinterpret_cast<uint64_t*>(smem + (size_t)NS * STAGE_BYTES);
    }
    __device__ __forceinline__ void init() {   // one thread
        for (int s = 0; s < NS; ++s) mbar_init(full + s, 1);
        mbar_fence_init();
    }
    __device__ __forceinline__ const unsigned char* stage(int s) const { return data + (size_t)s * STAGE_BYTES; }

    // Shared-memory reads of a stage at byte address sf: component cc of xbar / of u_k at row zz, column x.
    __device__ __forceinline__ static float xbar_at(uint32_t sf, int cc, int zz, int x) {
        return lds_f32(sf + 4u * ((cc * TZ + zz) * TX + x));
    }
    __device__ __forceinline__ static float u_at(uint32_t sf, int k, int cc, int zz, int x) {
        if (H) return lds_f16(sf + XBAR_BYTES + 2u * (((3 * k + cc) * TZ + zz) * TX + x));
        return lds_f32(sf + 4u * (((3 + 3 * k + cc) * TZ + zz) * TX + x));
    }

    // Tile of the volume that is group g's j-th tile in this CTA (may be >= the tile count).
    __device__ __forceinline__ static long long tile_of(int g, int j) {
        return (long long)blockIdx.x + ((long long)g + (long long)j * NG) * gridDim.x;
    }
    __device__ __forceinline__ static int stage_of(int g, int j) { return g * SPG + j % SPG; }
    __device__ __forceinline__ static uint32_t parity_of(int j) { return (uint32_t)(j / SPG) & 1u; }

    // Group leader: start the load of the group's j-th tile (nothing if the volume has no such tile).
    // map: all P planes in float (H = false) or xbar's three planes; umap: the half planes (H only).
    __device__ __forceinline__ void issue(const CUtensorMap* map, const CUtensorMap* umap, const Geom& G,
                                          long long n_tiles, int g, int j, uint64_t policy) const {
        const long long t = tile_of(g, j);
        if (t >= n_tiles) return;
        const int s = stage_of(g, j);
        const TileCoord c = tile_coord(G, TZ, t);
        mbar_arrive_expect_tx(full + s, STAGE_BYTES);
        tma_load_4d(data + (size_t)s * STAGE_BYTES, map, full + s, c.x0, c.y, c.z0, 0, policy);
        if (H) tma_load_4d(data + (size_t)s * STAGE_BYTES + XBAR_BYTES, umap, full + s, c.x0, c.y, c.z0, 0, policy);
    }
    // Group leader: start the load of tile t of the volume into stage s of the ring.
    __device__ __forceinline__ void issue_tile(const CUtensorMap* map, const CUtensorMap* umap, const Geom& G,
                                               long long t, int s, uint64_t policy) const {
        const TileCoord c = tile_coord(G, TZ, t);
        mbar_arrive_expect_tx(full + s, STAGE_BYTES);
        tma_load_4d(data + (size_t)s * STAGE_BYTES, map, full + s, c.x0, c.y, c.z0, 0, policy);
        if (H) tma_load_4d(data + (size_t)s * STAGE_BYTES + XBAR_BYTES, umap, full + s, c.x0, c.y, c.z0, 0, policy);
    }
    // Group leader, once: the first SPG tiles.
    __device__ __forceinline__ void prologue(const CUtensorMap* map, const CUtensorMap* umap, const Geom& G,
                                             long long n_tiles, int g, uint64_t policy) const {
        for (int j = 0; j < SPG; ++j) issue(map, umap, G, n_tiles, g, j, policy);
    }
};

// Reduced-precision storage of u_k: half(u_k / h * scale[k]), scale a power of two chosen at
// model_create so that the largest entry of u_k lands in [0.25, 0.5); inv[k] = 1 / scale[k].
// Eq. (1) then uses w_k * inv[k] (exact), and the K gradient sums are multiplied by inv[k].
struct FieldScale {
    float inv[KMAX];
};

// Largest magnitude of every plane of the fields (voxel units; as the kernels read them):
// |d_c| <= v[c] + sum_k |w_k| v[3 + 3k + c] bounds the displacement of Eq. (1) anywhere.
struct FieldMax {
    float v[3 * (KMAX + 1)];
};

// Summed-volume table of a 0/1 map over [0, ex) x [0, ey) x [0, ez): element ((z (ey + 1)) + y)(ex + 1) + x
// holds the number of ones in [0, x) x [0, y) x [0, z) (mod 2^32).  Ones in the inclusive box
// [xl, xh] x [yl, yh] x [zl, zh] (already clipped to the map, non-empty):
__device__ __forceinline__ unsigned box_count(const unsigned* __restrict__ I, int ex, int ey, int xl, int xh, int yl,
                                              int yh, int zl, int zh) {
    const unsigned px = (unsigned)(ex + 1), pp = px * (unsigned)(ey + 1);
    const unsigned x0 = (unsigned)xl, x1 = (unsigned)xh + 1u, y0 = (unsigned)yl * px, y1 = ((unsigned)yh + 1u) * px;
    const unsigned z0 = (unsigned)zl * pp, z1 = ((unsigned)zh + 1u) * pp;
    return __ldg(I + z1 + y1 + x1) - __ldg(I + z1 + y1 + x0) - __ldg(I + z1 + y0 + x1) - __ldg(I + z0 + y1 + x1) +
           __ldg(I + z1 + y0 + x0) + __ldg(I + z0 + y1 + x0) + __ldg(I + z0 + y0 + x1) - __ldg(I + z0 + y0 + x0);
}

// The tile flags cost a few dependent loads at the start of a launch: they are used where a CTA
// has at least this many tiles to win them back on.
constexpr int SKIP_MIN_TILES_PER_SM = 12;

// Reach of a tile's interpolation stencils: per axis the largest |floor(d)| any voxel can have,
// from the bound on |d| (a small margin covers the float rounding of Eq. (1)).
// Clamped to 2^20 voxels (beyond any grid every stencil is outside anyway; a huge or non-finite
// bound must not wrap the int box arithmetic of the tile flags: it then simply covers the volume).
__device__ __forceinline__ int reach_of(float dmax) { return (int)ceilf(fminf(dmax * 1.0001f + 0.001f, 1048576.f)); }

// Records of the voxels whose interpolation cell is not constant (single-solve path; warp.cu writes
// them, gradient.cu k_grad_gather reads them).  The warp kernel has, for every voxel of a trial
// volume, the eight taps of f0 and the three fractions in registers: G_j = df_j / dx_j is a function of
// those eleven numbers, and it is exactly 0 where the eight taps are equal.  So it writes, per trial
// slot, one record for every voxel whose taps differ (boundary voxels: 6 % at C2), and the gradient of
// the accepted candidate needs no second pass over the K+1 fields: G_j from the record, B_j and u_kj
// at the recorded voxels.  (The record holds the taps, not G_j: a warp row usually has one or two such
// voxels, and forming G_j there would cost the whole warp its 40 instructions for them; the gather
// forms it with every lane busy.)
// Layout per slot: a tile is cut into GROUP_WARPS sub-tiles (the voxels one warp of the consumer
// group handles: TX x TZ / GROUP_WARPS = `cap` of them, so a sub-tile cannot overflow); sub-tile s
// owns records s cap .. s cap + count[s] - 1, in the fixed order (lane, row).  A record is 48 bytes
// (three 16-byte stores / loads).
struct GradRecord {
    int xyz;           // x | y << 11 | z << 22 (pcamm_model_create: records only for nx, ny <= 2048, nz <= 1024)
    float tx, ty, tz;  // fractions of the displaced position in its cell (trilinear.cuh Taps: w1 = t, w0 = 1 - t)
    float c[8];        // the cell's taps of f0, in gather8's order
};
constexpr int RECORD_WORDS = 12;
constexpr int RECORD_MAX_XY = 2048, RECORD_MAX_Z = 1024;
constexpr int RECORD_MAX_FAN = 2;      // candidate slots per pass up to which the records are written (api.cu)
__device__ __forceinline__ int record_xyz(int x, int y, int z) { return x | y << 11 | z << 22; }
__device__ __forceinline__ int record_x(int w) { return w & 2047; }
__device__ __forceinline__ int record_y(int w) { return (w >> 11) & 2047; }
__device__ __forceinline__ int record_z(int w) { return (int)((unsigned)w >> 22); }
struct GradRecords {
    int* count;        // [n_sub]
    GradRecord* r;     // [n_sub * cap]
};
// (n_sub is a multiple of GROUP_WARPS = 8: the records start 16-byte aligned)
__host__ __device__ __forceinline__ long long grad_record_words(long long n_sub, long long plane) { return n_sub + RECORD_WORDS * plane; }
__host__ __device__ __forceinline__ GradRecords grad_records(int* base, long long n_sub, long long plane, int slot) {
    GradRecords r;
    r.count = base + (long long)slot * grad_record_words(n_sub, plane);
    r.r = reinterpret_cast<GradRecord*>(r.count + n_sub);
    return r;
}

__host__ __device__ constexpr int aos_pitch(int K) { return (3 * K + 3) / 4 * 4; }

// What the streaming kernels need to know about the model's fields.
struct FieldStream {
    const float* fields = nullptr;   // [3(K+1)][V]: xbar's planes, then u_1 .. u_K
    bool use_tma = false;            // false: register-staged generic kernels
    int n_sm = 1;                    // persistent grid size
    CUtensorMap map32, map16;        // boxes {TX, 1, 32 | 16, 3(K+1)}
    // reduced-precision storage: u_k in half, xbar in float
    bool half_u = false;
    const __half* u16 = nullptr;     // [3K][V]
    CUtensorMap xmap32, xmap16;      // xbar alone, boxes {TX, 1, 32 | 16, 3} of float
    CUtensorMap umap32, umap16;      // u16, boxes {TX, 1, 32 | 16, 3K} of half
    FieldScale scale = {};
    // one byte per interpolation cell (i0, j0, k0) in [-1, n-1]^3, element
    // ((k0+1)(ny+1) + (j0+1))(nx+1) + (i0+1): 0 if the cell's eight zero-padded taps of f0 are all
    // equal (then the image gradient is exactly 0 anywhere in the cell), else 1 (gradient.cu)
    const unsigned char* cellmap = nullptr;
    // summed-volume tables (box_count): of f0 != 0 over the voxel grid [nx][ny][nz], and of the
    // cell map over [nx + 1][ny + 1][nz + 1]; NULL: no tile is ever skipped (reading B8)
    const unsigned* f0_integral = nullptr;
    const unsigned* cell_integral = nullptr;
    FieldMax fmax = {};
    int skip_min_tiles_per_sm = SKIP_MIN_TILES_PER_SM;     // geometry.tile_skipping: 0 always, INT_MAX never
    // gradient records of the trial slots (GradRecords; NULL: none, the gradient makes its own pass)
    int* grad_rec = nullptr;
    // with the records: a copy of u_1 .. u_K with a voxel's 3 K values side by side, [V][aos_pitch(K)]
    // floats (zero padded), so that the gather over the records fetches them from two or three 32-byte
    // sectors instead of 3 K
    const float* u_aos = nullptr;
    // measurement: tiles whose fields the warp / gradient kernels really loaded, summed over the
    // launches since the host last cleared them ([0] warp, [1] gradient; one atomic per consumer group)
    unsigned long long* visited = nullptr;
};

// Tile extent along z and ring depth by K: a stage is 3(K+1) planes x TZ x TX floats and the
// ring has to fit in 227 KB of shared memory next to the kernel's own buffers.
#ifndef PCAMM_TZ_SMALL_K
#define PCAMM_TZ_SMALL_K 4      // largest K with 32-slice tiles (experiments: 0 = 16 slices for every K)
#endif
#ifndef PCAMM_MAX_SPG
#define PCAMM_MAX_SPG 2         // stages per consumer group, at most
#endif
template <int K> struct TileZ { static constexpr int value = K <= PCAMM_TZ_SMALL_K ? 32 : 16; };
// stages per consumer group that fit into budget_bytes, at most max_spg
template <int K, bool H = false>
constexpr int stages_per_group(int n_groups, int max_spg, int budget_bytes) {
    const int stage = (H ? 12 + 6 * K : 12 * (K + 1)) * TileZ<K>::value * TX;
    const int n = budget_bytes / stage / n_groups;
    return n < max_spg ? (n < 1 ? 1 : n) : max_spg;
}
template <int K>
__host__ __device__ __forceinline__ const CUtensorMap& field_map(const FieldStream& fs) {
    if (fs.half_u) return TileZ<K>::value == 32 ? fs.xmap32 : fs.xmap16;
    return TileZ<K>::value == 32 ? fs.map32 : fs.map16;
}
template <int K>
__host__ __device__ __forceinline__ const CUtensorMap& half_map(const FieldStream& fs) {
    if (!fs.half_u) return field_map<K>(fs);      // unused by the kernels then
    return TileZ<K>::value == 32 ? fs.umap32 : fs.umap16;
}

// Host: the tensor map of the fields [P][nz][ny][nx] (xbar's three planes first, then u_1 .. u_K)
// with box {TX, 1, tz, P}.  Returns false if the driver entry point is missing or the shape
// cannot be described (nx * 4 must be a multiple of 16 bytes).
// elem_bytes 4: float planes; 2: half planes.
bool make_field_map(const Geom& G, const void* fields, int planes, int tz, int elem_bytes, CUtensorMap* out,
                    std::string* why);

}  // namespace pcamm
