// a-1: fused DVF synthesis + trilinear warp.
//
//   x_j = xbar_j + sum_k u_kj w_k                  (section 2.1, Eq. 1; L80 Eq. 2 constraint)
//   f_j = trilinear(f0, idx_j + x_j / h)           ("found through trilinear
//                                                   interpolation"; pull-back, L99; readings A1, A2)
//
// The model keeps the fields in voxel units (xbar / h, u_k / h per component, divided once at
// pcamm_model_create), so Eq. (1) yields the displacement in voxels directly.
//
// One pass over the K+1 vector fields serves every active trial slot (candidate steps of a
// batched line search, or independent solves in flight): the fields of a voxel are loaded once
// into registers and the slot loop runs inside the thread.
//
// HBM layout: fields planar [3(K+1)][V] (xbar's planes, then u_1 .. u_K), exactly the caller's
// order.  The warped volume is written once, in the z-fastest ray layout of common.cuh that the
// projector reads at every gantry angle (or in the standard layout for the volume returned to
// the caller).
//
// k_warp_tma is the kernel of the solve: field tiles arrive in shared memory by TMA through the
// mbarrier ring of stream.cuh, consumer groups interpolate and store.  k_warp_generic (one
// register-staged tile per block) serves shapes TMA cannot describe (nx not a multiple of 4).
#include "internal.h"
#include "stream.cuh"
#include "trilinear.cuh"

namespace pcamm {

namespace {

constexpr int TILE = 32;
constexpr int ROWS = 4;        // voxels per thread (z rows tw, tw+8, tw+16, tw+24 of the tile)
constexpr int NTHREADS = 256;  // 32 x 8

// Trilinear interpolation of f0 at voxel (i,j,k) displaced by d voxels (d = x / h).
__device__ __forceinline__ float trilinear(const Geom& G, const float* __restrict__ f0, int i, int j, int k,
                                           float dx, float dy, float dz) {
    const Taps t = make_taps(G, i, j, k, dx, dy, dz);
    float c[8];
    gather8(G, f0, t, c);
    return combine8(t, c);
}

// Tile: 32 x by 32 z at fixed y.  Loads: lane = x (one 128 B line per plane and z).  Stores in the
// ray layout (RAY = true, what the projector reads): lane = z, through a 32x33 shared-memory
// tile, one 128 B line per (x, y); in the standard layout [z][y][x] (RAY = false: the volume
// handed back to the caller): lane = x.
template <int K, bool RAY>
__global__ void __launch_bounds__(NTHREADS)
k_warp_generic(const Geom G, const float* __restrict__ f0, const float* __restrict__ xbar, const float* __restrict__ u,
       const SlotState* __restrict__ slots, int nslots, float* __restrict__ vol_out, long long slot_stride,
       unsigned char* __restrict__ occ) {
    __shared__ float tile[TILE][TILE + 1];
    tl_begin(G.tl);
    const int lane = threadIdx.x & 31, tw = threadIdx.x >> 5;
    const int x0 = blockIdx.x * TILE, z0 = blockIdx.y * TILE, y = blockIdx.z;
    const int x = x0 + lane;
    const long long V = G.V;

    float xb[ROWS][3], uu[ROWS][K][3];
    bool in[ROWS];
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
        const int z = z0 + tw + 8 * r;
        in[r] = (x < G.nx) && (z < G.nz);
        const long long lin = ((long long)z * G.ny + y) * G.nx + x;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            xb[r][c] = in[r] ? __ldcs(xbar + c * V + lin) : 0.f;
#pragma unroll
            for (int k = 0; k < K; ++k) uu[r][k][c] = in[r] ? __ldcs(u + ((long long)k * 3 + c) * V + lin) : 0.f;
        }
    }

    for (int s = 0; s < nslots; ++s) {
        if (!slots[s].active) continue;               // uniform over the grid
        float w[K];
#pragma unroll
        for (int k = 0; k < K; ++k) w[k] = slots[s].w[k];
        float* out = vol_out + (long long)s * slot_stride;
        float val[ROWS];
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
            val[r] = 0.f;
            if (in[r]) {
                float d[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    float xs = xb[r][c];                    // Eq. (1)
#pragma unroll
                    for (int k = 0; k < K; ++k) xs = fmaf(uu[r][k][c], w[k], xs);
                    d[c] = xs;
                }
                val[r] = trilinear(G, f0, x, y, z0 + tw + 8 * r, d[0], d[1], d[2]);
            }
        }
        if (!RAY) {
#pragma unroll
            for (int r = 0; r < ROWS; ++r)
                if (in[r]) out[((long long)(z0 + tw + 8 * r) * G.ny + y) * G.nx + x] = val[r];
        } else {
            __syncthreads();
#pragma unroll
            for (int r = 0; r < ROWS; ++r) tile[tw + 8 * r][lane] = val[r];
            __syncthreads();
            const int zo = z0 + lane;
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const int xo = x0 + tw + 8 * r;
                const bool st = xo < G.nx && zo < G.nz;
                const float v = st ? tile[lane][tw + 8 * r] : 0.f;
                if (st) out[ray_layout_index(G, xo, y, zo)] = v;
                occ_record(G, occ + (long long)s * G.OCC, xo, y, z0, 32, v != 0.f);
            }
        }
    }
    tl_end(G.tl, TLK_WARP);
}

// ---------------------------------------------------------------- the TMA-fed kernel

// consumer groups: four where the stages of the 16-slice tiles (K = 5, 6) leave room for them
// and for the L1 lines of the f0 gathers, else three
#ifndef PCAMM_WARP_GROUPS
#define PCAMM_WARP_GROUPS 3
#endif
template <int K> struct WarpGroups { static constexpr int value = (K == 5 || K == 6) ? 4 : PCAMM_WARP_GROUPS; };
constexpr int AIR_WORDS = 64;      // air flags of up to 2048 tiles per consumer group (beyond: never skipped)
constexpr int SLOT_CACHE = 64;     // slots whose coefficients are kept in shared memory
template <int K> struct WarpThreads { static constexpr int value = 32 * WarpGroups<K>::value * GROUP_WARPS; };

constexpr int WSTATIC = 16 * 1024; // static shared memory of the kernel (transposition tiles, slot cache), rounded up
template <int K, bool H> struct WarpStages { static constexpr int value = stages_per_group<K, H>(WarpGroups<K>::value, PCAMM_MAX_SPG, 227 * 1024 - WSTATIC - 64); };

template <int K, bool H>
constexpr size_t warp_smem_bytes() {
    return FieldRing<3 * (K + 1), TileZ<K>::value, WarpGroups<K>::value, WarpStages<K, H>::value, H>::BYTES;
}

// H: u_k stored in half (stream.cuh FieldRing, FieldScale).  SKIP: with the tile flags of reading
// B8 (f0_integral != NULL); without them the loads simply follow the tile counter.  REC: also
// writes the gradient records of every slot (stream.cuh GradRecords; rec = their base).
template <int K, bool RAY, bool H, bool SKIP, bool REC>
__global__ void __launch_bounds__(WarpThreads<K>::value, 1)
k_warp_tma(const __grid_constant__ CUtensorMap fmap, const __grid_constant__ CUtensorMap umap, const FieldScale scale,
           const FieldMax fmax, const unsigned* __restrict__ f0_integral, const Geom G, const float* __restrict__ f0,
           const SlotState* __restrict__ slots, int nslots, float* __restrict__ vol_out, long long slot_stride,
           unsigned char* __restrict__ occ, unsigned long long* __restrict__ visited, int* __restrict__ rec) {
    constexpr int P = 3 * (K + 1), WTZ = TileZ<K>::value, WROWS = WTZ / GROUP_WARPS;
    constexpr int WNG = WarpGroups<K>::value;
    using Ring = FieldRing<P, WTZ, WNG, WarpStages<K, H>::value, H>;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ float tiles[WNG][WTZ][TX + 1];
    __shared__ int s_occ[WNG][2][TX];                      // per group: column x has something in z block 0 / 1
    __shared__ float s_w[SLOT_CACHE][K];                   // the slots' coefficients (constant during the launch)
    __shared__ int s_active[SLOT_CACHE];
    __shared__ int s_reach[3];                             // reach of the stencils, max over the active slots
    __shared__ int s_issue[WarpGroups<K>::value][2];
    __shared__ unsigned s_air[WarpGroups<K>::value][AIR_WORDS];   // per group: bit jt set = its jt-th tile is air
    tl_begin(G.tl);
    if (SKIP && threadIdx.x < 3) {
        float dmax = 0.f;
        for (int i = 0; i < nslots && i < SLOT_CACHE; ++i) {
            if (!slots[i].active) continue;
            float d = fmax.v[threadIdx.x];
            for (int k = 0; k < K; ++k) d = fmaf(fabsf(slots[i].w[k]), fmax.v[3 + 3 * k + threadIdx.x], d);
            dmax = fmaxf(dmax, d);
        }
        s_reach[threadIdx.x] = reach_of(dmax);
    }
    for (int i = threadIdx.x; i < nslots && i < SLOT_CACHE; i += blockDim.x) {
        s_active[i] = slots[i].active;
#pragma unroll
        for (int k = 0; k < K; ++k) s_w[i][k] = H ? slots[i].w[k] * scale.inv[k] : slots[i].w[k];
    }
    Ring ring;
    ring.bind(smem_raw);
    if (threadIdx.x == 0) {
        if (smem_u32(smem_raw) & 127u) __trap();           // TMA destinations must be 128 B aligned
        ring.init();
    }
    __syncthreads();
    const long long n_tiles = tile_count(G, WTZ);
    const long long n_sub = n_tiles * GROUP_WARPS, rec_plane = n_tiles * (TX * WTZ);
    constexpr int SUBCAP = TX * WROWS;                     // records a sub-tile (one warp's voxels of a tile) can hold
    const long long rec_stride_w = grad_record_words(n_sub, rec_plane);            // words per slot
    int* const rec_count = rec;                            // slot 0's counts and records (GradRecords)
    int* const rec_w = REC ? reinterpret_cast<int*>(grad_records(rec, n_sub, rec_plane, 0).r) : nullptr;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int last_active = -1;                                  // the last slot that reads the stage
    for (int i = 0; i < nslots; ++i)
        if (s_active[i]) last_active = i;
    if (last_active < 0) { tl_end(G.tl, TLK_WARP); return; }   // nothing to warp
    const int group = warp / GROUP_WARPS, tw = warp % GROUP_WARPS;
    const bool leader = tw == 0 && lane == 0;
    const uint64_t policy = l2_evict_first_policy();
    float(*tile)[TX + 1] = tiles[group];
    // A tile whose stencils can only reach zeros of f0 (summed-volume table of f0 != 0 over the
    // box the tile's voxels can be displaced into) is all zero whatever the fields say: its
    // fields are neither loaded nor read, it is written as zeros (reading B8: exact).
    // The flags of the group's tiles are worked out up front (one tile per thread, eight loads of
    // the table each) and kept as bit masks in shared memory, off the tiles' critical path.
    if (SKIP) {
        const int Rx = s_reach[0], Ry = s_reach[1], Rz = s_reach[2];
        const int gtid = threadIdx.x - group * GROUP_THREADS;
        for (int base = 0; base < AIR_WORDS * 32; base += GROUP_THREADS) {
            const int jt = base + gtid;
            const long long t = Ring::tile_of(group, jt);
            bool air = false;
            if (t < n_tiles) {
                const TileCoord c = tile_coord(G, WTZ, t);
                const int xl = max(c.x0 - Rx, 0), xh = min(c.x0 + TX + Rx, G.nx - 1);
                const int yl = max(c.y - Ry, 0), yh = min(c.y + 1 + Ry, G.ny - 1);
                const int zl = max(c.z0 - Rz, 0), zh = min(c.z0 + WTZ + Rz, G.nz - 1);
                air = xl > xh || yl > yh || zl > zh || box_count(f0_integral, G.nx, G.ny, xl, xh, yl, yh, zl, zh) == 0u;
            }
            const unsigned mask = __ballot_sync(0xffffffffu, air);
            if (lane == 0) s_air[group][jt >> 5] = mask;
            if (Ring::tile_of(group, base + GROUP_THREADS) >= n_tiles) break;     // uniform over the group
        }
        group_barrier(group);
    }
    auto tile_is_air = [&](int jt) -> bool {               // jt: the group's tile counter
        return SKIP && jt < AIR_WORDS * 32 && ((s_air[group][jt >> 5] >> (jt & 31)) & 1u) != 0u;
    };
    // The group's loads go through its stages in the order of its tiles that are not air.
    constexpr int SPG = WarpStages<K, H>::value;
    // (the leader's two counters live in shared memory: registers are what limits this kernel)
    if (leader) { s_issue[group][0] = 0; s_issue[group][1] = 0; }      // loads started, next tile counter to look at
    auto issue_next = [&]() {
        if (!SKIP) {                                       // the group's tiles in turn
            const int j_issue = s_issue[group][1]++;
            ring.issue(&fmap, &umap, G, n_tiles, group, j_issue, policy);
            return;
        }
        int n_issued = s_issue[group][0], j_issue = s_issue[group][1];
        for (;;) {
            const long long t2 = Ring::tile_of(group, j_issue);
            if (t2 >= n_tiles) break;
            if (tile_is_air(j_issue++)) continue;
            ring.issue_tile(&fmap, &umap, G, t2, group * SPG + n_issued % SPG, policy);
            ++n_issued;
            break;
        }
        s_issue[group][0] = n_issued; s_issue[group][1] = j_issue;
    };
    if (leader)
        for (int i = 0; i < SPG; ++i) issue_next();
    int n_loaded = 0, j = 0;                               // loads this group has consumed; its tile counter
    int n_written = 0;                                     // records this warp wrote (REC)
    for (long long t = Ring::tile_of(group, 0); t < n_tiles; t += (long long)WNG * gridDim.x, ++j) {
        const bool air = tile_is_air(j);                   // uniform over the group
        if (air) {                                         // zeros, straight to their places
            const TileCoord c = tile_coord(G, WTZ, t);
            for (int sl = 0; sl < nslots; ++sl) {
                if (!s_active[sl]) continue;
                float* out = vol_out + (long long)sl * slot_stride;
                if (REC && lane == 0) rec_count[(long long)sl * rec_stride_w + t * GROUP_WARPS + tw] = 0;   // f0 = 0 all around: G = 0
                if (!RAY) {
#pragma unroll
                    for (int r = 0; r < WROWS; ++r) {
                        const int x = c.x0 + lane, z = c.z0 + tw + GROUP_WARPS * r;
                        if (x < G.nx && z < G.nz) out[((long long)z * G.ny + c.y) * G.nx + x] = 0.f;
                    }
                } else {
                    const int zo = c.z0 + lane;
#pragma unroll
                    for (int r = 0; r < TX / GROUP_WARPS; ++r) {
                        const int xo = c.x0 + tw + GROUP_WARPS * r;
                        if (lane < WTZ && xo < G.nx && zo < G.nz) out[ray_layout_index(G, xo, c.y, zo)] = 0.f;
                    }
                    if (tw < WTZ / 16 && c.x0 + lane < G.nx && c.z0 + 16 * tw < G.nz)
                        occ[(long long)sl * G.OCC + occ_index(G, c.x0 + lane, c.y, (c.z0 >> 4) + tw)] = (unsigned char)0;
                }
            }
            continue;
        }
        {
            uint32_t sf = 0;
            if (!air) {
                const int nl = SKIP ? n_loaded : j;
                const int s = group * SPG + nl % SPG;
                mbar_wait(ring.full + s, (uint32_t)(nl / SPG) & 1u);
                sf = smem_u32(ring.stage(s));              // [P][WTZ][TX]
            }
            const TileCoord c = tile_coord(G, WTZ, t);
            const int x = c.x0 + lane;
            // which of the thread's rows are voxels of the grid
            unsigned in_grid = 0u;
#pragma unroll
            for (int r = 0; r < WROWS; ++r) in_grid |= (x < G.nx && c.z0 + tw + GROUP_WARPS * r < G.nz) ? 1u << r : 0u;
            for (int sl = 0; sl < nslots; ++sl) {
                if (!s_active[sl]) continue;               // uniform over the grid
                float w[K];
#pragma unroll
                for (int k = 0; k < K; ++k) w[k] = s_w[sl][k];
                float* out = vol_out + (long long)sl * slot_stride;
                // voxels of a ragged tile beyond the grid: TMA filled their fields with zeros, the
                // taps are clamped, the value is computed and not stored
                float val[WROWS];
#pragma unroll
                for (int r = 0; r < WROWS; ++r) val[r] = 0.f;
                if (!air) {
                Taps taps[WROWS];
#pragma unroll
                for (int r = 0; r < WROWS; ++r) {
                    const int zz = tw + GROUP_WARPS * r, z = c.z0 + zz;
                    float d[3];
#pragma unroll
                    for (int cc = 0; cc < 3; ++cc) {
                        float xs = Ring::xbar_at(sf, cc, zz, lane);                                // Eq. (1)
#pragma unroll
                        for (int k = 0; k < K; ++k) xs = fmaf(Ring::u_at(sf, k, cc, zz, lane), w[k], xs);
                        d[cc] = xs;
                    }
                    taps[r] = make_taps(G, x, c.y, z, d[0], d[1], d[2]);
                }
                if (sl == last_active) {                    // the fields of this tile are in registers: refill the
                    group_barrier(group);                   // stage while the gathers are under way
                    if (leader) issue_next();
                }
                float cv[WROWS][8];
#pragma unroll
                for (int r = 0; r < WROWS; ++r) gather8(G, f0, taps[r], cv[r]);    // 8 WROWS gathers in flight
#pragma unroll
                for (int r = 0; r < WROWS; ++r) val[r] = combine8(taps[r], cv[r]);
                if (REC) {
                    // the voxels of this warp whose cell is not constant (only they can have G_j != 0;
                    // PAPER.md:L95, reading A6), in the order (lane, row), into its sub-tile's records:
                    // a lane's rows with such a cell, the warp's running count of them, then each lane
                    // stores its records one behind the other
                    unsigned vmask = 0u;
#pragma unroll
                    for (int r = 0; r < WROWS; ++r) {
                        const bool diff = cv[r][1] != cv[r][0] || cv[r][2] != cv[r][0] || cv[r][3] != cv[r][0] || cv[r][4] != cv[r][0] ||
                                          cv[r][5] != cv[r][0] || cv[r][6] != cv[r][0] || cv[r][7] != cv[r][0];
                        vmask |= diff ? 1u << r : 0u;
                    }
                    vmask &= in_grid;
                    const int sub = (int)t * GROUP_WARPS + tw;
                    int n_rec = 0;
                    if (__any_sync(0xffffffffu, vmask != 0u)) {                  // uniform over the warp
                        const int cnt = __popc(vmask);
                        int incl = cnt;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const int v = __shfl_up_sync(0xffffffffu, incl, o);
                            if (lane >= o) incl += v;
                        }
                        n_rec = __shfl_sync(0xffffffffu, incl, 31);
                        if (vmask != 0u) {
                            int4* dst = reinterpret_cast<int4*>(reinterpret_cast<GradRecord*>(rec_w + (long long)sl * rec_stride_w) + sub * SUBCAP + (incl - cnt));
                            const int xyz0 = record_xyz(x, c.y, c.z0 + tw);
#pragma unroll
                            for (int r = 0; r < WROWS; ++r) {
                                if ((vmask >> r) & 1u) {
                                    dst[0] = make_int4(xyz0 + (GROUP_WARPS * r << 22), __float_as_int(taps[r].wx1), __float_as_int(taps[r].wy1), __float_as_int(taps[r].wz1));
                                    dst[1] = make_int4(__float_as_int(cv[r][0]), __float_as_int(cv[r][1]), __float_as_int(cv[r][2]), __float_as_int(cv[r][3]));
                                    dst[2] = make_int4(__float_as_int(cv[r][4]), __float_as_int(cv[r][5]), __float_as_int(cv[r][6]), __float_as_int(cv[r][7]));
                                    dst += 3;
                                }
                            }
                        }
                    }
                    if (lane == 0) rec_count[(long long)sl * rec_stride_w + sub] = n_rec;
                    n_written += n_rec;
                }
                }
                if (!RAY) {
#pragma unroll
                    for (int r = 0; r < WROWS; ++r)
                        if ((in_grid >> r) & 1u) out[((c.z0 + tw + GROUP_WARPS * r) * G.ny + c.y) * G.nx + x] = val[r];     // (V < 2^31)
                } else {
                    // occupancy (common.cuh): is anything non-zero in column x, z block of 16?  Rows
                    // zz = tw + 8 r: r = 0, 1 lie in the tile's first block, r = 2, 3 in its second.
                    bool nzb[2] = {false, false};
#pragma unroll
                    for (int r = 0; r < WROWS; ++r) nzb[r >> 1] |= val[r] != 0.f && ((in_grid >> r) & 1u);
                    if (tw < 2) s_occ[group][tw][lane] = 0;
                    group_barrier(group);
#pragma unroll
                    for (int r = 0; r < WROWS; ++r) tile[tw + GROUP_WARPS * r][lane] = val[r];
                    if (nzb[0]) s_occ[group][0][lane] = 1;
                    if (nzb[1]) s_occ[group][1][lane] = 1;
                    group_barrier(group);
                    // this thread's transposed stores: column c.x0 + tw + 8 r, level c.z0 + lane (elements < 2^31)
                    const int ray0 = (int)ray_layout_index(G, c.x0 + tw, c.y, c.z0 + lane), ray_step = GROUP_WARPS * G.nz;
                    const bool z_ok = lane < WTZ && c.z0 + lane < G.nz;
#pragma unroll
                    for (int r = 0; r < TX / GROUP_WARPS; ++r)
                        if (z_ok && c.x0 + tw + GROUP_WARPS * r < G.nx) out[ray0 + r * ray_step] = tile[lane][tw + GROUP_WARPS * r];
                    if (tw < WTZ / 16 && x < G.nx && c.z0 + 16 * tw < G.nz)
                        occ[(long long)sl * G.OCC + occ_index(G, x, c.y, (c.z0 >> 4) + tw)] = (unsigned char)s_occ[group][tw][lane];
                }
            }
            if (SKIP && !air) ++n_loaded;
        }
    }
    if (leader && visited) atomicAdd(visited, (unsigned long long)(SKIP ? n_loaded : j));
    if (REC && lane == 0 && visited && n_written) atomicAdd(visited + 3, (unsigned long long)n_written);
    tl_end(G.tl, TLK_WARP);
}

template <int K, bool RAY, bool H, bool REC>
void launch_tma(Seq& q, const Geom& G, const FieldStream& fs, const float* f0, const SlotState* slots,
                int nslots, float* vol_out, long long slot_stride, unsigned char* occ, int* rec) {
    static DeviceOnce configured;
    constexpr size_t smem = warp_smem_bytes<K, H>();
    const CUtensorMap& fmap = field_map<K>(fs);
    const CUtensorMap& umap = half_map<K>(fs);
    const int n_sm = fs.n_sm;
    {
        const cudaError_t e = configured.run([&] {
            cudaError_t r = cudaFuncSetAttribute(k_warp_tma<K, RAY, H, true, REC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (r == cudaSuccess)
                r = cudaFuncSetAttribute(k_warp_tma<K, RAY, H, false, REC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            return r;
        });
        if (e != cudaSuccess) { q.err = e; return; }
    }
    const long long nt = tile_count(G, TileZ<K>::value);
    const int grid = (int)(nt < n_sm ? nt : n_sm);
    // the tile flags cost a few dependent loads per launch: used where a CTA has tiles enough to win them back
    const unsigned* table = nt >= fs.skip_min_tiles_per_sm * (long long)n_sm ? fs.f0_integral : nullptr;
    for (int s0 = 0; s0 < nslots; s0 += SLOT_CACHE) {      // the kernel keeps up to SLOT_CACHE slots' coefficients on chip
        const int ns = nslots - s0 < SLOT_CACHE ? nslots - s0 : SLOT_CACHE;
        float* out = vol_out + (long long)s0 * slot_stride;
        unsigned char* oc = occ ? occ + (long long)s0 * G.OCC : occ;
        // the records of slot s0 onwards (GradRecords: one block of words per slot)
        int* rec_s0 = rec ? rec + (long long)s0 * grad_record_words(nt * GROUP_WARPS, nt * (TX * TileZ<K>::value)) : rec;
        if (table)
            q.launch(k_warp_tma<K, RAY, H, true, REC>, dim3(grid), dim3(WarpThreads<K>::value), smem, fmap, umap, fs.scale, fs.fmax,
                     table, G, f0, slots + s0, ns, out, slot_stride, oc, fs.visited, rec_s0);
        else
            q.launch(k_warp_tma<K, RAY, H, false, REC>, dim3(grid), dim3(WarpThreads<K>::value), smem, fmap, umap, fs.scale, fs.fmax,
                     table, G, f0, slots + s0, ns, out, slot_stride, oc, fs.visited, rec_s0);
    }
}

template <int K>
void launch_k(Seq& q, const Geom& G, const FieldStream& fs, const float* f0, const SlotState* slots, int nslots,
              int ray_layout, float* vol_out, long long slot_stride, unsigned char* occ, int* rec) {
    if (fs.use_tma) {
        // records only with the ray layout (the solve's trial volumes)
        const bool with_rec = rec && ray_layout;
        if (fs.half_u) {
            if (with_rec) launch_tma<K, true, true, true>(q, G, fs, f0, slots, nslots, vol_out, slot_stride, occ, rec);
            else if (ray_layout) launch_tma<K, true, true, false>(q, G, fs, f0, slots, nslots, vol_out, slot_stride, occ, nullptr);
            else launch_tma<K, false, true, false>(q, G, fs, f0, slots, nslots, vol_out, slot_stride, occ, nullptr);
        } else {
            if (with_rec) launch_tma<K, true, false, true>(q, G, fs, f0, slots, nslots, vol_out, slot_stride, occ, rec);
            else if (ray_layout) launch_tma<K, true, false, false>(q, G, fs, f0, slots, nslots, vol_out, slot_stride, occ, nullptr);
            else launch_tma<K, false, false, false>(q, G, fs, f0, slots, nslots, vol_out, slot_stride, occ, nullptr);
        }
        return;
    }
    const float* xbar = fs.fields;
    const float* u = fs.fields + 3 * G.V;
    dim3 grid((G.nx + TILE - 1) / TILE, (G.nz + TILE - 1) / TILE, G.ny);
    if (ray_layout) q.launch(k_warp_generic<K, true>, grid, dim3(NTHREADS), 0, G, f0, xbar, u, slots, nslots, vol_out, slot_stride, occ);
    else q.launch(k_warp_generic<K, false>, grid, dim3(NTHREADS), 0, G, f0, xbar, u, slots, nslots, vol_out, slot_stride, occ);
}

}  // namespace

void launch_warp(Seq& q, const Geom& G, const FieldStream& fs, const float* f0, const SlotState* slots, int nslots,
                 int ray_layout, float* vol_out, long long slot_stride, unsigned char* occ, int* rec) {
    switch (G.K) {
#define PCAMM_CASE(KK) \
    case KK: launch_k<KK>(q, G, fs, f0, slots, nslots, ray_layout, vol_out, slot_stride, occ, rec); break;
        PCAMM_CASE(1) PCAMM_CASE(2) PCAMM_CASE(3) PCAMM_CASE(4)
        PCAMM_CASE(5) PCAMM_CASE(6) PCAMM_CASE(7) PCAMM_CASE(8)
#undef PCAMM_CASE
        default: break;
    }
}

}  // namespace pcamm
