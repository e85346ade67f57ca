// a-3 (residual) and a-4: dJ/dw = 2 U^T (df/dx) P^T (P f - a y - b 1).
//
// The chain is evaluated voxel by voxel in one pass over the K+1 vector fields, and no
// volume-sized gradient is ever written:
//
//   B_j  = sum_i l_ij r_i          backprojection of the residual, gathered by the voxel: the exact
//                                  length of every ray through voxel box j (the same l_ij as the
//                                  projector: reading A4), times r_i
//   G_j  = df_j / dx_j             exact derivative of the trilinear interpolant (PAPER.md:L95:
//                                  "has to be consistent with the interpolation process"; A6)
//   g_k  = 2 sum_j B_j (G_j . u_kj)
//
// df/dx is block diagonal (voxel j's value depends on x_j only; reading A5), which is what allows
// the fusion.  Voxels whose eight taps make G_j = 0 skip the gather (their term is exactly 0).
//
// The gather uses the separable form of the ray/box intersection in the parameter alpha of
// S + alpha (D - S) with D on the flat detector: the in-plane slabs give an alpha-interval that
// depends on the detector column only, the z-slab one that depends on the row only, and
// l_ij = |D - S| * |intersection of the two|.  Per view, k_resid tabulates (d_x, d_y, 1/d_x,
// 1/d_y) per column, (d_z, 1/d_z) per row and rL_i = r_i |D_i - S| per pixel.
#include "internal.h"
#include "stream.cuh"
#include "trilinear.cuh"

namespace pcamm {

namespace {

constexpr int RT = 256;         // k_resid threads
constexpr int TILE = 32, ROWS = 4, GT = 256;
constexpr float PAR_INV = 1e30f; // 1/d for a ray parallel to a slab: [0, +big) or (-big, 0] keeps
                                 // the half-open inside test of reading A21

// r = p - a y - b (Eq. 2), rL = r |D - S|; tables of this view; partial sums of r^2.
// r_direct != NULL: r is taken from there (pcamm_backproject hook).  force: also for solves that
// have stopped (closing pass of a solve).
__global__ void __launch_bounds__(RT)
k_resid(const Geom G, const SolveState* __restrict__ solves, const SolveIn* __restrict__ in,
        int force, const float* __restrict__ p_slots, const float* __restrict__ r_direct, float* __restrict__ rL,
        float4* __restrict__ utab, float2* __restrict__ vtab, double* __restrict__ partials) {
    __shared__ double red[RT / 32];
    tl_begin(G.tl);
    const int b = blockIdx.y;
    const SolveState& st = solves[b];
    if (!needs_gradient(st) && !force) { tl_end(G.tl, TLK_RESID); return; }
    const View vw = st.view;
    const int pix = blockIdx.x * RT + threadIdx.x;
    double rr = 0.0;
    if (pix < G.npix) {
        const int iu = pix % G.nu, iv = pix / G.nu;
        const double uu = ((double)iu - 0.5 * (G.nu - 1) + (double)G.off_u) * (double)G.pu;
        const double vv = ((double)iv - 0.5 * (G.nv - 1) + (double)G.off_v) * (double)G.pv;
        const double L = sqrt((double)G.sdd * (double)G.sdd + uu * uu + vv * vv);
        double r;
        if (r_direct) r = (double)__ldg(r_direct + pix);
        else {
            const float* y = in[b].y;
            const double pv = (double)__ldg(p_slots + (long long)st.acc_slot * G.npix + pix);
            r = pv - st.a * (y ? (double)__ldg(y + pix) : 0.0) - st.b;
        }
        rr = r * r;
        rL[(long long)b * G.npix + pix] = (float)(r * L);
        if (pix < G.nu) {
            double dx, dy;
            ray_dir_inplane(G, vw.cs, vw.sn, pix, &dx, &dy);
            utab[(long long)b * G.nu + pix] = make_float4((float)dx, (float)dy, dx != 0.0 ? (float)(1.0 / dx) : PAR_INV,
                                                          dy != 0.0 ? (float)(1.0 / dy) : PAR_INV);
        }
        if (pix < G.nv) {
            const double vz = ((double)pix - 0.5 * (G.nv - 1) + (double)G.off_v) * (double)G.pv;
            vtab[(long long)b * G.nv + pix] = make_float2((float)vz, vz != 0.0 ? (float)(1.0 / vz) : PAR_INV);
        }
    }
    const double s = block_sum<RT>(rr, red);
    if (threadIdx.x == 0) partials[(long long)b * gridDim.x + blockIdx.x] = s;
    tl_end(G.tl, TLK_RESID);
}

// Per-view constants of the gather, in float.
struct GatherView {
    float cs, sn, Sx, Sy;     // source position (in-plane); S_z = 0
    float Wt, Wd;             // half extent of a voxel box across / along the central ray
    float sdd_ipu, sdd_ipv;   // sdd / pitch
    float cu, cv;             // pixel index of the detector origin
};

__device__ __forceinline__ GatherView make_gather_view(const Geom& G, const View& vw) {
    GatherView g;
    g.cs = (float)vw.cs; g.sn = (float)vw.sn;
    g.Sx = (float)((double)G.sad * vw.cs); g.Sy = (float)((double)G.sad * vw.sn);
    g.Wt = 0.5f * (G.hx * fabsf(g.sn) + G.hy * fabsf(g.cs));
    g.Wd = 0.5f * (G.hx * fabsf(g.cs) + G.hy * fabsf(g.sn));
    g.sdd_ipu = G.sdd / G.pu; g.sdd_ipv = G.sdd / G.pv;
    g.cu = 0.5f * (G.nu - 1) - G.off_u; g.cv = 0.5f * (G.nv - 1) - G.off_v;
    return g;
}

// B_j = sum_i l_ij r_i for the voxel centred at (xw, yw, zw) mm.
__device__ __forceinline__ float gather_voxel(const Geom& G, const GatherView& gv, const float* __restrict__ rL,
                                              const float4* __restrict__ utab, const float2* __restrict__ vtab,
                                              float xw, float yw, float zw) {
    const float ex = xw - gv.Sx, ey = yw - gv.Sy, ez = zw;             // voxel centre - source
    const float depth = -(ex * gv.cs + ey * gv.sn);                     // along the central ray
    const float t = ey * gv.cs - ex * gv.sn;                            // along u^
    // detector bounding rectangle of the box's shadow (perspective projection of a convex body:
    // extremes of t/depth and z/depth over the box are bounded by these four quotients)
    const float i1 = __frcp_rn(depth - gv.Wd), i2 = __frcp_rn(depth + gv.Wd);   // loop bounds only (0.01 px margin)
    const float tl = t - gv.Wt, th = t + gv.Wt, zl = ez - 0.5f * G.hz, zh = ez + 0.5f * G.hz;
    const float ulo = fminf(tl * i1, tl * i2) * gv.sdd_ipu + gv.cu, uhi = fmaxf(th * i1, th * i2) * gv.sdd_ipu + gv.cu;
    const float vlo = fminf(zl * i1, zl * i2) * gv.sdd_ipv + gv.cv, vhi = fmaxf(zh * i1, zh * i2) * gv.sdd_ipv + gv.cv;
    const int iu0 = max(0, (int)ceilf(ulo - 0.01f)), iu1 = min(G.nu - 1, (int)floorf(uhi + 0.01f));
    const int iv0 = max(0, (int)ceilf(vlo - 0.01f)), iv1 = min(G.nv - 1, (int)floorf(vhi + 0.01f));
    const float xl = ex - 0.5f * G.hx, xh = ex + 0.5f * G.hx, yl = ey - 0.5f * G.hy, yh = ey + 0.5f * G.hy;
    float acc = 0.f;
    // rows in chunks of NVB (usually one chunk): their z intervals once, then per column the NVB
    // residual loads are issued together (the gather is a latency chain otherwise)
    constexpr int NVB = 4;
    for (int ivb = iv0; ivb <= iv1; ivb += NVB) {
        float lo_z[NVB], hi_z[NVB];
#pragma unroll
        for (int bb = 0; bb < NVB; ++bb) {
            const int iv = min(ivb + bb, iv1);
            const float2 vd = __ldg(vtab + iv);
            const float az0 = zl * vd.y, az1 = zh * vd.y;
            const bool on = ivb + bb <= iv1;
            lo_z[bb] = on ? fminf(az0, az1) : 1.f;                 // an empty interval for rows beyond iv1
            hi_z[bb] = on ? fmaxf(az0, az1) : -1.f;
        }
#pragma unroll 2
        for (int iu = iu0; iu <= iu1; ++iu) {
            const float4 ud = __ldg(utab + iu);
            const float ax0 = xl * ud.z, ax1 = xh * ud.z, ay0 = yl * ud.w, ay1 = yh * ud.w;
            const float lo_u = fmaxf(fminf(ax0, ax1), fminf(ay0, ay1));
            const float hi_u = fminf(fmaxf(ax0, ax1), fmaxf(ay0, ay1));
            float rv[NVB];
#pragma unroll
            for (int bb = 0; bb < NVB; ++bb) rv[bb] = __ldg(rL + min(ivb + bb, iv1) * G.nu + iu);
#pragma unroll
            for (int bb = 0; bb < NVB; ++bb) {
                const float lo = fmaxf(lo_u, lo_z[bb]), hi = fminf(hi_u, hi_z[bb]);
                acc = fmaf(fmaxf(hi - lo, 0.f), rv[bb], acc);
            }
        }
    }
    return acc;
}

// G = d f / d x of the trilinear interpolant at voxel (i,j,k) displaced by d voxels, per voxel of
// displacement (the model's fields are in voxel units, so G . u_k needs no 1/h: (G/h) . (u h) = G . u).
__device__ __forceinline__ void trilinear_grad(const Geom& G, const float* __restrict__ f0, int i, int j, int k,
                                               float dx, float dy, float dz, float* gx, float* gy, float* gz) {
    const Taps t = make_taps(G, i, j, k, dx, dy, dz);
    float c[8];
    gather8(G, f0, t, c);
    grad8(t, c, gx, gy, gz);
}

template <int K>
__global__ void __launch_bounds__(GT)
k_grad_generic(const Geom G, const float* __restrict__ f0, const float* __restrict__ xbar, const float* __restrict__ u,
       const CtlBufs c, int B, const float* __restrict__ rL, const float4* __restrict__ utab,
       const float2* __restrict__ vtab, const float* __restrict__ bvol) {
    __shared__ double red[GT / 32];
    tl_begin(G.tl);
    const SolveState* __restrict__ solves = c.solves;
    double* __restrict__ partials = c.grad_part;
    const int lane = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int x0 = blockIdx.x * TILE, y0 = blockIdx.y * TILE, z = blockIdx.z;
    const int x = x0 + lane;
    const long long V = G.V;
    const int blk = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    const int nblk = gridDim.x * gridDim.y * gridDim.z;

    float xb[ROWS][3], uu[ROWS][K][3];
    bool in[ROWS];
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
        const int y = y0 + ty + 8 * r;
        in[r] = (x < G.nx) && (y < G.ny);
        const long long lin = ((long long)z * G.ny + y) * G.nx + x;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            xb[r][c] = in[r] ? __ldcs(xbar + c * V + lin) : 0.f;
#pragma unroll
            for (int k = 0; k < K; ++k) uu[r][k][c] = in[r] ? __ldcs(u + ((long long)k * 3 + c) * V + lin) : 0.f;
        }
    }
    const float xw = G.cx + ((float)x - 0.5f * (G.nx - 1)) * G.hx;
    const float zw = G.cz + ((float)z - 0.5f * (G.nz - 1)) * G.hz;

    for (int b = 0; b < B; ++b) {
        if (!needs_gradient(solves[b])) continue;       // uniform over the grid
        float w[K];
#pragma unroll
        for (int k = 0; k < K; ++k) w[k] = (float)solves[b].w[k];
        const GatherView gv = make_gather_view(G, solves[b].view);
        const float* rLb = rL + (long long)b * G.npix;
        const float4* ub = utab + (long long)b * G.nu;
        const float2* vb = vtab + (long long)b * G.nv;
        float acc[K];
#pragma unroll
        for (int k = 0; k < K; ++k) acc[k] = 0.f;
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
            if (!in[r]) continue;
            float d[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                float xs = xb[r][c];                    // Eq. (1)
#pragma unroll
                for (int k = 0; k < K; ++k) xs = fmaf(uu[r][k][c], w[k], xs);
                d[c] = xs;
            }
            const int y = y0 + ty + 8 * r;
            float gx, gy, gz;
            trilinear_grad(G, f0, x, y, z, d[0], d[1], d[2], &gx, &gy, &gz);
            if (gx == 0.f && gy == 0.f && gz == 0.f) continue;
            const float yw = G.cy + ((float)y - 0.5f * (G.ny - 1)) * G.hy;
            const float Bj = bvol ? __ldg(bvol + (long long)b * V + ((long long)z * G.ny + y) * G.nx + x)
                                  : gather_voxel(G, gv, rLb, ub, vb, xw, yw, zw);
#pragma unroll
            for (int k = 0; k < K; ++k)
                acc[k] = fmaf(Bj, gx * uu[r][k][0] + gy * uu[r][k][1] + gz * uu[r][k][2], acc[k]);
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const double s = block_sum<GT>((double)acc[k], red);
            if (threadIdx.x == 0) partials[((long long)b * nblk + blk) * KMAX + k] = s;
        }
    }
    tl_end(G.tl, TLK_GRAD);
}

int grad_grid(const Geom& G, const FieldStream& fs) {
    const long long nt = tile_count(G, G.K <= PCAMM_TZ_SMALL_K ? 32 : 16);      // TileZ<K>
    return (int)(nt < fs.n_sm ? nt : fs.n_sm);
}

// ---------------------------------------------------------------- the TMA-fed kernel
//
// Same ring as the warp kernel.  A consumer group works through a tile in batches of RB voxels
// per thread:
//   1. every thread forms G_j and q_kj = G_j . u_kj for its voxels (all their f0 gathers in flight
//      together);
//   2. the voxels with G_j != 0 are compacted into a shared-memory queue, in a fixed order
//      (ballot + prefix over the warps: no atomics, so the summation order is reproducible);
//   3. the queue is dealt out in full rounds of one entry per thread: each thread gathers B_j for
//      its entry and accumulates B_j q_kj; what does not fill a round waits for the next batch
//      (single solve) or is flushed (several solves in flight: their views differ).  Only
//      boundary voxels have G_j != 0 in piecewise-constant anatomy, so without the compaction
//      most lanes of a warp would idle through their neighbours' detector gathers.
// Per tile and solve the group's K sums are reduced in double and added to the group's slot of
// the partial-sum buffer; the control kernel adds the slots in index order.

// Consumer groups per CTA: three where their stages and queues fit into shared memory, else two.
constexpr int grad_groups_for(int K) {
    const int tz = K <= PCAMM_TZ_SMALL_K ? 32 : 16;                       // TileZ<K>
    const int stage = 3 * (K + 1) * tz * TX * 4;
    const int queue = GROUP_THREADS * 3 * (8 + 4 * K);                    // GradQueueCap x sizeof(QueueEntry)
    return 3 * (stage + queue) + 16 * 1024 <= 227 * 1024 ? 3 : 2;
}
template <int K> struct GradGroups { static constexpr int value = grad_groups_for(K); };
constexpr int GSTATIC = 12 * 1024;                  // static shared memory of the kernel, rounded up
constexpr int GRAD_SKIP_WORDS = 64;                 // skip flags of up to 2048 tiles per consumer group (beyond: never skipped)
constexpr int SOLVE_CACHE = 64;                     // solves whose constants are kept in shared memory

template <int K> struct GradBatch { static constexpr int value = 2; };     // RB

template <int K>
struct QueueEntry {
    int xy, z;        // x | y << 16; z
    float q[K];
};

// Entries of a group's queue: one batch of new ones plus what the last round left over.
template <int K> struct GradQueueCap { static constexpr int value = GROUP_THREADS * (GradBatch<K>::value + 1); };
template <int K>
constexpr size_t grad_queue_bytes() { return (size_t)GradGroups<K>::value * GradQueueCap<K>::value * sizeof(QueueEntry<K>); }
template <int K, bool H> struct GradStages {
    static constexpr int value = stages_per_group<K, H>(GradGroups<K>::value, PCAMM_MAX_SPG, 227 * 1024 - GSTATIC - (int)grad_queue_bytes<K>() - 64);
};
template <int K, bool H>
constexpr size_t grad_smem_bytes() {
    return FieldRing<3 * (K + 1), TileZ<K>::value, GradGroups<K>::value, GradStages<K, H>::value, H>::BYTES + 16 + grad_queue_bytes<K>();
}

// SINGLE: one solve (B = 1): the K sums stay in registers over all tiles of the CTA and are
// reduced once at the end; otherwise they are reduced per tile and solve.
// H: u_k stored in half (stream.cuh FieldRing, FieldScale).  SKIP: with the tile flags of reading
// B8 (cell_integral != NULL); without them the loads simply follow the tile counter.
template <int K, bool SINGLE, bool H, bool SKIP>
__global__ void __launch_bounds__(32 * GradGroups<K>::value * GROUP_WARPS, 1)
k_grad_tma(const __grid_constant__ CUtensorMap fmap, const __grid_constant__ CUtensorMap umap, const FieldScale scale,
           const FieldMax fmax, const unsigned* __restrict__ cell_integral, const Geom G, const float* __restrict__ f0,
           const unsigned char* __restrict__ cellmap, const CtlBufs c, int b0, int B, const float* __restrict__ rL, const float4* __restrict__ utab,
           const float2* __restrict__ vtab, const float* __restrict__ bvol, unsigned long long* __restrict__ visited) {
    constexpr int P = 3 * (K + 1), GTZ = TileZ<K>::value, GROWS = GTZ / GROUP_WARPS;
    const SolveState* __restrict__ solves = c.solves + b0;                 // solves b0 .. b0 + B - 1 in this launch
    constexpr int RB = GradBatch<K>::value, NB = GROWS / RB;
    static_assert(GROWS % RB == 0 && NB >= 1, "tile rows per thread must be a multiple of the batch");
    constexpr int GNG = GradGroups<K>::value;
    using Ring = FieldRing<P, GTZ, GNG, GradStages<K, H>::value, H>;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ int s_cnt[GNG][2][32];                      // double buffered over the batches
    __shared__ float s_red[GNG][GROUP_WARPS][K];
    __shared__ GatherView s_gv[SOLVE_CACHE];               // per solve, constant during the launch
    __shared__ float s_w[SOLVE_CACHE][K];
    __shared__ int s_running[SOLVE_CACHE];
    __shared__ int s_reach[3];                             // reach of the stencils, max over the running solves
    __shared__ int s_issue[GNG][2];
    __shared__ unsigned s_skip[GNG][GRAD_SKIP_WORDS];      // per group: bit jt set = nothing to do in its jt-th tile
    tl_begin(G.tl);
    if (SKIP && threadIdx.x < 3) {
        float dmax = 0.f;
        for (int b = 0; b < B; ++b) {
            if (!needs_gradient(solves[b])) continue;
            float d = fmax.v[threadIdx.x];
            for (int k = 0; k < K; ++k) d = fmaf(fabsf((float)solves[b].w[k]) * 1.000001f, fmax.v[3 + 3 * k + threadIdx.x], d);
            dmax = fmaxf(dmax, d);
        }
        s_reach[threadIdx.x] = reach_of(dmax);
    }
    for (int b = threadIdx.x; b < B; b += blockDim.x) {    // B <= SOLVE_CACHE (the launcher chunks)
        s_running[b] = needs_gradient(solves[b]);
        s_gv[b] = make_gather_view(G, solves[b].view);
#pragma unroll
        for (int k = 0; k < K; ++k) s_w[b][k] = H ? (float)solves[b].w[k] * scale.inv[k] : (float)solves[b].w[k];
    }
    Ring ring;
    ring.bind(smem_raw);
    QueueEntry<K>* queues = reinterpret_cast<QueueEntry<K>*>(smem_raw + ((Ring::BYTES + 15) & ~size_t(15)));
    if (threadIdx.x == 0) {
        if (smem_u32(smem_raw) & 127u) __trap();
        ring.init();
    }
    __syncthreads();
    const long long n_tiles = tile_count(G, GTZ);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int group = warp / GROUP_WARPS, tw = warp % GROUP_WARPS, gtid = threadIdx.x - group * GROUP_THREADS;
    constexpr int QCAP = GradQueueCap<K>::value;
    QueueEntry<K>* queue = queues + (size_t)group * QCAP;   // ring buffer: q_head .. q_head + q_n - 1 (mod QCAP)
    int q_head = 0, q_n = 0, parity = 0;                    // identical in every thread of the group
    const int nslot = gridDim.x * GNG, slot = blockIdx.x * GNG + group;   // this group's partial-sum slot
    double* __restrict__ partials = c.grad_part + (long long)b0 * nslot * KMAX;
    if (gtid < K)
        for (int b = 0; b < B; ++b) partials[((long long)b * nslot + slot) * KMAX + gtid] = 0.0;
    bool any_running = false;
    for (int b = 0; b < B; ++b) any_running |= s_running[b] != 0;
    if (!any_running) { tl_end(G.tl, TLK_GRAD); return; }  // uniform over the grid
    const bool leader = gtid == 0;
    const uint64_t policy = l2_evict_first_policy();
    // A tile all of whose voxels can only land in constant cells of f0 (summed-volume table of the
    // cell map over the box of cells the tile's voxels can be displaced into) has G_j = 0
    // everywhere: its fields are neither loaded nor read (reading B8: exact).  The flags of the
    // group's tiles are worked out up front, one tile per thread, and kept as bit masks.
    if (SKIP) {
        const int Rx = s_reach[0], Ry = s_reach[1], Rz = s_reach[2];
        for (int base = 0; base < GRAD_SKIP_WORDS * 32; base += GROUP_THREADS) {
            const int jt = base + gtid;
            const long long t = Ring::tile_of(group, jt);
            bool skip = false;
            if (t < n_tiles) {
                const TileCoord c = tile_coord(G, GTZ, t);
                const int xl = max(c.x0 - Rx + 1, 0), xh = min(c.x0 + TX + Rx, G.nx);
                const int yl = max(c.y - Ry + 1, 0), yh = min(c.y + 1 + Ry, G.ny);
                const int zl = max(c.z0 - Rz + 1, 0), zh = min(c.z0 + GTZ + Rz, G.nz);
                skip = xl > xh || yl > yh || zl > zh ||
                       box_count(cell_integral, G.nx + 1, G.ny + 1, xl, xh, yl, yh, zl, zh) == 0u;
            }
            const unsigned mask = __ballot_sync(0xffffffffu, skip);
            if (lane == 0) s_skip[group][jt >> 5] = mask;
            if (Ring::tile_of(group, base + GROUP_THREADS) >= n_tiles) break;     // uniform over the group
        }
        group_barrier(group);
    }
    auto tile_is_skipped = [&](int jt) -> bool {           // jt: the group's tile counter
        return SKIP && jt < GRAD_SKIP_WORDS * 32 && ((s_skip[group][jt >> 5] >> (jt & 31)) & 1u) != 0u;
    };
    // The group's loads go through its stages in the order of its tiles that are not skipped.
    constexpr int SPG = GradStages<K, H>::value;
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
            if (tile_is_skipped(j_issue++)) continue;
            ring.issue_tile(&fmap, &umap, G, t2, group * SPG + n_issued % SPG, policy);
            ++n_issued;
            break;
        }
        s_issue[group][0] = n_issued; s_issue[group][1] = j_issue;
    };
    if (leader)
        for (int i = 0; i < SPG; ++i) issue_next();

    float acc[K];
#pragma unroll
    for (int k = 0; k < K; ++k) acc[k] = 0.f;
    int j = 0, n_loaded = 0;                               // this group's tile counter; loads it has consumed
    for (long long t = Ring::tile_of(group, 0); t < n_tiles; t += (long long)GNG * gridDim.x, ++j) {
        if (tile_is_skipped(j)) continue;                  // uniform over the group
        {
            const int nl = SKIP ? n_loaded : j;
            const int s = group * SPG + nl % SPG;
            mbar_wait(ring.full + s, (uint32_t)(nl / SPG) & 1u);
            if (SKIP) ++n_loaded;
            const uint32_t sf = smem_u32(ring.stage(s));   // [P][GTZ][TX]
            const TileCoord c = tile_coord(G, GTZ, t);
            const int x = c.x0 + lane;
            for (int b = 0; b < B; ++b) {
                if (!s_running[b]) continue;               // uniform over the grid
                float w[K];
#pragma unroll
                for (int k = 0; k < K; ++k) w[k] = s_w[b][k];
                const GatherView gv = s_gv[b];
                const float* rLb = rL + (long long)b * G.npix;
                const float4* ub = utab + (long long)b * G.nu;
                const float2* vb = vtab + (long long)b * G.nv;
                if (!SINGLE) {
#pragma unroll
                    for (int k = 0; k < K; ++k) acc[k] = 0.f;
                }
                // 0. light pass over all the thread's voxels of the tile: the displacement (Eq. 1) and
                //    one byte of the cell map each, the loads of all of them in flight together.
                float dda[GROWS][3];
                unsigned char flaga[GROWS];
#pragma unroll
                for (int ra = 0; ra < GROWS; ++ra) {
                    const int zz = tw * GROWS + ra;
#pragma unroll
                    for (int cc = 0; cc < 3; ++cc) {
                        float xs = Ring::xbar_at(sf, cc, zz, lane);                                // Eq. (1)
#pragma unroll
                        for (int k = 0; k < K; ++k)
                            xs = fmaf(Ring::u_at(sf, k, cc, zz, lane), w[k], xs);
                        dda[ra][cc] = xs;
                    }
                    const int ci = x + (int)floorf(dda[ra][0]) + 1, cj = c.y + (int)floorf(dda[ra][1]) + 1,
                              ck = c.z0 + zz + (int)floorf(dda[ra][2]) + 1;
                    const bool inside = x < G.nx && c.z0 + zz < G.nz && (unsigned)ci <= (unsigned)G.nx &&
                                        (unsigned)cj <= (unsigned)G.ny && (unsigned)ck <= (unsigned)G.nz;
                    flaga[ra] = inside ? __ldg(cellmap + ((unsigned)ck * (unsigned)(G.ny + 1) + (unsigned)cj) * (unsigned)(G.nx + 1) + (unsigned)ci) : (unsigned char)0;   // (< 2^31 cells)
                }
#pragma unroll
                for (int bt = 0; bt < NB; ++bt) {
                    // 1. G_j and q_kj.  A voxel whose interpolation cell of f0 is constant (cell map)
                    //    has G_j = 0 exactly: a warp none of whose voxels of this batch needs more
                    //    skips the taps, the gathers and the derivative (most of the volume: air, the
                    //    inside of a homogeneous organ).
                    float dd[RB][3];
                    unsigned char flag[RB];
#pragma unroll
                    for (int rr = 0; rr < RB; ++rr) {
                        flag[rr] = flaga[bt * RB + rr];
#pragma unroll
                        for (int cc = 0; cc < 3; ++cc) dd[rr][cc] = dda[bt * RB + rr][cc];
                    }
                    bool mine = false;
#pragma unroll
                    for (int rr = 0; rr < RB; ++rr) mine |= flag[rr] != 0;
                    float q[RB][K];
                    unsigned masks[RB];
#pragma unroll
                    for (int rr = 0; rr < RB; ++rr) {
                        masks[rr] = 0u;
#pragma unroll
                        for (int k = 0; k < K; ++k) q[rr][k] = 0.f;
                    }
                    if (__any_sync(0xffffffffu, mine)) {                       // uniform over the warp
                        Taps taps[RB];
#pragma unroll
                        for (int rr = 0; rr < RB; ++rr)
                            taps[rr] = make_taps(G, x, c.y, c.z0 + tw * GROWS + bt * RB + rr,
                                                 dd[rr][0], dd[rr][1], dd[rr][2]);
                        float cv[RB][8];
#pragma unroll
                        for (int rr = 0; rr < RB; ++rr) gather8(G, f0, taps[rr], cv[rr]);
#pragma unroll
                        for (int rr = 0; rr < RB; ++rr) {
                            const int zz = tw * GROWS + bt * RB + rr;
                            float gx, gy, gz;
                            grad8(taps[rr], cv[rr], &gx, &gy, &gz);
#pragma unroll
                            for (int k = 0; k < K; ++k) {
                                q[rr][k] = gx * Ring::u_at(sf, k, 0, zz, lane) + gy * Ring::u_at(sf, k, 1, zz, lane) +
                                           gz * Ring::u_at(sf, k, 2, zz, lane);
                                if (H) q[rr][k] *= scale.inv[k];      // power of two: exact
                            }
                            const bool active = flag[rr] != 0 && (gx != 0.f || gy != 0.f || gz != 0.f);
                            masks[rr] = __ballot_sync(0xffffffffu, active);
                        }
                    }
                    if (lane == 0) {
#pragma unroll
                        for (int rr = 0; rr < RB; ++rr) s_cnt[group][parity][rr * GROUP_WARPS + tw] = __popc(masks[rr]);
                    }
                    group_barrier(group);
                    if (SINGLE && bt == NB - 1 && leader) issue_next();    // no more reads of the stage: refill it
                    // 2. compaction in the fixed order (row, warp, lane), appended to the queue
                    int cnt = lane < RB * GROUP_WARPS ? s_cnt[group][parity][lane] : 0, incl = cnt;
                    parity ^= 1;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int v = __shfl_up_sync(0xffffffffu, incl, o);
                        if (lane >= o) incl += v;
                    }
                    const int n_new = __shfl_sync(0xffffffffu, incl, 31);
#pragma unroll
                    for (int rr = 0; rr < RB; ++rr) {
                        const int base = __shfl_sync(0xffffffffu, incl - cnt, rr * GROUP_WARPS + tw);
                        if (masks[rr] >> lane & 1u) {
                            int pos = q_head + q_n + base + __popc(masks[rr] & ((1u << lane) - 1u));
                            if (pos >= QCAP) pos -= QCAP;
                            if (pos >= QCAP) pos -= QCAP;
                            QueueEntry<K>& e = queue[pos];
                            e.xy = x | c.y << 16;
                            e.z = c.z0 + tw * GROWS + bt * RB + rr;
#pragma unroll
                            for (int k = 0; k < K; ++k) e.q[k] = q[rr][k];
                        }
                    }
                    q_n += n_new;
                    group_barrier(group);
                    // 3. the detector gathers, one entry per thread and round
                    const int n_proc = SINGLE ? q_n / GROUP_THREADS * GROUP_THREADS : q_n;
                    for (int e = gtid; e < n_proc; e += GROUP_THREADS) {
                        int pos = q_head + e;
                        if (pos >= QCAP) pos -= QCAP;
                        if (pos >= QCAP) pos -= QCAP;
                        const QueueEntry<K> en = queue[pos];
                        const float xw = G.cx + ((float)(en.xy & 0xffff) - 0.5f * (G.nx - 1)) * G.hx;
                        const float yw = G.cy + ((float)(en.xy >> 16) - 0.5f * (G.ny - 1)) * G.hy;
                        const float zw = G.cz + ((float)en.z - 0.5f * (G.nz - 1)) * G.hz;
                        const float Bj = bvol ? __ldg(bvol + (long long)b * G.V + ((long long)en.z * G.ny + (en.xy >> 16)) * G.nx + (en.xy & 0xffff))
                                              : gather_voxel(G, gv, rLb, ub, vb, xw, yw, zw);
#pragma unroll
                        for (int k = 0; k < K; ++k) acc[k] = fmaf(Bj, en.q[k], acc[k]);
                    }
                    q_head += n_proc;
                    if (q_head >= QCAP) q_head -= QCAP;
                    if (q_head >= QCAP) q_head -= QCAP;
                    q_n -= n_proc;
                    // no barrier here: the next batch writes its entries only after its own first
                    // barrier, which no thread passes before every thread has left this loop
                }
                if (!SINGLE) {                              // the group's K sums of this tile and solve
#pragma unroll
                    for (int k = 0; k < K; ++k) {
                        float v = acc[k];
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                        if (lane == 0) s_red[group][tw][k] = v;
                    }
                    group_barrier(group);
                    if (gtid < K) {
                        double sum = 0.0;
#pragma unroll
                        for (int i = 0; i < GROUP_WARPS; ++i) sum += (double)s_red[group][i][gtid];
                        partials[((long long)b * nslot + slot) * KMAX + gtid] += sum;
                    }
                }
            }
            if (!SINGLE) {
                group_barrier(group);                       // every thread of the group is done with the stage
                if (leader) issue_next();
            }
        }
    }
    if (leader && visited) atomicAdd(visited + 1, (unsigned long long)(SKIP ? n_loaded : j));
    if (SINGLE) {                                           // the group's K sums over all its tiles
        if (s_running[0]) {                                 // what is left in the queue
            group_barrier(group);
            const GatherView gv = s_gv[0];
            if (gtid < q_n) {
                int pos = q_head + gtid;
                if (pos >= QCAP) pos -= QCAP;
                const QueueEntry<K> en = queue[pos];
                const float xw = G.cx + ((float)(en.xy & 0xffff) - 0.5f * (G.nx - 1)) * G.hx;
                const float yw = G.cy + ((float)(en.xy >> 16) - 0.5f * (G.ny - 1)) * G.hy;
                const float zw = G.cz + ((float)en.z - 0.5f * (G.nz - 1)) * G.hz;
                const float Bj = bvol ? __ldg(bvol + ((long long)en.z * G.ny + (en.xy >> 16)) * G.nx + (en.xy & 0xffff))
                                      : gather_voxel(G, gv, rL, utab, vtab, xw, yw, zw);
#pragma unroll
                for (int k = 0; k < K; ++k) acc[k] = fmaf(Bj, en.q[k], acc[k]);
            }
        }
        double sum[K];
#pragma unroll
        for (int k = 0; k < K; ++k) sum[k] = warp_sum((double)acc[k]);
        __shared__ double s_fin[GNG][GROUP_WARPS][K];
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < K; ++k) s_fin[group][tw][k] = sum[k];
        }
        group_barrier(group);
        if (gtid < K) {
            double tot = 0.0;
#pragma unroll
            for (int i = 0; i < GROUP_WARPS; ++i) tot += s_fin[group][i][gtid];
            partials[(long long)slot * KMAX + gtid] = tot;
        }
    }
    tl_end(G.tl, TLK_GRAD);
}

// ---------------------------------------------------------------- one solve: the gather over the records
//
// For a single solve the streaming pass above is not needed at all: the warp kernel that wrote the
// accepted candidate's trial volume had the eight taps of every voxel in registers and left a record
// (x, y, z, G_j) for every voxel with G_j != 0 (stream.cuh GradRecords; warp.cu).  What remains of
// a-4 is, per record: B_j by the voxel-driven detector gather (the same exact l_ij; or from the
// backprojection volume of the ray-marching variant), u_kj from the fields (3 K scattered loads),
// and acc_k += B_j (G_j . u_kj); per thread over its records, then warp -> block -> partial sums, all
// in fixed order.  No V-sized gradient volume exists at any point, and the K+1 fields are streamed
// once per line-search pass instead of once more per iteration.
constexpr int GG_WARPS = 8;        // warps of a gather block
constexpr int GG_THREADS = 32 * GG_WARPS;
constexpr int GG_ROUND = GG_THREADS;   // sub-tiles whose records a block flattens at a time: one count per thread
// blocks per SM (64 registers per thread for K <= 4, 80 beyond): the kernel lives on warps in flight
__host__ __device__ constexpr int gather_per_sm(int K) { return K <= 4 ? 4 : 3; }

// Block v takes sub-tiles v, v + grid, ...; their records are flattened (prefix of the counts,
// GG_ROUND sub-tiles at a time: usually all of the block's) and dealt one per thread, so that every
// lane has work whatever the counts.  One partial sum per block and k.
template <int K>
__global__ void __launch_bounds__(GG_THREADS, gather_per_sm(K))
k_grad_gather(const Geom G, const SolveState* __restrict__ solves, int* __restrict__ rec_base, long long n_sub, int cap,
              const float* __restrict__ fields, const float* __restrict__ u_aos, const float* rL, const float4* utab,
              const float2* vtab, const float* bvol, double* partials,
              unsigned long long* __restrict__ visited) {
    __shared__ double red[GG_WARPS][K];
    __shared__ int s_pref[GG_ROUND + 1];
    __shared__ int s_wsum[GG_WARPS];
    tl_begin(G.tl);
    const int b = blockIdx.y;                                               // the solve (grid.y solves in flight)
    if (!needs_gradient(solves[b])) { tl_end(G.tl, TLK_GRAD); return; }    // uniform over the block
    const GradRecords rec = grad_records(rec_base, n_sub, n_sub * cap, solves[b].acc_slot);   // of the accepted candidate
    const GatherView gv = make_gather_view(G, solves[b].view);
    rL += (long long)b * G.npix; utab += (long long)b * G.nu; vtab += (long long)b * G.nv;
    if (bvol) bvol += (long long)b * G.V;
    partials += (long long)b * gridDim.x * KMAX;
    const float* __restrict__ u = fields + 3 * G.V;                          // u_1 .. u_K, planar, voxel units
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float acc[K];
#pragma unroll
    for (int k = 0; k < K; ++k) acc[k] = 0.f;
    long long n_gathered = 0;
    for (long long t0 = blockIdx.x; t0 < n_sub; t0 += (long long)gridDim.x * GG_ROUND) {
        // the counts of this round's sub-tiles t0, t0 + grid, ... and their exclusive prefix
        const long long t = t0 + (long long)threadIdx.x * gridDim.x;
        int incl = t < n_sub ? __ldcg(rec.count + t) : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        if (lane == 31) s_wsum[warp] = incl;
        __syncthreads();                                   // (every thread is done with the previous round's prefix)
        int before = 0, total = 0;
#pragma unroll
        for (int i = 0; i < GG_WARPS; ++i) {
            const int v = s_wsum[i];
            before += i < warp ? v : 0;
            total += v;
        }
        s_pref[threadIdx.x + 1] = before + incl;
        if (threadIdx.x == 0) s_pref[0] = 0;
        __syncthreads();
        n_gathered += total;
        for (int e = threadIdx.x; e < total; e += GG_THREADS) {
            int lo = 0, hi = GG_ROUND;                      // sub-tile index i with pref[i] <= e < pref[i + 1]
#pragma unroll
            for (int step = 0; step < 8; ++step) {
                const int mid = (lo + hi) >> 1;
                if (s_pref[mid] <= e) lo = mid; else hi = mid;
            }
            const long long idx = (t0 + (long long)lo * gridDim.x) * cap + (e - s_pref[lo]);
            const int4* rp = reinterpret_cast<const int4*>(rec.r + idx);             // one 48-byte record
            const int4 rw = __ldcg(rp), c03 = __ldcg(rp + 1), c47 = __ldcg(rp + 2);
            const int x = record_x(rw.x), y = record_y(rw.x), z = record_z(rw.x);
            // G_j from the taps and fractions the warp kernel had (trilinear.cuh: the same arithmetic)
            Taps tp;
            tp.base = 0u;
            tp.wx1 = __int_as_float(rw.y); tp.wy1 = __int_as_float(rw.z); tp.wz1 = __int_as_float(rw.w);
            tp.wx0 = 1.f - tp.wx1; tp.wy0 = 1.f - tp.wy1; tp.wz0 = 1.f - tp.wz1;
            const float cv[8] = {__int_as_float(c03.x), __int_as_float(c03.y), __int_as_float(c03.z), __int_as_float(c03.w),
                                 __int_as_float(c47.x), __int_as_float(c47.y), __int_as_float(c47.z), __int_as_float(c47.w)};
            float gx, gy, gz;
            grad8(tp, cv, &gx, &gy, &gz);
            if (gx == 0.f && gy == 0.f && gz == 0.f) continue;                       // contributes an exact 0
            const long long lin = ((long long)z * G.ny + y) * G.nx + x;
            float q[K];                                     // q_kj = G_j . u_kj (fields in voxel units: no 1/h, reading B4)
            if (u_aos) {                                    // uniform over the grid
                constexpr int P = aos_pitch(K);
                float uu[P];
                const float4* ua = reinterpret_cast<const float4*>(u_aos + lin * P);
#pragma unroll
                for (int i = 0; i < P / 4; ++i) {
                    const float4 v = __ldg(ua + i);
                    uu[4 * i] = v.x; uu[4 * i + 1] = v.y; uu[4 * i + 2] = v.z; uu[4 * i + 3] = v.w;
                }
#pragma unroll
                for (int k = 0; k < K; ++k) q[k] = gx * uu[3 * k] + gy * uu[3 * k + 1] + gz * uu[3 * k + 2];
            } else {
#pragma unroll
                for (int k = 0; k < K; ++k)
                    q[k] = gx * __ldg(u + (3 * k) * G.V + lin) + gy * __ldg(u + (3 * k + 1) * G.V + lin) + gz * __ldg(u + (3 * k + 2) * G.V + lin);
            }
            float Bj;
            if (bvol) Bj = __ldg(bvol + lin);
            else {
                const float xw = G.cx + ((float)x - 0.5f * (G.nx - 1)) * G.hx;
                const float yw = G.cy + ((float)y - 0.5f * (G.ny - 1)) * G.hy;
                const float zw = G.cz + ((float)z - 0.5f * (G.nz - 1)) * G.hz;
                Bj = gather_voxel(G, gv, rL, utab, vtab, xw, yw, zw);
            }
#pragma unroll
            for (int k = 0; k < K; ++k) acc[k] = fmaf(Bj, q[k], acc[k]);
        }
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const double sv = warp_sum((double)acc[k]);
        if (lane == 0) red[warp][k] = sv;
    }
    __syncthreads();
    if (threadIdx.x < K) {
        double tot = 0.0;
#pragma unroll
        for (int i = 0; i < GG_WARPS; ++i) tot += red[i][threadIdx.x];
        partials[(long long)blockIdx.x * KMAX + threadIdx.x] = tot;
    }
    if (threadIdx.x == 0 && visited) atomicAdd(visited + 2, (unsigned long long)n_gathered);
    tl_end(G.tl, TLK_GRAD);
}

// The cell map of FieldStream: one thread per interpolation cell.
__global__ void __launch_bounds__(256)
k_build_cellmap(const Geom G, const float* __restrict__ f0, unsigned char* __restrict__ cellmap) {
    const long long n = (long long)(G.nx + 1) * (G.ny + 1) * (G.nz + 1);
    const long long lin = (long long)blockIdx.x * 256 + threadIdx.x;
    if (lin >= n) return;
    const int i0 = (int)(lin % (G.nx + 1)) - 1, j0 = (int)((lin / (G.nx + 1)) % (G.ny + 1)) - 1,
              k0 = (int)(lin / ((long long)(G.nx + 1) * (G.ny + 1))) - 1;
    float first = 0.f;
    bool varies = false;
#pragma unroll
    for (int t = 0; t < 8; ++t) {
        const int i = i0 + (t & 1), j = j0 + ((t >> 1) & 1), k = k0 + (t >> 2);
        const bool in = (unsigned)i < (unsigned)G.nx && (unsigned)j < (unsigned)G.ny && (unsigned)k < (unsigned)G.nz;
        const float v = in ? f0[((long long)k * G.ny + j) * G.nx + i] : 0.f;      // zero padding (reading A2)
        if (t == 0) first = v;
        else varies |= v != first;
    }
    cellmap[lin] = varies ? 1 : 0;
}

// Hook: B = P^T r as a volume (view of solve 0).
__global__ void __launch_bounds__(256)
k_backproject(const Geom G, const SolveState* __restrict__ solves, const float* __restrict__ rL,
              const float4* __restrict__ utab, const float2* __restrict__ vtab, float* __restrict__ out) {
    const GatherView gv = make_gather_view(G, solves[0].view);
    const long long lin = (long long)blockIdx.x * 256 + threadIdx.x;
    if (lin >= G.V) return;
    const int i = (int)(lin % G.nx), j = (int)((lin / G.nx) % G.ny), k = (int)(lin / ((long long)G.nx * G.ny));
    const float xw = G.cx + ((float)i - 0.5f * (G.nx - 1)) * G.hx;
    const float yw = G.cy + ((float)j - 0.5f * (G.ny - 1)) * G.hy;
    const float zw = G.cz + ((float)k - 0.5f * (G.nz - 1)) * G.hz;
    out[lin] = gather_voxel(G, gv, rL, utab, vtab, xw, yw, zw);
}

template <int K, bool H>
void launch_tma(Seq& q, const Geom& G, const FieldStream& fs, const float* f0, const CtlBufs& c, int B,
                const float* rL, const float4* utab, const float2* vtab, const float* bvol) {
    static DeviceOnce configured;
    constexpr size_t smem = grad_smem_bytes<K, H>();
    {
        const cudaError_t e0 = configured.run([&] {
            cudaError_t e = cudaSuccess;
            auto set = [&](auto kernel) { if (e == cudaSuccess) e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); };
            set(k_grad_tma<K, true, H, true>); set(k_grad_tma<K, true, H, false>);
            set(k_grad_tma<K, false, H, true>); set(k_grad_tma<K, false, H, false>);
            return e;
        });
        if (e0 != cudaSuccess) { q.err = e0; return; }
    }
    constexpr int GNG = GradGroups<K>::value, GTHREADS = 32 * GNG * GROUP_WARPS;
    const int grid = grad_grid(G, fs);
    // the flags cost a few dependent loads per launch: only where a CTA has tiles enough to win them back
    const unsigned* skip_table = tile_count(G, TileZ<K>::value) >= fs.skip_min_tiles_per_sm * (long long)fs.n_sm ? fs.cell_integral : nullptr;
    if (fs.grad_rec) {                                  // the warp kernel left the records: gather only
        if (B > 65535) { q.err = cudaErrorInvalidValue; return; }
        const long long n_sub = tile_count(G, TileZ<K>::value) * GROUP_WARPS;
        // a plain edge into the gather: launched programmatically behind k_resid at the top level of the graph it
        // took 65 us instead of 38 (timeline; the other kernels are indifferent or gain)
        q.plain_next = true;
        q.launch(k_grad_gather<K>, dim3(grad_gather_blocks(G, fs), B), dim3(GG_THREADS), 0, G, (const SolveState*)c.solves, fs.grad_rec, n_sub,
                 TX * TileZ<K>::value / GROUP_WARPS, fs.fields, fs.u_aos, rL, utab, vtab, bvol, c.grad_part, fs.visited);
        return;
    }
    if (B == 1) {
        q.launch(skip_table ? k_grad_tma<K, true, H, true> : k_grad_tma<K, true, H, false>, dim3(grid), dim3(GTHREADS), smem, field_map<K>(fs), half_map<K>(fs), fs.scale, fs.fmax, skip_table, G, f0,
                 fs.cellmap, c, 0, 1, rL, utab, vtab, bvol, fs.visited);
        return;
    }
    for (int b0 = 0; b0 < B; b0 += SOLVE_CACHE) {       // the kernel keeps up to SOLVE_CACHE solves' constants on chip
        const int nb = B - b0 < SOLVE_CACHE ? B - b0 : SOLVE_CACHE;
        q.launch(skip_table ? k_grad_tma<K, false, H, true> : k_grad_tma<K, false, H, false>, dim3(grid), dim3(GTHREADS), smem, field_map<K>(fs), half_map<K>(fs), fs.scale, fs.fmax, skip_table, G, f0,
                 fs.cellmap, c, b0, nb, rL + (long long)b0 * G.npix, utab + (long long)b0 * G.nu,
                 vtab + (long long)b0 * G.nv, bvol ? bvol + (long long)b0 * G.V : bvol, fs.visited);
    }
}

template <int K>
void launch_k(Seq& q, const Geom& G, const FieldStream& fs, const float* f0, const CtlBufs& c, int B,
              const float* rL, const float4* utab, const float2* vtab, const float* bvol) {
    if (fs.use_tma) {
        if (fs.half_u) launch_tma<K, true>(q, G, fs, f0, c, B, rL, utab, vtab, bvol);
        else launch_tma<K, false>(q, G, fs, f0, c, B, rL, utab, vtab, bvol);
        return;
    }
    dim3 grid((G.nx + TILE - 1) / TILE, (G.ny + TILE - 1) / TILE, G.nz);
    q.launch(k_grad_generic<K>, grid, dim3(GT), 0, G, f0, fs.fields, fs.fields + 3 * G.V, c, B, rL, utab, vtab, bvol);
}

}  // namespace

int resid_blocks(const Geom& G) { return (G.npix + RT - 1) / RT; }

void launch_build_cellmap(cudaStream_t st, const Geom& G, const float* f0, unsigned char* cellmap) {
    const long long n = (long long)(G.nx + 1) * (G.ny + 1) * (G.nz + 1);
    k_build_cellmap<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(G, f0, cellmap);
}
// partial-sum slots per solve: two per persistent CTA (TMA kernel), else one per block
int grad_gather_blocks(const Geom& G, const FieldStream& fs) { return fs.n_sm * gather_per_sm(G.K); }

int grad_blocks(const Geom& G, const FieldStream& fs) {
    if (fs.use_tma) return grad_grid(G, fs) * grad_groups_for(G.K);
    return ((G.nx + TILE - 1) / TILE) * ((G.ny + TILE - 1) / TILE) * G.nz;
}

void launch_resid(Seq& q, const Geom& G, const SolveState* solves, const SolveIn* in, int B, int force,
                  const float* p, const float* r_direct, float* rL, float4* utab, float2* vtab, double* partials) {
    q.launch(k_resid, dim3(resid_blocks(G), B), dim3(RT), 0, G, solves, in, force, p, r_direct, rL, utab, vtab,
             partials);
}

void launch_grad(Seq& q, const Geom& G, const FieldStream& fs, const float* f0, const CtlBufs& c, int B,
                 const float* rL, const float4* utab, const float2* vtab, const float* bvol, int mode) {
    switch (G.K) {
#define PCAMM_CASE(KK) \
    case KK: launch_k<KK>(q, G, fs, f0, c, B, rL, utab, vtab, bvol); break;
        PCAMM_CASE(1) PCAMM_CASE(2) PCAMM_CASE(3) PCAMM_CASE(4)
        PCAMM_CASE(5) PCAMM_CASE(6) PCAMM_CASE(7) PCAMM_CASE(8)
#undef PCAMM_CASE
        default: break;
    }
    CtlBufs cc = c;                             // the control step that follows the gradient (control.cu) adds as many
    if (fs.use_tma && fs.grad_rec) cc.grad_blocks = grad_gather_blocks(G, fs);     // partial sums as the kernel left
    launch_ctl_after_grad(q, G, cc, mode);
}

void launch_backproject(Seq& q, const Geom& G, const SolveState* solves, const float* rL, const float4* utab,
                        const float2* vtab, float* vol_out) {
    q.launch(k_backproject, dim3((unsigned)((G.V + 255) / 256)), dim3(256), 0, G, solves, rL, utab, vtab, vol_out);
}

}  // namespace pcamm
