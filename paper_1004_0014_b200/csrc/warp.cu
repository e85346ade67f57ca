// a-1: fused DVF synthesis + trilinear warp.
//
//   x_j = xbar_j + sum_k u_kj w_k                  (section 2.1, Eq. 1; L80 Eq. 2 constraint)
//   f_j = trilinear(f0, idx_j + x_j / h)           ("found through trilinear
//                                                   interpolation"; pull-back, L99; readings A1, A2)
//
// One pass over the K+1 vector fields serves every active trial slot (candidate steps of a
// batched line search, or independent solves in flight): the fields of a voxel are loaded once
// into registers and the slot loop runs inside the thread.
//
// HBM layout: fields planar [3][V] / [K][3][V] exactly as the caller gave them; a warp reads 32
// consecutive x of one row per load instruction (one 128 B line per plane and row).  The warped
// volume is written once, in the z-fastest ray layout of common.cuh that the projector reads at
// every gantry angle (or in the standard layout for the volume returned to the caller).
#include "internal.h"

namespace pcamm {

namespace {

constexpr int TILE = 32;
constexpr int ROWS = 4;        // voxels per thread (z rows tw, tw+8, tw+16, tw+24 of the tile)
constexpr int NTHREADS = 256;  // 32 x 8

// f0 with zero padding outside the grid (reading A2).
__device__ __forceinline__ float f0_tap(const float* __restrict__ f0, int nx, int ny, int nz, int i, int j, int k) {
    if ((unsigned)i < (unsigned)nx && (unsigned)j < (unsigned)ny && (unsigned)k < (unsigned)nz)
        return __ldg(f0 + ((long long)k * ny + j) * nx + i);
    return 0.f;
}

// Trilinear interpolation of f0 at voxel (i,j,k) displaced by d voxels (d = x / h).
// floor() and the fractional part are taken of the displacement alone, so that the lattice
// position never enters a float32 sum (idx + d would lose 1e-5 voxel at idx ~ 256).
__device__ __forceinline__ float trilinear(const float* __restrict__ f0, int nx, int ny, int nz, int i, int j, int k,
                                           float dx, float dy, float dz) {
    const float fx = floorf(dx), fy = floorf(dy), fz = floorf(dz);
    const float tx = dx - fx, ty = dy - fy, tz = dz - fz;
    const int i0 = i + (int)fx, j0 = j + (int)fy, k0 = k + (int)fz;
    float c000, c100, c010, c110, c001, c101, c011, c111;
    if (i0 >= 0 && i0 + 1 < nx && j0 >= 0 && j0 + 1 < ny && k0 >= 0 && k0 + 1 < nz) {
        const float* p = f0 + ((long long)k0 * ny + j0) * nx + i0;
        const long long sy = nx, sz = (long long)nx * ny;
        c000 = __ldg(p);           c100 = __ldg(p + 1);
        c010 = __ldg(p + sy);      c110 = __ldg(p + sy + 1);
        c001 = __ldg(p + sz);      c101 = __ldg(p + sz + 1);
        c011 = __ldg(p + sz + sy); c111 = __ldg(p + sz + sy + 1);
    } else {
        c000 = f0_tap(f0, nx, ny, nz, i0, j0, k0);         c100 = f0_tap(f0, nx, ny, nz, i0 + 1, j0, k0);
        c010 = f0_tap(f0, nx, ny, nz, i0, j0 + 1, k0);     c110 = f0_tap(f0, nx, ny, nz, i0 + 1, j0 + 1, k0);
        c001 = f0_tap(f0, nx, ny, nz, i0, j0, k0 + 1);     c101 = f0_tap(f0, nx, ny, nz, i0 + 1, j0, k0 + 1);
        c011 = f0_tap(f0, nx, ny, nz, i0, j0 + 1, k0 + 1); c111 = f0_tap(f0, nx, ny, nz, i0 + 1, j0 + 1, k0 + 1);
    }
    const float X0 = 1.f - tx, Y0 = 1.f - ty, Z0 = 1.f - tz;
    // sum_abc c_abc X_a Y_b Z_c, x innermost
    const float r00 = c000 * X0 + c100 * tx, r10 = c010 * X0 + c110 * tx;
    const float r01 = c001 * X0 + c101 * tx, r11 = c011 * X0 + c111 * tx;
    return (r00 * Y0 + r10 * ty) * Z0 + (r01 * Y0 + r11 * ty) * tz;
}

// Tile: 32 x by 32 z at fixed y.  Loads: lane = x (one 128 B line per plane and z).  Stores in the
// ray layout (RAY = true, what the projector reads): lane = z, through a 32x33 shared-memory
// tile, one 128 B line per (x, y); in the standard layout [z][y][x] (RAY = false: the volume
// handed back to the caller): lane = x.
template <int K, bool RAY>
__global__ void __launch_bounds__(NTHREADS)
k_warp(const Geom G, const float* __restrict__ f0, const float* __restrict__ xbar, const float* __restrict__ u,
       const SlotState* __restrict__ slots, int nslots, float* __restrict__ vol_out, long long slot_stride) {
    __shared__ float tile[TILE][TILE + 1];
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
                val[r] = trilinear(f0, G.nx, G.ny, G.nz, x, y, z0 + tw + 8 * r,
                                   __fdiv_rn(d[0], G.hx), __fdiv_rn(d[1], G.hy), __fdiv_rn(d[2], G.hz));
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
                if (xo < G.nx && zo < G.nz) out[ray_layout_index(G, xo, y, zo)] = tile[lane][tw + 8 * r];
            }
        }
    }
}

template <int K>
void launch_k(Seq& q, const Geom& G, const float* f0, const float* xbar, const float* u, const SlotState* slots,
              int nslots, int ray_layout, float* vol_out, long long slot_stride) {
    dim3 grid((G.nx + TILE - 1) / TILE, (G.nz + TILE - 1) / TILE, G.ny);
    if (ray_layout) q.launch(k_warp<K, true>, grid, dim3(NTHREADS), 0, G, f0, xbar, u, slots, nslots, vol_out, slot_stride);
    else q.launch(k_warp<K, false>, grid, dim3(NTHREADS), 0, G, f0, xbar, u, slots, nslots, vol_out, slot_stride);
}

}  // namespace

void launch_warp(Seq& q, const Geom& G, const float* f0, const float* xbar, const float* u, const SlotState* slots,
                 int nslots, int ray_layout, float* vol_out, long long slot_stride) {
    switch (G.K) {
#define PCAMM_CASE(KK) \
    case KK: launch_k<KK>(q, G, f0, xbar, u, slots, nslots, ray_layout, vol_out, slot_stride); break;
        PCAMM_CASE(1) PCAMM_CASE(2) PCAMM_CASE(3) PCAMM_CASE(4)
        PCAMM_CASE(5) PCAMM_CASE(6) PCAMM_CASE(7) PCAMM_CASE(8)
#undef PCAMM_CASE
        default: break;
    }
}

}  // namespace pcamm
