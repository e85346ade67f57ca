// The 8-tap trilinear stencil shared by a-1 (warp.cu: the interpolated value) and a-4
// (gradient.cu: its exact derivative with respect to the displacement).
//
//   f(q) = sum_abc c_abc X_a Y_b Z_c,   c_abc = f0(i0 + (a,b,c)), f0 = 0 outside the grid
//   ("found through trilinear interpolation"; readings A2, A6, B1).
#pragma once

#include "common.cuh"

namespace pcamm {

// One axis of the 8-tap stencil: the cell index i0 = i + floor(d), the fraction t = d - floor(d),
// the two tap indices clamped into the grid and the two weights, zeroed where the tap lies
// outside the grid (reading A2: f0 = 0 there).  floor() and the fraction are taken of the
// displacement alone, so that the lattice position never enters a float32 sum (idx + d would
// lose 1e-5 voxel at idx ~ 256).  Branch-free, so that the gathers of several voxels can be in
// flight together.
struct AxisTaps {
    int i0, i1;       // clamped tap indices
    float w0, w1;     // (1 - t), t, or 0 outside the grid
    float m0, m1;     // 1 inside the grid, 0 outside
};

__device__ __forceinline__ AxisTaps axis_taps(int i, float d, int n) {
    const float fl = floorf(d);
    const float t = d - fl;
    const int a = i + (int)fl, b = a + 1;
    AxisTaps r;
    r.m0 = (unsigned)a < (unsigned)n ? 1.f : 0.f;
    r.m1 = (unsigned)b < (unsigned)n ? 1.f : 0.f;
    r.w0 = (1.f - t) * r.m0;
    r.w1 = t * r.m1;
    r.i0 = min(max(a, 0), n - 1);
    r.i1 = min(max(b, 0), n - 1);
    return r;
}

// The 8-tap stencil of one voxel, split into address set-up, gather and combination so that a
// thread can have the gathers of all its voxels in flight before it consumes the first.
struct Taps {
    unsigned r00, r10, r01, r11;    // element offsets of the four x rows (y0 z0, y1 z0, y0 z1, y1 z1)
    int x0, x1;                     // clamped x indices
    float wx0, wx1, wy0, wy1, wz0, wz1;
    float mx0, mx1, my0, my1, mz0, mz1;   // used by the derivative only
};

__device__ __forceinline__ Taps make_taps(int nx, int ny, int nz, int i, int j, int k, float dx, float dy, float dz) {
    const AxisTaps X = axis_taps(i, dx, nx), Y = axis_taps(j, dy, ny), Z = axis_taps(k, dz, nz);
    Taps t;
    t.r00 = (unsigned)((Z.i0 * ny + Y.i0) * nx); t.r10 = (unsigned)((Z.i0 * ny + Y.i1) * nx);
    t.r01 = (unsigned)((Z.i1 * ny + Y.i0) * nx); t.r11 = (unsigned)((Z.i1 * ny + Y.i1) * nx);
    t.x0 = X.i0; t.x1 = X.i1;
    t.wx0 = X.w0; t.wx1 = X.w1; t.wy0 = Y.w0; t.wy1 = Y.w1; t.wz0 = Z.w0; t.wz1 = Z.w1;
    t.mx0 = X.m0; t.mx1 = X.m1; t.my0 = Y.m0; t.my1 = Y.m1; t.mz0 = Z.m0; t.mz1 = Z.m1;
    return t;
}

__device__ __forceinline__ void gather8(const float* __restrict__ f0, const Taps& t, float* c) {
    c[0] = __ldg(f0 + (t.r00 + t.x0)); c[1] = __ldg(f0 + (t.r00 + t.x1));
    c[2] = __ldg(f0 + (t.r10 + t.x0)); c[3] = __ldg(f0 + (t.r10 + t.x1));
    c[4] = __ldg(f0 + (t.r01 + t.x0)); c[5] = __ldg(f0 + (t.r01 + t.x1));
    c[6] = __ldg(f0 + (t.r11 + t.x0)); c[7] = __ldg(f0 + (t.r11 + t.x1));
}

// sum_abc c_abc X_a Y_b Z_c, x innermost.
__device__ __forceinline__ float combine8(const Taps& t, const float* c) {
    const float v00 = c[0] * t.wx0 + c[1] * t.wx1, v10 = c[2] * t.wx0 + c[3] * t.wx1;
    const float v01 = c[4] * t.wx0 + c[5] * t.wx1, v11 = c[6] * t.wx0 + c[7] * t.wx1;
    return (v00 * t.wy0 + v10 * t.wy1) * t.wz0 + (v01 * t.wy0 + v11 * t.wy1) * t.wz1;
}

// d f / d q (per voxel of displacement) of the same interpolant: forward differences along the
// four parallel cell edges per axis, bilinearly weighted ("has to be consistent with
// the interpolation process"; reading A6).  A tap outside the grid counts as 0 (masks).
__device__ __forceinline__ void grad8(const Taps& t, const float* c, float* gx, float* gy, float* gz) {
    const float dx00 = t.mx1 * c[1] - t.mx0 * c[0], dx10 = t.mx1 * c[3] - t.mx0 * c[2];
    const float dx01 = t.mx1 * c[5] - t.mx0 * c[4], dx11 = t.mx1 * c[7] - t.mx0 * c[6];
    *gx = (t.wy0 * dx00 + t.wy1 * dx10) * t.wz0 + (t.wy0 * dx01 + t.wy1 * dx11) * t.wz1;
    const float dy00 = t.my1 * c[2] - t.my0 * c[0], dy10 = t.my1 * c[3] - t.my0 * c[1];
    const float dy01 = t.my1 * c[6] - t.my0 * c[4], dy11 = t.my1 * c[7] - t.my0 * c[5];
    *gy = (t.wx0 * dy00 + t.wx1 * dy10) * t.wz0 + (t.wx0 * dy01 + t.wx1 * dy11) * t.wz1;
    const float dz00 = t.mz1 * c[4] - t.mz0 * c[0], dz10 = t.mz1 * c[5] - t.mz0 * c[1];
    const float dz01 = t.mz1 * c[6] - t.mz0 * c[2], dz11 = t.mz1 * c[7] - t.mz0 * c[3];
    *gz = (t.wx0 * dz00 + t.wx1 * dz10) * t.wy0 + (t.wx0 * dz01 + t.wx1 * dz11) * t.wy1;
}

}  // namespace pcamm
