// The 8-tap trilinear stencil shared by a-1 (warp.cu: the interpolated value) and a-4
// (gradient.cu: its exact derivative with respect to the displacement).
//
//   f(q) = sum_abc c_abc X_a Y_b Z_c,   c_abc = f0(i0 + (a,b,c)), f0 = 0 outside the grid
//   ("found through trilinear interpolation"; readings A2, A6, B1).
#pragma once

#include "common.cuh"

namespace pcamm {

// f0 is read from a copy with a border of two zero voxels on every side (Geom::fnx, fny, fpp:
// voxel (i,j,k) at ((k + 2) fny + (j + 2)) fnx + (i + 2)), so that reading A2 (f0 = 0 outside the
// grid) needs neither masks nor per-tap clamps: the cell index is clamped once per axis into
// [-2, n], where both of its taps lie in the border.
//
// One axis: the cell index a = i + floor(d) (clamped) and the fraction t = d - floor(d).  floor()
// and the fraction are taken of the displacement alone, so that the lattice position never enters
// a float32 sum (idx + d would lose 1e-5 voxel at idx ~ 256).  Branch-free, so that the gathers
// of several voxels can be in flight together.
struct AxisTaps {
    int a;
    float t;
};

__device__ __forceinline__ AxisTaps axis_taps(int i, float d, int n) {
    const float fl = floorf(d);
    AxisTaps r;
    r.t = d - fl;
    r.a = min(max(i + (int)fl, -2), n);
    return r;
}

// The 8-tap stencil of one voxel, split into address set-up, gather and combination so that a
// thread can have the gathers of all its voxels in flight before it consumes the first.
struct Taps {
    unsigned base;                  // element offset of tap (0,0,0) in the padded f0
    float wx0, wx1, wy0, wy1, wz0, wz1;
};

__device__ __forceinline__ Taps make_taps(const Geom& G, int i, int j, int k, float dx, float dy, float dz) {
    const AxisTaps X = axis_taps(i, dx, G.nx), Y = axis_taps(j, dy, G.ny), Z = axis_taps(k, dz, G.nz);
    Taps t;
    t.base = (unsigned)(((Z.a + 2) * G.fny + (Y.a + 2)) * G.fnx + (X.a + 2));
    t.wx0 = 1.f - X.t; t.wx1 = X.t; t.wy0 = 1.f - Y.t; t.wy1 = Y.t; t.wz0 = 1.f - Z.t; t.wz1 = Z.t;
    return t;
}

// c[0..7]: taps (x0,y0,z0), (x1,y0,z0), (x0,y1,z0), (x1,y1,z0), (x0,y0,z1), ...; f0p: the padded copy.
__device__ __forceinline__ void gather8(const Geom& G, const float* __restrict__ f0p, const Taps& t, float* c) {
    // 32-bit element offsets (the padded copy has fewer than 2^31 elements): one add and one widening
    // multiply-add per tap pair instead of 64-bit pointer sums
    const unsigned b10 = t.base + (unsigned)G.fnx, b01 = t.base + (unsigned)G.fpp, b11 = b01 + (unsigned)G.fnx;
    const float* p00 = f0p + t.base;
    const float* p10 = f0p + b10;
    const float* p01 = f0p + b01;
    const float* p11 = f0p + b11;
    c[0] = __ldg(p00); c[1] = __ldg(p00 + 1);
    c[2] = __ldg(p10); c[3] = __ldg(p10 + 1);
    c[4] = __ldg(p01); c[5] = __ldg(p01 + 1);
    c[6] = __ldg(p11); c[7] = __ldg(p11 + 1);
}

// sum_abc c_abc X_a Y_b Z_c, x innermost.
__device__ __forceinline__ float combine8(const Taps& t, const float* c) {
    const float v00 = c[0] * t.wx0 + c[1] * t.wx1, v10 = c[2] * t.wx0 + c[3] * t.wx1;
    const float v01 = c[4] * t.wx0 + c[5] * t.wx1, v11 = c[6] * t.wx0 + c[7] * t.wx1;
    return (v00 * t.wy0 + v10 * t.wy1) * t.wz0 + (v01 * t.wy0 + v11 * t.wy1) * t.wz1;
}

// d f / d q (per voxel of displacement) of the same interpolant: forward differences along the
// four parallel cell edges per axis, bilinearly weighted ("has to be consistent with
// the interpolation process"; reading A6).  A tap outside the grid is a 0 of the border.
__device__ __forceinline__ void grad8(const Taps& t, const float* c, float* gx, float* gy, float* gz) {
    const float dx00 = c[1] - c[0], dx10 = c[3] - c[2], dx01 = c[5] - c[4], dx11 = c[7] - c[6];
    *gx = (t.wy0 * dx00 + t.wy1 * dx10) * t.wz0 + (t.wy0 * dx01 + t.wy1 * dx11) * t.wz1;
    const float dy00 = c[2] - c[0], dy10 = c[3] - c[1], dy01 = c[6] - c[4], dy11 = c[7] - c[5];
    *gy = (t.wx0 * dy00 + t.wx1 * dy10) * t.wz0 + (t.wx0 * dy01 + t.wx1 * dy11) * t.wz1;
    const float dz00 = c[4] - c[0], dz10 = c[5] - c[1], dz01 = c[6] - c[2], dz11 = c[7] - c[3];
    *gz = (t.wx0 * dz00 + t.wx1 * dz10) * t.wy0 + (t.wx0 * dz01 + t.wx1 * dz11) * t.wy1;
}

}  // namespace pcamm
