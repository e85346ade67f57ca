// Shared device structs and helpers of the CUDA path.  No code here is shared with oracle/.
//
// Notation follows the paper (section 2): f0 reference volume, xbar mean DVF, u_k
// eigenvector fields, w PCA coefficients, y measured projection, P_theta projector, (a, b)
// intensity fit, J cost, g = dJ/dw, mu step size.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/pcamm.h"

namespace pcamm {

constexpr int KMAX = PCAMM_KMAX;
constexpr int MAXBT = PCAMM_MAX_BACKTRACKS;
constexpr int TRACE_CAP = 1024;  // iterations recorded in the device-side traces

// Measurement (pcamm_tune "timeline"): start and end of every kernel of a solve on the device's
// global timer, taken inside the kernels (first block in, last block out).  The kernels of a solve
// run strictly one after the other, so one running event index serves them all.
constexpr int TL_CAP = 2048;
enum { TLK_YSUMS = 0, TLK_BEGIN, TLK_VIEW, TLK_WARP, TLK_PROJECT, TLK_CTL_PROJ, TLK_RESID, TLK_GRAD, TLK_CTL_GRAD,
       TLK_ITER_END, TLK_FINAL, TLK_INVERT };
struct Timeline {
    unsigned n, done;
    unsigned pad[2];
    unsigned long long t0[TL_CAP], t1[TL_CAP];      // ns; t0 preset to ~0, t1 to 0
    int kind[TL_CAP];
};
__device__ __forceinline__ unsigned long long global_timer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ bool tl_first_thread() { return (threadIdx.x | threadIdx.y | threadIdx.z) == 0; }
// Programmatic dependent launch (internal.h Seq, pcamm_tune "pdl"): inside the solve graph a kernel
// may be launched, and its blocks become resident, while its predecessor drains; the blocks wait here
// until the predecessor has completed and its writes are visible.  Nothing a previous kernel wrote
// may be read, and nothing it read may be overwritten, before this; every kernel of the graph calls
// it first thing (through tl_begin), so the order of all memory effects is that of the plain graph.
// Once through, the kernel lets its own dependents be launched: they wait the same way, and at most
// one kernel is ever resident ahead of the running one.  (Launched without a programmatic edge both
// instructions do nothing.)
__device__ __forceinline__ void grid_dependency_wait() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
// at the top of a kernel, by every block
__device__ __forceinline__ void tl_begin(Timeline* tl) {
    grid_dependency_wait();
    if (tl && tl_first_thread()) {
        const unsigned e = *(volatile unsigned*)&tl->n;
        if (e < TL_CAP) atomicMin(&tl->t0[e], global_timer_ns());
    }
}
// wherever a block leaves the kernel (uniform over the block)
__device__ __forceinline__ void tl_end(Timeline* tl, int kind) {
    if (!tl) return;
    __syncthreads();
    if (tl_first_thread()) {
        const unsigned e = *(volatile unsigned*)&tl->n;
        if (e < TL_CAP) atomicMax(&tl->t1[e], global_timer_ns());
        __threadfence();
        const unsigned nblk = gridDim.x * gridDim.y * gridDim.z;
        if (atomicAdd(&tl->done, 1u) == nblk - 1u) {
            tl->done = 0u;
            if (e < TL_CAP) tl->kind[e] = kind;
            __threadfence();
            *(volatile unsigned*)&tl->n = e + 1u;
        }
    }
}

// Model-constant geometry (passed to kernels by value).
struct Geom {
    Timeline* tl;             // NULL unless the timeline knob was on when the model was created
    int nx, ny, nz;
    long long V;
    int pnx, pny;             // in-plane size of a ray-layout volume: nx + 2, ny + 2 (zero border)
    long long PV;             // elements of one ray-layout volume: pnx * pny * nz
    int occ_pitch;            // occupancy bytes per voxel column of the ray layout (one per 16 z, padded to 8)
    long long OCC;            // occupancy bytes of one trial volume: pnx * pny * occ_pitch
    int fnx, fny, fpp;        // padded f0 (two zero voxels on every side): nx + 4, ny + 4, fnx * fny (trilinear.cuh)
    float hx, hy, hz;
    float ihx, ihy, ihz;      // 1 / h
    float cx, cy, cz;         // world position of the volume centre
    double lox, loy, loz;     // world position of the volume's low corner
    double ihz_d, Szi;        // 1 / hz and the source plane z = 0 in voxel-corner units, -loz / hz (project.cu)
    int K;
    int nu, nv, npix;
    float pu, pv, sad, sdd, off_u, off_v;
    unsigned tile_mx, tile_my; // ceil(2^32 / tiles along x), ceil(2^32 / ny): tile index -> coordinates without divisions (stream.cuh tile_coord; 0: divide)
    int projector;            // 0: Siddon's exact path lengths (project.cu), 1: fixed-step ray marching (raymarch.cu)
    float rm_step_mm;         // nominal step of the ray marching
};

// Angle-dependent part of the geometry of one solve, computed on the device in double.
struct View {
    double cs, sn;
};

// Ray layout of a trial volume (what the projector reads): z fastest, one voxel of zero border
// in x and y,   element (x, y, z) at ((y + 1) * pnx + (x + 1)) * nz + z.
// All rays of one detector column share their in-plane path, so a warp takes 32 consecutive
// detector rows of one column: its lanes sit in the same (x, y) voxel column and read
// neighbouring z, i.e. one or two 128 B lines per load, whatever the gantry angle.
__host__ __device__ __forceinline__ long long ray_layout_index(const Geom& G, int x, int y, int z) {
    return ((long long)(y + 1) * G.pnx + (x + 1)) * G.nz + z;
}

// Occupancy of a trial volume: one byte per voxel column (x, y) of the ray layout and range of 16
// z, non-zero iff some voxel there is non-zero.  Written by whoever writes the volume (every
// byte exactly once per pass; the border columns stay 0), read by the projector to skip the slabs
// of a ray that lie in air: their contribution is an exact +0.
__device__ __forceinline__ long long occ_index(const Geom& G, int x, int y, int zt16) {
    return ((long long)(y + 1) * G.pnx + (x + 1)) * G.occ_pitch + zt16;
}
// A warp holding tz = 16 or 32 consecutive z (lane = z - z0, z0 a multiple of tz) of column (x, y):
// records the one or two 16-ranges.
__device__ __forceinline__ void occ_record(const Geom& G, unsigned char* __restrict__ occ, int x, int y, int z0,
                                           int tz, bool nonzero) {
    const unsigned bal = __ballot_sync(0xffffffffu, nonzero);
    if ((threadIdx.x & 31) == 0 && x < G.nx) {
        const int zt = z0 >> 4;
        occ[occ_index(G, x, y, zt)] = (bal & 0xffffu) ? 1 : 0;
        if (tz == 32 && z0 + 16 < G.nz) occ[occ_index(G, x, y, zt + 1)] = (bal >> 16) ? 1 : 0;
    }
}

// Per view and detector column: the in-plane part of the slab traversal (project.cu).
struct ColHdr {
    double lam0;              // (M_b - S_m) / g_m at the entry plane of the first slab
    double kap;               // 1 / |g_m|: ray parameter per slab, in units of (D - S) per voxel
    float dxy2;               // in-plane part of |D - S|^2, mm^2
    int n_slabs;              // slabs in which the column's rays can be inside the volume in-plane
    int dT;                   // voxel-column offset ((y + 1) pnx + (x + 1) units) to the next column across a transverse plane
    int axis;                 // 0: marches along x, 1: along y
};

// Per view, column and slab: the voxel column (i, j) the ray is in when it enters the slab, as the
// column index (j + 1) pnx + (i + 1) of the ray layout, and the share tt of the slab's path before
// the transverse plane crossing (1 if none in this slab), stored in units of 2^-32 of the slab
// like the z crossing counters.
struct SlabEntry {
    int col;
    float tt;
};

// Host -> device, one copy per call.
struct CallOpts {
    int B, C;                 // solves in flight, candidate steps evaluated per trial round (the fan width)
    int max_iter, max_backtracks, batched, inv_max_iter;
    double grad_tol, armijo_c, armijo_beta, init_step_vox, inv_tol;
    double hmin_sqrtV;        // min(h) * sqrt(V): the 1-voxel-rms step scale (reading A7)
};

struct SolveIn {
    const float* y;           // measured projection of this solve (device)
    float angle;
    float w_init[KMAX];
    float a, b;               // used by the pcamm_eval hook only
};

struct SolveState {
    View view;
    double w[KMAX], g[KMAX];
    double a, b, Sy, Syy;
    double Jn, J0, J, g2, mu, mu_prev;
    double fit_a, fit_b;      // pcamm_eval hook: least-squares (a, b) for the evaluated p
    int iter, status, running, trialing, t, acc_slot;
};

struct SolveTrace {
    double J[TRACE_CAP + 1], gnorm[TRACE_CAP], mu[TRACE_CAP];
    int bt[TRACE_CAP];
};

// The loop of a solve is flat: its body is {residual, gradient, warp, projection}.  A solve in the
// middle of a line search (trialing) skips the first two; one whose step has just been accepted
// needs the residual and the gradient of its next iteration.
__device__ __forceinline__ bool needs_gradient(const SolveState& st) { return st.running && !st.trialing; }

// One trial evaluation: candidate c of solve b, slot s = b * C + c.
struct SlotState {
    float w[KMAX];
    int active, solve;
    double mu, J, Sp, Syp;
};

// Loop condition mirrored to plain memory so that the host-driven mode can read it, and the
// number of kernels the device-side loop has launched.
struct LoopFlags {
    int loop_cond, pad0;
    long long n_launch;
};

// Control step run by the last block of a projection (control.cuh) ...
constexpr int THEN_NONE = 0, THEN_INIT = 1, THEN_TRIAL = 2, THEN_EVAL = 3;
// ... and of a gradient pass.
constexpr int GRAD_NONE = 0, GRAD_SOLVE = 1, GRAD_EVAL = 2;

// Device buffers of the control steps.
struct CtlBufs {
    CallOpts* opts;
    SolveIn* in;
    SolveState* solves;
    SolveTrace* traces;
    SlotState* slots;
    LoopFlags* flags;
    int* seg_ticket;     // [S][nu]: blocks of a detector column that are done (self-resetting)
    double* ysum_part;   // [B][ysum_blocks][2]
    double* proj_part;   // [S][project_blocks][3]
    double* resid_part;  // [B][resid_blocks]
    double* grad_part;   // [B][grad_blocks][K]
    int ysum_blocks, proj_blocks, resid_blocks, grad_blocks;
};

// In-plane direction D - S of the rays of detector column iu (independent of the row).
__device__ __forceinline__ void ray_dir_inplane(const Geom& G, double cs, double sn, int iu, double* dx, double* dy) {
    const double uu = ((double)iu - 0.5 * (G.nu - 1) + (double)G.off_u) * (double)G.pu;
    *dx = -(double)G.sdd * cs - uu * sn;
    *dy = -(double)G.sdd * sn + uu * cs;
}

// ---------------------------------------------------------------- reductions

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over a block of NT threads (NT multiple of 32, <= 1024); result valid in thread 0.
// Fixed order: lanes by butterfly, warps in index order -> deterministic.
template <int NT>
__device__ __forceinline__ double block_sum(double v, double* smem /* [NT/32] */) {
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();  // protect smem reuse between successive calls
    if (lane == 0) smem[wid] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NT / 32; ++i) s += smem[i];
    }
    return s;
}

}  // namespace pcamm
