// a-2: cone-beam forward projection p = P_theta f  (section 2.2, Eq. 2;
// "P is a projection matrix which computes the projection image of f").
//
// Reading A3: p_i = sum_j l_ij f_j with l_ij the exact length of the source -> pixel-centre
// segment inside voxel box j (Siddon's radiological path).  The oracle merges and sorts all plane
// crossings; this kernel computes the same sum slab by slab:
//
//   the ray marches along its dominant in-plane axis m (|d_m|/h_m largest; t = the other in-plane
//   axis).  Between the planes M = i and M = i+1 (voxel-corner index units) it moves by
//   |sT| <= 1 voxels in t and |sZ| <= 1 voxels in z, so it crosses at most one t-plane and one
//   z-plane inside the slab: at most three voxels, whose shares tau of the slab length follow
//   from where those two crossings fall.  Summed over slabs this is exactly Siddon's sum; most
//   slabs hold a single voxel (one load, one add) and neighbouring rays read neighbouring
//   addresses.
//
// Layout: rays marching along y read the standard volume [z][y][x] (t = x is contiguous), rays
// marching along x read the in-plane transposed copy [z][x][y] (t = y contiguous), both written
// by the warp kernel.  One thread per ray, one warp per 32 consecutive u of a detector row, a
// block per 32 x 8 detector tile: a warp's loads of one slab fall into one or two 128 B lines.
//
// Ray set-up (source, direction, entry, first crossings, crossing spacing) is done in double; the
// march itself is integer (fixed-point crossing counters) plus one float multiply-add per piece.
//
// a-3 (first half): the same kernel forms r_i = p_i - a y_i - b and the per-block partial sums of
// p, y p and r^2 (Eq. 2, L91-93 Eq. 4) in double.
#include "internal.h"

namespace pcamm {

namespace {

constexpr int TU = 32, TV = 8, NT = TU * TV;

// One ray in the frame of its marching axis.  Slab n (n = 0 .. n_slabs-1, counted from the source
// side) is the n-th voxel layer along the marching axis that the ray meets; q in [n, n+1] is the
// ray parameter inside it.  The crossings of transverse (t) and axial (z) voxel planes are tracked
// as 32.32 fixed-point values of q: hi word = slab in which the crossing falls, lo word = share of
// that slab's path before it.  The first crossing and the spacing 1/|slope| come from the double
// precision set-up, so that a crossing's slab and share do not depend on float rounding of a
// position (for a ray almost parallel to a plane family that rounding, divided by the slope,
// would misplace the crossing by whole slabs).
struct Ray {
    int axis;                       // 0: marches along x (reads [z][x][y]); 1: along y (reads [z][y][x])
    int i_start, n_slabs, step;     // first layer index, count, +1 / -1
    int Nm, Nt, Nz;
    int j0, k0, dirT, dirZ;         // voxel of the entry point; direction of change at a crossing
    unsigned long long QT, dQT, QZ, dQZ;
    float Ls;                       // mm of path per slab
};

constexpr double FIX = 4294967296.0;            // 2^32
constexpr double QMAX = 1073741824.0;           // crossings beyond any volume are parked here (2^30 slabs)

__device__ __forceinline__ void first_crossing(double P0, double s, int* idx0, int* dir, unsigned long long* Q,
                                               unsigned long long* dQ) {
    const double fl = floor(P0);
    *idx0 = (int)fl;
    if (s == 0.0) { *dir = 0; *Q = (unsigned long long)(QMAX * FIX); *dQ = 0ull; return; }
    *dir = s > 0.0 ? 1 : -1;
    const double plane = s > 0.0 ? fl + 1.0 : fl;
    const double q = fmin(fmax((plane - P0) / s, 0.0), QMAX);
    const double d = fmin(1.0 / fabs(s), QMAX);
    *Q = (unsigned long long)(q * FIX + 0.5);
    *dQ = (unsigned long long)(d * FIX + 0.5);
    if (*dQ < (1ull << 32)) *dQ = 1ull << 32;   // |s| <= 1: never two crossings in one slab
}

__device__ __forceinline__ Ray make_ray(const Geom& G, const View& vw, int iu, int iv) {
    Ray r;
    double dx, dy;
    ray_dir_inplane(G, vw.cs, vw.sn, iu, &dx, &dy);                       // D - S
    const double dz = ((double)iv - 0.5 * (G.nv - 1) + (double)G.off_v) * (double)G.pv;
    const double Sx = (double)G.sad * vw.cs, Sy = (double)G.sad * vw.sn;
    const double L = sqrt(dx * dx + dy * dy + dz * dz);
    const double gx = dx / (double)G.hx, gy = dy / (double)G.hy, gz = dz / (double)G.hz;
    const double Sxi = (Sx - G.lox) / (double)G.hx, Syi = (Sy - G.loy) / (double)G.hy, Szi = (0.0 - G.loz) / (double)G.hz;
    double gm, gt, Sm, St;
    if (fabs(gx) >= fabs(gy)) { r.axis = 0; gm = gx; gt = gy; Sm = Sxi; St = Syi; r.Nm = G.nx; r.Nt = G.ny; }
    else                      { r.axis = 1; gm = gy; gt = gx; Sm = Syi; St = Sxi; r.Nm = G.ny; r.Nt = G.nx; }
    r.Nz = G.nz;
    const double sT = gt / gm, sZ = gz / gm;            // per unit of the marching coordinate M
    const double T0 = St - Sm * sT, Z0 = Szi - Sm * sZ; // at the plane M = 0
    r.step = gm > 0.0 ? 1 : -1;
    r.Ls = (float)(L / fabs(gm));
    // layers in which the ray can be inside the volume (conservative by one; exactness comes from
    // the per-voxel range test in the sink)
    double Mlo = 0.0, Mhi = (double)r.Nm;
    bool empty = false;
    if (sT != 0.0) {
        const double m0 = (0.0 - T0) / sT, m1 = ((double)r.Nt - T0) / sT;
        Mlo = fmax(Mlo, fmin(m0, m1)); Mhi = fmin(Mhi, fmax(m0, m1));
    } else if (!(T0 >= 0.0 && T0 < (double)r.Nt)) empty = true;
    if (sZ != 0.0) {
        const double m0 = (0.0 - Z0) / sZ, m1 = ((double)r.Nz - Z0) / sZ;
        Mlo = fmax(Mlo, fmin(m0, m1)); Mhi = fmin(Mhi, fmax(m0, m1));
    } else if (!(Z0 >= 0.0 && Z0 < (double)r.Nz)) empty = true;
    int ifirst = (int)floor(Mlo) - 1, ilast = (int)ceil(Mhi);
    ifirst = max(ifirst, 0); ilast = min(ilast, r.Nm - 1);
    r.n_slabs = 0; r.i_start = 0; r.j0 = r.k0 = r.dirT = r.dirZ = 0; r.QT = r.dQT = r.QZ = r.dQZ = 0ull;
    if (empty || !(Mlo <= Mhi) || ilast < ifirst) return r;
    r.n_slabs = ilast - ifirst + 1;
    r.i_start = r.step > 0 ? ifirst : ilast;
    const double Mb = r.step > 0 ? (double)ifirst : (double)(ilast + 1);   // entry plane of the first slab
    first_crossing(T0 + sT * Mb, sT * r.step, &r.j0, &r.dirT, &r.QT, &r.dQT);
    first_crossing(Z0 + sZ * Mb, sZ * r.step, &r.k0, &r.dirZ, &r.QZ, &r.dQZ);
    return r;
}

// Calls sink(i, j, k, tau) for every (layer i, transverse j, axial k) piece, source side first;
// tau = share of the slab's path length.
template <class Sink>
__device__ __forceinline__ void march(const Ray& r, Sink& sink) {
    int i = r.i_start, j = r.j0, k = r.k0;
    unsigned long long QT = r.QT, QZ = r.QZ;
    const float inv32 = 2.3283064365386963e-10f;   // 2^-32
    for (int n = 0; n < r.n_slabs; ++n, i += r.step) {
        const bool ct = (unsigned)(QT >> 32) == (unsigned)n, cz = (unsigned)(QZ >> 32) == (unsigned)n;
        if (!ct && !cz) { sink(i, j, k, 1.f); continue; }
        const float tt = ct ? __uint2float_rn((unsigned)QT) * inv32 : 1.f;
        const float tz = cz ? __uint2float_rn((unsigned)QZ) * inv32 : 1.f;
        const int je = ct ? j + r.dirT : j, ke = cz ? k + r.dirZ : k;
        const float t1 = fminf(tt, tz), t2 = fmaxf(tt, tz);
        sink(i, j, k, t1);
        const bool tfirst = tt < tz;
        sink(i, tfirst ? je : j, tfirst ? k : ke, t2 - t1);
        if (ct && cz) sink(i, je, ke, 1.f - t2);
        j = je; k = ke;
        if (ct) QT += r.dQT;
        if (cz) QZ += r.dQZ;
    }
}

struct AccSink {
    const float* __restrict__ vol;
    int Nm, Nt, Nz;
    float acc;
    __device__ __forceinline__ void operator()(int i, int j, int k, float tau) {
        if ((unsigned)j < (unsigned)Nt && (unsigned)k < (unsigned)Nz)
            acc = fmaf(tau, __ldg(vol + (k * Nm + i) * Nt + j), acc);
    }
};

__global__ void __launch_bounds__(NT)
k_project(const Geom G, const SlotState* __restrict__ slots, const SolveState* __restrict__ solves,
          const SolveIn* __restrict__ in, const float* __restrict__ vol_std, const float* __restrict__ vol_tr,
          long long slot_stride, float* __restrict__ p_out, double* __restrict__ partials) {
    __shared__ double red[NT / 32];
    const int s = blockIdx.z;
    if (!slots[s].active) return;
    const int b = slots[s].solve;
    const View vw = solves[b].view;
    const int tiles_u = (G.nu + TU - 1) / TU;
    const int iu = (blockIdx.x % tiles_u) * TU + (threadIdx.x & 31);
    const int iv = (blockIdx.x / tiles_u) * TV + (threadIdx.x >> 5);
    double vp = 0.0, vyp = 0.0, vrr = 0.0;
    if (iu < G.nu && iv < G.nv) {
        const Ray r = make_ray(G, vw, iu, iv);
        AccSink sink;
        sink.vol = (r.axis == 0 ? vol_tr : vol_std) + (long long)s * slot_stride;
        sink.Nm = r.Nm; sink.Nt = r.Nt; sink.Nz = r.Nz; sink.acc = 0.f;
        march(r, sink);
        const float p = sink.acc * r.Ls;
        const int pix = iv * G.nu + iu;
        p_out[(long long)s * G.npix + pix] = p;
        const float* y = in[b].y;
        const double yv = y ? (double)__ldg(y + pix) : 0.0;
        const double res = (double)p - solves[b].a * yv - solves[b].b;   // Eq. (2) residual
        vp = (double)p; vyp = yv * (double)p; vrr = res * res;
    }
    const int nblk = gridDim.x;
    double* out = partials + ((long long)s * nblk + blockIdx.x) * 3;
    const double sp = block_sum<NT>(vp, red);
    const double syp = block_sum<NT>(vyp, red);
    const double srr = block_sum<NT>(vrr, red);
    if (threadIdx.x == 0) { out[0] = sp; out[1] = syp; out[2] = srr; }
}

// In-plane transpose [z][y][x] -> [z][x][y] (hook path only: the solve's volumes are written in
// both layouts by the warp kernel).
__global__ void __launch_bounds__(256)
k_transpose(const Geom G, const float* __restrict__ src, float* __restrict__ dst) {
    __shared__ float tile[32][33];
    const int lane = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32, z = blockIdx.z;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int y = y0 + ty + 8 * r, x = x0 + lane;
        tile[ty + 8 * r][lane] = (x < G.nx && y < G.ny) ? src[((long long)z * G.ny + y) * G.nx + x] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int x = x0 + ty + 8 * r, y = y0 + lane;
        if (x < G.nx && y < G.ny) dst[((long long)z * G.nx + x) * G.ny + y] = tile[lane][ty + 8 * r];
    }
}

struct RecSink {
    int axis, cap, n;
    int Nt, Nz;
    float Ls, eps;
    int* ijk;
    float* len;
    __device__ __forceinline__ void operator()(int i, int j, int k, float tau) {
        if (!((unsigned)j < (unsigned)Nt && (unsigned)k < (unsigned)Nz)) return;
        const float l = tau * Ls;
        if (!(l > eps)) return;     // zero-length pieces are dropped (reading A22)
        if (n < cap) {
            ijk[3 * n + 0] = axis == 0 ? i : j;
            ijk[3 * n + 1] = axis == 0 ? j : i;
            ijk[3 * n + 2] = k;
            len[n] = l;
        }
        ++n;
    }
};

__global__ void k_traverse(const Geom G, const SolveState* __restrict__ solves, int iu, int iv, int cap, int* ijk,
                           float* len, int* n_out) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const Ray r = make_ray(G, solves[0].view, iu, iv);
    RecSink sink;
    sink.axis = r.axis; sink.cap = cap; sink.n = 0; sink.Nt = r.Nt; sink.Nz = r.Nz; sink.Ls = r.Ls;
    sink.eps = 1e-6f * fminf(G.hx, fminf(G.hy, G.hz));
    sink.ijk = ijk; sink.len = len;
    march(r, sink);
    *n_out = sink.n;
}

}  // namespace

int project_blocks(const Geom& G) { return ((G.nu + TU - 1) / TU) * ((G.nv + TV - 1) / TV); }

void launch_project(Seq& q, const Geom& G, const SlotState* slots, const SolveState* solves, const SolveIn* in,
                    int nslots, const float* vol_std, const float* vol_tr, long long slot_stride, float* p,
                    double* partials) {
    q.launch(k_project, dim3(project_blocks(G), 1, nslots), dim3(NT), 0, G, slots, solves, in, vol_std, vol_tr,
             slot_stride, p, partials);
}

void launch_transpose(Seq& q, const Geom& G, const float* vol_std, float* vol_tr) {
    q.launch(k_transpose, dim3((G.nx + 31) / 32, (G.ny + 31) / 32, G.nz), dim3(256), 0, G, vol_std, vol_tr);
}

void launch_traverse(Seq& q, const Geom& G, const SolveState* solves, int iu, int iv, int cap, int* ijk, float* len,
                     int* n_out) {
    q.launch(k_traverse, dim3(1), dim3(32), 0, G, solves, iu, iv, cap, ijk, len, n_out);
}

}  // namespace pcamm
