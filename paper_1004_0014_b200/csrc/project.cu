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
//   from where those two crossings fall.  Summed over slabs this is exactly Siddon's sum.
//
// Split of the work.  On a flat detector whose rows are parallel to the rotation axis, all rays
// of one detector column share their in-plane path; the gantry angle is fixed for the whole
// solve (P varies per angle, not per iteration).  So the in-plane traversal is
// tabulated ONCE per solve (k_view_tables: per column and slab the voxel column the ray is in
// and the share tt of the slab before its t-plane crossing, evaluated directly in double), and
// the projector, which runs once per line-search trial, only tracks the z crossings per ray (32.32
// fixed-point counters set up in double) and accumulates at most three pieces per slab.
//
// Mapping: one thread per ray, one warp per 32 consecutive detector rows of ONE column.  The
// lanes of a warp are in the same (x, y) voxel column and ~11 neighbouring z, so with the
// z-fastest ray layout of the trial volumes (common.cuh) every load of a warp falls into one or
// two 128 B lines at any gantry angle; the table entry of a slab is one broadcast 8-byte load;
// the trip count is uniform over the warp.  The volume was just written by the warp kernel and is
// L2/L1-resident: this kernel is bound by instruction issue, not by HBM.
//
// The rays are cut into segments of SEG slabs (one block per segment of 4 columns x 32 rows);
// the block of a ray group that finishes last adds the segments and forms the a-3 sums.
#include "internal.h"

namespace pcamm {

namespace {

constexpr int PW = 4;             // warps (= detector columns) per block
constexpr int NT = 32 * PW;
constexpr int SEG = 64;           // slabs per block (a multiple of the march's group size)

constexpr double FIX = 4294967296.0;            // 2^32
constexpr double QMAX = 1073741824.0;           // crossings beyond any volume are parked here (2^30 slabs)

// ------------------------------------------------------------------ per-view tables (once per solve)

struct ColSetup {
    int axis, Nm, Nt, step, dirT, n_slabs, i_start;
    double sT, T0, Mb, gm, Sm;
};

__device__ __forceinline__ ColSetup col_setup(const Geom& G, const View& vw, int iu, double* dxy2) {
    ColSetup c;
    double dx, dy;
    ray_dir_inplane(G, vw.cs, vw.sn, iu, &dx, &dy);                       // D - S, in-plane
    *dxy2 = dx * dx + dy * dy;
    const double Sx = (double)G.sad * vw.cs, Sy = (double)G.sad * vw.sn;
    const double gx = dx / (double)G.hx, gy = dy / (double)G.hy;
    const double Sxi = (Sx - G.lox) / (double)G.hx, Syi = (Sy - G.loy) / (double)G.hy;
    double gt, St;
    if (fabs(gx) >= fabs(gy)) { c.axis = 0; c.gm = gx; gt = gy; c.Sm = Sxi; St = Syi; c.Nm = G.nx; c.Nt = G.ny; }
    else                      { c.axis = 1; c.gm = gy; gt = gx; c.Sm = Syi; St = Sxi; c.Nm = G.ny; c.Nt = G.nx; }
    c.sT = gt / c.gm;                                   // t per unit of the marching coordinate M
    c.T0 = St - c.Sm * c.sT;                            // t at the plane M = 0
    c.step = c.gm > 0.0 ? 1 : -1;
    const double s = c.sT * c.step;
    c.dirT = s > 0.0 ? 1 : (s < 0.0 ? -1 : 0);
    // layers in which the in-plane ray overlaps [0, Nt): analytic range, widened by one, then
    // shrunk with the same expression the entries use
    double Mlo = 0.0, Mhi = (double)c.Nm;
    bool empty = false;
    if (c.sT != 0.0) {
        const double m0 = (0.0 - c.T0) / c.sT, m1 = ((double)c.Nt - c.T0) / c.sT;
        Mlo = fmax(Mlo, fmin(m0, m1)); Mhi = fmin(Mhi, fmax(m0, m1));
    } else if (!(c.T0 >= 0.0 && c.T0 < (double)c.Nt)) empty = true;
    int ifirst = (int)floor(Mlo) - 1, ilast = (int)ceil(Mhi);
    ifirst = max(ifirst, 0); ilast = min(ilast, c.Nm - 1);
    if (empty || !(Mlo <= Mhi)) ilast = ifirst - 1;
    auto Tat = [&](int M) { return fma(c.sT, (double)M, c.T0); };
    auto incl = [&](int i) {
        const double a = Tat(i), b = Tat(i + 1);
        return fmax(a, b) >= 0.0 && fmin(a, b) < (double)c.Nt;
    };
    while (ifirst <= ilast && !incl(ifirst)) ++ifirst;
    while (ilast >= ifirst && !incl(ilast)) --ilast;
    c.n_slabs = max(ilast - ifirst + 1, 0);
    c.i_start = c.step > 0 ? ifirst : ilast;
    c.Mb = c.step > 0 ? (double)ifirst : (double)(ilast + 1);            // entry plane of the first slab
    return c;
}

// grid (nu, B); the threads of a block share the column and take slabs n = tid, tid + NT, ...
__global__ void __launch_bounds__(128)
k_view_tables(const Geom G, const SolveState* __restrict__ solves, ColHdr* __restrict__ hdr,
              SlabEntry* __restrict__ tab, int max_slabs) {
    const int iu = blockIdx.x, b = blockIdx.y;
    const View vw = solves[b].view;
    double dxy2;
    const ColSetup c = col_setup(G, vw, iu, &dxy2);
    const int strideT = (c.axis == 0 ? G.pnx : 1) * G.nz;
    if (threadIdx.x == 0) {
        ColHdr h;
        h.lam0 = (c.Mb - c.Sm) / c.gm;
        h.kap = 1.0 / fabs(c.gm);
        h.dxy2 = (float)dxy2;
        h.n_slabs = c.n_slabs;
        h.dT = c.dirT * strideT;
        h.axis = c.axis;
        hdr[(long long)b * G.nu + iu] = h;
    }
    SlabEntry* row = tab + ((long long)b * G.nu + iu) * max_slabs;
    const double s = c.sT * c.step;
    for (int n = threadIdx.x; n < c.n_slabs; n += blockDim.x) {
        const int Me = (int)c.Mb + c.step * n;                    // plane through which the slab is entered
        const int i = c.i_start + c.step * n;                     // layer index of the slab
        const double Te = fma(c.sT, (double)Me, c.T0), Tx = fma(c.sT, (double)(Me + c.step), c.T0);
        const double fl = floor(Te);
        const int j = (int)fl;
        double tt = 1.0;
        if (s > 0.0) { if (Tx >= fl + 1.0) tt = (fl + 1.0 - Te) / s; }
        else if (s < 0.0) { if (Tx < fl) tt = (fl - Te) / s; }
        tt = fmin(fmax(tt, 0.0), 1.0);
        const int jx = c.axis == 0 ? i : j, jy = c.axis == 0 ? j : i;
        SlabEntry e;
        e.off0 = ((jy + 1) * G.pnx + (jx + 1)) * G.nz;
        e.tt = (float)(tt * 4294967296.0);       // in units of 2^-32 of the slab (see march)
        row[n] = e;
    }
    // null entries up to the end of the (padded) row: a zero-valued border column whose
    // transverse neighbours are inside the buffer, no crossing
    for (int n = c.n_slabs + threadIdx.x; n < max_slabs; n += blockDim.x) {
        SlabEntry e;
        e.off0 = G.pnx * G.nz;            // (x, y) = (-1, 0)
        e.tt = 4294967296.f;
        row[n] = e;
    }
}

// ------------------------------------------------------------------ per-ray z tracking and the march

// The crossings of axial (z) voxel planes are tracked as 32.32 fixed-point values of the slab
// coordinate q: hi word = slab in which the crossing falls, lo word = share of that slab's path
// before it.  The first crossing and the spacing 1/|slope| come from a double precision set-up,
// so that a crossing's slab and share do not depend on float rounding of a position (for a ray
// almost parallel to the planes that rounding, divided by the slope, would misplace the crossing
// by whole slabs).
struct RayZ {
    int k, dirZ;
    unsigned long long QZ, dQZ;
    float Ls;                       // mm of path per slab
    int kmin, kmax;                 // bounds of the axial indices met in n_slabs slabs
};

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

// z state of the ray of row iv at the entry of slab n0 of its column (slabs are then counted
// from there), for a march of n slabs.
__device__ __forceinline__ RayZ make_ray_z(const Geom& G, const ColHdr& h, int iv, int n0, int n) {
    RayZ r;
    const double dz = ((double)iv - 0.5 * (G.nv - 1) + (double)G.off_v) * (double)G.pv;
    const double gz = dz / (double)G.hz;
    const double Szi = (0.0 - G.loz) / (double)G.hz;                      // the source is in the plane z = 0
    const double sz = gz * h.kap;                                         // z per slab
    first_crossing(fma(gz, fma(h.kap, (double)n0, h.lam0), Szi), sz, &r.k, &r.dirZ, &r.QZ, &r.dQZ);
    r.Ls = (float)(sqrt((double)h.dxy2 + dz * dz) * h.kap);            // mm per slab
    const int ncross = (int)(fabs(sz) * (double)n) + 2;                   // conservative
    r.kmin = r.dirZ < 0 ? r.k - ncross : r.k;
    r.kmax = r.dirZ > 0 ? r.k + ncross : r.k;
    return r;
}

// Runs the slabs of one ray, source side first, U at a time.  Per piece the sink is asked first
// to fetch (off = element offset of the voxel column (i, j), k = axial index) and later to add
// (off, k, tau = share of the slab's path length, fetched value): all fetches of a group of U
// slabs are issued before the first add, and the table entries of the next group are loaded
// while this one is worked on.  Rows are padded with null entries (zero-valued border column,
// tt = 1) to a multiple of U plus one group, so there is no remainder loop.  Pieces of zero
// share are passed on (the sink ignores or drops them).
constexpr int U = 4;

template <class Sink>
__device__ __forceinline__ void march(const SlabEntry* __restrict__ row, int n_slabs, int dT, RayZ r, Sink& sink) {
    const int4* row4 = reinterpret_cast<const int4*>(row);          // two entries per 16 B
    int k = r.k;
    unsigned qlo = (unsigned)r.QZ, qhi = (unsigned)(r.QZ >> 32);     // next z crossing: slab, share * 2^32
    const unsigned dlo = (unsigned)r.dQZ, dhi = (unsigned)(r.dQZ >> 32);
    int4 ea = __ldg(row4), eb = __ldg(row4 + 1);
    for (int n0 = 0; n0 < n_slabs; n0 += U) {
        const int4 na = __ldg(row4 + (n0 >> 1) + 2), nb = __ldg(row4 + (n0 >> 1) + 3);   // next group
        const int off0s[U] = {ea.x, ea.z, eb.x, eb.z};
        const float tts[U] = {__int_as_float(ea.y), __int_as_float(ea.w), __int_as_float(eb.y), __int_as_float(eb.w)};
        int pi[U][3], pk[U][3];
        float pt[U][3], pv[U][3];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            // shares are kept in units of 2^-32 of a slab (the table's tt is stored that way and the
            // crossing counter's low word is one already): the caller scales the sum once
            const float tt = tts[u];
            const bool cz = qhi == (unsigned)(n0 + u);
            const float tz = cz ? __uint2float_rn(qlo) : 4294967296.f;
            const int dk = cz ? r.dirZ : 0;
            const float t1 = fminf(tt, tz), t2 = fmaxf(tt, tz);
            const bool tfirst = tt < tz;
            const int i0 = off0s[u] + k;
            pi[u][0] = i0;                          pk[u][0] = k;                    pt[u][0] = t1;
            pi[u][1] = i0 + (tfirst ? dT : dk);     pk[u][1] = tfirst ? k : k + dk;  pt[u][1] = t2 - t1;
            pi[u][2] = i0 + dT + dk;                pk[u][2] = k + dk;               pt[u][2] = 4294967296.f - t2;
#pragma unroll
            for (int i = 0; i < 3; ++i) pv[u][i] = sink.fetch(pi[u][i], pk[u][i]);
            k += dk;
            asm("{\n"
                ".reg .pred p;\n"
                "setp.ne.s32 p, %2, 0;\n"
                "@p add.cc.u32 %0, %0, %3;\n"
                "@p addc.u32 %1, %1, %4;\n"
                "}\n"
                : "+r"(qlo), "+r"(qhi)
                : "r"((int)cz), "r"(dlo), "r"(dhi));
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
#pragma unroll
            for (int i = 0; i < 3; ++i) sink.add(pi[u][i], pk[u][i], pt[u][i], pv[u][i]);
        }
        ea = na; eb = nb;
    }
}

// CHECK = false: the caller has established that the ray stays inside [0, nz) for the whole
// march (no per-piece test).
template <bool CHECK>
struct AccSink {
    const float* __restrict__ vol;
    int Nz;
    float acc;
    __device__ __forceinline__ float fetch(int idx, int k) const {      // idx = column offset + k
        return (!CHECK || (unsigned)k < (unsigned)Nz) ? __ldg(vol + (unsigned)idx) : 0.f;
    }
    __device__ __forceinline__ void add(int, int, float tau, float v) { acc = fmaf(tau, v, acc); }
};

// Grid: (columns / PW, row groups of 32, slots x segments).  A block marches SEG slabs of its
// rays: the rows of the grid are cut into segments so that there are several times more blocks
// than fit on the GPU at once and the hardware block scheduler keeps every SM busy to the end
// (with one block per ray group everything is resident at once and the last third of the
// kernel runs half empty: profiles/r01).  Segment s of a ray starts from the exact z state at
// its first slab (double precision set-up) and writes its partial line integral to
// pseg[slot][s][iu][iv]; the last block of the ray group adds the segments in index order.
__global__ void __launch_bounds__(NT)
k_project(const Geom G, const SlotState* __restrict__ slots, const SolveState* __restrict__ solves,
          const SolveIn* __restrict__ in, const ColHdr* __restrict__ hdr, const SlabEntry* __restrict__ tab,
          int max_slabs, int n_seg, const float* __restrict__ vol, const unsigned char* __restrict__ occ,
          float* pseg, float* __restrict__ p_out, double* __restrict__ partials, int* seg_ticket) {
    __shared__ double red[NT / 32];
    __shared__ int s_last;
    const int s = blockIdx.z / n_seg, seg = blockIdx.z % n_seg;
    if (!slots[s].active) return;                            // uniform over the block
    const int b = slots[s].solve;
    const int iu = blockIdx.x * PW + (threadIdx.x >> 5);
    const int iv = blockIdx.y * 32 + (threadIdx.x & 31);
    const bool col_ok = iu < G.nu, ray_ok = col_ok && iv < G.nv;
    ColHdr h;
    h.n_slabs = 0; h.dT = 0; h.lam0 = 0.0; h.kap = 0.0; h.dxy2 = 0.f; h.axis = 0;
    if (col_ok) h = hdr[(long long)b * G.nu + iu];
    int n0 = seg * SEG, n = min(h.n_slabs - n0, SEG);
    const SlabEntry* row = tab + ((long long)b * G.nu + (col_ok ? iu : 0)) * max_slabs + n0;
    float p = 0.f;
    if (n > 0) {
        // Slabs in air add an exact +0: trim the segment to the span of slabs whose voxel columns
        // hold something (occupancy written with the volume; the lanes share the column, so the
        // test is split over them and the result is uniform over the warp).
        {
            const unsigned long long* ow = reinterpret_cast<const unsigned long long*>(occ + (long long)s * G.OCC);
            const int words = G.occ_pitch >> 3, lane = threadIdx.x & 31;
            unsigned long long span = 0ull;
#pragma unroll
            for (int part = 0; part < SEG / 32; ++part) {
                const int sl = part * 32 + lane;
                bool o = false;
                if (sl < n) {
                    const int off0 = __ldg(&row[sl].off0);
                    const int c0 = off0 / G.nz, c1 = (off0 + h.dT) / G.nz;
                    for (int wd = 0; wd < words; ++wd)
                        o |= (__ldg(ow + (long long)c0 * words + wd) | __ldg(ow + (long long)c1 * words + wd)) != 0ull;
                }
                span |= (unsigned long long)__ballot_sync(0xffffffffu, o) << (32 * part);
            }
            if (span == 0ull) n = 0;
            else {
                const int first = (__ffsll((long long)span) - 1) & ~(U - 1);
                const int last = 63 - __clzll((long long)span);
                n = min(n, (last & ~(U - 1)) + U) - first;
                n0 += first;
                row += first;
            }
        }
    }
    if (ray_ok && n > 0) {
        const RayZ r = make_ray_z(G, h, iv, n0, n);
        const float* base = vol + (long long)s * G.PV;
        asm volatile("" : "+l"(base));       // one base pointer; 32-bit offsets in the loop
        float acc;
        if (r.kmin >= 0 && r.kmax < G.nz) {
            AccSink<false> sink{base, G.nz, 0.f};
            march(row, n, h.dT, r, sink);
            acc = sink.acc;
        } else {
            AccSink<true> sink{base, G.nz, 0.f};
            march(row, n, h.dT, r, sink);
            acc = sink.acc;
        }
        p = acc * (r.Ls * 2.3283064365386963e-10f);      // the shares were summed in units of 2^-32
    }
    float* my_seg = pseg + (((long long)s * n_seg + seg) * G.nu + (col_ok ? iu : 0)) * G.nv + (ray_ok ? iv : 0);
    if (ray_ok && n_seg > 1) *my_seg = p;

    // The block of this ray group (PW columns x 32 rows) that finishes last adds the segments in
    // index order and forms a-3 for its rays: r_i = p_i - a y_i - b with the per-group partial sums
    // of p, y p and r^2 (Eq. 2, L91-93 Eq. 4) in double.
    const int ngroups = gridDim.x * gridDim.y, grp = blockIdx.y * gridDim.x + blockIdx.x;
    if (n_seg > 1) {
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) {
            int* t = seg_ticket + (long long)s * ngroups + grp;
            const int k = atomicAdd(t, 1);
            s_last = k == n_seg - 1;
            if (s_last) *t = 0;
        }
        __syncthreads();
        if (!s_last) return;
        __threadfence();
        if (ray_ok) {
            p = 0.f;
            for (int g = 0; g < n_seg; ++g)
                p += __ldcg(pseg + (((long long)s * n_seg + g) * G.nu + iu) * G.nv + iv);
        }
    }
    double vp = 0.0, vyp = 0.0, vrr = 0.0;
    if (ray_ok) {
        const int pix = iv * G.nu + iu;
        p_out[(long long)s * G.npix + pix] = p;
        const float* y = in[b].y;
        const double yv = y ? (double)__ldg(y + pix) : 0.0;
        const double res = (double)p - solves[b].a * yv - solves[b].b;   // Eq. (2) residual
        vp = (double)p; vyp = yv * (double)p; vrr = res * res;
    }
    double* out = partials + ((long long)s * ngroups + grp) * 3;
    const double sp = block_sum<NT>(vp, red);
    const double syp = block_sum<NT>(vyp, red);
    const double srr = block_sum<NT>(vrr, red);
    if (threadIdx.x == 0) { out[0] = sp; out[1] = syp; out[2] = srr; }
}

// Standard [z][y][x] -> ray layout (hook path only: the solve's volumes are written in the ray
// layout by the warp kernel).  Tile: 32 x by 32 z at fixed y.
__global__ void __launch_bounds__(256)
k_to_ray_layout(const Geom G, const float* __restrict__ src, float* __restrict__ dst, unsigned char* __restrict__ occ) {
    __shared__ float tile[32][33];
    const int lane = threadIdx.x & 31, tw = threadIdx.x >> 5;
    const int x0 = blockIdx.x * 32, z0 = blockIdx.y * 32, y = blockIdx.z;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int z = z0 + tw + 8 * r, x = x0 + lane;
        tile[tw + 8 * r][lane] = (x < G.nx && z < G.nz) ? src[((long long)z * G.ny + y) * G.nx + x] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int x = x0 + tw + 8 * r, z = z0 + lane;
        const bool st = x < G.nx && z < G.nz;
        const float v = st ? tile[lane][tw + 8 * r] : 0.f;
        if (st) dst[ray_layout_index(G, x, y, z)] = v;
        occ_record(G, occ, x, y, z0, 32, v != 0.f);
    }
}

struct RecSink {
    int cap, n;
    int nx, ny, nz, pnx;
    float Ls, eps;
    int* ijk;
    float* len;
    __device__ __forceinline__ float fetch(int, int) const { return 0.f; }
    __device__ __forceinline__ void add(int idx, int k, float tau_raw, float) {
        if (!((unsigned)k < (unsigned)nz)) return;
        const float tau = tau_raw * 2.3283064365386963e-10f;                // shares come in units of 2^-32
        const int col = (idx - k) / nz, jy = col / pnx - 1, jx = col % pnx - 1;
        if (!((unsigned)jx < (unsigned)nx && (unsigned)jy < (unsigned)ny)) return;      // zero border
        const float l = tau * Ls;
        if (!(l > eps)) return;     // zero-length pieces are dropped (reading A22)
        if (n < cap) {
            ijk[3 * n + 0] = jx;
            ijk[3 * n + 1] = jy;
            ijk[3 * n + 2] = k;
            len[n] = l;
        }
        ++n;
    }
};

// One ray through the projector's own tables and march (pcamm_traverse).
__global__ void k_traverse(const Geom G, const ColHdr* __restrict__ hdr, const SlabEntry* __restrict__ tab,
                           int max_slabs, int iu, int iv, int cap, int* ijk, float* len, int* n_out) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const ColHdr h = hdr[iu];
    RecSink sink;
    sink.cap = cap; sink.n = 0; sink.nx = G.nx; sink.ny = G.ny; sink.nz = G.nz; sink.pnx = G.pnx;
    sink.eps = 1e-6f * fminf(G.hx, fminf(G.hy, G.hz));
    sink.Ls = 0.f;
    sink.ijk = ijk; sink.len = len;
    if (h.n_slabs > 0) {
        const RayZ r = make_ray_z(G, h, iv, 0, h.n_slabs);
        sink.Ls = r.Ls;
        march(tab + (long long)iu * max_slabs, h.n_slabs, h.dT, r, sink);
    }
    *n_out = sink.n;
}

}  // namespace

int project_blocks(const Geom& G) { return ((G.nu + PW - 1) / PW) * ((G.nv + 31) / 32); }
// slabs per table row: the longest march, rounded up to the group size, plus one group read ahead
int max_slabs(const Geom& G) { return ((G.nx > G.ny ? G.nx : G.ny) + U - 1) / U * U + U; }
int project_segments(const Geom& G) { return ((G.nx > G.ny ? G.nx : G.ny) + SEG - 1) / SEG; }

void launch_view_tables(Seq& q, const Geom& G, const SolveState* solves, int B, ColHdr* hdr, SlabEntry* tab) {
    q.launch(k_view_tables, dim3(G.nu, B), dim3(128), 0, G, solves, hdr, tab, max_slabs(G));
}

void launch_project(Seq& q, const Geom& G, const CtlBufs& c, int nslots, const ColHdr* hdr, const SlabEntry* tab,
                    const float* vol, const unsigned char* occ, float* pseg, float* p, int then,
                    cudaGraphConditionalHandle h, int use_cond) {
    const int n_seg = project_segments(G);
    q.launch(k_project, dim3((G.nu + PW - 1) / PW, (G.nv + 31) / 32, nslots * n_seg), dim3(NT), 0, G,
             (const SlotState*)c.slots, (const SolveState*)c.solves, (const SolveIn*)c.in, hdr, tab, max_slabs(G), n_seg, vol,
             occ, pseg, p, c.proj_part, c.seg_ticket);
    launch_ctl_after_project(q, G, c, then, h, use_cond);
}

void launch_to_ray_layout(Seq& q, const Geom& G, const float* vol_std, float* vol_ray, unsigned char* occ) {
    q.launch(k_to_ray_layout, dim3((G.nx + 31) / 32, (G.nz + 31) / 32, G.ny), dim3(256), 0, G, vol_std, vol_ray, occ);
}

void launch_traverse(Seq& q, const Geom& G, const ColHdr* hdr, const SlabEntry* tab, int iu, int iv, int cap,
                     int* ijk, float* len, int* n_out) {
    q.launch(k_traverse, dim3(1), dim3(32), 0, G, hdr, tab, max_slabs(G), iu, iv, cap, ijk, len, n_out);
}

}  // namespace pcamm
