// a-2: cone-beam forward projection p = P_theta f  (section 2.2, Eq. 2;
// "P is a projection matrix which computes the projection image of f").
//
// Reading A3: p_i = sum_j l_ij f_j with l_ij the exact length of the source -> pixel-centre
// segment inside voxel box j (Siddon's radiological path).  The oracle merges and sorts all plane
// crossings of every ray; this file computes the same sums from the structure of a flat detector
// whose columns are parallel to the rotation axis:
//
//   the ray marches along its dominant in-plane axis m (|d_m|/h_m largest; t = the other in-plane
//   axis) through the slabs between the planes M = i and M = i+1 (voxel-corner index units).  ALL
//   rays of one detector column share their in-plane path: in slab n they are in voxel column A_n
//   for the share tt_n of the slab and in the transverse neighbour B_n for the rest (|sT| <= 1:
//   at most one transverse crossing per slab).  The rows of the column differ only in WHERE they
//   cross the axial (z) planes.  With the per-level path integral
//
//       S_k(q) = integral_0^q f[column(s)][k] ds       (q in slabs; piecewise linear in q)
//
//   the line integral of a ray that is in level k_0 until its crossing q_1, in k_1 until q_2, ...
//   is  Ls * sum_m [ S_{k_m}(q_{m+1}) - S_{k_m}(q_m) ]  (Ls = mm of path per slab): exactly
//   Siddon's sum, regrouped.
//
// Split of the work.  The gantry angle is fixed for the whole solve (P varies per
// angle, not per iteration), so the in-plane traversal is tabulated ONCE per solve (k_view_tables:
// per column and slab the voxel column A_n and the share tt_n, evaluated directly in double).
// The projector, which runs once per line-search trial, takes one block per (detector column,
// segment of CH slabs):
//   phase 1  each warp scans SC slabs for every level at once (lanes = z, coalesced 128-bit loads
//            of the z-fastest ray layout, all loads of the scan in flight together) and leaves the
//            knots of S_k (slab entry, transverse crossing, slab exit; prefix restarted per warp)
//            in shared memory: (levels x slabs) work, shared by all rows of the column, instead of
//            (rows x slabs) gathers;
//   phase 2  one thread per row: the z crossings of its ray (32.32 fixed-point counters set up in
//            double) are walked in order; each costs one interpolated look-up of two levels'
//            knots, each scan adds its end knot at the ray's current level.
// The block of a column that finishes last adds the segments and forms the a-3 sums.
#include "internal.h"

namespace pcamm {

namespace {

constexpr int PT = 384;           // threads of a projector block
constexpr int PWARPS = PT / 32;   // = scans per block (one per warp)

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
    tl_begin(G.tl);
    const int iu = blockIdx.x, b = blockIdx.y;
    const View vw = solves[b].view;
    double dxy2;
    const ColSetup c = col_setup(G, vw, iu, &dxy2);
    const int strideT = c.axis == 0 ? G.pnx : 1;
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
        e.col = (jy + 1) * G.pnx + (jx + 1);
        e.tt = (float)(tt * 4294967296.0);       // in units of 2^-32 of the slab
        row[n] = e;
    }
    // null entries up to the end of the (padded) row: a zero-valued border column whose
    // transverse neighbours are inside the buffer, no crossing
    for (int n = c.n_slabs + threadIdx.x; n < max_slabs; n += blockDim.x) {
        SlabEntry e;
        e.col = G.pnx;                    // (x, y) = (-1, 0)
        e.tt = 4294967296.f;
        row[n] = e;
    }
    tl_end(G.tl, TLK_VIEW);
}

// ------------------------------------------------------------------ per-ray z tracking

// The crossings of axial (z) voxel planes are tracked as 32.32 fixed-point values of the slab
// coordinate q: hi word = slab in which the crossing falls, lo word = share of that slab's path
// before it.  The first crossing and the spacing 1/|slope| come from a double precision set-up,
// so that a crossing's slab and share do not depend on float rounding of a position (for a ray
// almost parallel to the planes that rounding, divided by the slope, would misplace the crossing
// by whole slabs).
struct RayZ {
    int k, dirZ;                    // level at the entry of the first slab; +1 / -1 / 0 per crossing
    unsigned long long QZ, dQZ;     // next crossing and the spacing of the crossings
};

// z state of the ray of row iv at the entry of slab n0 of its column (slabs are then counted
// from there).  first_crossing() with the divisions by the slope replaced by one reciprocal.
__device__ __forceinline__ RayZ make_ray_z(const Geom& G, const ColHdr& h, int iv, int n0) {
    RayZ r;
    const double dz = ((double)iv - 0.5 * (G.nv - 1) + (double)G.off_v) * (double)G.pv;
    const double gz = dz * G.ihz_d;
    const double sz = gz * h.kap;                                         // z per slab
    const double P0 = fma(gz, fma(h.kap, (double)n0, h.lam0), G.Szi);     // z (voxel-corner units) at the slab's entry
    const double fl = floor(P0);
    r.k = (int)fl;
    if (sz == 0.0) { r.dirZ = 0; r.QZ = (unsigned long long)(QMAX * FIX); r.dQZ = 0ull; return r; }
    r.dirZ = sz > 0.0 ? 1 : -1;
    const double inv = 1.0 / fabs(sz);
    const double dist = sz > 0.0 ? fl + 1.0 - P0 : P0 - fl;               // to the next plane, in voxels
    const double q = fmin(dist * inv, QMAX), d = fmin(inv, QMAX);
    r.QZ = (unsigned long long)(q * FIX + 0.5);
    r.dQZ = (unsigned long long)(d * FIX + 0.5);
    if (r.dQZ < (1ull << 32)) r.dQZ = 1ull << 32;                         // |sz| <= 1 (reading B2)
    return r;
}

// mm of path per slab of the ray of row iv in the column of header h
__device__ __forceinline__ float ray_slab_length(const Geom& G, const ColHdr& h, int iv) {
    const double dz = ((double)iv - 0.5 * (G.nv - 1) + (double)G.off_v) * (double)G.pv;
    return (float)(sqrt((double)h.dxy2 + dz * dz) * h.kap);
}

// ------------------------------------------------------------------ the pieces of one ray, in order
//
// pcamm_traverse: the ordered voxels and lengths of one ray, from the same table entries and the
// same crossing counters the projector integrates over.  Per slab at most three pieces: the
// transverse crossing (share tt of the table) and the z crossing (share tz of the counter) cut it.
struct RecSink {
    int cap, n;
    int nx, ny, nz, pnx;
    float Ls, eps;
    int* ijk;
    float* len;
    __device__ __forceinline__ void add(int col, int k, float tau_raw) {
        if (!((unsigned)k < (unsigned)nz)) return;
        const float tau = tau_raw * 2.3283064365386963e-10f;                // shares come in units of 2^-32
        const int jy = col / pnx - 1, jx = col % pnx - 1;
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

__device__ __forceinline__ void walk_pieces(const SlabEntry* __restrict__ row, int n_slabs, int dT, RayZ r, RecSink& sink) {
    int k = r.k;
    unsigned long long Q = r.QZ;
    for (int n = 0; n < n_slabs; ++n) {
        const SlabEntry e = row[n];
        const float tt = e.tt;                                        // units of 2^-32 of the slab
        const bool cz = (unsigned)(Q >> 32) == (unsigned)n;
        const float tz = cz ? __uint2float_rn((unsigned)Q) : 4294967296.f;
        const int dk = cz ? r.dirZ : 0;
        const float t1 = fminf(tt, tz), t2 = fmaxf(tt, tz);
        const bool tfirst = tt < tz;
        sink.add(e.col, k, t1);
        sink.add(tfirst ? e.col + dT : e.col, tfirst ? k : k + dk, t2 - t1);
        sink.add(e.col + dT, k + dk, 4294967296.f - t2);
        k += dk;
        if (cz) Q += r.dQZ;
    }
}

// ------------------------------------------------------------------ the projector

// Knots of one scan: 2 SC + 1 rows (entry of slab 0, its transverse crossing, entry of slab 1, ...,
// exit of slab SC - 1) of NZP floats: level k at element 4 + k, four zero floats in front (level -1
// and alignment) and at least four behind (level nz): a ray outside the volume in z reads zeros.
__host__ __device__ __forceinline__ int knot_pitch(int nz) { return (nz + 3) / 4 * 4 + 8; }

// chunks per segment: their air masks (2 SC bits each) share one 32-bit ballot
__host__ __device__ constexpr int max_cps(int sc) { return 32 / (2 * sc); }

__device__ __forceinline__ void add64(unsigned& lo, unsigned& hi, unsigned dlo, unsigned dhi) {
    asm("add.cc.u32 %0, %0, %2;\n\taddc.u32 %1, %1, %3;" : "+r"(lo), "+r"(hi) : "r"(dlo), "r"(dhi));
}

// Grid: (detector columns, segments x row blocks, slots).  A block takes the rows
// rb RPT PT .. + RPT PT - 1 of its column through the n_chunks chunks (of CH = PWARPS SC slabs) of
// its segment; the ray state lives in registers from chunk to chunk.  VEC: levels per lane and load
// (4 where nz is a multiple of 4, else 1).  Segment g writes the sums of all its rows (in slabs,
// not yet mm) to pseg[slot][g][iu][iv]; the block of the column that finishes last adds the
// segments in index order and multiplies by the path length per slab.
//
// Per chunk: (1) the scans, one per warp; (2) the prefix of the scans' end knots over the chunk,
// P[c][k] = S_k at the entry of scan c, so that S_k(q) = P[c][k] + (the scan's own knots); (3) per
// ray the crossings that fall into the chunk, in order: S_k(q) - S_{k+dirZ}(q) each, and S at the
// chunk's exit at the level the ray has by then.
template <int VEC, int SC, int RPT>
__global__ void __launch_bounds__(PT, SC == 4 ? 3 : 4)
k_project(const Geom G, const CtlBufs c, int slot0, const ColHdr* __restrict__ hdr, const SlabEntry* __restrict__ tab,
          int max_slabs, int n_seg, int n_chunks, int NZP, const float* __restrict__ vol,
          const unsigned char* __restrict__ occ, float* pseg, float* __restrict__ p_out) {
    constexpr int CH = PWARPS * SC, NKNOT = 2 * SC + 1;
    constexpr int LOG_SC = SC == 4 ? 2 : (SC == 2 ? 1 : 0);
    extern __shared__ __align__(16) float s_knots[];        // [PWARPS][NKNOT][NZP], then P [PWARPS + 1][NZP]
    __shared__ float s_tt[CH];
    __shared__ float2 s_inv[CH];                             // 1 / tt and 1 / (1 - tt) (0 where there is nothing to divide)
    __shared__ int s_air[PWARPS];
    __shared__ double red[PT / 32];
    __shared__ int s_last;
    tl_begin(G.tl);
    int seg = blockIdx.y, rb = 0;
    if (seg >= n_seg) { rb = seg / n_seg; seg -= rb * n_seg; }
    const int iu = blockIdx.x, s = slot0 + blockIdx.z;
    const SlotState* __restrict__ slots = c.slots;
    const SolveState* __restrict__ solves = c.solves;
    int* seg_ticket = c.seg_ticket;
    double* __restrict__ partials = c.proj_part;
    if (!slots[s].active) { tl_end(G.tl, TLK_PROJECT); return; }     // uniform over the block
    const int b = slots[s].solve;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int p_off = PWARPS * NKNOT * NZP;                  // start of P in s_knots
    const int kw = warp * NKNOT * NZP;                       // this warp's knot rows
    const ColHdr h = hdr[b * G.nu + iu];
    const int n0 = seg * n_chunks * CH;
    const SlabEntry* rows = tab + ((long long)b * G.nu + iu) * max_slabs + n0 + warp * SC;   // this warp's first scan
    const float* base = vol + (long long)s * G.PV;
    const int dTe = h.dT * G.nz;                             // element offset of the transverse neighbour

    // the rays of this thread: level (+ 4: index into a knot row), next crossing (relative to slab n0), running sum
    int rk[RPT], rdir[RPT];
    unsigned rqlo[RPT], rqhi[RPT], rdlo[RPT], rdhi[RPT];
    float racc[RPT];
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
        const int iv = (rb * RPT + r) * PT + threadIdx.x;
        rk[r] = 4; rdir[r] = 0; rqlo[r] = 0u; rqhi[r] = 0xffffffffu; rdlo[r] = rdhi[r] = 0u; racc[r] = 0.f;
        if (iv < G.nv && n0 < h.n_slabs) {
            const RayZ z = make_ray_z(G, h, iv, n0);
            rk[r] = z.k + 4; rdir[r] = z.dirZ;
            rqlo[r] = (unsigned)z.QZ; rqhi[r] = (unsigned)(z.QZ >> 32);
            rdlo[r] = (unsigned)z.dQZ; rdhi[r] = (unsigned)(z.dQZ >> 32);
        }
    }
    // Slabs in air add an exact +0 (reading B8).  Per scan of this warp in every chunk of the segment:
    // the occupancy of the column the ray is in and, if it crosses into the transverse neighbour,
    // of that one.  Lane = (chunk, slab, A | B): bit 2 SC j + 2 i of the mask says that slab i of the
    // warp's scan in chunk j has something in A, the next bit the same for B.
    unsigned masks;
    {
        const int words = G.occ_pitch >> 3;
        const unsigned long long* ow = reinterpret_cast<const unsigned long long*>(occ + (long long)s * G.OCC);
        const int j = lane / (2 * SC), i = (lane / 2) % SC;
        bool has = false;
        if (j < n_chunks && n0 + j * CH < h.n_slabs) {
            const SlabEntry e = rows[j * CH + i];
            if ((lane & 1) == 0 || e.tt < 4294967296.f) {
                const unsigned long long* o = ow + (e.col + (lane & 1) * h.dT) * words;
                for (int wd = 0; wd < words; ++wd) has |= __ldg(o + wd) != 0ull;
            }
        }
        masks = __ballot_sync(0xffffffffu, has);
    }
    {   // the zero levels -1 and nz of this warp's knot rows (and the padding), never written again
        const int wpad = NZP - 4 - G.nz;
        if (lane < 4 + wpad) {
            const int e = lane < 4 ? lane : G.nz + lane;
#pragma unroll
            for (int i = 0; i < NKNOT; ++i) s_knots[kw + i * NZP + e] = 0.f;
        }
        if (warp == 0 && lane < 4 + wpad) {                  // and of the prefix rows
            const int e = lane < 4 ? lane : G.nz + lane;
            for (int i = 0; i <= PWARPS; ++i) s_knots[p_off + i * NZP + e] = 0.f;
        }
    }

    for (int j = 0; j < n_chunks; ++j) {
        if (n0 + j * CH >= h.n_slabs) break;                 // uniform over the block
        // ---- (1) warp w scans slabs n0 + j CH + w SC .. + SC - 1 (null entries behind the column's
        //      last slab: a zero-valued border column without occupancy)
        const unsigned m = (masks >> (2 * SC * j)) & ((1u << (2 * SC)) - 1u);
        const SlabEntry* row = rows + j * CH;
        if (lane < SC) {
            const float tt = row[lane].tt, ot = 4294967296.f - tt;
            s_tt[warp * SC + lane] = tt;
            s_inv[warp * SC + lane] = make_float2(tt > 0.f ? __fdividef(1.f, tt) : 0.f, ot > 0.f ? __fdividef(1.f, ot) : 0.f);
        }
        if (lane == 0) s_air[warp] = m == 0u;
        if (m != 0u) {                                       // uniform over the warp
            for (int zp = 0; zp < G.nz; zp += 32 * VEC) {
                const int z = zp + lane * VEC;
                const bool ok = z < G.nz;
                const float* bz = base + (ok ? z : 0);       // lanes beyond the last level load level 0 and store nothing
                float A[SC][VEC], Bv[SC][VEC];
#pragma unroll
                for (int i = 0; i < SC; ++i) {               // every load of the scan before the first use
                    const float* pa = bz + __ldg(&row[i].col) * G.nz;       // broadcast load
#pragma unroll
                    for (int v = 0; v < VEC; ++v) { A[i][v] = 0.f; Bv[i][v] = 0.f; }
                    if ((m >> (2 * i)) & 1u) {               // uniform over the warp
                        if (VEC == 4) {
                            const float4 va = __ldg(reinterpret_cast<const float4*>(pa));
                            A[i][0] = va.x; A[i][1 % VEC] = va.y; A[i][2 % VEC] = va.z; A[i][3 % VEC] = va.w;
                        } else A[i][0] = __ldg(pa);
                    }
                    if ((m >> (2 * i + 1)) & 1u) {
                        if (VEC == 4) {
                            const float4 vb = __ldg(reinterpret_cast<const float4*>(pa + dTe));
                            Bv[i][0] = vb.x; Bv[i][1 % VEC] = vb.y; Bv[i][2 % VEC] = vb.z; Bv[i][3 % VEC] = vb.w;
                        } else Bv[i][0] = __ldg(pa + dTe);
                    }
                }
                __syncwarp();                                // s_tt of this warp's slabs (written above)
                float S[VEC];
#pragma unroll
                for (int v = 0; v < VEC; ++v) S[v] = 0.f;
                float* dst = s_knots + kw + 4 + z;
                auto put = [&]() {
                    if (ok) {
                        if (VEC == 4) *reinterpret_cast<float4*>(dst) = make_float4(S[0], S[1 % VEC], S[2 % VEC], S[3 % VEC]);
                        else dst[0] = S[0];
                    }
                    dst += NZP;
                };
#pragma unroll
                for (int i = 0; i < SC; ++i) {
                    const float tt = s_tt[warp * SC + i];
                    const float ta = tt * 2.3283064365386963e-10f;          // the table's shares are in units of 2^-32
                    const float tb = (4294967296.f - tt) * 2.3283064365386963e-10f;
                    put();
#pragma unroll
                    for (int v = 0; v < VEC; ++v) S[v] = fmaf(ta, A[i][v], S[v]);
                    put();
#pragma unroll
                    for (int v = 0; v < VEC; ++v) S[v] = fmaf(tb, Bv[i][v], S[v]);
                }
                put();
            }
        } else {                                             // an air scan: its end knots are zeros (for the prefix)
            for (int i = lane; i < G.nz; i += 32) s_knots[kw + 2 * SC * NZP + 4 + i] = 0.f;
        }
        const int any = __syncthreads_or(m != 0u);
        // ---- (2) prefix of the scans' end knots, per level
        if (any) {                                           // uniform over the block
            for (int i = threadIdx.x; i < G.nz; i += PT) {
                float run = 0.f;
                const float* e = s_knots + 2 * SC * NZP + 4 + i;
                float* pp = s_knots + p_off + 4 + i;
                pp[0] = 0.f;
#pragma unroll
                for (int c = 0; c < PWARPS; ++c) {
                    run += e[c * NKNOT * NZP];
                    pp[(c + 1) * NZP] = run;
                }
            }
            __syncthreads();
        }
        // ---- (3) the crossings of this thread's rays that fall into the chunk
        const unsigned end = (unsigned)((j + 1) * CH);
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            if (!any) {                                      // nothing to add: the crossings only move the level
                while (rqhi[r] < end) { rk[r] += rdir[r]; add64(rqlo[r], rqhi[r], rdlo[r], rdhi[r]); }
                continue;
            }
            int k = rk[r];
            unsigned qlo = rqlo[r], qhi = rqhi[r];
            float acc = racc[r];
            const int dir = rdir[r], ktop = G.nz + 4;
            while (qhi < end) {
                // crossing from level k to k + dir at share tz of slab qhi: S_k(q) - S_{k + dir}(q),
                // S linear between the knots on either side of q
                const int rel = (int)qhi - j * CH, c = rel >> LOG_SC;
                const int ka = min(max(k, 3), ktop), kb = min(max(k + dir, 3), ktop);
                const int pc = p_off + c * NZP;
                float dv = s_knots[pc + ka] - s_knots[pc + kb];
                if (!s_air[c]) {
                    const float tz = __uint2float_rn(qlo), tt = s_tt[rel];
                    const float2 inv = s_inv[rel];
                    const bool before = tz < tt;
                    const float lam = before ? tz * inv.x : (tz - tt) * inv.y;
                    const int k0 = (c * NKNOT + 2 * (rel & (SC - 1)) + (before ? 0 : 1)) * NZP;
                    const float a0 = s_knots[k0 + ka], a1 = s_knots[k0 + NZP + ka];
                    const float b0 = s_knots[k0 + kb], b1 = s_knots[k0 + NZP + kb];
                    dv += (a0 - b0) + ((a1 - a0) - (b1 - b0)) * lam;
                }
                acc += dv;
                k += dir;
                add64(qlo, qhi, rdlo[r], rdhi[r]);
            }
            acc += s_knots[p_off + PWARPS * NZP + min(max(k, 3), ktop)];
            rk[r] = k; rqlo[r] = qlo; rqhi[r] = qhi; racc[r] = acc;
        }
        __syncthreads();                                     // the next chunk's scans overwrite the knots
    }

    // The block of this column that finishes last adds the segments in index order and forms a-3
    // for its rays: r_i = p_i - a y_i - b with the per-column partial sums of p, y p and r^2
    // (Eq. 2, L91-93 Eq. 4) in double.
    const int n_part = gridDim.y;                            // segments x row blocks of this column
    if (n_part > 1) {
        float* my = pseg + (((long long)s * n_seg + seg) * G.nu + iu) * G.nv;
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            const int iv = (rb * RPT + r) * PT + threadIdx.x;
            if (iv < G.nv) my[iv] = racc[r];
        }
        __syncthreads();                                     // the block's stores are ordered before thread 0's fence
        if (threadIdx.x == 0) {
            // release: the block's stores (ordered before this thread by the barrier) are visible to whoever
            // reads the ticket after it; acquire: the last block sees the other blocks' stores.  One
            // acq_rel atomic instead of a full fence on either side of a relaxed one.
            int* t = seg_ticket + s * G.nu + iu;
            int k;
            asm volatile("atom.add.acq_rel.gpu.s32 %0, [%1], 1;" : "=r"(k) : "l"(t) : "memory");
            s_last = k == n_part - 1;
            if (s_last) *t = 0;                              // for the next launch (kernel boundaries order it)
        }
        __syncthreads();
        if (!s_last) { tl_end(G.tl, TLK_PROJECT); return; }
    }
    double vp = 0.0, vyp = 0.0, vrr = 0.0;
    const float* y = c.in[b].y;
    const double fa = solves[b].a, fb = solves[b].b;
    auto finish = [&](int iv, float acc) {
        const long long pix = (long long)iv * G.nu + iu;
        const float p = acc * ray_slab_length(G, h, iv);
        p_out[(long long)s * G.npix + pix] = p;
        const double yv = y ? (double)__ldg(y + pix) : 0.0;
        const double res = (double)p - fa * yv - fb;                      // Eq. (2) residual
        vp += (double)p; vyp += yv * (double)p; vrr += res * res;
    };
    if (n_part > 1) {
        const float* ps = pseg + ((long long)s * n_seg * G.nu + iu) * G.nv;
        const long long gstride = (long long)G.nu * G.nv;
        for (int iv = threadIdx.x; iv < G.nv; iv += PT) {
            float acc = 0.f;
            for (int g = 0; g < n_seg; ++g) acc += __ldcg(ps + g * gstride + iv);
            finish(iv, acc);
        }
    } else {                                                 // this block had the whole column
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            const int iv = r * PT + threadIdx.x;
            if (iv < G.nv) finish(iv, racc[r]);
        }
    }
    double* out = partials + ((long long)s * G.nu + iu) * 3;
    const double sp = block_sum<PT>(vp, red);
    const double syp = block_sum<PT>(vyp, red);
    const double srr = block_sum<PT>(vrr, red);
    if (threadIdx.x == 0) { out[0] = sp; out[1] = syp; out[2] = srr; }
    tl_end(G.tl, TLK_PROJECT);
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

// One ray through the projector's own tables and crossing counters (pcamm_traverse).
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
        const RayZ r = make_ray_z(G, h, iv, 0);
        sink.Ls = ray_slab_length(G, h, iv);
        walk_pieces(tab + (long long)iu * max_slabs, h.n_slabs, h.dT, r, sink);
    }
    *n_out = sink.n;
}

}  // namespace

// Slabs per scan: the most whose knots leave room for three blocks per SM (the block's shared memory
// is PWARPS (2 SC + 1) knot rows and PWARPS + 1 prefix rows of knot_pitch(nz) floats).
int g_scan_slabs = 0;                                       // 0: automatic (pcamm_tune "project_scan_slabs")
int scan_slabs(const Geom& G) {
    const size_t row = sizeof(float) * (size_t)knot_pitch(G.nz);
    if (g_scan_slabs == 1 || g_scan_slabs == 2 || g_scan_slabs == 4) {
        if (row * (PWARPS * (2 * g_scan_slabs + 2) + 1) <= 200 * 1024) return g_scan_slabs;
    }
    if (row * (PWARPS * 10 + 1) <= 75 * 1024) return 4;
    if (row * (PWARPS * 6 + 1) <= 75 * 1024) return 2;
    return 1;
}
size_t project_smem(const Geom& G) {
    return sizeof(float) * (size_t)knot_pitch(G.nz) * (PWARPS * (2 * scan_slabs(G) + 2) + 1);
}
bool project_fits(const Geom& G) { return project_smem(G) <= 200 * 1024; }

// partial-sum groups per slot: one per detector column
int project_blocks(const Geom& G) { return G.nu; }
// chunks (of PWARPS scans) of the longest march
int project_chunks(const Geom& G) {
    const int ch = PWARPS * scan_slabs(G);
    return ((G.nx > G.ny ? G.nx : G.ny) + ch - 1) / ch;
}
// Chunks per block: a column's march is cut into segments so that the grid has several waves of
// blocks (the ray set-up is paid once per segment and ray).
int g_chunks_per_segment = 0;                              // 0: automatic (pcamm_tune "project_chunks_per_segment")
int chunks_per_segment(const Geom& G) {
    const int nc = project_chunks(G);
    const int mc = max_cps(scan_slabs(G)), cap = nc < mc ? nc : mc;
    if (g_chunks_per_segment > 0) return g_chunks_per_segment < cap ? g_chunks_per_segment : cap;
    int cps = cap;                                         // the fewest segments that still give >= 1024 blocks
    while (cps > 1 && (long long)G.nu * ((nc + cps - 1) / cps) * ((G.nv + 2 * PT - 1) / (2 * PT)) < 1024) --cps;
    return cps;
}
// upper bound (scratch is sized for one chunk per segment)
int project_segments(const Geom& G) { return project_chunks(G); }
// slabs per table row: whole chunks (null entries behind the column's last slab)
int max_slabs(const Geom& G) { return project_chunks(G) * PWARPS * scan_slabs(G); }

void launch_view_tables(Seq& q, const Geom& G, const SolveState* solves, int B, ColHdr* hdr, SlabEntry* tab) {
    q.launch(k_view_tables, dim3(G.nu, B), dim3(128), 0, G, solves, hdr, tab, max_slabs(G));
}

template <int VEC, int SC, int RPT>
void launch_project_t(Seq& q, const Geom& G, const CtlBufs& c, int nslots, const ColHdr* hdr, const SlabEntry* tab,
                      const float* vol, const unsigned char* occ, float* pseg, float* p) {
    static DeviceOnce configured;
    const size_t smem = project_smem(G);
    const cudaError_t e = configured.run([&] {
        return cudaFuncSetAttribute(k_project<VEC, SC, RPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    });
    if (e != cudaSuccess) { q.err = e; return; }
    const int cps = chunks_per_segment(G), n_seg = (project_chunks(G) + cps - 1) / cps;
    const int row_blocks = (G.nv + RPT * PT - 1) / (RPT * PT);
    for (int s0 = 0; s0 < nslots; s0 += 65535) {              // gridDim.z
        const int ns = nslots - s0 < 65535 ? nslots - s0 : 65535;
        q.launch(k_project<VEC, SC, RPT>, dim3(G.nu, n_seg * row_blocks, ns), dim3(PT), smem, G, c, s0, hdr, tab,
                 max_slabs(G), n_seg, cps, knot_pitch(G.nz), vol, occ, pseg, p);
    }
}

void launch_project(Seq& q, const Geom& G, const CtlBufs& c, int nslots, const ColHdr* hdr, const SlabEntry* tab,
                    const float* vol, const unsigned char* occ, float* pseg, float* p, int then,
                    cudaGraphConditionalHandle h, int use_cond, int n_before) {
    const int n_mark = q.n_kernels;
    if (G.projector == 1) {                                  // the ray-marching variant (raymarch.cu)
        launch_project_rm(q, G, c, nslots, vol, p);
        launch_ctl_after_project(q, G, c, then, h, use_cond, q.n_kernels - n_mark + n_before);
        return;
    }
    const int sc = scan_slabs(G);
    const bool v4 = G.nz % 4 == 0, one = G.nv <= PT;
#define PCAMM_PROJ(VEC, SC) \
    do { if (one) launch_project_t<VEC, SC, 1>(q, G, c, nslots, hdr, tab, vol, occ, pseg, p); \
         else launch_project_t<VEC, SC, 2>(q, G, c, nslots, hdr, tab, vol, occ, pseg, p); } while (0)
    if (sc == 4) { if (v4) PCAMM_PROJ(4, 4); else PCAMM_PROJ(1, 4); }
    else if (sc == 2) { if (v4) PCAMM_PROJ(4, 2); else PCAMM_PROJ(1, 2); }
    else { if (v4) PCAMM_PROJ(4, 1); else PCAMM_PROJ(1, 1); }
#undef PCAMM_PROJ
    // the control step that follows the projection (control.cu); n_before + the kernels launched here
    launch_ctl_after_project(q, G, c, then, h, use_cond, q.n_kernels - n_mark + n_before);
}

void launch_to_ray_layout(Seq& q, const Geom& G, const float* vol_std, float* vol_ray, unsigned char* occ) {
    q.launch(k_to_ray_layout, dim3((G.nx + 31) / 32, (G.nz + 31) / 32, G.ny), dim3(256), 0, G, vol_std, vol_ray, occ);
}

void launch_traverse(Seq& q, const Geom& G, const ColHdr* hdr, const SlabEntry* tab, int iu, int iv, int cap,
                     int* ijk, float* len, int* n_out) {
    q.launch(k_traverse, dim3(1), dim3(32), 0, G, hdr, tab, max_slabs(G), iu, iv, cap, ijk, len, n_out);
}

}  // namespace pcamm
