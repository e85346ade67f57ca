// CPU ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, double-precision implementation of the per-projection solve of
// Li et al., "Real-time volumetric image reconstruction and 3D tumor
// localization based on a single x-ray projection image for lung cancer
// radiotherapy".  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
// code with the CUDA path (paper_1004_0014_b200/csrc) and is written from the
// paper plus the readings A1..A23 listed in DESIGN.md.
//
// Every function follows the cited passage step by step; nothing is blocked,
// fused or reordered.  OpenMP (optional) only splits independent voxels / rays
// across threads; the per-thread partial sums are combined in thread order.
//
// Pins (tests/test_oracle_*.py): brute-force ray/box intersection, chord closed
// forms, adjoint dot-product, identity / integer-shift / affine-ramp warps,
// finite differences of J, exact intensity fits, planted coefficients, closed-
// form DVF inversion; for the ray-marching variant of P (reading C1): uniform and
// affine volumes in closed form, a dense matrix built separately, the adjoint
// identity, finite differences of J.  No function here is "parity unpinned".
//
// Inputs are the float32 arrays the GPU path consumes, up-cast to double.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

struct OrcGeom {
    int32_t nx, ny, nz;          // volume, x fastest
    double hx, hy, hz;           // voxel size, mm
    double cx, cy, cz;           // world position of the volume centre (isocentre = origin), mm
    int32_t K;                   // number of eigenvector fields
    int32_t nu, nv;              // detector, u fastest
    double pu, pv;               // pixel pitch, mm
    double sad, sdd;             // source-axis / source-detector distance, mm
    double off_u, off_v;         // detector offsets in pixels
};

struct OrcOpts {
    int32_t max_iter;            // PAPER.md:L125 uses 10
    double grad_tol;             // stop if ||g||_2 <= grad_tol
    double armijo_c, armijo_beta;
    int32_t max_backtracks;
    double init_step_vox;        // reading A7
    int32_t batched_linesearch;  // evaluate the whole candidate fan, take the largest passing step
    int32_t inv_max_iter;
    double inv_tol_mm;           // reading A13
};

struct OrcResult {
    int32_t iters, status;       // status: 1 max_iter, 2 grad_tol, 3 line search failed, -5 singular fit
    double J0, J, a, b;
};

static int g_threads = 1;
void orc_set_threads(int n) { g_threads = n < 1 ? 1 : n; }

// Which discretisation of P the projector, the backprojector and everything built on them use
// (PAPER.md:L82 says only "projection matrix"): 0 = Siddon's exact radiological path (reading A3,
// the default), 1 = fixed-step trilinear ray marching (reading C1 below) with
// the nominal step step_mm.
static int g_projector = 0;
static double g_step_mm = 1.0;
void orc_set_projector(int kind, double step_mm) { g_projector = kind == 1 ? 1 : 0; if (step_mm > 0) g_step_mm = step_mm; }
int orc_get_projector() { return g_projector; }
int orc_get_threads() { return g_threads; }
int orc_max_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"

namespace {

inline int64_t nvox(const OrcGeom& g) { return (int64_t)g.nx * g.ny * g.nz; }
inline int64_t npix(const OrcGeom& g) { return (int64_t)g.nu * g.nv; }

// Reference image with zero padding outside the grid (reading A2).
inline double F0(const float* f0, const OrcGeom& g, int64_t i, int64_t j, int64_t k) {
    if (i < 0 || j < 0 || k < 0 || i >= g.nx || j >= g.ny || k >= g.nz) return 0.0;
    return (double)f0[(k * g.ny + j) * g.nx + i];
}

// Trilinear interpolation of f0 at index coordinates q and its exact derivative
// with respect to q (SURVEY 8(a) formulas; readings A6, A17).
inline void trilinear(const float* f0, const OrcGeom& g, const double q[3], double* val, double dq[3]) {
    const double fx = std::floor(q[0]), fy = std::floor(q[1]), fz = std::floor(q[2]);
    const int64_t i0 = (int64_t)fx, j0 = (int64_t)fy, k0 = (int64_t)fz;
    const double tx = q[0] - fx, ty = q[1] - fy, tz = q[2] - fz;
    double c[2][2][2];  // c[a][b][c] = F0(i0+a, j0+b, k0+c)
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b)
            for (int cc = 0; cc < 2; ++cc) c[a][b][cc] = F0(f0, g, i0 + a, j0 + b, k0 + cc);
    const double X[2] = {1.0 - tx, tx}, Y[2] = {1.0 - ty, ty}, Z[2] = {1.0 - tz, tz};
    double v = 0.0, dx = 0.0, dy = 0.0, dz = 0.0;
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b)
            for (int cc = 0; cc < 2; ++cc) v += c[a][b][cc] * X[a] * Y[b] * Z[cc];
    for (int b = 0; b < 2; ++b)
        for (int cc = 0; cc < 2; ++cc) dx += Y[b] * Z[cc] * (c[1][b][cc] - c[0][b][cc]);
    for (int a = 0; a < 2; ++a)
        for (int cc = 0; cc < 2; ++cc) dy += X[a] * Z[cc] * (c[a][1][cc] - c[a][0][cc]);
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) dz += X[a] * Y[b] * (c[a][b][1] - c[a][b][0]);
    *val = v;
    if (dq) { dq[0] = dx; dq[1] = dy; dq[2] = dz; }
}

// Eq. (1): x_j = xbar_j + sum_k u_kj w_k  (mm), at voxel lin.
inline void dvf_at_voxel(const OrcGeom& g, const float* xbar, const float* u, const double* w,
                         int64_t lin, double x[3]) {
    const int64_t V = nvox(g);
    for (int c = 0; c < 3; ++c) {
        double s = (double)xbar[c * V + lin];
        for (int k = 0; k < g.K; ++k) s += (double)u[((int64_t)k * 3 + c) * V + lin] * w[k];
        x[c] = s;
    }
}

// Pull-back sampling position in index units: q_j = idx_j + x_j / h (reading A1).
inline void sample_pos(const OrcGeom& g, int64_t i, int64_t j, int64_t k, const double x[3], double q[3]) {
    q[0] = (double)i + x[0] / g.hx;
    q[1] = (double)j + x[1] / g.hy;
    q[2] = (double)k + x[2] / g.hz;
}

struct Ray { double S[3], d[3], L; };

// Cone-beam geometry at gantry angle theta (reading A14).
inline Ray make_ray(const OrcGeom& g, double theta, int iu, int iv) {
    const double c = std::cos(theta), s = std::sin(theta);
    Ray r;
    r.S[0] = g.sad * c; r.S[1] = g.sad * s; r.S[2] = 0.0;
    const double Cx = -(g.sdd - g.sad) * c, Cy = -(g.sdd - g.sad) * s;
    const double uu = ((double)iu - (g.nu - 1) / 2.0 + g.off_u) * g.pu;
    const double vv = ((double)iv - (g.nv - 1) / 2.0 + g.off_v) * g.pv;
    const double D[3] = {Cx + uu * (-s), Cy + uu * c, vv};
    for (int a = 0; a < 3; ++a) r.d[a] = D[a] - r.S[a];
    r.L = std::sqrt(r.d[0] * r.d[0] + r.d[1] * r.d[1] + r.d[2] * r.d[2]);
    return r;
}

struct Seg { int32_t i, j, k; double len; };

// Siddon's exact radiological path (reading A3): the parametric values of all
// plane crossings inside the volume are merged and sorted; each consecutive
// pair is one segment, whose voxel is read off its midpoint.  Segments no
// longer than eps_mm are dropped: 0 for the line integrals (every positive
// length counts), 1e-6 min(h) for the reported index lists (ties, reading A22).
// Returns the smallest gap (mm) between consecutive crossings in *min_gap
// (for the degenerate-ray filter).
void siddon(const OrcGeom& g, const Ray& r, std::vector<Seg>& out, double* min_gap, double eps_mm = 0.0) {
    out.clear();
    if (min_gap) *min_gap = INFINITY;
    const int N[3] = {g.nx, g.ny, g.nz};
    const double h[3] = {g.hx, g.hy, g.hz};
    const double lo[3] = {g.cx - g.nx * g.hx / 2.0, g.cy - g.ny * g.hy / 2.0, g.cz - g.nz * g.hz / 2.0};
    double amin = 0.0, amax = 1.0;
    bool par[3];
    for (int c = 0; c < 3; ++c) {
        par[c] = std::fabs(r.d[c]) < 1e-12 * r.L;   // reading A21
        if (par[c]) {
            const double hi = lo[c] + N[c] * h[c];
            if (r.S[c] < lo[c] || r.S[c] >= hi) return;
            continue;
        }
        const double a0 = (lo[c] - r.S[c]) / r.d[c], a1 = (lo[c] + N[c] * h[c] - r.S[c]) / r.d[c];
        amin = std::max(amin, std::min(a0, a1));
        amax = std::min(amax, std::max(a0, a1));
    }
    if (!(amin < amax)) return;
    std::vector<double> al;
    al.push_back(amin);
    for (int c = 0; c < 3; ++c) {
        if (par[c]) continue;
        for (int n = 0; n <= N[c]; ++n) {
            const double a = (lo[c] + n * h[c] - r.S[c]) / r.d[c];
            if (a > amin && a < amax) al.push_back(a);
        }
    }
    al.push_back(amax);
    std::sort(al.begin(), al.end());
    const double eps = eps_mm;
    for (size_t m = 0; m + 1 < al.size(); ++m) {
        const double len = (al[m + 1] - al[m]) * r.L;
        if (min_gap && len < *min_gap) *min_gap = len;
        if (!(len > eps)) continue;
        const double am = 0.5 * (al[m] + al[m + 1]);
        int idx[3];
        for (int c = 0; c < 3; ++c) {
            const double p = r.S[c] + am * r.d[c];
            int64_t ii = (int64_t)std::floor((p - lo[c]) / h[c]);
            idx[c] = (int)std::min<int64_t>(std::max<int64_t>(ii, 0), N[c] - 1);
        }
        out.push_back({idx[0], idx[1], idx[2], len});
    }
}

inline void world_to_index(const OrcGeom& g, const double r[3], double q[3]) {
    q[0] = (r[0] - g.cx) / g.hx + (g.nx - 1) / 2.0;
    q[1] = (r[1] - g.cy) / g.hy + (g.ny - 1) / 2.0;
    q[2] = (r[2] - g.cz) / g.hz + (g.nz - 1) / 2.0;
}

// DVF of Eq. (1) at an off-grid world point: trilinear interpolation of the
// synthesised field, coordinates clamped to the grid (reading A13).
void dvf_at_point(const OrcGeom& g, const float* xbar, const float* u, const double* w,
                  const double r[3], double x[3]) {
    double q[3];
    world_to_index(g, r, q);
    const int N[3] = {g.nx, g.ny, g.nz};
    int64_t i0[3];
    double t[3];
    for (int c = 0; c < 3; ++c) {
        double qc = std::min(std::max(q[c], 0.0), (double)(N[c] - 1));
        int64_t f = (int64_t)std::floor(qc);
        if (f > N[c] - 2) f = N[c] - 2;
        if (f < 0) f = 0;
        i0[c] = f;
        t[c] = qc - (double)f;
        if (N[c] == 1) t[c] = 0.0;
    }
    x[0] = x[1] = x[2] = 0.0;
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b)
            for (int cc = 0; cc < 2; ++cc) {
                const double wgt = (a ? t[0] : 1.0 - t[0]) * (b ? t[1] : 1.0 - t[1]) * (cc ? t[2] : 1.0 - t[2]);
                if (wgt == 0.0) continue;
                const int64_t i = std::min<int64_t>(i0[0] + a, N[0] - 1), j = std::min<int64_t>(i0[1] + b, N[1] - 1),
                              k = std::min<int64_t>(i0[2] + cc, N[2] - 1);
                double xv[3];
                dvf_at_voxel(g, xbar, u, w, (k * g.ny + j) * g.nx + i, xv);
                for (int c = 0; c < 3; ++c) x[c] += wgt * xv[c];
            }
}

// ---- fixed-step trilinear ray marching (north_star "fixed-step or Siddon
// traversal"; PAPER.md:L82 leaves the discretisation of P open).  Reading C1:
//
//   p_i = d_i sum_{m = 0}^{M_i - 1} (T f)(E_i + (m + 1/2) d_i e_i)
//
// where [E_i, X_i] is the part of the ray source -> pixel centre i inside the box spanned by the
// voxel CENTRES (where trilinear interpolation T f of the voxel-centre values is defined without
// any padding rule), L_i its length, e_i the unit direction, M_i = ceil(L_i / step) and
// d_i = L_i / M_i <= step: the midpoint rule on M_i equal steps.  A ray that misses the box, or an
// axis with a single voxel layer (a box of no thickness), gives 0.
//
// The matrix entries are l_ij = d_i sum_m (weight of voxel j in T at sample m); both P and P^T walk
// the same samples through this one enumerator, so P^T is the exact transpose.
// fn(lin, weight): called for each of the 8 taps of each sample, weight = d_i * trilinear weight.
template <class Fn>
void rm_samples(const OrcGeom& g, const Ray& r, double step_mm, Fn fn) {
    const int N[3] = {g.nx, g.ny, g.nz};
    const double h[3] = {g.hx, g.hy, g.hz};
    const double ctr[3] = {g.cx, g.cy, g.cz};
    double lo[3], amin = 0.0, amax = 1.0;
    for (int c = 0; c < 3; ++c) {
        if (N[c] < 2) return;
        lo[c] = ctr[c] - (N[c] - 1) / 2.0 * h[c];                        // centre of voxel 0
        const double hi = ctr[c] + (N[c] - 1) / 2.0 * h[c];              // centre of voxel N - 1
        if (std::fabs(r.d[c]) < 1e-12 * r.L) {
            if (r.S[c] < lo[c] || r.S[c] > hi) return;
            continue;
        }
        const double a0 = (lo[c] - r.S[c]) / r.d[c], a1 = (hi - r.S[c]) / r.d[c];
        amin = std::max(amin, std::min(a0, a1));
        amax = std::min(amax, std::max(a0, a1));
    }
    if (!(amin < amax)) return;
    const double L = (amax - amin) * r.L;
    const int64_t M = (int64_t)std::ceil(L / step_mm);
    if (M < 1) return;
    const double d = L / (double)M, da = (amax - amin) / (double)M;
    for (int64_t m = 0; m < M; ++m) {
        const double al = amin + ((double)m + 0.5) * da;
        int64_t i0[3];
        double t[3];
        for (int c = 0; c < 3; ++c) {
            const double q = (r.S[c] + al * r.d[c] - lo[c]) / h[c];      // index coordinates, in [0, N - 1]
            int64_t f = (int64_t)std::floor(q);
            f = std::min<int64_t>(std::max<int64_t>(f, 0), N[c] - 2);
            i0[c] = f;
            t[c] = q - (double)f;
        }
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b)
                for (int cc = 0; cc < 2; ++cc) {
                    const double wgt = (a ? t[0] : 1.0 - t[0]) * (b ? t[1] : 1.0 - t[1]) * (cc ? t[2] : 1.0 - t[2]);
                    fn(((i0[2] + cc) * g.ny + (i0[1] + b)) * g.nx + (i0[0] + a), d * wgt);
                }
    }
}

}  // namespace

extern "C" {

// f = warp(f0, xbar + U w): Eq. (1), Eq. (2) constraint, trilinear pull-back.
void orc_warp(const OrcGeom* g, const float* f0, const float* xbar, const float* u, const double* w, double* f_out) {
    const OrcGeom& G = *g;
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int64_t k = 0; k < G.nz; ++k)
        for (int64_t j = 0; j < G.ny; ++j)
            for (int64_t i = 0; i < G.nx; ++i) {
                const int64_t lin = (k * G.ny + j) * G.nx + i;
                double x[3], q[3], v;
                dvf_at_voxel(G, xbar, u, w, lin, x);
                sample_pos(G, i, j, k, x, q);
                trilinear(f0, G, q, &v, nullptr);
                f_out[lin] = v;
            }
}

// G_j = d f_j / d x_j (1/mm), [3][V]: exact derivative of the trilinear interpolant (A6).
void orc_warp_grad(const OrcGeom* g, const float* f0, const float* xbar, const float* u, const double* w, double* G_out) {
    const OrcGeom& G = *g;
    const int64_t V = nvox(G);
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int64_t k = 0; k < G.nz; ++k)
        for (int64_t j = 0; j < G.ny; ++j)
            for (int64_t i = 0; i < G.nx; ++i) {
                const int64_t lin = (k * G.ny + j) * G.nx + i;
                double x[3], q[3], v, dq[3];
                dvf_at_voxel(G, xbar, u, w, lin, x);
                sample_pos(G, i, j, k, x, q);
                trilinear(f0, G, q, &v, dq);
                G_out[0 * V + lin] = dq[0] / G.hx;
                G_out[1 * V + lin] = dq[1] / G.hy;
                G_out[2 * V + lin] = dq[2] / G.hz;
            }
}

// One ray's ordered voxel list and intersection lengths (test hook for the traversal pin).
int orc_traverse(const OrcGeom* g, double theta, int iu, int iv, int cap, int32_t* ijk_out, double* len_out,
                 int32_t* n_out, double* min_gap_out) {
    std::vector<Seg> segs;
    double mg;
    siddon(*g, make_ray(*g, theta, iu, iv), segs, &mg, 1e-6 * std::min(g->hx, std::min(g->hy, g->hz)));
    *n_out = (int32_t)segs.size();
    if (min_gap_out) *min_gap_out = mg;
    for (size_t m = 0; m < segs.size() && (int)m < cap; ++m) {
        ijk_out[3 * m + 0] = segs[m].i; ijk_out[3 * m + 1] = segs[m].j; ijk_out[3 * m + 2] = segs[m].k;
        len_out[m] = segs[m].len;
    }
    return (int)segs.size() <= cap ? 0 : 1;
}

// p = P_theta f: p_i = sum_j l_ij f_j (Eq. 2; reading A3).
void orc_project(const OrcGeom* g, const double* f, double theta, double* p_out) {
    const OrcGeom& G = *g;
    if (g_projector == 1) {                            // reading C1: p_i = sum_j l_ij f_j with the ray-marching l_ij
#pragma omp parallel for num_threads(g_threads) schedule(static)
        for (int64_t pix = 0; pix < npix(G); ++pix) {
            double s = 0.0;
            rm_samples(G, make_ray(G, theta, (int)(pix % G.nu), (int)(pix / G.nu)), g_step_mm,
                       [&](int64_t lin, double wgt) { s += wgt * f[lin]; });
            p_out[pix] = s;
        }
        return;
    }
#pragma omp parallel num_threads(g_threads)
    {
        std::vector<Seg> segs;
#pragma omp for schedule(static)
        for (int64_t pix = 0; pix < npix(G); ++pix) {
            siddon(G, make_ray(G, theta, (int)(pix % G.nu), (int)(pix / G.nu)), segs, nullptr);
            double s = 0.0;
            for (const Seg& sg : segs) s += sg.len * f[((int64_t)sg.k * G.ny + sg.j) * G.nx + sg.i];
            p_out[pix] = s;
        }
    }
}

// B = P_theta^T r: B_j = sum_i l_ij r_i, the transpose of the same l_ij (reading A4).
void orc_backproject(const OrcGeom* g, const double* r, double theta, double* B_out) {
    const OrcGeom& G = *g;
    const int64_t V = nvox(G);
    const int T = g_threads;
    std::vector<std::vector<double>> part(T > 1 ? T : 0);
    std::memset(B_out, 0, sizeof(double) * V);
#pragma omp parallel num_threads(T)
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        double* acc = B_out;
        if (T > 1) { part[tid].assign(V, 0.0); acc = part[tid].data(); }
        std::vector<Seg> segs;
#pragma omp for schedule(static)
        for (int64_t pix = 0; pix < npix(G); ++pix) {
            if (g_projector == 1) {                    // reading C1: the transpose of the same ray-marching l_ij
                const double ri = r[pix];
                rm_samples(G, make_ray(G, theta, (int)(pix % G.nu), (int)(pix / G.nu)), g_step_mm,
                           [&](int64_t lin, double wgt) { acc[lin] += wgt * ri; });
                continue;
            }
            siddon(G, make_ray(G, theta, (int)(pix % G.nu), (int)(pix / G.nu)), segs, nullptr);
            for (const Seg& sg : segs) acc[((int64_t)sg.k * G.ny + sg.j) * G.nx + sg.i] += sg.len * r[pix];
        }
    }
    if (T > 1)
        for (int t = 0; t < T; ++t)
            if (!part[t].empty())
                for (int64_t j = 0; j < V; ++j) B_out[j] += part[t][j];
}

// Step 2, Eq. (4): (a, b)^T = (Y^T Y)^-1 Y^T p, Y = [y, 1].  Returns -5 when y is constant (reading A8).
int orc_lsfit(int64_t n, const double* p, const float* y, double* a, double* b) {
    double Sy = 0, Syy = 0, Sp = 0, Syp = 0;
    for (int64_t i = 0; i < n; ++i) {
        const double yi = (double)y[i];
        Sy += yi; Syy += yi * yi; Sp += p[i]; Syp += yi * p[i];
    }
    const double det = Syy * (double)n - Sy * Sy;
    if (!(det > 1e-12 * Syy * (double)n)) return -5;
    *a = (Syp * (double)n - Sy * Sp) / det;
    *b = (Syy * Sp - Sy * Syp) / det;
    return 0;
}

// Eq. (2): J = || p - a y - b 1 ||_2^2 over all pixels (reading A10).
double orc_cost(int64_t n, const double* p, const float* y, double a, double b) {
    double J = 0;
    for (int64_t i = 0; i < n; ++i) {
        const double r = p[i] - a * (double)y[i] - b;
        J += r * r;
    }
    return J;
}

// dJ/dw = 2 U^T (df/dx) P^T (P f - a y - b 1)  (readings A4-A6).  p must be P f(w).
void orc_gradient(const OrcGeom* g, const float* f0, const float* xbar, const float* u, const double* w,
                  double a, double b, const double* p, const float* y, double theta, double* g_out) {
    const OrcGeom& G = *g;
    const int64_t V = nvox(G), N = npix(G);
    std::vector<double> r(N), B(V), Gr(3 * V);
    for (int64_t i = 0; i < N; ++i) r[i] = p[i] - a * (double)y[i] - b;
    orc_backproject(g, r.data(), theta, B.data());
    orc_warp_grad(g, f0, xbar, u, w, Gr.data());
    for (int k = 0; k < G.K; ++k) {
        double s = 0.0;
        for (int64_t j = 0; j < V; ++j) {
            double dot = 0.0;
            for (int c = 0; c < 3; ++c) dot += Gr[c * V + j] * (double)u[((int64_t)k * 3 + c) * V + j];
            s += B[j] * dot;
        }
        g_out[k] = 2.0 * s;
    }
}

// Tumour localisation: fixed-point inversion of the pull-back DVF (ref 13; reading A13).
// r_{m+1} = r0 - x(r_m), r_0 = r0.
void orc_invert(const OrcGeom* g, const float* xbar, const float* u, const double* w, int M, const float* r0,
                int max_iter, double tol_mm, double* r_out, int32_t* iters_out) {
    for (int m = 0; m < M; ++m) {
        const double R0[3] = {(double)r0[3 * m], (double)r0[3 * m + 1], (double)r0[3 * m + 2]};
        double r[3] = {R0[0], R0[1], R0[2]};
        int it = 0;
        for (; it < max_iter; ++it) {
            double x[3];
            dvf_at_point(*g, xbar, u, w, r, x);
            const double rn[3] = {R0[0] - x[0], R0[1] - x[1], R0[2] - x[2]};
            const double dr = std::sqrt((rn[0] - r[0]) * (rn[0] - r[0]) + (rn[1] - r[1]) * (rn[1] - r[1]) +
                                        (rn[2] - r[2]) * (rn[2] - r[2]));
            r[0] = rn[0]; r[1] = rn[1]; r[2] = rn[2];
            if (dr < tol_mm) { ++it; break; }
        }
        r_out[3 * m] = r[0]; r_out[3 * m + 1] = r[1]; r_out[3 * m + 2] = r[2];
        if (iters_out) iters_out[m] = it;
    }
}

// The DVF of Eq. (1) at arbitrary world points (test hook for the inversion pins).
void orc_dvf_at_points(const OrcGeom* g, const float* xbar, const float* u, const double* w, int M,
                       const double* pts, double* x_out) {
    for (int m = 0; m < M; ++m) dvf_at_point(*g, xbar, u, w, pts + 3 * m, x_out + 3 * m);
}

// The alternating algorithm of PAPER.md:L84-95 (Eq. 3 with Armijo's rule, then Eq. 4), readings A7-A9.
// forced_mu (or NULL): replay mode, iteration n takes exactly the step forced_mu[n] (A16 level ii).
// Trace arrays (or NULL): J_trace[max_iter+1], gnorm_trace/mu_trace/bt_trace[max_iter].
int orc_solve(const OrcGeom* g, const float* f0, const float* xbar, const float* u, const float* y, double theta,
              const double* w0, const OrcOpts* o, const double* forced_mu, double* w_out, double* f_out,
              double* p_out, OrcResult* res, double* J_trace, double* gnorm_trace, double* mu_trace,
              int32_t* bt_trace) {
    const OrcGeom& G = *g;
    const int K = G.K;
    const int64_t V = nvox(G), N = npix(G);
    std::vector<double> w(w0, w0 + K), f(V), p(N), ft(V), pt(N), gk(K), wt(K);
    const double hmin = std::min(G.hx, std::min(G.hy, G.hz));
    double a = 0, b = 0;
    orc_warp(g, f0, xbar, u, w.data(), f.data());
    orc_project(g, f.data(), theta, p.data());
    if (orc_lsfit(N, p.data(), y, &a, &b) != 0) { res->status = -5; res->iters = 0; return -5; }
    res->J0 = orc_cost(N, p.data(), y, a, b);
    int status = 1, n = 0;
    double mu_prev = 0.0;
    for (; n < o->max_iter; ++n) {
        const double Jn = orc_cost(N, p.data(), y, a, b);
        if (J_trace) J_trace[n] = Jn;
        orc_gradient(g, f0, xbar, u, w.data(), a, b, p.data(), y, theta, gk.data());
        double g2 = 0;
        for (int k = 0; k < K; ++k) g2 += gk[k] * gk[k];
        const double gn = std::sqrt(g2);
        if (gnorm_trace) gnorm_trace[n] = gn;
        if (gn <= o->grad_tol) { status = 2; break; }
        double mu = (n == 0) ? o->init_step_vox * hmin * std::sqrt((double)V) / gn : 2.0 * mu_prev;
        bool accepted = false;
        int t = 0;
        if (forced_mu) {
            mu = forced_mu[n];
            for (int k = 0; k < K; ++k) wt[k] = w[k] - mu * gk[k];
            orc_warp(g, f0, xbar, u, wt.data(), ft.data());
            orc_project(g, ft.data(), theta, pt.data());
            accepted = true;
        } else if (o->batched_linesearch) {
            // evaluate mu beta^t for every t, take the largest passing (= first passing in sequential order)
            std::vector<double> fb(V), pb(N);
            int best = -1;
            for (int tt = o->max_backtracks - 1; tt >= 0; --tt) {
                const double m = mu * std::pow(o->armijo_beta, tt);
                for (int k = 0; k < K; ++k) wt[k] = w[k] - m * gk[k];
                orc_warp(g, f0, xbar, u, wt.data(), fb.data());
                orc_project(g, fb.data(), theta, pb.data());
                if (orc_cost(N, pb.data(), y, a, b) <= Jn - o->armijo_c * m * g2) { best = tt; ft = fb; pt = pb; }
            }
            if (best >= 0) { accepted = true; t = best; mu = mu * std::pow(o->armijo_beta, best); }
            else t = o->max_backtracks;
        } else {
            for (; t < o->max_backtracks; ++t) {
                for (int k = 0; k < K; ++k) wt[k] = w[k] - mu * gk[k];
                orc_warp(g, f0, xbar, u, wt.data(), ft.data());
                orc_project(g, ft.data(), theta, pt.data());
                if (orc_cost(N, pt.data(), y, a, b) <= Jn - o->armijo_c * mu * g2) { accepted = true; break; }
                mu *= o->armijo_beta;
            }
        }
        if (bt_trace) bt_trace[n] = t;
        if (!accepted) { if (mu_trace) mu_trace[n] = 0.0; status = 3; break; }
        if (mu_trace) mu_trace[n] = mu;
        for (int k = 0; k < K; ++k) w[k] -= mu * gk[k];                   // Eq. (3)
        f.swap(ft); p.swap(pt);
        if (orc_lsfit(N, p.data(), y, &a, &b) != 0) { status = -5; break; }  // Eq. (4)
        mu_prev = mu;
    }
    res->iters = n;
    res->status = status;
    res->a = a; res->b = b;
    res->J = orc_cost(N, p.data(), y, a, b);
    if (J_trace) J_trace[n] = res->J;
    for (int k = 0; k < K; ++k) w_out[k] = w[k];
    if (f_out) std::memcpy(f_out, f.data(), sizeof(double) * V);
    if (p_out) std::memcpy(p_out, p.data(), sizeof(double) * N);
    return status;
}

}  // extern "C"
