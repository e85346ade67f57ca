// a-2 / a-4, second discretisation of P (PAPER.md:L82 says only "P is a
// projection matrix"; north_star: "fixed-step or Siddon traversal"): fixed-step trilinear ray
// marching, reading C1 (pcamm_geometry.projector = 1):
//
//   p_i = d_i sum_{m = 0}^{M_i - 1} (T f)(E_i + (m + 1/2) d_i e_i)
//
// [E_i, X_i] = the part of the ray source -> pixel centre i inside the box spanned by the voxel
// centres, L_i its length, M_i = ceil(L_i / step), d_i = L_i / M_i, T f the trilinear interpolant of
// the voxel-centre values.  P^T is the exact transpose: the same samples and weights, scattered.
//
// Both kernels are ray-driven, one thread per ray, a block per detector column (the rays of a
// column share their in-plane positions, so the lanes of a warp read the same (x, y) voxel columns
// of the z-fastest ray layout).  The sample position is formed in double, so that the cell a sample
// falls into never depends on float rounding; the interpolation itself is float.  The transpose
// scatters with atomic adds into a volume B that the gradient kernel then reads instead of
// gathering (the order of the adds is not fixed: results of this variant are reproducible to
// rounding, not bitwise).  This variant is the simple ray-driven form; the regrouping that makes
// the Siddon projector fast (project.cu) is not applied to it.
//
// Where the gradient of a single solve is a gather over the records the warp kernel left
// (stream.cuh GradRecords), B is read at the recorded voxels only: k_record_mask turns the records
// of the accepted candidate into one bit per voxel, and the scatter then skips every add to a voxel
// nobody will read (at C2 94 % of them; the sums at the others are what they would have been).
#include "internal.h"

namespace pcamm {

namespace {

constexpr int RT = 256;          // threads of a block (rows of one detector column, strided)

struct RmRay {
    double q0[3], dq[3];         // index coordinates of the chord's entry and their change per unit of alpha
    double a0, da;               // alpha at the entry, alpha per step
    int M;                       // steps (0: the ray misses)
    float d;                     // mm per step
};

// the chord of ray (iu, iv) in the box of voxel centres, and its steps
__device__ __forceinline__ RmRay rm_ray(const Geom& G, const View& vw, int iu, int iv) {
    RmRay r;
    r.M = 0; r.d = 0.f; r.a0 = 0.0; r.da = 0.0;
    double dx, dy;
    ray_dir_inplane(G, vw.cs, vw.sn, iu, &dx, &dy);
    const double dz = ((double)iv - 0.5 * (G.nv - 1) + (double)G.off_v) * (double)G.pv;
    const double S[3] = {(double)G.sad * vw.cs, (double)G.sad * vw.sn, 0.0}, d[3] = {dx, dy, dz};
    const int N[3] = {G.nx, G.ny, G.nz};
    const double h[3] = {(double)G.hx, (double)G.hy, (double)G.hz};
    const double ctr[3] = {(double)G.cx, (double)G.cy, (double)G.cz};
    const double len = sqrt(dx * dx + dy * dy + dz * dz);
    double amin = 0.0, amax = 1.0;
    bool miss = false;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (N[c] < 2) { miss = true; continue; }
        const double lo = ctr[c] - 0.5 * (N[c] - 1) * h[c], hi = ctr[c] + 0.5 * (N[c] - 1) * h[c];
        r.q0[c] = (S[c] - lo) / h[c];
        r.dq[c] = d[c] / h[c];
        if (fabs(d[c]) < 1e-12 * len) {
            if (S[c] < lo || S[c] > hi) miss = true;
            continue;
        }
        const double a = (lo - S[c]) / d[c], b = (hi - S[c]) / d[c];
        amin = fmax(amin, fmin(a, b));
        amax = fmin(amax, fmax(a, b));
    }
    if (miss || !(amin < amax)) return r;
    const double L = (amax - amin) * len;
    const double Md = ceil(L / (double)G.rm_step_mm);
    if (!(Md >= 1.0) || Md > 1e8) return r;
    r.M = (int)Md;
    r.d = (float)(L / Md);
    r.a0 = amin;
    r.da = (amax - amin) / Md;
    return r;
}

// cell and fractions of sample m
struct RmSample { int i, j, k; float tx, ty, tz; };
__device__ __forceinline__ RmSample rm_sample(const Geom& G, const RmRay& r, int m) {
    const double al = fma((double)m + 0.5, r.da, r.a0);
    const double qx = fma(al, r.dq[0], r.q0[0]), qy = fma(al, r.dq[1], r.q0[1]), qz = fma(al, r.dq[2], r.q0[2]);
    RmSample s;
    s.i = min(max((int)floor(qx), 0), G.nx - 2);
    s.j = min(max((int)floor(qy), 0), G.ny - 2);
    s.k = min(max((int)floor(qz), 0), G.nz - 2);
    s.tx = (float)(qx - (double)s.i); s.ty = (float)(qy - (double)s.j); s.tz = (float)(qz - (double)s.k);
    return s;
}

// p[s] = P f[s] (volumes in the ray layout) and the a-3 partial sums of the column.  grid (nu, slots).
__global__ void __launch_bounds__(RT)
k_project_rm(const Geom G, const CtlBufs c, int slot0, const float* __restrict__ vol, float* __restrict__ p_out) {
    __shared__ double red[RT / 32];
    tl_begin(G.tl);
    const int iu = blockIdx.x, s = slot0 + blockIdx.y;
    if (!c.slots[s].active) { tl_end(G.tl, TLK_PROJECT); return; }     // uniform over the block
    const int b = c.slots[s].solve;
    const View vw = c.solves[b].view;
    const float* __restrict__ f = vol + (long long)s * G.PV;
    const float* y = c.in[b].y;
    const double fa = c.solves[b].a, fb = c.solves[b].b;
    const int sx = G.nz, sy = G.pnx * G.nz;                            // ray layout: z fastest, then x, then y
    double vp = 0.0, vyp = 0.0, vrr = 0.0;
    for (int iv = threadIdx.x; iv < G.nv; iv += RT) {
        const RmRay r = rm_ray(G, vw, iu, iv);
        float acc = 0.f;
        for (int m = 0; m < r.M; ++m) {
            const RmSample q = rm_sample(G, r, m);
            const float* p0 = f + ((q.j + 1) * G.pnx + (q.i + 1)) * G.nz + q.k;
            const float c000 = __ldg(p0), c001 = __ldg(p0 + 1), c100 = __ldg(p0 + sx), c101 = __ldg(p0 + sx + 1);
            const float c010 = __ldg(p0 + sy), c011 = __ldg(p0 + sy + 1), c110 = __ldg(p0 + sy + sx), c111 = __ldg(p0 + sy + sx + 1);
            // c[x][y][z]; interpolate along z, then x, then y
            const float z00 = fmaf(q.tz, c001 - c000, c000), z10 = fmaf(q.tz, c101 - c100, c100);
            const float z01 = fmaf(q.tz, c011 - c010, c010), z11 = fmaf(q.tz, c111 - c110, c110);
            const float x0 = fmaf(q.tx, z10 - z00, z00), x1 = fmaf(q.tx, z11 - z01, z01);
            acc += fmaf(q.ty, x1 - x0, x0);
        }
        const float p = acc * r.d;
        const long long pix = (long long)iv * G.nu + iu;
        p_out[(long long)s * G.npix + pix] = p;
        const double yv = y ? (double)__ldg(y + pix) : 0.0;
        const double res = (double)p - fa * yv - fb;                      // Eq. (2) residual
        vp += (double)p; vyp += yv * (double)p; vrr += res * res;
    }
    double* out = c.proj_part + ((long long)s * G.nu + iu) * 3;
    const double sp = block_sum<RT>(vp, red);
    const double syp = block_sum<RT>(vyp, red);
    const double srr = block_sum<RT>(vrr, red);
    if (threadIdx.x == 0) { out[0] = sp; out[1] = syp; out[2] = srr; }
    tl_end(G.tl, TLK_PROJECT);
}

// B[b] += P^T r for the solves that need a gradient (B zeroed beforehand); rL = r |D - S| as
// k_resid leaves it.  r_direct: one view, solve 0 (the pcamm_backproject hook).  grid (nu, B).
__global__ void __launch_bounds__(RT)
k_backproject_rm(const Geom G, const SolveState* __restrict__ solves, int force, const float* __restrict__ rL,
                 float* __restrict__ bvol, const unsigned* __restrict__ mask) {
    tl_begin(G.tl);
    const int iu = blockIdx.x, b = blockIdx.y;
    if (!needs_gradient(solves[b]) && !force) { tl_end(G.tl, TLK_RESID); return; }
    const View vw = solves[b].view;
    float* __restrict__ B = bvol + (long long)b * G.V;
    const int sx = 1, sy = G.nx;
    const long long sz = (long long)G.nx * G.ny;
    for (int iv = threadIdx.x; iv < G.nv; iv += RT) {
        const RmRay r = rm_ray(G, vw, iu, iv);
        if (r.M == 0) continue;
        const double uu = ((double)iu - 0.5 * (G.nu - 1) + (double)G.off_u) * (double)G.pu;
        const double vv = ((double)iv - 0.5 * (G.nv - 1) + (double)G.off_v) * (double)G.pv;
        const double Lds = sqrt((double)G.sdd * (double)G.sdd + uu * uu + vv * vv);
        const float rd = (float)((double)__ldg(rL + (long long)b * G.npix + (long long)iv * G.nu + iu) / Lds) * r.d;
        if (rd == 0.f) continue;
        for (int m = 0; m < r.M; ++m) {
            const RmSample q = rm_sample(G, r, m);
            const long long l0 = ((long long)q.k * G.ny + q.j) * G.nx + q.i;
            float* p0 = B + l0;
            const float wx0 = 1.f - q.tx, wy0 = 1.f - q.ty, wz0 = (1.f - q.tz) * rd, wz1 = q.tz * rd;
            if (mask) {                                                    // uniform over the grid
                auto add = [&](long long off, float v) {
                    const long long l = l0 + off;
                    if ((__ldg(mask + (l >> 5)) >> (unsigned)(l & 31)) & 1u) atomicAdd(p0 + off, v);
                };
                add(0, wx0 * wy0 * wz0);            add(sx, q.tx * wy0 * wz0);
                add(sy, wx0 * q.ty * wz0);          add(sy + sx, q.tx * q.ty * wz0);
                add(sz, wx0 * wy0 * wz1);           add(sz + sx, q.tx * wy0 * wz1);
                add(sz + sy, wx0 * q.ty * wz1);     add(sz + sy + sx, q.tx * q.ty * wz1);
                continue;
            }
            atomicAdd(p0, wx0 * wy0 * wz0);           atomicAdd(p0 + sx, q.tx * wy0 * wz0);
            atomicAdd(p0 + sy, wx0 * q.ty * wz0);     atomicAdd(p0 + sy + sx, q.tx * q.ty * wz0);
            atomicAdd(p0 + sz, wx0 * wy0 * wz1);      atomicAdd(p0 + sz + sx, q.tx * wy0 * wz1);
            atomicAdd(p0 + sz + sy, wx0 * q.ty * wz1); atomicAdd(p0 + sz + sy + sx, q.tx * q.ty * wz1);
        }
    }
    tl_end(G.tl, TLK_RESID);
}

__global__ void __launch_bounds__(256)
k_zero_bvol(const Geom G, const SolveState* __restrict__ solves, int force, float4* __restrict__ bvol4, long long n4_per_solve,
            float* __restrict__ bvol, long long V) {
    grid_dependency_wait();
    const int b = blockIdx.y;
    if (!needs_gradient(solves[b]) && !force) return;
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (n4_per_solve > 0) {
        if (i < n4_per_solve) bvol4[b * n4_per_solve + i] = make_float4(0.f, 0.f, 0.f, 0.f);
    } else if (i < V) bvol[b * V + i] = 0.f;
}

// One bit per voxel (bit lin & 31 of word lin >> 5, lin = (z ny + y) nx + x): set where the accepted
// candidate of solve 0 has a gradient record.  One warp per sub-tile of records; the words are
// cleared beforehand (k_zero_words).
__global__ void __launch_bounds__(256)
k_record_mask(const Geom G, const SolveState* __restrict__ solves, int force, int* __restrict__ rec_base, long long n_sub, int cap,
              unsigned* __restrict__ mask) {
    grid_dependency_wait();
    if (!needs_gradient(solves[0]) && !force) return;
    const GradRecords rec = grad_records(rec_base, n_sub, n_sub * cap, solves[0].acc_slot);
    const long long sub = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (sub >= n_sub) return;
    const int n = __ldcg(rec.count + sub);
    for (int e = threadIdx.x & 31; e < n; e += 32) {
        const int w = __ldcg(&rec.r[sub * cap + e].xyz);
        const long long lin = ((long long)record_z(w) * G.ny + record_y(w)) * G.nx + record_x(w);
        atomicOr(mask + (lin >> 5), 1u << (unsigned)(lin & 31));
    }
}

__global__ void __launch_bounds__(256)
k_zero_words(const SolveState* __restrict__ solves, int force, unsigned* __restrict__ words, long long n) {
    grid_dependency_wait();
    if (!needs_gradient(solves[0]) && !force) return;
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i < n) words[i] = 0u;
}

}  // namespace

void launch_project_rm(Seq& q, const Geom& G, const CtlBufs& c, int nslots, const float* vol, float* p) {
    for (int s0 = 0; s0 < nslots; s0 += 65535) {
        const int ns = nslots - s0 < 65535 ? nslots - s0 : 65535;
        q.launch(k_project_rm, dim3(G.nu, ns), dim3(RT), 0, G, c, s0, vol, p);
    }
}

long long record_mask_words(const Geom& G) { return (G.V + 31) / 32; }

void launch_backproject_rm(Seq& q, const Geom& G, const SolveState* solves, int B, int force, const float* rL, float* bvol,
                           int* rec, long long n_sub, int cap, unsigned* mask) {
    const bool v4 = G.V % 4 == 0;
    const long long n = v4 ? G.V / 4 : G.V;
    const bool masked = B == 1 && rec && mask;          // one solve whose gradient gathers over the records
    if (masked) {
        const long long nw = record_mask_words(G);
        q.launch(k_zero_words, dim3((unsigned)((nw + 255) / 256)), dim3(256), 0, solves, force, mask, nw);
        q.launch(k_record_mask, dim3((unsigned)((n_sub + 7) / 8)), dim3(256), 0, G, solves, force, rec, n_sub, cap, mask);
    }
    for (int b0 = 0; b0 < B; b0 += 65535) {
        const int nb = B - b0 < 65535 ? B - b0 : 65535;
        q.launch(k_zero_bvol, dim3((unsigned)((n + 255) / 256), nb), dim3(256), 0, G, solves + b0, force,
                 reinterpret_cast<float4*>(bvol + (long long)b0 * G.V), v4 ? n : 0LL, bvol + (long long)b0 * G.V, G.V);
        q.launch(k_backproject_rm, dim3(G.nu, nb), dim3(RT), 0, G, solves + b0, force, rL + (long long)b0 * G.npix,
                 bvol + (long long)b0 * G.V, (const unsigned*)(masked ? mask : nullptr));
    }
}

}  // namespace pcamm
