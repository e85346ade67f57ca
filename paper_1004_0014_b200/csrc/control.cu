// a-3 (second half), a-5 and a-6: the scalar side of the alternating algorithm, kept on the device.
//
//   step 1 (Eq. 3):  w_{n+1} = w_n - mu_n dJ/dw_n, mu_n by Armijo's rule (L95)
//   step 2 (Eq. 4):  (a, b)^T = (Y^T Y)^-1 Y^T P f_{n+1},  Y = [y, 1]
//   stop:         ||dJ/dw|| small or max_iter reached
//   tumour:     r_{m+1} = r0 - x(r_m)  (fixed-point inverse of the pull-back DVF)
//
// Readings A7 (Armijo constants, first step = init_step_vox voxels rms, later 2 x the accepted
// step), A8 (initial (a, b) = fit at w0; singular fit), A9, A13 are listed in DESIGN.md.
//
// Each control kernel is one block; thread b owns solve b.  All scalars are double.  The kernels
// also decide whether the enclosing device-side while-loops of the solve graph continue
// (cudaGraphSetConditional) and mirror those decisions into LoopFlags for the host-driven mode.
#include "internal.h"

namespace pcamm {

namespace {

constexpr int CT = 256;   // threads of a control block
constexpr int YT = 256;

__global__ void __launch_bounds__(YT)
k_ysums(const Geom G, const SolveIn* __restrict__ in, double* __restrict__ part) {
    __shared__ double red[YT / 32];
    const int b = blockIdx.y;
    const float* y = in[b].y;
    double s = 0.0, ss = 0.0;
    if (y)
        for (int i = blockIdx.x * YT + threadIdx.x; i < G.npix; i += gridDim.x * YT) {
            const double v = (double)__ldg(y + i);
            s += v; ss += v * v;
        }
    const double S = block_sum<YT>(s, red), SS = block_sum<YT>(ss, red);
    if (threadIdx.x == 0) {
        double* o = part + ((long long)b * gridDim.x + blockIdx.x) * 2;
        o[0] = S; o[1] = SS;
    }
}

// Step 2, Eq. (4) as the 2x2 normal equations of Y = [y, 1].  false: y constant (reading A8).
__device__ bool lsfit(double n, double Sy, double Syy, double Sp, double Syp, double* a, double* b) {
    const double det = Syy * n - Sy * Sy;
    if (!(det > 1e-12 * Syy * n)) return false;
    *a = (Syp * n - Sy * Sp) / det;
    *b = (Syy * Sp - Sy * Syp) / det;
    return true;
}

__device__ void set_view(const Geom& G, float angle, View* vw) {
    const double th = (double)angle;
    vw->cs = cos(th); vw->sn = sin(th);
}

// Candidates st.t, st.t + 1, ... (at most C per round, fewer at the end of the backtrack budget) of
// the Armijo sequence mu0 beta^t into the solve's slots; st.mu is the step of candidate st.t and
// every later one follows by repeated multiplication, whatever the fan width, so that a fan of
// any width takes exactly the steps sequential backtracking would.
__device__ void trial_w(const SolveState& st, int K, double mu, SlotState* sl);
__device__ void make_round(const SolveState& st, int K, const CallOpts& o, SlotState* slots_b) {
    double mu = st.mu;
    for (int cnd = 0; cnd < o.C; ++cnd) {
        if (st.t + cnd < o.max_backtracks) trial_w(st, K, mu, &slots_b[cnd]);
        else slots_b[cnd].active = 0;
        mu *= o.armijo_beta;
    }
}

__device__ void trial_w(const SolveState& st, int K, double mu, SlotState* sl) {
    for (int k = 0; k < K; ++k) sl->w[k] = (float)(st.w[k] - mu * st.g[k]);   // Eq. (3), candidate
    sl->mu = mu;
    sl->active = 1;
}

// mode 0: start of a solve.  mode 1: pcamm_eval (a, b given).  mode 2: hooks that only need the
// view and w in slot 0.
__global__ void __launch_bounds__(CT)
k_begin(const Geom G, const CallOpts* __restrict__ opts, const SolveIn* __restrict__ in, SolveState* solves,
        SlotState* slots, LoopFlags* flags, int mode) {
    const int B = opts->B, C = opts->C;
    for (int b = threadIdx.x; b < B; b += CT) {
        SolveState& st = solves[b];
        set_view(G, in[b].angle, &st.view);
        for (int k = 0; k < KMAX; ++k) { st.w[k] = k < G.K ? (double)in[b].w_init[k] : 0.0; st.g[k] = 0.0; }
        st.a = mode == 1 ? (double)in[b].a : 0.0;
        st.b = mode == 1 ? (double)in[b].b : 0.0;
        st.Sy = st.Syy = 0.0;
        st.Jn = st.J = st.g2 = st.mu = st.mu_prev = 0.0;
        st.J0 = nan("");
        st.fit_a = st.fit_b = 0.0;
        st.iter = 0; st.status = 0; st.running = mode == 1 ? 1 : 0; st.trialing = 0; st.t = 0;
        st.acc_slot = b * C;
        for (int c = 0; c < C; ++c) {
            SlotState& sl = slots[b * C + c];
            sl.solve = b; sl.active = 0; sl.mu = 0.0; sl.J = sl.Sp = sl.Syp = 0.0;
            for (int k = 0; k < KMAX; ++k) sl.w[k] = 0.f;
        }
        SlotState& s0 = slots[b * C];
        for (int k = 0; k < G.K; ++k) s0.w[k] = in[b].w_init[k];
        s0.active = 1;
    }
    if (threadIdx.x == 0) { flags->iter_cond = 0; flags->trial_cond = 0; flags->n_launch = 0; flags->ticket = 0u; }
}

// Sum of n partials with the given stride, by the whole control block (fixed order); the result
// is broadcast to all threads.
__device__ double coop_sum(const double* part, int n, int stride, double* red /* [CT/32 + 1] */) {
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += CT) v += __ldcg(part + (long long)i * stride);   // written by other blocks
    const double s = block_sum<CT>(v, red);
    if (threadIdx.x == 0) red[CT / 32] = s;
    __syncthreads();
    return red[CT / 32];
}

struct Sums3 { double a, b, c; };

// The three projection sums of slot s in one pass (one round trip to L2, one exchange).
__device__ Sums3 sum_proj(const double* part, int nblk, int s, double* red /* unused */) {
    __shared__ double ex[3][CT / 32];
    __shared__ double tot[3];
    (void)red;
    const double* p = part + (long long)s * nblk * 3;
    double v0 = 0.0, v1 = 0.0, v2 = 0.0;
    for (int i = threadIdx.x; i < nblk; i += CT) {
        v0 += __ldcg(p + 3 * i); v1 += __ldcg(p + 3 * i + 1); v2 += __ldcg(p + 3 * i + 2);
    }
    v0 = warp_sum(v0); v1 = warp_sum(v1); v2 = warp_sum(v2);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();                       // ex / tot may still be read from a previous call
    if (lane == 0) { ex[0][wid] = v0; ex[1][wid] = v1; ex[2][wid] = v2; }
    __syncthreads();
    if (threadIdx.x < 3) {
        double t = 0.0;
#pragma unroll
        for (int i = 0; i < CT / 32; ++i) t += ex[threadIdx.x][i];
        tot[threadIdx.x] = t;
    }
    __syncthreads();
    Sums3 r;
    r.a = tot[0]; r.b = tot[1]; r.c = tot[2];
    return r;
}

__device__ void publish(LoopFlags* flags, int iter_cond, int trial_cond, int launched) {
    flags->iter_cond = iter_cond;
    flags->trial_cond = trial_cond;
    flags->n_launch += launched;
}

// After the initial evaluation at w0: Sy, Syy, the first fit (reading A8), loop start.
__device__ void ctl_init_body(const Geom& G, const CtlBufs& c, cudaGraphConditionalHandle h_iter, int use_cond) {
    __shared__ double red[CT / 32 + 1];
    int any_running = 0;
    const CallOpts& o = *c.opts;
    for (int b = 0; b < o.B; ++b) {
        SolveState& st = c.solves[b];
        const double* yp = c.ysum_part + (long long)b * c.ysum_blocks * 2;
        const double Sy = coop_sum(yp, c.ysum_blocks, 2, red), Syy = coop_sum(yp + 1, c.ysum_blocks, 2, red);
        const int s0 = b * o.C;
        const Sums3 sp = sum_proj(c.proj_part, c.proj_blocks, s0, red);
        if (threadIdx.x != 0) continue;
        st.Sy = Sy; st.Syy = Syy;
        c.slots[s0].Sp = sp.a; c.slots[s0].Syp = sp.b;
        c.slots[s0].active = 0;
        if (!isfinite(Sy) || !isfinite(Syy)) st.status = PCAMM_E_NONFINITE;
        else if (!lsfit((double)G.npix, Sy, Syy, sp.a, sp.b, &st.a, &st.b)) st.status = PCAMM_E_SINGULAR;
        st.acc_slot = s0;
        st.iter = 0;
        if (st.status == 0 && o.max_iter <= 0) st.status = PCAMM_S_MAXITER;
        st.running = st.status == 0;
        any_running |= st.running;
    }
    if (threadIdx.x == 0) {
        publish(c.flags, any_running, 0, 6);
        if (use_cond) cudaGraphSetConditional(h_iter, any_running);
    }
}

// After the residual and gradient kernels of iteration n: J_n, g, stopping rule, first candidate(s).
__global__ void __launch_bounds__(CT)
k_ctl_grad(const Geom G, CtlBufs c, cudaGraphConditionalHandle h_trial, int use_cond) {
    __shared__ double ex[KMAX + 1][CT / 32];
    __shared__ double tot[KMAX + 1];
    int any_trial = 0, any_running = 0;
    const CallOpts o = *c.opts;
    const int K = G.K;
    for (int b = 0; b < o.B; ++b) {
        SolveState st = c.solves[b];                   // worked on in registers; thread 0 writes it back
        if (!st.running) continue;                                                        // uniform
        const int n = st.iter;
        // J_n and the K gradient sums in one pass over the partial sums (fixed order)
        {
            double v[KMAX + 1];
#pragma unroll
            for (int k = 0; k <= KMAX; ++k) v[k] = 0.0;
            const double* rp = c.resid_part + (long long)b * c.resid_blocks;
            for (int i = threadIdx.x; i < c.resid_blocks; i += CT) v[KMAX] += __ldcg(rp + i);
            const double* gp = c.grad_part + (long long)b * c.grad_blocks * KMAX;
            for (int i = threadIdx.x; i < c.grad_blocks; i += CT) {
#pragma unroll
                for (int k = 0; k < KMAX; ++k)
                    if (k < K) v[k] += __ldcg(gp + (long long)i * KMAX + k);
            }
            const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
            __syncthreads();
#pragma unroll
            for (int k = 0; k <= KMAX; ++k) {
                const double w = warp_sum(v[k]);
                if (lane == 0) ex[k][wid] = w;
            }
            __syncthreads();
            if (threadIdx.x <= KMAX) {
                double t = 0.0;
#pragma unroll
                for (int i = 0; i < CT / 32; ++i) t += ex[threadIdx.x][i];
                tot[threadIdx.x] = t;
            }
            __syncthreads();
        }
        if (threadIdx.x != 0) continue;
        const double Jn = tot[KMAX];
        double gk[KMAX];
        for (int k = 0; k < K; ++k) gk[k] = tot[k];
        st.Jn = Jn;                                                                       // Eq. (2)
        if (n == 0) st.J0 = st.Jn;
        double g2 = 0.0;
        for (int k = 0; k < K; ++k) {
            st.g[k] = 2.0 * gk[k];
            g2 += st.g[k] * st.g[k];
        }
        st.g2 = g2;
        const double gn = sqrt(g2);
        if (n < TRACE_CAP) { c.traces[b].J[n] = st.Jn; c.traces[b].gnorm[n] = gn; }
        if (gn <= o.grad_tol || !isfinite(gn)) {
            st.status = isfinite(gn) ? PCAMM_S_GRADTOL : PCAMM_E_NONFINITE;
            st.running = 0; st.trialing = 0;
            c.solves[b] = st;
            continue;
        }
        st.mu = n == 0 ? o.init_step_vox * o.hmin_sqrtV / gn : 2.0 * st.mu_prev;         // reading A7
        st.t = 0;
        st.trialing = 1;
        make_round(st, K, o, &c.slots[b * o.C]);
        any_trial = 1;
        any_running = 1;
        c.solves[b] = st;
    }
    if (threadIdx.x == 0) {
        publish(c.flags, any_running, any_trial, 3);
        if (use_cond) cudaGraphSetConditional(h_trial, any_trial);
    }
}

// After warp + projection of the candidate(s): Armijo's inequality, Eq. (3) update, Eq. (4) fit.
__device__ void ctl_trial_body(const Geom& G, const CtlBufs& c, cudaGraphConditionalHandle h_trial, int use_cond) {
    __shared__ double red[CT / 32 + 1];
    int any_trial = 0, any_running = 0;
    const CallOpts o = *c.opts;
    const int K = G.K;
    for (int b = 0; b < o.B; ++b) {
        // the state is worked on in registers (one round trip to L2 each way, instead of one per
        // field touched); thread 0 writes it back
        SolveState st = c.solves[b];
        if (st.running && !st.trialing) any_running = 1;
        if (!st.trialing) continue;                                                       // uniform
        const int n = st.iter;
        int acc = -1;
        double acc_mu = 0.0, acc_Sp = 0.0, acc_Syp = 0.0;
        bool failed = false;
        // the round's candidates st.t .. st.t + C - 1 have been evaluated: the first that passes is
        // the one sequential backtracking would have accepted (reading A7)
        int n_cand = o.max_backtracks - st.t;
        if (n_cand > o.C) n_cand = o.C;
        double mu_last = st.mu;
        for (int cnd = 0; cnd < n_cand; ++cnd) {
            const int s = b * o.C + cnd;
            const Sums3 sp = sum_proj(c.proj_part, c.proj_blocks, s, red);
            if (threadIdx.x != 0) continue;
            const double mu_s = c.slots[s].mu;
            c.slots[s].Sp = sp.a; c.slots[s].Syp = sp.b; c.slots[s].J = sp.c;
            if (acc < 0 && sp.c <= st.Jn - o.armijo_c * mu_s * st.g2) {                   // Armijo (L95)
                acc = s; acc_mu = mu_s; acc_Sp = sp.a; acc_Syp = sp.b;
                st.t += cnd;
            }
            c.slots[s].active = 0;
            mu_last = mu_s;
        }
        if (threadIdx.x != 0) continue;
        if (acc < 0) {
            st.t += n_cand;
            st.mu = mu_last * o.armijo_beta;
            if (st.t >= o.max_backtracks) failed = true;
            else make_round(st, K, o, &c.slots[b * o.C]);
        }
        if (acc >= 0) {
            const double mu = acc_mu;
            for (int k = 0; k < K; ++k) st.w[k] -= mu * st.g[k];                          // Eq. (3)
            st.mu_prev = mu;
            st.acc_slot = acc;
            if (n < TRACE_CAP) { c.traces[b].mu[n] = mu; c.traces[b].bt[n] = st.t; }
            st.iter = n + 1;
            st.trialing = 0;
            if (!lsfit((double)G.npix, st.Sy, st.Syy, acc_Sp, acc_Syp, &st.a, &st.b)) {   // Eq. (4)
                st.status = PCAMM_E_SINGULAR; st.running = 0;
            } else if (st.iter >= o.max_iter) { st.status = PCAMM_S_MAXITER; st.running = 0; }
        } else if (failed) {
            if (n < TRACE_CAP) { c.traces[b].mu[n] = 0.0; c.traces[b].bt[n] = st.t; }
            st.status = PCAMM_S_LINESEARCH;
            st.running = 0; st.trialing = 0;
        }
        if (st.trialing) any_trial = 1;
        if (st.running) any_running = 1;
        c.solves[b] = st;                                                                 // thread 0 only gets here
    }
    if (threadIdx.x == 0) {
        publish(c.flags, any_running, any_trial, 3);
        if (use_cond) cudaGraphSetConditional(h_trial, any_trial);
    }
}

// Last kernel of the iteration body: decides whether the outer while-loop runs again.
__global__ void k_ctl_iter_end(CtlBufs c, cudaGraphConditionalHandle h_iter, int use_cond) {
    if (threadIdx.x == 0) {
        c.flags->n_launch += 1;
        if (use_cond) cudaGraphSetConditional(h_iter, c.flags->iter_cond);
    }
}

// After the closing residual pass: J at exit, final w into the output slots.
__global__ void __launch_bounds__(CT)
k_ctl_final(const Geom G, CtlBufs c, SlotState* out_slots) {
    __shared__ double red[CT / 32 + 1];
    const CallOpts& o = *c.opts;
    for (int b = 0; b < o.B; ++b) {
        SolveState& st = c.solves[b];
        const double J = coop_sum(c.resid_part + (long long)b * c.resid_blocks, c.resid_blocks, 1, red);
        if (threadIdx.x != 0) continue;
        st.J = J;
        if (isnan(st.J0)) st.J0 = st.J;
        if (st.iter <= TRACE_CAP) c.traces[b].J[st.iter] = st.J;
        SlotState& sl = out_slots[b];
        for (int k = 0; k < KMAX; ++k) sl.w[k] = k < G.K ? (float)st.w[k] : 0.f;
        sl.active = 1; sl.solve = b; sl.mu = 0.0; sl.J = st.J; sl.Sp = sl.Syp = 0.0;
    }
    if (threadIdx.x == 0) c.flags->n_launch += 3;
}

// pcamm_eval: stage 0 after the projection (J at the given (a, b), fit of Eq. 4), stage 1 after
// the gradient.
__device__ void ctl_eval_body(const Geom& G, const CtlBufs& c, int stage) {
    __shared__ double red[CT / 32 + 1];
    const CallOpts& o = *c.opts;
    for (int b = 0; b < o.B; ++b) {
        SolveState& st = c.solves[b];
        if (stage == 0) {
            const double* yp = c.ysum_part + (long long)b * c.ysum_blocks * 2;
            const double Sy = coop_sum(yp, c.ysum_blocks, 2, red), Syy = coop_sum(yp + 1, c.ysum_blocks, 2, red);
            const Sums3 sp = sum_proj(c.proj_part, c.proj_blocks, b * o.C, red);
            if (threadIdx.x != 0) continue;
            st.Sy = Sy; st.Syy = Syy;
            st.J = sp.c;
            st.fit_a = st.fit_b = nan("");
            lsfit((double)G.npix, Sy, Syy, sp.a, sp.b, &st.fit_a, &st.fit_b);
            st.acc_slot = b * o.C;
        } else {
            const double Jn = coop_sum(c.resid_part + (long long)b * c.resid_blocks, c.resid_blocks, 1, red);
            double gk[KMAX];
            for (int k = 0; k < G.K; ++k)
                gk[k] = coop_sum(c.grad_part + (long long)b * c.grad_blocks * KMAX + k, c.grad_blocks, KMAX, red);
            if (threadIdx.x != 0) continue;
            st.Jn = Jn;
            for (int k = 0; k < G.K; ++k) st.g[k] = 2.0 * gk[k];
        }
    }
}

__global__ void __launch_bounds__(CT)
k_ctl_eval_grad(const Geom G, CtlBufs c) { ctl_eval_body(G, c, 1); }

// The control step that follows a projection (then = THEN_INIT / THEN_TRIAL / THEN_EVAL): one block.
__global__ void __launch_bounds__(CT)
k_ctl_after_project(const Geom G, CtlBufs c, int then, cudaGraphConditionalHandle h, int use_cond) {
    if (then == THEN_INIT) ctl_init_body(G, c, h, use_cond);
    else if (then == THEN_TRIAL) ctl_trial_body(G, c, h, use_cond);
    else ctl_eval_body(G, c, 0);
}

// a-6.  One warp per (landmark, solve).  x(r) is the trilinear interpolation of the synthesised
// DVF of Eq. (1) at the off-grid point r, coordinates clamped to the grid (reading A13); the
// 8 (K+1) (tap, field) pairs are spread over the lanes.
__global__ void __launch_bounds__(32)
k_invert(const Geom G, const float* __restrict__ xbar, const float* __restrict__ u, const CallOpts* __restrict__ opts,
         const SolveState* __restrict__ solves, int M, const float* __restrict__ r0s, double* __restrict__ r_out) {
    const int m = blockIdx.x, b = blockIdx.y, lane = threadIdx.x;
    const int K = G.K;
    const long long V = G.V;
    const double R0[3] = {(double)r0s[3 * m], (double)r0s[3 * m + 1], (double)r0s[3 * m + 2]};
    double r[3] = {R0[0], R0[1], R0[2]};
    const int N[3] = {G.nx, G.ny, G.nz};
    const double h[3] = {(double)G.hx, (double)G.hy, (double)G.hz};
    const double ctr[3] = {(double)G.cx, (double)G.cy, (double)G.cz};
    const int max_iter = opts->inv_max_iter;
    const double tol = opts->inv_tol;
    for (int it = 0; it < max_iter; ++it) {
        int i0[3];
        double t[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double q = (r[c] - ctr[c]) / h[c] + 0.5 * (N[c] - 1);
            q = fmin(fmax(q, 0.0), (double)(N[c] - 1));
            int f = (int)floor(q);
            if (f > N[c] - 2) f = N[c] - 2;
            if (f < 0) f = 0;
            i0[c] = f;
            t[c] = N[c] == 1 ? 0.0 : q - (double)f;
        }
        double part[3] = {0.0, 0.0, 0.0};
        for (int idx = lane; idx < 8 * (K + 1); idx += 32) {
            const int tap = idx & 7, fld = idx >> 3;
            const int a = tap & 1, bb = (tap >> 1) & 1, cc = tap >> 2;
            const double wgt = (a ? t[0] : 1.0 - t[0]) * (bb ? t[1] : 1.0 - t[1]) * (cc ? t[2] : 1.0 - t[2]);
            if (wgt == 0.0) continue;
            const int i = min(i0[0] + a, N[0] - 1), j = min(i0[1] + bb, N[1] - 1), k = min(i0[2] + cc, N[2] - 1);
            const long long lin = ((long long)k * G.ny + j) * G.nx + i;
            const double coef = wgt * (fld == 0 ? 1.0 : solves[b].w[fld - 1]);
            const float* base = fld == 0 ? xbar : u + (long long)(fld - 1) * 3 * V;
#pragma unroll
            for (int c = 0; c < 3; ++c) part[c] += coef * (double)__ldg(base + c * V + lin);
        }
        double x[3];                                   // the model's fields are in voxel units: x (mm) = field * h
#pragma unroll
        for (int c = 0; c < 3; ++c) x[c] = warp_sum(part[c]) * h[c];
        double d2 = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double rn = R0[c] - x[c];
            d2 += (rn - r[c]) * (rn - r[c]);
            r[c] = rn;
        }
        if (sqrt(d2) < tol) break;   // identical on all lanes (butterfly sum)
    }
    if (lane == 0) {
        double* o = r_out + ((long long)b * M + m) * 3;
        o[0] = r[0]; o[1] = r[1]; o[2] = r[2];
    }
}

}  // namespace

int ysum_blocks(const Geom& G) { return min(64, (G.npix + YT - 1) / YT); }

void launch_ysums(Seq& q, const Geom& G, const CtlBufs& c, int B) {
    q.launch(k_ysums, dim3(c.ysum_blocks, B), dim3(YT), 0, G, (const SolveIn*)c.in, c.ysum_part);
}

void launch_begin(Seq& q, const Geom& G, const CtlBufs& c, int mode) {
    q.launch(k_begin, dim3(1), dim3(CT), 0, G, (const CallOpts*)c.opts, (const SolveIn*)c.in, c.solves, c.slots,
             c.flags, mode);
}

void launch_ctl_grad(Seq& q, const Geom& G, const CtlBufs& c, cudaGraphConditionalHandle h_trial, int use_cond) {
    q.launch(k_ctl_grad, dim3(1), dim3(CT), 0, G, c, h_trial, use_cond);
}

void launch_ctl_iter_end(Seq& q, const CtlBufs& c, cudaGraphConditionalHandle h_iter, int use_cond) {
    q.launch(k_ctl_iter_end, dim3(1), dim3(32), 0, c, h_iter, use_cond);
}

void launch_ctl_final(Seq& q, const Geom& G, const CtlBufs& c, SlotState* out_slots) {
    q.launch(k_ctl_final, dim3(1), dim3(CT), 0, G, c, out_slots);
}

void launch_ctl_eval_grad(Seq& q, const Geom& G, const CtlBufs& c) {
    q.launch(k_ctl_eval_grad, dim3(1), dim3(CT), 0, G, c);
}

void launch_ctl_after_project(Seq& q, const Geom& G, const CtlBufs& c, int then, cudaGraphConditionalHandle h,
                              int use_cond) {
    if (then == THEN_NONE) return;
    q.launch(k_ctl_after_project, dim3(1), dim3(CT), 0, G, c, then, h, use_cond);
}

void launch_invert(Seq& q, const Geom& G, const float* xbar, const float* u, const CtlBufs& c, int B, int M,
                   const float* r0, double* r_out) {
    if (M <= 0) return;
    q.launch(k_invert, dim3(M, B), dim3(32), 0, G, xbar, u, (const CallOpts*)c.opts, (const SolveState*)c.solves, M,
             r0, r_out);
}

}  // namespace pcamm
