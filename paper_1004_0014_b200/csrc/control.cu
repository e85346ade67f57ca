// The single-block kernels of a solve that are not folded into a streaming kernel: sums of y, the
// start of a call, the closing step, and a-6:
//
//   tumour:     r_{m+1} = r0 - x(r_m)  (fixed-point inverse of the pull-back DVF)
//
// The control steps of the alternating algorithm (Armijo test, Eq. 3 update, Eq. 4 fit, stopping
// rule) are the device functions of control.cuh, run by the last block of the projector / of the
// gradient kernel.  Reading A13 (landmark inversion) is listed in DESIGN.md.
#include "internal.h"
#include "control.cuh"

namespace pcamm {

namespace {

constexpr int YT = 256;

__global__ void __launch_bounds__(YT)
k_ysums(const Geom G, const SolveIn* __restrict__ in, double* __restrict__ part) {
    __shared__ double red[YT / 32];
    tl_begin(G.tl);
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
    tl_end(G.tl, TLK_YSUMS);
}

__device__ void set_view(const Geom& G, float angle, View* vw) {
    const double th = (double)angle;
    vw->cs = cos(th); vw->sn = sin(th);
}

// mode 0: start of a solve.  mode 1: pcamm_eval (a, b given).  mode 2: hooks that only need the
// view and w in slot 0.
__global__ void __launch_bounds__(CT)
k_begin(const Geom G, const CallOpts* __restrict__ opts, const SolveIn* __restrict__ in, SolveState* solves,
        SlotState* slots, LoopFlags* flags, int mode) {
    tl_begin(G.tl);
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
    if (threadIdx.x == 0) { flags->loop_cond = 0; flags->n_launch = 0; }
    tl_end(G.tl, TLK_BEGIN);
}

// The control step that follows a projection (then = THEN_INIT / THEN_TRIAL / THEN_EVAL): one block.
// In graph mode the decision it leaves in LoopFlags becomes the condition of the solve graph's
// while-node.
__global__ void __launch_bounds__(CT)
k_ctl_after_project(const Geom G, CtlBufs c, int then, cudaGraphConditionalHandle h_loop, int use_cond, int n_seq) {
    __shared__ CtlShared sh;
    tl_begin(G.tl);
    put_word(&sh.o, get_word((const CallOpts*)c.opts));
    __syncthreads();
    if (then == THEN_INIT) ctl_init_body(sh, G, c, n_seq);
    else if (then == THEN_TRIAL) ctl_trial_body(sh, G, c, n_seq);
    else ctl_eval_body(sh, G, c, 0);
    if (use_cond && threadIdx.x == 0) cudaGraphSetConditional(h_loop, c.flags->loop_cond);
    tl_end(G.tl, TLK_CTL_PROJ);
}

// The control step that follows a gradient pass (mode = GRAD_SOLVE / GRAD_EVAL): one block.  (The
// loop condition it may change is handed over by the step after the projection, which always
// follows in the same loop body.)
__global__ void __launch_bounds__(CT)
k_ctl_after_grad(const Geom G, CtlBufs c, int mode) {
    __shared__ CtlShared sh;
    tl_begin(G.tl);
    put_word(&sh.o, get_word((const CallOpts*)c.opts));
    __syncthreads();
    if (mode == GRAD_SOLVE) ctl_grad_body(sh, G, c);
    else ctl_eval_body(sh, G, c, 1);
    tl_end(G.tl, TLK_CTL_GRAD);
}

// After the closing residual pass: J at exit, final w into the output slots.
__global__ void __launch_bounds__(CT)
k_ctl_final(const Geom G, CtlBufs c, SlotState* out_slots, int n_seq) {
    __shared__ CtlShared sh;
    tl_begin(G.tl);
    const int B = c.opts->B;
    for (int b = 0; b < B; ++b) {
        SolveState& st = c.solves[b];
        double vj[1];
        load_partials<1, 4>(c.resid_part + (long long)b * c.resid_blocks, c.resid_blocks, 1, vj);
        reduce_partials<1>(sh, vj, 0);
        if (threadIdx.x != 0) continue;
        st.J = sh.res[0][0];
        if (isnan(st.J0)) st.J0 = st.J;
        if (st.iter <= TRACE_CAP) c.traces[b].J[st.iter] = st.J;
        SlotState& sl = out_slots[b];
        for (int k = 0; k < KMAX; ++k) sl.w[k] = k < G.K ? (float)st.w[k] : 0.f;
        sl.active = 1; sl.solve = b; sl.mu = 0.0; sl.J = st.J; sl.Sp = sl.Syp = 0.0;
    }
    if (threadIdx.x == 0) c.flags->n_launch += n_seq;
    tl_end(G.tl, TLK_FINAL);
}

// a-6.  One warp per (landmark, solve).  x(r) is the trilinear interpolation of the synthesised
// DVF of Eq. (1) at the off-grid point r, coordinates clamped to the grid (reading A13); the
// 8 (K+1) (tap, field) pairs are spread over the lanes.
__global__ void __launch_bounds__(32)
k_invert(const Geom G, const float* __restrict__ xbar, const float* __restrict__ u, const CallOpts* __restrict__ opts,
         const SolveState* __restrict__ solves, int M, const float* __restrict__ r0s, double* __restrict__ r_out) {
    tl_begin(G.tl);
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
    tl_end(G.tl, TLK_INVERT);
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

void launch_ctl_after_project(Seq& q, const Geom& G, const CtlBufs& c, int then, cudaGraphConditionalHandle h,
                              int use_cond, int n_before) {
    if (then == THEN_NONE) return;
    q.launch(k_ctl_after_project, dim3(1), dim3(CT), 0, G, c, then, h, use_cond, n_before + 1);
}

void launch_ctl_after_grad(Seq& q, const Geom& G, const CtlBufs& c, int mode) {
    if (mode == GRAD_NONE) return;
    q.launch(k_ctl_after_grad, dim3(1), dim3(CT), 0, G, c, mode);
}

void launch_ctl_final(Seq& q, const Geom& G, const CtlBufs& c, SlotState* out_slots, int n_seq) {
    q.launch(k_ctl_final, dim3(1), dim3(CT), 0, G, c, out_slots, n_seq);
}

void launch_invert(Seq& q, const Geom& G, const float* xbar, const float* u, const CtlBufs& c, int B, int M,
                   const float* r0, double* r_out) {
    if (M <= 0) return;
    q.launch(k_invert, dim3(M, B), dim3(32), 0, G, xbar, u, (const CallOpts*)c.opts, (const SolveState*)c.solves, M,
             r0, r_out);
}

}  // namespace pcamm
