// a-3 (second half) and a-5: the scalar side of the alternating algorithm, as device functions.
//
//   step 1 (Eq. 3):  w_{n+1} = w_n - mu_n dJ/dw_n, mu_n by Armijo's rule (L95)
//   step 2 (Eq. 4):  (a, b)^T = (Y^T Y)^-1 Y^T P f_{n+1},  Y = [y, 1]
//   stop:         ||dJ/dw|| small or max_iter reached
//
// Readings A7 (Armijo constants, first step = init_step_vox voxels rms, later 2 x the accepted
// step), A8 (initial (a, b) = fit at w0; singular fit), A9 are listed in DESIGN.md.
//
// A control step is run by ONE block (any multiple of 32 threads up to 1024; control.cu launches
// them as single-block kernels behind the projection / the gradient pass).  Thread 0 owns the state;
// all scalars are double.  The steps also decide whether the loop of the solve runs again
// (LoopFlags::loop_cond, handed to the graph's while-node by the kernel that ran the step).
//
// (Running the steps in the last block of the projector / gradient kernel instead was measured with
// the in-kernel timeline: the step takes as long there, every dependent read of other blocks'
// partial sums being a 0.6 us round trip, and carrying the control code slowed the streaming part
// of those kernels by 10 to 40 %.)
//
// The loop of a solve is flat: its body is {residual, gradient, warp, projection}.  A solve that is
// in the middle of a line search (trialing) skips the first two; one whose step has just been
// accepted takes them and starts the next line search in the same body.
#pragma once

#include "common.cuh"

namespace pcamm {

constexpr int CT = 256;   // threads of a control block

// Step 2, Eq. (4) as the 2x2 normal equations of Y = [y, 1].  false: y constant (reading A8).
__device__ __forceinline__ bool lsfit(double n, double Sy, double Syy, double Sp, double Syp, double* a, double* b) {
    const double det = Syy * n - Sy * Sy;
    if (!(det > 1e-12 * Syy * n)) return false;
    *a = (Syp * n - Sy * Sp) / det;
    *b = (Syy * Sp - Sy * Syp) / det;
    return true;
}

__device__ __forceinline__ void trial_w(const SolveState& st, int K, double mu, SlotState* sl) {
    for (int k = 0; k < K; ++k) sl->w[k] = (float)(st.w[k] - mu * st.g[k]);   // Eq. (3), candidate
    sl->mu = mu;
    sl->active = 1;
}

// Candidates st.t, st.t + 1, ... (at most C per round, fewer at the end of the backtrack budget) of
// the Armijo sequence mu0 beta^t into the solve's slots; st.mu is the step of candidate st.t and
// every later one follows by repeated multiplication, whatever the fan width, so that a fan of
// any width takes exactly the steps sequential backtracking would.
__device__ __forceinline__ void make_round(const SolveState& st, int K, const CallOpts& o, SlotState* slots_b) {
    double mu = st.mu;
    for (int cnd = 0; cnd < o.C; ++cnd) {
        if (st.t + cnd < o.max_backtracks) trial_w(st, K, mu, &slots_b[cnd]);
        else slots_b[cnd].active = 0;
        mu *= o.armijo_beta;
    }
}

// ---------------------------------------------------------------- the control block's tools
//
// What a control step costs is its chain of DEPENDENT global reads: a read of what other blocks have
// just written is a 0.6 us round trip (measured with the in-kernel timeline).
// So a step first issues every load it can need (options, state, all partial sums) in one batch,
// then reduces and computes out of shared memory, then stores.

struct CtlShared {
    double ex[CT / 32][8];     // per warp and quantity
    double res[2][8];          // totals of up to two sums
    SolveState st;             // the solve being worked on (thread 0 computes, the block copies)
    CallOpts o;
};

// word t of *src (a struct of at most CT words), to be stored with put_word after the other loads
template <class T>
__device__ __forceinline__ int get_word(const T* src) {
    static_assert(sizeof(T) % 4 == 0 && sizeof(T) / 4 <= CT, "one word per thread");
    return threadIdx.x < sizeof(T) / 4 ? __ldcg(reinterpret_cast<const int*>(src) + threadIdx.x) : 0;
}
template <class T>
__device__ __forceinline__ void put_word(T* dst, int w) {
    if (threadIdx.x < sizeof(T) / 4) reinterpret_cast<int*>(dst)[threadIdx.x] = w;
}

// Partial sums of NQ quantities held by this thread (records t, t + CT, ... of n): all its loads in
// flight together.  R = records per thread the registers hold (n <= R CT, else the rest follows in
// further batches).
template <int NQ, int R>
__device__ __forceinline__ void load_partials(const double* part, int n, int stride, double* v /* [NQ] */) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) v[q] = 0.0;
    for (int i0 = threadIdx.x; i0 < n; i0 += R * CT) {
        double a[R][NQ];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = i0 + r * CT;
#pragma unroll
            for (int q = 0; q < NQ; ++q) a[r][q] = i < n ? __ldcg(part + (long long)i * stride + q) : 0.0;   // written by other blocks
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
#pragma unroll
            for (int q = 0; q < NQ; ++q) v[q] += a[r][q];
        }
    }
}

// Block totals of NQ per-thread values into sh.res[which][0 .. NQ): lanes by butterfly, warps in
// index order (fixed order).  Ends with a barrier.
template <int NQ>
__device__ __forceinline__ void reduce_partials(CtlShared& sh, const double* v, int which) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();                       // ex may still be read from a previous call
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const double w = warp_sum(v[q]);
        if (lane == 0) sh.ex[wid][q] = w;
    }
    __syncthreads();
    if (threadIdx.x < NQ) {
        double t = 0.0;
#pragma unroll
        for (int i = 0; i < CT / 32; ++i) t += sh.ex[i][threadIdx.x];
        sh.res[which][threadIdx.x] = t;
    }
    __syncthreads();
}

__device__ __forceinline__ void publish(LoopFlags* flags, int loop_cond, int launched) {
    flags->loop_cond = loop_cond;
    flags->n_launch += launched;
}

// After the initial evaluation at w0: Sy, Syy, the first fit (reading A8), loop start.
// n_seq: kernels of the sequence this step closes (launch accounting).
__device__ __forceinline__ void ctl_init_body(CtlShared& sh, const Geom& G, const CtlBufs& c, int n_seq) {
    int any_running = 0;
    const int B = sh.o.B, C = sh.o.C;
    for (int b = 0; b < B; ++b) {
        const int s0 = b * C;
        double vy[2], vp[3];
        load_partials<2, 1>(c.ysum_part + (long long)b * c.ysum_blocks * 2, c.ysum_blocks, 2, vy);
        load_partials<3, 2>(c.proj_part + (long long)s0 * c.proj_blocks * 3, c.proj_blocks, 3, vp);
        reduce_partials<2>(sh, vy, 0);
        reduce_partials<3>(sh, vp, 1);
        if (threadIdx.x != 0) continue;
        SolveState& st = c.solves[b];
        const double Sy = sh.res[0][0], Syy = sh.res[0][1], Sp = sh.res[1][0], Syp = sh.res[1][1];
        st.Sy = Sy; st.Syy = Syy;
        c.slots[s0].Sp = Sp; c.slots[s0].Syp = Syp;
        c.slots[s0].active = 0;
        if (!isfinite(Sy) || !isfinite(Syy)) st.status = PCAMM_E_NONFINITE;
        else if (!lsfit((double)G.npix, Sy, Syy, Sp, Syp, &st.a, &st.b)) st.status = PCAMM_E_SINGULAR;
        st.acc_slot = s0;
        st.iter = 0;
        if (st.status == 0 && sh.o.max_iter <= 0) st.status = PCAMM_S_MAXITER;
        st.running = st.status == 0;
        st.trialing = 0;
        any_running |= st.running;
    }
    if (threadIdx.x == 0) publish(c.flags, any_running, n_seq);
}

// After the residual and gradient kernels of iteration n, for the solves that took them: J_n, g,
// stopping rule, first candidate(s).
__device__ __forceinline__ void ctl_grad_body(CtlShared& sh, const Geom& G, const CtlBufs& c) {
    int any_running = 0;
    const CallOpts& o = sh.o;
    const int K = G.K;
    for (int b = 0; b < o.B; ++b) {
        // the state and every partial sum in one batch of loads (whether or not this solve needs them)
        const int word = get_word(&c.solves[b]);
        double vj[1], vg[KMAX];
        load_partials<1, 4>(c.resid_part + (long long)b * c.resid_blocks, c.resid_blocks, 1, vj);
        load_partials<KMAX, 2>(c.grad_part + (long long)b * c.grad_blocks * KMAX, c.grad_blocks, KMAX, vg);
        __syncthreads();                               // sh.st of the previous solve has been copied out
        put_word(&sh.st, word);
        reduce_partials<1>(sh, vj, 0);
        reduce_partials<KMAX>(sh, vg, 1);
        SolveState& st = sh.st;
        const int running = st.running, trialing = st.trialing;
        __syncthreads();                               // every thread has read the state before thread 0 changes it
        if (running && trialing) any_running = 1;
        if (!(running && !trialing)) continue;                                            // uniform
        if (threadIdx.x == 0) {
            const int n = st.iter;
            st.Jn = sh.res[0][0];                                                         // Eq. (2)
            if (n == 0) st.J0 = st.Jn;
            double g2 = 0.0;
            for (int k = 0; k < K; ++k) {
                st.g[k] = 2.0 * sh.res[1][k];
                g2 += st.g[k] * st.g[k];
            }
            st.g2 = g2;
            const double gn = sqrt(g2);
            if (n < TRACE_CAP) { c.traces[b].J[n] = st.Jn; c.traces[b].gnorm[n] = gn; }
            if (gn <= o.grad_tol || !isfinite(gn)) {
                st.status = isfinite(gn) ? PCAMM_S_GRADTOL : PCAMM_E_NONFINITE;
                st.running = 0; st.trialing = 0;
            } else {
                st.mu = n == 0 ? o.init_step_vox * o.hmin_sqrtV / gn : 2.0 * st.mu_prev;  // reading A7
                st.t = 0;
                st.trialing = 1;
                make_round(st, K, o, &c.slots[b * o.C]);
                any_running = 1;
            }
        }
        __syncthreads();
        put_word(&c.solves[b], threadIdx.x < sizeof(SolveState) / 4 ? reinterpret_cast<const int*>(&sh.st)[threadIdx.x] : 0);
    }
    if (threadIdx.x == 0) c.flags->loop_cond = any_running;
}

// After warp + projection of the candidate(s): Armijo's inequality, Eq. (3) update, Eq. (4) fit.
__device__ __forceinline__ void ctl_trial_body(CtlShared& sh, const Geom& G, const CtlBufs& c, int n_seq) {
    int any_running = 0;
    const CallOpts& o = sh.o;
    const int K = G.K;
    for (int b = 0; b < o.B; ++b) {
        // the state and the first candidate's sums in one batch of loads
        const int word = get_word(&c.solves[b]);
        double vp[3];
        load_partials<3, 2>(c.proj_part + (long long)b * o.C * c.proj_blocks * 3, c.proj_blocks, 3, vp);
        const double mu_first = threadIdx.x == 0 ? __ldcg(&c.slots[b * o.C].mu) : 0.0;
        __syncthreads();
        put_word(&sh.st, word);
        reduce_partials<3>(sh, vp, 0);
        SolveState& st = sh.st;                        // thread 0 writes it, the block copies it back
        const int trialing = st.trialing, running = st.running, n = st.iter, t0 = st.t;
        double mu_last = st.mu;
        __syncthreads();                               // every thread has read the state before thread 0 changes it
        if (!trialing) { any_running |= running; continue; }                              // uniform
        int acc = -1;
        double acc_mu = 0.0, acc_Sp = 0.0, acc_Syp = 0.0;
        // the round's candidates t0 .. t0 + C - 1 have been evaluated: the first that passes is
        // the one sequential backtracking would have accepted (reading A7)
        int n_cand = o.max_backtracks - t0;
        if (n_cand > o.C) n_cand = o.C;
        for (int cnd = 0; cnd < n_cand; ++cnd) {
            const int s = b * o.C + cnd;
            if (cnd > 0) {
                load_partials<3, 2>(c.proj_part + (long long)s * c.proj_blocks * 3, c.proj_blocks, 3, vp);
                reduce_partials<3>(sh, vp, 0);
            }
            if (threadIdx.x != 0) continue;
            const double mu_s = cnd == 0 ? mu_first : c.slots[s].mu;
            const double Sp = sh.res[0][0], Syp = sh.res[0][1], Js = sh.res[0][2];
            c.slots[s].Sp = Sp; c.slots[s].Syp = Syp; c.slots[s].J = Js;
            if (acc < 0 && Js <= st.Jn - o.armijo_c * mu_s * st.g2) {                     // Armijo (L95)
                acc = s; acc_mu = mu_s; acc_Sp = Sp; acc_Syp = Syp;
                st.t = t0 + cnd;
            }
            c.slots[s].active = 0;
            mu_last = mu_s;
        }
        if (threadIdx.x == 0) {
            if (acc >= 0) {
                const double mu = acc_mu;
                for (int k = 0; k < K; ++k) st.w[k] -= mu * st.g[k];                      // Eq. (3)
                st.mu_prev = mu;
                st.acc_slot = acc;
                if (n < TRACE_CAP) { c.traces[b].mu[n] = mu; c.traces[b].bt[n] = st.t; }
                st.iter = n + 1;
                st.trialing = 0;
                if (!lsfit((double)G.npix, st.Sy, st.Syy, acc_Sp, acc_Syp, &st.a, &st.b)) {   // Eq. (4)
                    st.status = PCAMM_E_SINGULAR; st.running = 0;
                } else if (st.iter >= o.max_iter) { st.status = PCAMM_S_MAXITER; st.running = 0; }
            } else {
                st.t = t0 + n_cand;
                st.mu = mu_last * o.armijo_beta;
                if (st.t >= o.max_backtracks) {
                    if (n < TRACE_CAP) { c.traces[b].mu[n] = 0.0; c.traces[b].bt[n] = st.t; }
                    st.status = PCAMM_S_LINESEARCH;
                    st.running = 0; st.trialing = 0;
                } else make_round(st, K, o, &c.slots[b * o.C]);
            }
            any_running |= st.running;
        }
        __syncthreads();
        put_word(&c.solves[b], threadIdx.x < sizeof(SolveState) / 4 ? reinterpret_cast<const int*>(&sh.st)[threadIdx.x] : 0);
    }
    if (threadIdx.x == 0) publish(c.flags, any_running, n_seq);
}

// pcamm_eval: stage 0 after the projection (J at the given (a, b), fit of Eq. 4), stage 1 after
// the gradient.
__device__ __forceinline__ void ctl_eval_body(CtlShared& sh, const Geom& G, const CtlBufs& c, int stage) {
    const int B = sh.o.B, C = sh.o.C;
    for (int b = 0; b < B; ++b) {
        SolveState& st = c.solves[b];
        if (stage == 0) {
            double vy[2], vp[3];
            load_partials<2, 1>(c.ysum_part + (long long)b * c.ysum_blocks * 2, c.ysum_blocks, 2, vy);
            load_partials<3, 2>(c.proj_part + (long long)b * C * c.proj_blocks * 3, c.proj_blocks, 3, vp);
            reduce_partials<2>(sh, vy, 0);
            reduce_partials<3>(sh, vp, 1);
            if (threadIdx.x != 0) continue;
            st.Sy = sh.res[0][0]; st.Syy = sh.res[0][1];
            st.J = sh.res[1][2];
            st.fit_a = st.fit_b = nan("");
            lsfit((double)G.npix, st.Sy, st.Syy, sh.res[1][0], sh.res[1][1], &st.fit_a, &st.fit_b);
            st.acc_slot = b * C;
        } else {
            double vj[1], vg[KMAX];
            load_partials<1, 4>(c.resid_part + (long long)b * c.resid_blocks, c.resid_blocks, 1, vj);
            load_partials<KMAX, 2>(c.grad_part + (long long)b * c.grad_blocks * KMAX, c.grad_blocks, KMAX, vg);
            reduce_partials<1>(sh, vj, 0);
            reduce_partials<KMAX>(sh, vg, 1);
            if (threadIdx.x != 0) continue;
            st.Jn = sh.res[0][0];
            for (int k = 0; k < G.K; ++k) st.g[k] = 2.0 * sh.res[1][k];
        }
    }
}

}  // namespace pcamm
