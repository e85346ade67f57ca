/* pcamm.h -- C ABI of the B200 per-projection PCA lung-motion solve.
 *
 * Method: Li, Jia, Lewis, Gu, Folkerts, Men, Jiang, "Real-time volumetric image reconstruction and
 * 3D tumor localization based on a single x-ray projection image for lung cancer radiotherapy"
 * (PAPER.md).  Citations below are PAPER.md line numbers plus the section / equation they fall in;
 * "reading A<n>" refers to the list of readings in DESIGN.md.
 *
 * The library minimises (section 2.2, Eq. 2)
 *
 *        J(w, a, b) = || P_theta f(x, f0) - a y - b 1 ||_2^2     s.t.   x = xbar + U w
 *
 * by the alternating algorithm of PAPER.md:L84-95 (Eq. 3: gradient step on w with Armijo's rule,
 * Eq. 4: closed-form (a, b)), and localises landmarks through the fixed-point inverse of the
 * pull-back DVF (section 2.3).  Every step runs in CUDA kernels for sm_100a;
 * there is no CPU fallback.  All calls are blocking with respect to their host outputs.
 *
 * Conventions
 *   volume   [nz][ny][nx] float32, x fastest; voxel (i,j,k) centre in world mm is
 *            (cx + (i-(nx-1)/2) hx, cy + (j-(ny-1)/2) hy, cz + (k-(nz-1)/2) hz); z = rotation axis.
 *   fields   DVFs are pull-back, in mm: f(r) = f0(r + x(r)) (reading A1), stored
 *            planar [3][nz][ny][nx] (component 0 = x).
 *   detector [nv][nu] float32, u fastest.  At gantry angle theta the source is
 *            S = sad (cos theta, sin theta, 0), the detector centre C = -(sdd-sad)(cos theta, sin theta, 0),
 *            u^ = (-sin theta, cos theta, 0), v^ = (0,0,1); pixel (iu,iv) centre is
 *            C + (iu-(nu-1)/2+off_u) pu u^ + (iv-(nv-1)/2+off_v) pv v^   (reading A14).
 *   P        Siddon's exact radiological path, one ray per pixel centre: p_i = sum_j l_ij f_j with
 *            l_ij the length in mm of the source->pixel segment inside voxel box j (reading A3);
 *            P^T is the transpose of the same l_ij (reading A4).
 *   *_dev    CUDA device pointers (caller-owned);  *_host  host pointers (caller-owned).
 *   stream   a cudaStream_t passed as void* (NULL = default stream).
 *
 * Return codes: 0 OK; < 0 hard error (PCAMM_E_*); > 0 soft status of a solve (PCAMM_S_*), also
 * stored in pcamm_info.status.  No exception crosses the ABI.  pcamm_last_error() returns a
 * thread-local message for the last hard error on the calling thread.
 */
#ifndef PCAMM_H
#define PCAMM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PCAMM_KMAX 8            /* maximum number of eigenvector fields K */
#define PCAMM_MAX_BACKTRACKS 16 /* upper bound on pcamm_opts.max_backtracks */

#define PCAMM_OK 0
#define PCAMM_E_INVALID (-1)    /* invalid argument / size mismatch / unsupported geometry */
#define PCAMM_E_CUDA (-2)       /* CUDA runtime error (message in pcamm_last_error) */
#define PCAMM_E_NOMEM (-3)      /* device allocation failed */
#define PCAMM_E_NONFINITE (-4)  /* non-finite value in an input checked at this call */
#define PCAMM_E_SINGULAR (-5)   /* intensity fit singular: y is constant (reading A8) */
#define PCAMM_S_MAXITER 1       /* stopped on max_iter */
#define PCAMM_S_GRADTOL 2       /* stopped on ||g||_2 <= grad_tol */
#define PCAMM_S_LINESEARCH 3    /* no candidate step satisfied Armijo's inequality */

typedef struct pcamm_model pcamm_model; /* opaque; immutable after create except for its scratch */

typedef struct {
    int32_t nx, ny, nz;   /* volume size, x fastest */
    float hx, hy, hz;     /* voxel size, mm */
    float cx, cy, cz;     /* world position of the volume centre, mm (isocentre = origin) */
    int32_t K;            /* number of eigenvector fields, 1..PCAMM_KMAX (Eq. 1) */
    int32_t nu, nv;       /* detector size, u fastest */
    float pu, pv;         /* pixel pitch, mm */
    float sad, sdd;       /* source-axis and source-detector distance, mm */
    float off_u, off_v;   /* detector offset in pixels */
    int32_t max_batch;    /* largest B of pcamm_reconstruct_batch (>= 1); scratch is sized for it */
    int32_t max_candidates; /* 1, or >= opts.max_backtracks to allow batched_linesearch */
    int32_t field_storage;  /* 0 (default): x-bar and u_k kept in float32.  1: u_k kept in
                               half precision, each scaled by a power of two so that its entries keep 11
                               significant bits; x-bar stays float32.  Halves the dominant HBM stream of the
                               warp and gradient kernels; the model then IS the rounded one (every step,
                               the landmark inversion included, uses the rounded u_k; pcamm_model_fields
                               returns them).  Needs nx % 8 == 0. */
    int32_t tile_skipping;  /* the warp and gradient kernels skip, exactly, the tiles of the volume that can only
                               see zeros / constant cells of f0 (reading B8): 0 (default) where the
                               volume has tiles enough per SM to win back the flags' set-up (a few dependent
                               loads per launch), 1 always, 2 never */
    int32_t projector;      /* discretisation of P (PAPER.md:L82 says only "projection matrix"): 0 (default)
                               Siddon's exact radiological path (reading A3); 1 fixed-step trilinear ray
                               marching (reading C1): p_i = d_i sum_m (T f)(sample m), the
                               midpoint rule on M_i = ceil(L_i / step) equal steps d_i = L_i / M_i over the part
                               of the ray inside the box spanned by the voxel centres, T f the trilinear
                               interpolant; P^T is the exact transpose (scattered with atomic adds: results
                               reproducible to rounding, not bitwise).  pcamm_traverse needs projector 0 */
    float ray_step_vox;     /* projector 1: nominal step in units of the smallest voxel edge; 0 = default 0.5 */
} pcamm_geometry;

typedef struct {
    int32_t max_iter;       /* default 10 */
    float grad_tol;         /* stop if ||g||_2 <= grad_tol; default 0 = off */
    float armijo_c;         /* default 1e-4 (reading A7) */
    float armijo_beta;      /* default 0.5 */
    int32_t max_backtracks; /* default 8 */
    float init_step_vox;    /* first trial moves the DVF by this many voxels rms; default 1 (A7) */
    int32_t batched_linesearch; /* 0: sequential backtracking; 1: evaluate all max_backtracks candidates
                                   at once and take the largest passing step (config C3); F >= 2:
                                   F candidates per pass, the next F if none passes.  The accepted
                                   step is the same in every mode; needs max_candidates >= the fan */
    int32_t inv_max_iter;   /* default 50 (reading A13) */
    float inv_tol_mm;       /* default 1e-4 */
    int32_t loop_mode;      /* 0 (default): the whole solve is one CUDA graph with device-side
                               while-loops, no host round trip per trial;
                               1: the host drives the same kernels and reads one status word per
                               step (debug aid; same arithmetic) */
} pcamm_opts;

typedef struct {
    int32_t iters, status;
    double J0, J;           /* cost after the initial intensity fit / at exit (Eq. 2) */
    double a, b;            /* intensity fit at exit (Eq. 4) */
    /* optional traces, caller-allocated host arrays or NULL:
       J_trace[max_iter+1], gnorm_trace[max_iter], mu_trace[max_iter], backtracks_trace[max_iter] */
    double* J_trace;
    double* gnorm_trace;
    double* mu_trace;
    int32_t* backtracks_trace;
} pcamm_info;

/* Fills *opts with the defaults listed above. */
void pcamm_default_opts(pcamm_opts* opts);

/* Build a model: copies f0 [nz][ny][nx], the mean DVF [3][nz][ny][nx] and the K eigenvector fields
 * [K][3][nz][ny][nx] (mm; Eq. 1) into library-owned device memory, allocates all
 * scratch for geometry->max_batch x max_candidates evaluations, and stores the n_landmarks
 * reference positions [M][3] (mm).  The caller may free its inputs on return.
 * Geometry restrictions (else PCAMM_E_INVALID): the source and the detector plane lie outside
 * the volume's bounding sphere, and a ray moves at most one voxel in z per voxel along its
 * dominant in-plane axis (true for any circular cone-beam geometry with sane voxel aspect). */
int pcamm_model_create(const pcamm_geometry* geometry, const float* f0_dev, const float* mean_dvf_dev,
                       const float* eig_dvf_dev, int32_t n_landmarks, const float* landmarks_mm_host,
                       void* stream, pcamm_model** out);
void pcamm_model_destroy(pcamm_model* model);

/* The motion model as the solve uses it, in mm and in model_create's layout: mean_dvf_out_dev
 * [3][nz][ny][nx], eig_dvf_out_dev [K][3][nz][ny][nx].  With field_storage = 0 these are the
 * inputs again (to float rounding of x / h * h); with field_storage = 1 the u_k are the values the
 * stored halves stand for. */
int pcamm_model_fields(pcamm_model* model, float* mean_dvf_out_dev, float* eig_dvf_out_dev, void* stream);

/* The per-projection solve (sections 2.2-2.3).  y_dev [nv][nu] is the measured
 * projection, w_init_host [K] the start (the previous frame's w).  Outputs:
 * w_out_host [K]; volume_out_dev [nz][ny][nx] = f(w) or NULL; landmarks_out_host [M][3] mm or
 * NULL; info or NULL.  Returns a PCAMM_S_* status or a PCAMM_E_* error. */
int pcamm_reconstruct(pcamm_model* model, const float* y_dev, float angle_rad, const float* w_init_host,
                      const pcamm_opts* opts, float* w_out_host, float* volume_out_dev,
                      float* landmarks_out_host, pcamm_info* info, void* stream);

/* Same, with the measured projection in host memory: the host->device copy of y is part of the
 * call (used for end-to-end timing). */
int pcamm_reconstruct_host(pcamm_model* model, const float* y_host, float angle_rad,
                           const float* w_init_host, const pcamm_opts* opts, float* w_out_host,
                           float* volume_out_dev, float* landmarks_out_host, pcamm_info* info,
                           void* stream);

/* B independent solves in flight (different angles, projections and starts), advanced in lock
 * step so that every pass over the K+1 vector fields serves all B of them.  Arrays are the
 * single-solve ones with a leading [B]; info is an array of B or NULL.  Returns 0 when every
 * solve ended with a soft status, else the first hard error. */
int pcamm_reconstruct_batch(pcamm_model* model, int32_t B, const float* y_dev, const float* angles_rad_host,
                            const float* w_init_host, const pcamm_opts* opts, float* w_out_host,
                            float* volumes_out_dev, float* landmarks_out_host, pcamm_info* info,
                            void* stream);

/* ---- PCA motion model from training DVFs ----
 *
 * PAPER.md:L63-69 (section 2.1, Eq. 1): x(t) ~ xbar + sum_k u_k w_k(t) with xbar "the sample mean
 * vector" and u_k the "eigenvectors corresponding to the largest eigenvalues"; the
 * samples are the DVFs of the training phases relative to the reference phase.
 * dvfs_dev [N][n_per_sample] float32 (n_per_sample = 3 nx ny nz for [3][nz][ny][nx] fields), N in
 * [2, PCAMM_PCA_MAX_SAMPLES], 1 <= K <= min(PCAMM_KMAX, N - 1).  Outputs, in the layout
 * pcamm_model_create takes: mean_out_dev [n_per_sample] = (1/N) sum_i D_i; eig_out_dev
 * [K][n_per_sample], unit L2 norm each, u_k = sum_i v_ik (D_i - xbar) / sqrt(lambda_k) for the
 * eigenpairs (lambda_k, v_k) of the N x N scatter matrix <D_i - xbar, D_j - xbar> (no 1/(N-1)),
 * lambda descending (reading A12).  Sign: u_k . (D_sign_ref - xbar) >= 0 (sign_ref = -1: sample
 * N/2, the end-of-inhale phase of the recipe); if that product is exactly 0 the training
 * coefficient of largest magnitude is positive (reading B10).  Host outputs or NULL:
 * eigenvalues_out_host [N] (double), coeffs_out_host [N][K] = u_k . (D_i - xbar) (double).
 * Errors: PCAMM_E_SINGULAR if lambda_K <= 1e-6 lambda_1 (below what float32 products resolve),
 * PCAMM_E_NONFINITE for non-finite samples.
 * pass_ms_out_host [2] or NULL: device time in ms of the two passes over the samples (scatter
 * matrix; fields), CUDA events on `stream` (for bench.py).  Blocking. */
#define PCAMM_PCA_MAX_SAMPLES 16
int pcamm_pca_fit(int64_t n_per_sample, int32_t N, int32_t K, const float* dvfs_dev, int32_t sign_ref,
                  float* mean_out_dev, float* eig_out_dev, double* eigenvalues_out_host,
                  double* coeffs_out_host, float* pass_ms_out_host, void* stream);

/* ---- frame stream: consecutive projections of one treatment ----
 *
 * PAPER.md:L141 (section 4): "We initialized the PCA coefficients to those at its previous frame
 * considering the high-frequency image acquisition (6 Hz) relative to breathing."
 * PAPER.md:L154 (section 5): "we can also use the predicted PCA coefficients from previous
 * histories to serve as the initial guess for optimization."  The paper names no predictor;
 * reading B9: the start of frame n is the polynomial of degree `order` through the last
 * order + 1 solved frames (their time stamps t and results w), evaluated at the new frame's t:
 *   order 0 = the previous frame's w (L141); 1 = linear; 2 = quadratic extrapolation;
 *   PCAMM_PREDICT_NONE = every frame starts from w0.
 * With fewer solved frames than order + 1 the degree drops to what the history allows; the first
 * frame starts from w0; equal time stamps among the frames used fall back to order 0.  The
 * prediction is K scalars of host arithmetic in double, rounded to float (w_init is float).
 * A fixed-angle sequence (fluoroscopy: "the projection matrix will be constant")
 * is the same call with a constant angle_rad. */
#define PCAMM_PREDICT_NONE (-1)
#define PCAMM_PREDICT_MAX_ORDER 2

/* The predictor alone (host arithmetic, no device): history of n frames, oldest first, time stamps
 * t_host [n] and results w_host [n][K]; w0_host [K] or NULL (= 0); w_pred_host [K]. */
int pcamm_predict_w(int32_t order, int32_t K, int32_t n, const double* t_host, const float* w_host,
                    const float* w0_host, double t, float* w_pred_host);

typedef struct pcamm_frames pcamm_frames; /* opaque; holds the history, refers to (does not own) the model */

/* w0_host [K] or NULL (= 0).  The model must outlive the stream. */
int pcamm_frames_create(pcamm_model* model, int32_t order, const float* w0_host, pcamm_frames** out);
void pcamm_frames_destroy(pcamm_frames* frames);
/* Forget the history (the next frame starts from w0 again). */
int pcamm_frames_reset(pcamm_frames* frames);
/* Number of solved frames held (at most PCAMM_PREDICT_MAX_ORDER + 1 are kept). */
int32_t pcamm_frames_count(const pcamm_frames* frames);
/* The start the next pcamm_frames_push at time t would use: w_pred_host [K]. */
int pcamm_frames_predict(const pcamm_frames* frames, double t, float* w_pred_host);
/* Solve the frame measured at time t (any unit, non-decreasing) from the predicted start and
 * append (t, w) to the history.  y [nv][nu] is a device pointer, or a host pointer if y_on_host
 * != 0 (then the host->device copy is part of the call).  w_init_out_host [K] or NULL receives
 * the start that was used; the other arguments are pcamm_reconstruct's.  A hard error leaves
 * the history as it was. */
int pcamm_frames_push(pcamm_frames* frames, const float* y, int32_t y_on_host, float angle_rad, double t,
                      const pcamm_opts* opts, float* w_out_host, float* w_init_out_host, float* volume_out_dev,
                      float* landmarks_out_host, pcamm_info* info, void* stream);

/* ---- function-level hooks (parity tests; reading A16 level i) ---- */

/* f = warp(f0, xbar + U w): Eq. 1 + trilinear pull-back. */
int pcamm_warp(pcamm_model* model, const float* w_host, float* volume_out_dev, void* stream);

/* p = P_theta f for a caller-supplied volume [nz][ny][nx] (Eq. 2). */
int pcamm_project(pcamm_model* model, const float* volume_dev, float angle_rad, float* proj_out_dev,
                  void* stream);

/* B = P_theta^T r for a caller-supplied detector image r [nv][nu]: backprojection onto the voxel
 * grid, [nz][ny][nx] (reading A4).  Test hook for the adjoint identity; the solve
 * itself never materialises this volume. */
int pcamm_backproject(pcamm_model* model, const float* r_dev, float angle_rad, float* volume_out_dev,
                      void* stream);

/* One evaluation at (w, a, b): p = P f(w) (written to proj_out_dev if not NULL),
 * J = ||p - a y - b||^2 (Eq. 2), grad[k] = dJ/dw_k, and the least-squares
 * (a, b) of Eq. 4 for this p in ab_fit_out[2] (or NULL). */
int pcamm_eval(pcamm_model* model, const float* y_dev, float angle_rad, const float* w_host, float a,
               float b, double* J_out, double* grad_out, double* ab_fit_out, float* proj_out_dev,
               void* stream);

/* Ordered voxel list and intersection lengths (mm) of one ray, source side first, segments of
 * zero length dropped (reading A22).  Runs the projector's own traversal code on the device. */
int pcamm_traverse(pcamm_model* model, float angle_rad, int32_t iu, int32_t iv, int32_t cap,
                   int32_t* ijk_out_host, float* len_out_host, int32_t* n_out, void* stream);

/* Landmark positions r with r + x(r) = r0 by r_{m+1} = r0 - x(r_m) (A13). */
int pcamm_localise(pcamm_model* model, const float* w_host, int32_t inv_max_iter, float inv_tol_mm,
                   float* landmarks_out_host, void* stream);

/* Timing hook for bench.py: launches the given kernel of one evaluation `reps` times on `stream`
 * with the model's scratch (inputs taken as they stand from the last pcamm_eval) and returns the
 * average device time per launch in milliseconds, measured with CUDA events on that stream.
 * which: 0 = warp (a-1), 1 = project (a-2), 2 = gradient (a-4). */
int pcamm_time_kernel(pcamm_model* model, int32_t which, int32_t reps, float* ms_out, void* stream);

/* For pcamm_time_kernel: makes the first nslots (<= max_batch * max_candidates) trial slots active
 * with the coefficients w_host [nslots][K], so that the warp and projection kernels are timed over
 * as many candidate steps per launch as the solve evaluates per line-search pass.  Call it after
 * pcamm_eval (which leaves one slot active and resets this to 1). */
int pcamm_time_slots(pcamm_model* model, int32_t nslots, const float* w_host, void* stream);

/* What the two streaming kernels really loaded (reading B8: tiles whose stencils can only see zeros
 * of f0 / constant cells are skipped, exactly).  out[0], out[1] = field tiles loaded by the warp and
 * by the gradient kernel in all launches since the counters were last reset (one tile = out[3]
 * voxels, all 3(K+1) field planes); out[2] = tiles of the whole volume (0: the generic kernels are
 * in use, which visit everything and count nothing).  With gradient records (pcamm_tune
 * "grad_records", the default for a single solve) the gradient loads no field tiles: out[4] = records
 * its gather went through, out[5] = records the warp kernel wrote (48 bytes each), same launches.
 * reset != 0 clears the counters. */
int pcamm_tile_counts(pcamm_model* model, int32_t reset, int64_t* out /* [6] */, void* stream);

/* Measurement knob (process-wide; set it before pcamm_model_create: a model's solve graphs keep the
 * launch configuration they were built with).  Returns PCAMM_E_INVALID for an unknown name.
 *   "project_chunks_per_segment"  chunks of the projector's march a block works through
 *                                 (0 = automatic, the default);
 *   "project_scan_slabs"          slabs per scan of the projector: 1, 2 or 4 (0 = automatic);
 *   "grad_records"                0: the gradient of a single solve makes its own pass over the K+1 fields
 *                                 (1, the default: in models created with max_candidates <= 2 whose
 *                                 records (48 bytes per voxel, trial slot and solve in flight) fit into
 *                                 three fifths of the free device memory, the warp kernel leaves records of
 *                                 the voxels whose interpolation cell is not constant and the gradient is
 *                                 a gather over them);
 *   "grad_aos"                    0: the gather over the records reads u_k from the field planes (1, the
 *                                 default: models with records also hold u_1 .. u_K with a voxel's 3 K values
 *                                 side by side, 4 ceil(3 K / 4) floats per voxel, which the gather reads);
 *   "pdl"                         0: plain kernel -> kernel edges in the solve graphs (1, the default:
 *                                 programmatic dependent launch, the next kernel's blocks are launched
 *                                 while the previous kernel drains and wait for its completion on the
 *                                 device; same order of memory effects);
 *   "static_passes"               line-search passes laid out as plain kernel nodes in front of the solve
 *                                 graph's while-loop (the loop takes the passes beyond): -1, the default,
 *                                 = min(max_iter, 16) when opts.grad_tol = 0 (a solve then takes max_iter
 *                                 iterations of at least one pass each) and 0 otherwise; 0 .. 64 forces it;
 *   "timeline"                    1: models created from now on record, inside their kernels, the
 *                                 start and end of every kernel of a solve (pcamm_timeline). */
int pcamm_tune(const char* name, int32_t value);

/* Kernel timeline of the model's last solve (timeline knob): per kernel, in launch order, its kind
 * (0 ysums, 1 begin, 2 view tables, 3 warp, 4 project, 5 control after a projection, 6 residual,
 * 7 gradient, 8 control after the gradient, 9 unused, 10 final, 11 tumour inversion) and
 * its start (first block in) and end (last block out) in microseconds on the device's global timer,
 * relative to the first kernel's start.  *n_out = kernels recorded (at most 2048; arrays filled up
 * to cap). */
int pcamm_timeline(pcamm_model* model, int32_t cap, int32_t* kind_out, double* start_us_out, double* end_us_out,
                   int32_t* n_out, void* stream);

/* Number of kernels launched by this library on the calling thread since the last reset
 * (host-side launch count; kernels inside device-side loops are counted from the device's
 * iteration counters after each solve). */
int64_t pcamm_launch_count(int32_t reset);

/* a-3 for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the intensity fit of Eq. 4 and the cost of Eq. 2
 * of one projection pair, with no model and no allocation of any kind: every
 * intermediate lives in one file-scope device array of 41 216 bytes (csrc/noalloc.cu), which every
 * GPU that loads the library holds until the process exits.
 *   p_dev, y_dev  [npix] float, device: the computed and the measured projection (any layout, the
 *                 same for both); read only
 *   npix          1 .. PCAMM_STATIC_MAX_PIXELS; beyond that PCAMM_E_INVALID (the array holds no more)
 *   out_dev       [8] double, device, owned by the caller: a, b (Eq. 4), J = sum (p - a y - b)^2 at
 *                 that (a, b), sum p, sum y, sum y^2, sum y p, status (PCAMM_OK, PCAMM_E_SINGULAR: y is
 *                 constant, then a = b = 0; PCAMM_E_NONFINITE: a sum is not finite) as a double
 * Asynchronous on `stream` (one memset and two kernels; nothing is synchronised, nothing read back):
 * out_dev is valid once the stream has reached the end of the call.  Sums in double in a fixed
 * order: the same inputs give the same bits.  The scratch array is shared by every call on a device
 * and keeps the last call's contents; what must start at zero is cleared on the stream at the start
 * of each call.  Calls that overlap on the GPU (different streams or threads, same device) race on it
 * and give wrong results: serialise them.  Returns PCAMM_OK, PCAMM_E_INVALID (NULL argument, size) or
 * PCAMM_E_CUDA. */
#define PCAMM_STATIC_MAX_PIXELS (1 << 22)
int pcamm_fit_cost_static(const float* p_dev, const float* y_dev, int64_t npix, double* out_dev, void* stream);

const char* pcamm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PCAMM_H */
