// C ABI of libpcamm (include/pcamm.h): model life cycle, the solve as one CUDA graph with
// device-side while-loops (or driven from the host, opts.loop_mode = 1), and the function-level
// hooks.  Argument marshalling and kernel sequencing only: every step of the hot path runs in the
// kernels of warp.cu, project.cu, gradient.cu and control.cu.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <string>
#include <vector>

#include "internal.h"

namespace pcamm {

static thread_local std::string g_error;
static thread_local long long g_launches = 0;
int g_timeline = 0;
constexpr int STATIC_PASSES_MAX = 16;
int g_static_passes = -1; // pcamm_tune "static_passes": -1 automatic (get_graph's caller)
int g_pdl = 1;            // pcamm_tune "pdl": programmatic kernel -> kernel edges in the solve graphs built from then on
int g_grad_aos = 1;       // pcamm_tune "grad_aos": 0 = the gather over the records reads u_k from the planes
int g_grad_records = 1;   // pcamm_tune "grad_records": 0 = the gradient of a single solve makes its own pass over the fields

void set_error(const std::string& msg) { g_error = msg; }
void count_launch(long long n) { g_launches += n; }

namespace {

struct GraphRec {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
};

__global__ void k_count_nonfinite(const float* __restrict__ a, long long n, unsigned long long* count) {
    unsigned long long c = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        if (!isfinite(a[i])) ++c;
    if (c) atomicAdd(count, c);
}

// Fields to voxel units, once at create: plane p holds component p % 3, divided by h of that
// axis (IEEE division: a displacement of exactly n voxels stays exactly n).
__global__ void k_fields_to_voxel_units(float* __restrict__ fields, long long V, int planes, float hx, float hy, float hz) {
    const long long n = V * planes;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int c = (int)((i / V) % 3);
        fields[i] = __fdiv_rn(fields[i], c == 0 ? hx : (c == 1 ? hy : hz));
    }
}

// u_1 .. u_K, planar [3 K][V], to [V][pitch] with a voxel's 3 K values side by side (FieldStream::u_aos).
__global__ void k_u_to_aos(const float* __restrict__ u, long long V, int K, int pitch, float* __restrict__ out) {
    const long long n = V * pitch;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const long long v = i / pitch;
        const int c = (int)(i - v * pitch);
        out[i] = c < 3 * K ? u[(long long)c * V + v] : 0.f;
    }
}

// f0 with a border of two zero voxels on every side (trilinear.cuh); out is zeroed beforehand.
__global__ void k_pad_f0(const float* __restrict__ f0, Geom G, float* __restrict__ out) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < G.V; i += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(i % G.nx), y = (int)((i / G.nx) % G.ny), z = (int)(i / ((long long)G.nx * G.ny));
        out[((long long)(z + 2) * G.fny + (y + 2)) * G.fnx + (x + 2)] = f0[i];
    }
}

// Reduced-precision storage.  max |u_k| per eigenvector field (bit pattern of a
// non-negative float orders like an unsigned integer).
__global__ void k_field_absmax(const float* __restrict__ u, long long n_per_k, int K, unsigned int* __restrict__ out) {
    for (int k = 0; k < K; ++k) {
        float mx = 0.f;
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_per_k; i += (long long)gridDim.x * blockDim.x)
            mx = fmaxf(mx, fabsf(u[(long long)k * n_per_k + i]));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        if ((threadIdx.x & 31) == 0) atomicMax(out + k, __float_as_uint(mx));
    }
}
// u16 = half(u * scale[k]); u is overwritten by the value the half stands for, u16 / scale[k]
// (exact in float), so that every other reader of the fields sees what the streaming kernels see.
__global__ void k_quantise_fields(float* __restrict__ u, __half* __restrict__ u16, long long n_per_k, int K,
                                  FieldScale scale, FieldScale inv) {
    const long long n = n_per_k * K;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int k = (int)(i / n_per_k);
        const __half h = __float2half_rn(u[i] * scale.inv[k]);
        u16[i] = h;
        u[i] = __half2float(h) * inv.inv[k];
    }
}
// max |value| of every plane of the fields (voxel units).
__global__ void k_plane_absmax(const float* __restrict__ fields, long long V, int planes, unsigned int* __restrict__ out) {
    for (int p = 0; p < planes; ++p) {
        float mx = 0.f;
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += (long long)gridDim.x * blockDim.x)
            mx = fmaxf(mx, fabsf(fields[(long long)p * V + i]));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        if ((threadIdx.x & 31) == 0) atomicMax(out + p, __float_as_uint(mx));
    }
}

// Fields as the solve uses them, back in mm.
__global__ void k_fields_to_mm(const float* __restrict__ fields, long long V, int planes, float hx, float hy, float hz,
                               float* __restrict__ out) {
    const long long n = V * planes;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int c = (int)((i / V) % 3);
        out[i] = fields[i] * (c == 0 ? hx : (c == 1 ? hy : hz));
    }
}

}  // namespace

bool make_field_map(const Geom& G, const void* fields, int planes, int tz, int elem_bytes, CUtensorMap* out,
                    std::string* why) {
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    const cuuint64_t eb = (cuuint64_t)elem_bytes;
    if ((G.nx * eb) % 16 != 0) { if (why) *why = "a row of nx elements is not a multiple of 16 bytes"; return false; }
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        if (why) *why = "cuTensorMapEncodeTiled is not available";
        return false;
    }
    const cuuint64_t dims[4] = {(cuuint64_t)G.nx, (cuuint64_t)G.ny, (cuuint64_t)G.nz, (cuuint64_t)planes};
    const cuuint64_t strides[3] = {(cuuint64_t)G.nx * eb, (cuuint64_t)G.nx * G.ny * eb, (cuuint64_t)G.V * eb};
    const cuuint32_t box[4] = {(cuuint32_t)TX, 1u, (cuuint32_t)tz, (cuuint32_t)planes};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUresult r = ((EncodeFn)fn)(out, elem_bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                                      4, (void*)fields, dims, strides, box, estr,
                                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                      CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { if (why) *why = "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")"; return false; }
    return true;
}

}  // namespace pcamm

using namespace pcamm;

struct pcamm_model {
    pcamm_geometry geo;
    Geom G;
    int M = 0, Bmax = 1, Cmax = 1, S = 1;
    // model (device)
    float* f0p = nullptr;           // f0 with its zero border: what the warp and gradient kernels gather from
    float *f0 = nullptr, *fields = nullptr, *xbar = nullptr, *u = nullptr, *lm0 = nullptr;   // xbar, u: views of fields
    __half* u16 = nullptr;          // reduced-precision copy of u (geometry.field_storage = 1), else NULL
    FieldStream fs;
    // scratch (device)
    unsigned char* cellmap = nullptr;   // FieldStream::cellmap
    unsigned *f0_integral = nullptr, *cell_integral = nullptr;   // summed-volume tables (stream.cuh box_count)
    unsigned char* occ = nullptr;       // occupancy of the trial volumes [S][OCC] (common.cuh)
    float *vol = nullptr, *pseg = nullptr, *p = nullptr, *rL = nullptr;   // vol: trial volumes, ray layout [S][PV]
    float* bvol = nullptr;          // projector 1: backprojection volumes P^T r, [B][V] (raymarch.cu), else NULL
    unsigned* rec_mask = nullptr;   // projector 1 with gradient records: one bit per voxel, record_mask_words(G) words
    ColHdr* col_hdr = nullptr;      // [B][nu]
    SlabEntry* slab_tab = nullptr;  // [B][nu][max_slabs]
    float4* utab = nullptr;
    float2* vtab = nullptr;
    char* in_block = nullptr;
    size_t in_block_bytes = 0, in_off = 0;
    CtlBufs c = {};
    SlotState* out_slots = nullptr;
    double* lm_out = nullptr;
    int* trav_ijk = nullptr;
    float* trav_len = nullptr;
    int* trav_n = nullptr;
    int trav_cap = 0;
    unsigned long long* nonfinite = nullptr;
    unsigned long long* visited = nullptr;   // FieldStream::visited
    Timeline* tl = nullptr;                  // kernel timeline of the last solve (timeline knob), else NULL
    int time_slots = 1;                      // trial slots pcamm_time_kernel launches over (pcamm_time_slots)
    float* y_stage = nullptr;   // device copy of a host-side measured projection (pcamm_reconstruct_host)
    // pinned host staging
    char* h_in = nullptr;
    SolveState* h_solves = nullptr;
    SolveTrace* h_traces = nullptr;
    LoopFlags* h_flags = nullptr;
    double* h_lm = nullptr;
    int* h_trav = nullptr;
    std::map<long long, GraphRec> graphs;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    std::vector<void*> dev_allocs, host_allocs;
};

namespace {

#define CUDA_TRY(expr)                                                                         \
    do {                                                                                       \
        cudaError_t e_ = (expr);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            set_error(std::string(#expr) + ": " + cudaGetErrorString(e_));                     \
            return e_ == cudaErrorMemoryAllocation ? PCAMM_E_NOMEM : PCAMM_E_CUDA;             \
        }                                                                                      \
    } while (0)

int invalid(const std::string& msg) {
    set_error(msg);
    return PCAMM_E_INVALID;
}

template <class T>
cudaError_t dalloc(pcamm_model* m, T** ptr, size_t count) {
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, count * sizeof(T) > 0 ? count * sizeof(T) : 16);
    if (e == cudaSuccess) { m->dev_allocs.push_back(p); *ptr = (T*)p; }
    return e;
}

template <class T>
cudaError_t halloc(pcamm_model* m, T** ptr, size_t count) {
    void* p = nullptr;
    cudaError_t e = cudaMallocHost(&p, count * sizeof(T) > 0 ? count * sizeof(T) : 16);
    if (e == cudaSuccess) { m->host_allocs.push_back(p); *ptr = (T*)p; }
    return e;
}

CallOpts* h_opts(pcamm_model* m) { return (CallOpts*)m->h_in; }
SolveIn* h_solve_in(pcamm_model* m) { return (SolveIn*)(m->h_in + m->in_off); }

int check_seq(const Seq& q, const char* what) {
    if (q.err != cudaSuccess) {
        set_error(std::string(what) + ": " + cudaGetErrorString(q.err));
        return PCAMM_E_CUDA;
    }
    return PCAMM_OK;
}

// Candidate steps evaluated per line-search pass: 0 -> 1 (sequential), 1 -> all max_backtracks
// at once, F >= 2 -> F (the next F follow if none passes).
int fan_width(const pcamm_opts& o) {
    if (o.batched_linesearch <= 0) return 1;
    if (o.batched_linesearch == 1) return o.max_backtracks;
    return o.batched_linesearch < o.max_backtracks ? o.batched_linesearch : o.max_backtracks;
}

int resolve_opts(const pcamm_model* m, const pcamm_opts* user, pcamm_opts* o) {
    pcamm_default_opts(o);
    if (user) *o = *user;
    if (o->max_iter < 0) return invalid("opts.max_iter < 0");
    if (o->max_backtracks < 1 || o->max_backtracks > MAXBT) return invalid("opts.max_backtracks out of range");
    if (!(o->armijo_beta > 0.f && o->armijo_beta < 1.f)) return invalid("opts.armijo_beta must be in (0, 1)");
    if (!(o->armijo_c >= 0.f) || !(o->init_step_vox > 0.f)) return invalid("opts.armijo_c / init_step_vox");
    if (o->batched_linesearch < 0) return invalid("opts.batched_linesearch < 0");
    if (fan_width(*o) > m->Cmax)
        return invalid("batched_linesearch needs geometry.max_candidates >= the fan width");
    if (o->inv_max_iter < 0) return invalid("opts.inv_max_iter < 0");
    return PCAMM_OK;
}

void fill_call(pcamm_model* m, const pcamm_opts& o, int B, int C) {
    CallOpts* c = h_opts(m);
    c->B = B; c->C = C;
    c->max_iter = o.max_iter; c->max_backtracks = o.max_backtracks; c->batched = o.batched_linesearch ? 1 : 0;
    c->inv_max_iter = o.inv_max_iter;
    c->grad_tol = (double)o.grad_tol; c->armijo_c = (double)o.armijo_c; c->armijo_beta = (double)o.armijo_beta;
    c->init_step_vox = (double)o.init_step_vox; c->inv_tol = (double)o.inv_tol_mm;
    const Geom& G = m->G;
    const double hmin = std::fmin((double)G.hx, std::fmin((double)G.hy, (double)G.hz));
    c->hmin_sqrtV = hmin * std::sqrt((double)G.V);
}

int push_call(pcamm_model* m, int B, cudaStream_t st) {
    CUDA_TRY(cudaMemcpyAsync(m->in_block, m->h_in, m->in_off + sizeof(SolveIn) * (size_t)B, cudaMemcpyHostToDevice, st));
    return PCAMM_OK;
}

// ---- the kernel sequences of a solve (shared by the graph and the host-driven mode)
//
//   head:       sums of y, begin, per-view tables, warp + projection at w0 (-> first fit)
//   loop body:  residual, gradient (-> J_n, g, first candidates), warp, projection (-> Armijo test,
//               Eq. 3 update, Eq. 4 fit); a solve in the middle of a line search skips the first two
//   tail:       closing residual (J at exit), final, landmark inversion
// A single-block control step (control.cuh) follows every projection and every gradient pass.

// P^T r of the ray-marching variant for the solves that need a gradient; where the gradient of the one solve
// gathers over the records, only at the recorded voxels (raymarch.cu)
void backproject_rm(pcamm_model* m, Seq& q, int B, int force, float* bvol, bool all_voxels) {
    const Geom& G = m->G;
    const int tz = G.K <= PCAMM_TZ_SMALL_K ? 32 : 16;                     // TileZ<K>
    const bool masked = !all_voxels && B == 1 && m->fs.grad_rec;
    launch_backproject_rm(q, G, m->c.solves, B, force, m->rL, bvol, masked ? m->fs.grad_rec : nullptr,
                          tile_count(G, tz) * GROUP_WARPS, TX * tz / GROUP_WARPS, masked ? m->rec_mask : nullptr);
}

void seq_head(pcamm_model* m, Seq& q, int B, int C, cudaGraphConditionalHandle h_loop, int use_cond) {
    const Geom& G = m->G;
    launch_ysums(q, G, m->c, B);
    launch_begin(q, G, m->c, 0);
    launch_view_tables(q, G, m->c.solves, B, m->col_hdr, m->slab_tab);
    launch_warp(q, G, m->fs, m->f0p, m->c.slots, B * C, 1, m->vol, G.PV, m->occ, m->fs.grad_rec);
    launch_project(q, G, m->c, B * C, m->col_hdr, m->slab_tab, m->vol, m->occ, m->pseg, m->p, THEN_INIT, h_loop, use_cond,
                   q.n_kernels);
}

void seq_body(pcamm_model* m, Seq& q, int B, int C, cudaGraphConditionalHandle h_loop, int use_cond) {
    const Geom& G = m->G;
    const int n0 = q.n_kernels;
    launch_resid(q, G, m->c.solves, m->c.in, B, 0, m->p, nullptr, m->rL, m->utab, m->vtab, m->c.resid_part);
    if (G.projector == 1) backproject_rm(m, q, B, 0, m->bvol, false);
    launch_grad(q, G, m->fs, m->f0p, m->c, B, m->rL, m->utab, m->vtab, m->bvol, GRAD_SOLVE);
    launch_warp(q, G, m->fs, m->f0p, m->c.slots, B * C, 1, m->vol, G.PV, m->occ, m->fs.grad_rec);
    launch_project(q, G, m->c, B * C, m->col_hdr, m->slab_tab, m->vol, m->occ, m->pseg, m->p, THEN_TRIAL, h_loop, use_cond,
                   q.n_kernels - n0);
}

void seq_tail(pcamm_model* m, Seq& q, int B) {
    const Geom& G = m->G;
    const int n0 = q.n_kernels;
    launch_resid(q, G, m->c.solves, m->c.in, B, 1, m->p, nullptr, m->rL, m->utab, m->vtab, m->c.resid_part);
    launch_ctl_final(q, G, m->c, m->out_slots, q.n_kernels - n0 + 1 + (m->M > 0 ? 1 : 0));
    launch_invert(q, G, m->xbar, m->u, m->c, B, m->M, m->lm0, m->lm_out);
}

// n_static: line-search passes laid out as plain kernel nodes in front of the while-loop (pcamm_tune
// "static_passes"); the loop then takes whatever passes remain.  Every kernel of a pass looks at its
// solves' state first, so a pass behind the end of a solve does nothing.
int get_graph(pcamm_model* m, int B, int C, int n_static, GraphRec** out) {
    const long long key = ((long long)n_static * 8192 + B) * 1024 + C;
    auto it = m->graphs.find(key);
    if (it != m->graphs.end()) { *out = &it->second; return PCAMM_OK; }
    GraphRec rec;
    CUDA_TRY(cudaGraphCreate(&rec.graph, 0));
    cudaGraphConditionalHandle h_loop;
    CUDA_TRY(cudaGraphConditionalHandleCreate(&h_loop, rec.graph, 0, cudaGraphCondAssignDefault));
    Seq q;
    q.graph = rec.graph;
    q.pdl = g_pdl != 0;
    seq_head(m, q, B, C, h_loop, 1);
    for (int i = 0; i < n_static; ++i) seq_body(m, q, B, C, h_loop, 1);
    Seq body = q.add_while(h_loop);             // iterations and their line searches
    // (two or more passes per evaluation of the loop condition were measured and are slower: 2.81 / 2.84 / 2.87 ms
    // per C2 solve with 2 / 3 / 4 against 2.74 ms with one)
    seq_body(m, body, B, C, h_loop, 1);
    seq_tail(m, q, B);
    int rc;
    if ((rc = check_seq(q, "graph build")) || (rc = check_seq(body, "graph build (loop body)"))) {
        cudaGraphDestroy(rec.graph);
        return rc;
    }
    cudaError_t e = cudaGraphInstantiate(&rec.exec, rec.graph, 0);
    if (e != cudaSuccess) {
        set_error(std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e));
        cudaGraphDestroy(rec.graph);
        return PCAMM_E_CUDA;
    }
    m->graphs[key] = rec;
    *out = &m->graphs[key];
    return PCAMM_OK;
}

int read_flags(pcamm_model* m, cudaStream_t st) {
    CUDA_TRY(cudaMemcpyAsync(m->h_flags, m->c.flags, sizeof(LoopFlags), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return PCAMM_OK;
}

int run_host_loop(pcamm_model* m, int B, int C, cudaStream_t st) {
    Seq q;
    q.stream = st;
    int rc;
    seq_head(m, q, B, C, 0, 0);
    if ((rc = check_seq(q, "solve head")) || (rc = read_flags(m, st))) return rc;
    while (m->h_flags->loop_cond) {
        seq_body(m, q, B, C, 0, 0);
        if ((rc = check_seq(q, "loop body")) || (rc = read_flags(m, st))) return rc;
    }
    seq_tail(m, q, B);
    return check_seq(q, "solve tail");
}

int solve_impl(pcamm_model* m, int B, const float* y_dev, const float* angles, const float* w_init,
               const pcamm_opts* user_opts, float* w_out, float* volumes_out, float* lm_out, pcamm_info* info,
               cudaStream_t st) {
    if (!m) return invalid("model is NULL");
    if (B < 1 || B > m->Bmax) return invalid("B outside [1, geometry.max_batch]");
    if (!y_dev || !angles || !w_init || !w_out) return invalid("NULL argument");
    pcamm_opts o;
    int rc = resolve_opts(m, user_opts, &o);
    if (rc) return rc;
    const Geom& G = m->G;
    const int C = fan_width(o);
    fill_call(m, o, B, C);
    SolveIn* in = h_solve_in(m);
    for (int b = 0; b < B; ++b) {
        in[b].y = y_dev + (size_t)b * G.npix;
        in[b].angle = angles[b];
        if (!std::isfinite(angles[b])) return invalid("angle is not finite");
        for (int k = 0; k < KMAX; ++k) in[b].w_init[k] = k < G.K ? w_init[b * G.K + k] : 0.f;
        for (int k = 0; k < G.K; ++k)
            if (!std::isfinite(w_init[b * G.K + k])) { set_error("w_init is not finite"); return PCAMM_E_NONFINITE; }
        in[b].a = in[b].b = 0.f;
    }
    if ((rc = push_call(m, B, st))) return rc;
    if (m->tl) {       // fresh timeline: no events, starts at the largest time, ends at 0
        CUDA_TRY(cudaMemsetAsync(m->tl, 0, sizeof(Timeline), st));
        CUDA_TRY(cudaMemsetAsync(m->tl->t0, 0xff, sizeof(m->tl->t0), st));
    }
    if (o.loop_mode == 0) {
        GraphRec* g = nullptr;
        // Passes in front of the loop: with the stopping rule off (grad_tol = 0) a solve takes max_iter iterations,
        // each at least one line-search pass, so that many passes can be plain nodes (2 us from kernel to kernel
        // instead of the 7 to 9 us an evaluation of the loop condition costs); the loop takes the passes beyond.
        // With grad_tol on, the count is not known and a pass behind the end of a solve still costs its six
        // launches (about 20 us): none then.  (A line search that fails ends a solve early too: rare.)
        const int auto_static = o.grad_tol > 0.f ? 0 : (o.max_iter < STATIC_PASSES_MAX ? o.max_iter : STATIC_PASSES_MAX);
        const int n_static = g_static_passes < 0 ? auto_static : (g_static_passes < o.max_iter ? g_static_passes : o.max_iter);
        if ((rc = get_graph(m, B, C, n_static, &g))) return rc;
        CUDA_TRY(cudaGraphLaunch(g->exec, st));
    } else {
        if ((rc = run_host_loop(m, B, C, st))) return rc;
    }
    if (volumes_out) {
        Seq q;
        q.stream = st;
        launch_warp(q, G, m->fs, m->f0p, m->out_slots, B, 0, volumes_out, G.V, nullptr, nullptr);
        if ((rc = check_seq(q, "final warp"))) return rc;
    }
    CUDA_TRY(cudaMemcpyAsync(m->h_solves, m->c.solves, sizeof(SolveState) * B, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(m->h_flags, m->c.flags, sizeof(LoopFlags), cudaMemcpyDeviceToHost, st));
    if (lm_out && m->M > 0)
        CUDA_TRY(cudaMemcpyAsync(m->h_lm, m->lm_out, sizeof(double) * 3 * m->M * B, cudaMemcpyDeviceToHost, st));
    bool want_trace = false;
    if (info)
        for (int b = 0; b < B; ++b)
            want_trace |= info[b].J_trace || info[b].gnorm_trace || info[b].mu_trace || info[b].backtracks_trace;
    if (want_trace)
        CUDA_TRY(cudaMemcpyAsync(m->h_traces, m->c.traces, sizeof(SolveTrace) * B, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (o.loop_mode == 0) count_launch(m->h_flags->n_launch);
    int first_err = 0;
    for (int b = 0; b < B; ++b) {
        const SolveState& s = m->h_solves[b];
        for (int k = 0; k < G.K; ++k) w_out[b * G.K + k] = (float)s.w[k];
        if (s.status < 0 && !first_err) {
            first_err = s.status;
            set_error(s.status == PCAMM_E_SINGULAR ? "intensity fit singular: y is constant"
                                                   : "non-finite value in y or in the gradient");
        }
        if (info) {
            pcamm_info& I = info[b];
            I.iters = s.iter; I.status = s.status; I.J0 = s.J0; I.J = s.J; I.a = s.a; I.b = s.b;
            const SolveTrace& t = m->h_traces[b];
            const int n = s.iter < TRACE_CAP ? s.iter : TRACE_CAP;
            const int ng = (s.status == PCAMM_S_GRADTOL || s.status == PCAMM_S_LINESEARCH) && n < TRACE_CAP ? n + 1 : n;
            if (I.J_trace) std::memcpy(I.J_trace, t.J, sizeof(double) * (n + 1));
            if (I.gnorm_trace) std::memcpy(I.gnorm_trace, t.gnorm, sizeof(double) * (ng < o.max_iter ? ng : o.max_iter));
            if (I.mu_trace) std::memcpy(I.mu_trace, t.mu, sizeof(double) * n);
            if (I.backtracks_trace) std::memcpy(I.backtracks_trace, t.bt, sizeof(int) * n);
        }
    }
    if (lm_out)
        for (int i = 0; i < 3 * m->M * B; ++i) lm_out[i] = (float)m->h_lm[i];
    if (first_err) return first_err;
    return B == 1 ? m->h_solves[0].status : PCAMM_OK;
}

// Common start of the hooks: one solve slot, view from `angle`, w into slot 0.
int hook_begin(pcamm_model* m, const float* y_dev, float angle, const float* w, float a, float b, int mode,
               cudaStream_t st, Seq& q) {
    pcamm_opts o;
    pcamm_default_opts(&o);
    fill_call(m, o, 1, 1);
    SolveIn* in = h_solve_in(m);
    in[0].y = y_dev;
    in[0].angle = angle;
    for (int k = 0; k < KMAX; ++k) in[0].w_init[k] = (w && k < m->G.K) ? w[k] : 0.f;
    in[0].a = a; in[0].b = b;
    int rc = push_call(m, 1, st);
    if (rc) return rc;
    q.stream = st;
    launch_begin(q, m->G, m->c, mode);
    return check_seq(q, "begin");
}

}  // namespace

namespace pcamm {
int model_K(const pcamm_model* m) { return m->G.K; }
}  // namespace pcamm

extern "C" {

void pcamm_default_opts(pcamm_opts* o) {
    if (!o) return;
    o->max_iter = 10;
    o->grad_tol = 0.f;
    o->armijo_c = 1e-4f;
    o->armijo_beta = 0.5f;
    o->max_backtracks = 8;
    o->init_step_vox = 1.f;
    o->batched_linesearch = 0;
    o->inv_max_iter = 50;
    o->inv_tol_mm = 1e-4f;
    o->loop_mode = 0;
}

const char* pcamm_last_error(void) { return g_error.c_str(); }

int64_t pcamm_launch_count(int32_t reset) {
    const long long n = g_launches;
    if (reset) g_launches = 0;
    return n;
}

void pcamm_model_destroy(pcamm_model* m) {
    if (!m) return;
    for (auto& kv : m->graphs) {
        if (kv.second.exec) cudaGraphExecDestroy(kv.second.exec);
        if (kv.second.graph) cudaGraphDestroy(kv.second.graph);
    }
    if (m->ev0) cudaEventDestroy(m->ev0);
    if (m->ev1) cudaEventDestroy(m->ev1);
    for (void* p : m->dev_allocs) cudaFree(p);
    for (void* p : m->host_allocs) cudaFreeHost(p);
    delete m;
}

int pcamm_model_create(const pcamm_geometry* g, const float* f0_dev, const float* mean_dvf_dev, const float* eig_dvf_dev,
                       int32_t n_landmarks, const float* landmarks_mm_host, void* stream, pcamm_model** out) {
    if (out) *out = nullptr;
    if (!g || !f0_dev || !mean_dvf_dev || !eig_dvf_dev || !out) return invalid("NULL argument");
    if (g->nx < 1 || g->ny < 1 || g->nz < 1 || g->nu < 1 || g->nv < 1) return invalid("sizes must be positive");
    if (!(g->hx > 0 && g->hy > 0 && g->hz > 0 && g->pu > 0 && g->pv > 0)) return invalid("voxel / pixel sizes must be positive");
    if (g->K < 1 || g->K > KMAX) return invalid("K outside [1, PCAMM_KMAX]");
    if (g->projector != 0 && g->projector != 1) return invalid("geometry.projector must be 0 or 1");
    if (!(g->ray_step_vox >= 0.f) || !std::isfinite(g->ray_step_vox)) return invalid("geometry.ray_step_vox must be >= 0");
    if (n_landmarks < 0 || (n_landmarks > 0 && !landmarks_mm_host)) return invalid("landmarks");
    const long long V = (long long)g->nx * g->ny * g->nz;
    if ((long long)(g->nx + 4) * (g->ny + 4) * (g->nz + 4) >= (1LL << 31) || (long long)g->nu * g->nv >= (1LL << 31)) return invalid("volume or detector too large");
    // the gradient kernel's voxel queue packs (x, y) into 16 + 15 bits
    if (g->nx >= 65536 || g->ny >= 32768) return invalid("nx must be < 65536 and ny < 32768");
    const int Bmax = g->max_batch < 1 ? 1 : g->max_batch;
    const int Cmax = g->max_candidates < 1 ? 1 : g->max_candidates;
    if (Cmax > MAXBT || Bmax > 4096) return invalid("max_batch / max_candidates too large");
    if (!(g->sad > 0 && g->sdd > g->sad)) return invalid("need 0 < sad < sdd");
    // source and detector plane outside the volume's bounding sphere about the isocentre
    const double ex = 0.5 * g->nx * (double)g->hx, ey = 0.5 * g->ny * (double)g->hy, ez = 0.5 * g->nz * (double)g->hz;
    const double R = std::sqrt((double)g->cx * g->cx + (double)g->cy * g->cy + (double)g->cz * g->cz) +
                     std::sqrt(ex * ex + ey * ey + ez * ez);
    if (!(R < 0.999 * g->sad && R < 0.999 * ((double)g->sdd - g->sad)))
        return invalid("source or detector inside the volume's bounding sphere");
    // at most one voxel in z per voxel along the dominant in-plane axis
    const double vmax = (0.5 * (g->nv - 1) + std::fabs((double)g->off_v)) * g->pv;
    if (!(vmax / g->hz <= (double)g->sdd / std::sqrt((double)g->hx * g->hx + (double)g->hy * g->hy)))
        return invalid("cone angle too steep for the voxel aspect ratio (z-slope > 1 voxel per slab)");

    {
        Geom Gz = {};
        Gz.nz = g->nz;
        if (!project_fits(Gz)) return invalid("nz too large for the projector's shared-memory knots");
    }
    pcamm_model* m = new (std::nothrow) pcamm_model();
    if (!m) { set_error("out of host memory"); return PCAMM_E_NOMEM; }
    m->G.tl = nullptr;
    m->geo = *g;
    m->M = n_landmarks; m->Bmax = Bmax; m->Cmax = Cmax; m->S = Bmax * Cmax;
    Geom& G = m->G;
    G.nx = g->nx; G.ny = g->ny; G.nz = g->nz; G.V = V;
    G.pnx = g->nx + 2; G.pny = g->ny + 2; G.PV = (long long)G.pnx * G.pny * g->nz;
    G.fnx = g->nx + 4; G.fny = g->ny + 4; G.fpp = G.fnx * G.fny;
    G.occ_pitch = ((g->nz + 15) / 16 + 7) / 8 * 8;
    G.OCC = (long long)G.pnx * G.pny * G.occ_pitch;
    G.hx = g->hx; G.hy = g->hy; G.hz = g->hz;
    G.ihx = 1.f / g->hx; G.ihy = 1.f / g->hy; G.ihz = 1.f / g->hz;
    G.cx = g->cx; G.cy = g->cy; G.cz = g->cz;
    G.lox = (double)g->cx - ex; G.loy = (double)g->cy - ey; G.loz = (double)g->cz - ez;
    G.ihz_d = 1.0 / (double)g->hz; G.Szi = (0.0 - G.loz) / (double)g->hz;
    tile_multipliers(G);
    G.projector = g->projector;
    G.rm_step_mm = (g->ray_step_vox > 0.f ? g->ray_step_vox : 0.5f) * std::fmin(g->hx, std::fmin(g->hy, g->hz));
    G.K = g->K; G.nu = g->nu; G.nv = g->nv; G.npix = g->nu * g->nv;
    G.pu = g->pu; G.pv = g->pv; G.sad = g->sad; G.sdd = g->sdd; G.off_u = g->off_u; G.off_v = g->off_v;

    cudaStream_t st = (cudaStream_t)stream;
    const size_t S = (size_t)m->S, B = (size_t)Bmax;
    m->in_off = (sizeof(CallOpts) + 63) / 64 * 64;
    m->in_block_bytes = m->in_off + sizeof(SolveIn) * B;
    m->c.ysum_blocks = ysum_blocks(G);
    m->c.proj_blocks = project_blocks(G);
    m->c.resid_blocks = resid_blocks(G);
    {   // sized for either gradient kernel; the count in use is fixed once the field stream is known
        int dev = 0, n_sm = 1;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        m->fs.n_sm = n_sm > 0 ? n_sm : 1;
        FieldStream generic = m->fs, tma = m->fs;
        generic.use_tma = false; tma.use_tma = true;
        m->c.grad_blocks = std::max(std::max(grad_blocks(G, generic), grad_blocks(G, tma)), grad_gather_blocks(G, m->fs));
    }
    m->trav_cap = G.nx + G.ny + G.nz + 8;
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t r) { if (e == cudaSuccess) e = r; return r == cudaSuccess; };
    ok(dalloc(m, &m->f0, (size_t)V)) && ok(dalloc(m, &m->f0p, (size_t)(g->nx + 4) * (g->ny + 4) * (g->nz + 4))) && ok(dalloc(m, &m->cellmap, (size_t)(g->nx + 1) * (g->ny + 1) * (g->nz + 1))) && ok(dalloc(m, &m->fields, 3 * (size_t)V * (G.K + 1))) && ok(dalloc(m, &m->lm0, 3 * (size_t)(m->M > 0 ? m->M : 1))) &&
        ok(dalloc(m, &m->vol, S * (size_t)G.PV)) && ok(dalloc(m, &m->occ, S * (size_t)G.OCC)) && ok(dalloc(m, &m->col_hdr, B * G.nu)) &&
        ok(dalloc(m, &m->slab_tab, B * G.nu * (size_t)max_slabs(G))) && ok(dalloc(m, &m->p, S * G.npix)) && ok(dalloc(m, &m->pseg, S * G.npix * (size_t)project_segments(G))) &&
        ok(dalloc(m, &m->rL, B * G.npix)) && ok(dalloc(m, &m->utab, B * G.nu)) && ok(dalloc(m, &m->vtab, B * G.nv)) &&
        ok(dalloc(m, &m->in_block, m->in_block_bytes)) && ok(dalloc(m, &m->c.solves, B)) &&
        ok(dalloc(m, &m->c.traces, B)) && ok(dalloc(m, &m->c.slots, S)) && ok(dalloc(m, &m->c.flags, 1)) &&
        ok(dalloc(m, &m->c.ysum_part, B * m->c.ysum_blocks * 2)) &&
        ok(dalloc(m, &m->c.proj_part, S * m->c.proj_blocks * 3)) && ok(dalloc(m, &m->c.seg_ticket, S * m->c.proj_blocks)) &&
        ok(dalloc(m, &m->c.resid_part, B * m->c.resid_blocks)) &&
        ok(dalloc(m, &m->c.grad_part, B * m->c.grad_blocks * KMAX)) && ok(dalloc(m, &m->out_slots, B)) &&
        ok(dalloc(m, &m->lm_out, 3 * B * (size_t)(m->M > 0 ? m->M : 1))) &&
        ok(dalloc(m, &m->trav_ijk, 3 * (size_t)m->trav_cap)) && ok(dalloc(m, &m->trav_len, (size_t)m->trav_cap)) &&
        ok(dalloc(m, &m->trav_n, 1)) && ok(dalloc(m, &m->nonfinite, 1)) && ok(dalloc(m, &m->visited, 4)) && ok(dalloc(m, &m->y_stage, (size_t)G.npix)) &&
        ok(halloc(m, &m->h_in, m->in_block_bytes)) && ok(halloc(m, &m->h_solves, B)) &&
        ok(halloc(m, &m->h_traces, B)) && ok(halloc(m, &m->h_flags, 1)) &&
        ok(halloc(m, &m->h_lm, 3 * B * (size_t)(m->M > 0 ? m->M : 1))) &&
        ok(halloc(m, &m->h_trav, 4 * (size_t)m->trav_cap + 4)) &&
        ok(cudaEventCreate(&m->ev0)) && ok(cudaEventCreate(&m->ev1));
    if (e != cudaSuccess) {
        set_error(std::string("allocation failed: ") + cudaGetErrorString(e));
        cudaGetLastError();
        pcamm_model_destroy(m);
        return e == cudaErrorMemoryAllocation ? PCAMM_E_NOMEM : PCAMM_E_CUDA;
    }
    if (g->projector == 1) {
        e = dalloc(m, &m->bvol, B * (size_t)V);
        if (e == cudaSuccess) e = dalloc(m, &m->rec_mask, (size_t)record_mask_words(G));
        if (e != cudaSuccess) { set_error("allocation failed (backprojection volumes)"); cudaGetLastError(); pcamm_model_destroy(m); return PCAMM_E_NOMEM; }
    }
    if (g_timeline) {
        e = dalloc(m, &m->tl, 1);
        if (e != cudaSuccess) { set_error("allocation failed (timeline)"); pcamm_model_destroy(m); return PCAMM_E_NOMEM; }
        G.tl = m->tl;
    }
    m->xbar = m->fields;
    m->u = m->fields + 3 * (size_t)V;
    m->c.opts = (CallOpts*)m->in_block;
    m->c.in = (SolveIn*)(m->in_block + m->in_off);
    std::memset(m->h_in, 0, m->in_block_bytes);

    auto fail = [&](int rc) { pcamm_model_destroy(m); return rc; };
#define TRY_OR_FAIL(expr)                                                                       \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess) {                                                                \
            set_error(std::string(#expr) + ": " + cudaGetErrorString(e_));                      \
            return fail(PCAMM_E_CUDA);                                                          \
        }                                                                                       \
    } while (0)
    TRY_OR_FAIL(cudaMemcpyAsync(m->f0, f0_dev, sizeof(float) * V, cudaMemcpyDeviceToDevice, st));
    TRY_OR_FAIL(cudaMemcpyAsync(m->xbar, mean_dvf_dev, sizeof(float) * 3 * V, cudaMemcpyDeviceToDevice, st));
    TRY_OR_FAIL(cudaMemcpyAsync(m->u, eig_dvf_dev, sizeof(float) * 3 * V * G.K, cudaMemcpyDeviceToDevice, st));
    if (m->M > 0)
        TRY_OR_FAIL(cudaMemcpyAsync(m->lm0, landmarks_mm_host, sizeof(float) * 3 * m->M, cudaMemcpyHostToDevice, st));
    TRY_OR_FAIL(cudaMemsetAsync(m->vol, 0, sizeof(float) * S * (size_t)G.PV, st));   // zero border, never written
    TRY_OR_FAIL(cudaMemsetAsync(m->occ, 0, S * (size_t)G.OCC, st));                   // likewise
    TRY_OR_FAIL(cudaMemsetAsync(m->nonfinite, 0, sizeof(unsigned long long), st));
    TRY_OR_FAIL(cudaMemsetAsync(m->visited, 0, 4 * sizeof(unsigned long long), st));
    m->fs.visited = m->visited;
    TRY_OR_FAIL(cudaMemsetAsync(m->c.solves, 0, sizeof(SolveState) * B, st));
    TRY_OR_FAIL(cudaMemsetAsync(m->c.slots, 0, sizeof(SlotState) * S, st));
    TRY_OR_FAIL(cudaMemsetAsync(m->c.flags, 0, sizeof(LoopFlags), st));
    TRY_OR_FAIL(cudaMemsetAsync(m->c.seg_ticket, 0, sizeof(int) * S * m->c.proj_blocks, st));
    k_count_nonfinite<<<592, 256, 0, st>>>(m->f0, V, m->nonfinite);
    k_count_nonfinite<<<592, 256, 0, st>>>(m->xbar, 3 * V, m->nonfinite);
    k_count_nonfinite<<<592, 256, 0, st>>>(m->u, 3 * V * G.K, m->nonfinite);
    k_fields_to_voxel_units<<<1184, 256, 0, st>>>(m->fields, V, 3 * (G.K + 1), G.hx, G.hy, G.hz);
    TRY_OR_FAIL(cudaMemsetAsync(m->f0p, 0, sizeof(float) * (size_t)G.fpp * (g->nz + 4), st));
    k_pad_f0<<<1184, 256, 0, st>>>(m->f0, G, m->f0p);
    launch_build_cellmap(st, G, m->f0, m->cellmap);
    m->fs.cellmap = m->cellmap;
    unsigned long long bad = 0;
    TRY_OR_FAIL(cudaMemcpyAsync(&bad, m->nonfinite, sizeof(bad), cudaMemcpyDeviceToHost, st));
    TRY_OR_FAIL(cudaStreamSynchronize(st));
#undef TRY_OR_FAIL
    if (m->M > 0)
        for (int i = 0; i < 3 * m->M; ++i)
            if (!std::isfinite(landmarks_mm_host[i])) bad++;
    if (bad) {
        set_error("non-finite value in f0, the DVF fields or the landmarks");
        return fail(PCAMM_E_NONFINITE);
    }
    // the streaming kernels' view of the fields: TMA tensor map (else the generic kernels)
    m->fs.fields = m->fields;
    std::string why;
    m->fs.use_tma = make_field_map(G, m->fields, 3 * (G.K + 1), 32, 4, &m->fs.map32, &why) &&
                    make_field_map(G, m->fields, 3 * (G.K + 1), 16, 4, &m->fs.map16, &why);
    if (g->field_storage == 1) {
        // u_k in half: scale[k] = the power of two that puts max |u_k| (voxel units) into [8192, 16384),
        // so that entries down to 2^-28 of the largest stay normal halves with 11 significant bits
        if (G.nx % 8 != 0) { set_error("field_storage = 1 needs nx to be a multiple of 8"); return fail(PCAMM_E_INVALID); }
        unsigned int* d_max = nullptr;
        unsigned int h_max[KMAX] = {};
        cudaError_t e2 = dalloc(m, &m->u16, 3 * (size_t)V * G.K);
        if (e2 == cudaSuccess) e2 = dalloc(m, &d_max, (size_t)KMAX);
        if (e2 == cudaSuccess) e2 = cudaMemsetAsync(d_max, 0, sizeof(unsigned int) * KMAX, st);
        if (e2 == cudaSuccess) {
            k_field_absmax<<<1184, 256, 0, st>>>(m->u, 3 * V, G.K, d_max);
            e2 = cudaMemcpyAsync(h_max, d_max, sizeof(unsigned int) * KMAX, cudaMemcpyDeviceToHost, st);
        }
        if (e2 == cudaSuccess) e2 = cudaStreamSynchronize(st);
        if (e2 != cudaSuccess) { set_error(std::string("field quantisation: ") + cudaGetErrorString(e2)); return fail(PCAMM_E_CUDA); }
        FieldScale scale = {}, inv = {};
        for (int k = 0; k < KMAX; ++k) {
            float mx;
            std::memcpy(&mx, &h_max[k], sizeof(float));
            int ex = 0;
            if (k < G.K && mx > 0.f) std::frexp(mx, &ex);       // mx = f * 2^ex, f in [0.5, 1)
            scale.inv[k] = (k < G.K && mx > 0.f) ? std::ldexp(1.f, 14 - ex) : 1.f;
            inv.inv[k] = 1.f / scale.inv[k];
        }
        k_quantise_fields<<<1184, 256, 0, st>>>(m->u, m->u16, 3 * V, G.K, scale, inv);
        m->fs.scale = inv;
        m->fs.u16 = m->u16;
        m->fs.half_u = make_field_map(G, m->fields, 3, 32, 4, &m->fs.xmap32, &why) &&
                       make_field_map(G, m->fields, 3, 16, 4, &m->fs.xmap16, &why) &&
                       make_field_map(G, m->u16, 3 * G.K, 32, 2, &m->fs.umap32, &why) &&
                       make_field_map(G, m->u16, 3 * G.K, 16, 2, &m->fs.umap16, &why);
        e2 = cudaStreamSynchronize(st);
        if (e2 != cudaSuccess || !m->fs.half_u || !m->fs.use_tma) {
            set_error("field_storage = 1: " + (e2 != cudaSuccess ? std::string(cudaGetErrorString(e2)) : why));
            return fail(e2 != cudaSuccess ? PCAMM_E_CUDA : PCAMM_E_INVALID);
        }
    } else if (g->field_storage != 0) {
        set_error("geometry.field_storage must be 0 or 1");
        return fail(PCAMM_E_INVALID);
    }
    if (g->tile_skipping < 0 || g->tile_skipping > 2) { set_error("geometry.tile_skipping must be 0, 1 or 2"); return fail(PCAMM_E_INVALID); }
    if (m->fs.use_tma && g->tile_skipping != 2) {
        // what lets the streaming kernels skip tiles that can only see zeros (reading B8): the
        // largest magnitude of every field plane (bounds the displacement for any w) and the
        // summed-volume tables of f0 != 0 and of the cell map, built on the host once
        const int planes = 3 * (G.K + 1);
        unsigned int* d_max = nullptr;
        unsigned int h_max[3 * (KMAX + 1)] = {};
        std::vector<float> h_f0((size_t)V);
        const size_t ncell = (size_t)(g->nx + 1) * (g->ny + 1) * (g->nz + 1);
        std::vector<unsigned char> h_cell(ncell);
        cudaError_t e3 = dalloc(m, &d_max, (size_t)planes);
        if (e3 == cudaSuccess) e3 = dalloc(m, &m->f0_integral, ncell);
        if (e3 == cudaSuccess) e3 = dalloc(m, &m->cell_integral, (size_t)(g->nx + 2) * (g->ny + 2) * (g->nz + 2));
        if (e3 == cudaSuccess) e3 = cudaMemsetAsync(d_max, 0, sizeof(unsigned int) * planes, st);
        if (e3 == cudaSuccess) {
            k_plane_absmax<<<1184, 256, 0, st>>>(m->fields, V, planes, d_max);
            e3 = cudaMemcpyAsync(h_max, d_max, sizeof(unsigned int) * planes, cudaMemcpyDeviceToHost, st);
        }
        if (e3 == cudaSuccess) e3 = cudaMemcpyAsync(h_f0.data(), m->f0, sizeof(float) * (size_t)V, cudaMemcpyDeviceToHost, st);
        if (e3 == cudaSuccess) e3 = cudaMemcpyAsync(h_cell.data(), m->cellmap, ncell, cudaMemcpyDeviceToHost, st);
        if (e3 == cudaSuccess) e3 = cudaStreamSynchronize(st);
        if (e3 == cudaSuccess) {
            for (int p = 0; p < planes; ++p) std::memcpy(&m->fs.fmax.v[p], &h_max[p], sizeof(float));
            // table over [0, ex) x [0, ey) x [0, ez) of a 0/1 map given by `one(x, y, z)`
            auto build = [](int ex, int ey, int ez, auto one) {
                const size_t px = (size_t)ex + 1, pp = px * ((size_t)ey + 1);
                std::vector<unsigned> I(pp * ((size_t)ez + 1), 0u);
                for (int z = 0; z < ez; ++z)
                    for (int y = 0; y < ey; ++y) {
                        unsigned row = 0;                 // ones in [0, x] of this row
                        for (int x = 0; x < ex; ++x) {
                            row += one(x, y, z) ? 1u : 0u;
                            I[(z + 1) * pp + (y + 1) * px + (x + 1)] =
                                row + I[(z + 1) * pp + y * px + (x + 1)] + I[z * pp + (y + 1) * px + (x + 1)] - I[z * pp + y * px + (x + 1)];
                        }
                    }
                return I;
            };
            const int nx = g->nx, ny = g->ny;
            const std::vector<unsigned> If = build(g->nx, g->ny, g->nz, [&](int x, int y, int z) {
                return h_f0[((size_t)z * ny + y) * nx + x] != 0.f;
            });
            const std::vector<unsigned> Ic = build(g->nx + 1, g->ny + 1, g->nz + 1, [&](int x, int y, int z) {
                return h_cell[((size_t)z * (ny + 1) + y) * (nx + 1) + x] != 0;
            });
            e3 = cudaMemcpyAsync(m->f0_integral, If.data(), sizeof(unsigned) * If.size(), cudaMemcpyHostToDevice, st);
            if (e3 == cudaSuccess) e3 = cudaMemcpyAsync(m->cell_integral, Ic.data(), sizeof(unsigned) * Ic.size(), cudaMemcpyHostToDevice, st);
            if (e3 == cudaSuccess) e3 = cudaStreamSynchronize(st);
        }
        if (e3 != cudaSuccess) { set_error(std::string("summed-volume tables: ") + cudaGetErrorString(e3)); return fail(PCAMM_E_CUDA); }
        m->fs.f0_integral = m->f0_integral;
        m->fs.cell_integral = m->cell_integral;
        m->fs.skip_min_tiles_per_sm = g->tile_skipping == 1 ? 0 : (g->tile_skipping == 2 ? (1 << 30) : SKIP_MIN_TILES_PER_SM);
    }
    m->c.grad_blocks = grad_blocks(G, m->fs);
    // Records pay where few candidates share a pass (each candidate slot costs the warp kernel about a sixth
    // more, the gather saves one pass over the fields per iteration and solve: a win for one or two candidates,
    // a loss for the fan of eight), and they take 48 V bytes per trial slot: models with max_candidates <= 2
    // get them if all their slots' records fit into three fifths of what is free on the device now.
    size_t rec_bytes = 0, free_b = 0, total_b = 0;
    {
        const int tz = G.K <= PCAMM_TZ_SMALL_K ? 32 : 16;                     // TileZ<K>
        const long long n_tiles = tile_count(G, tz);
        rec_bytes = sizeof(int) * (size_t)grad_record_words(n_tiles * GROUP_WARPS, n_tiles * (TX * tz)) * (size_t)m->S;
        if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { free_b = 0; cudaGetLastError(); }
    }
    if (m->fs.use_tma && g_grad_records && Cmax <= RECORD_MAX_FAN && rec_bytes <= free_b / 5 * 3 && G.nx <= RECORD_MAX_XY &&
        G.ny <= RECORD_MAX_XY && G.nz <= RECORD_MAX_Z) {
        // gradient records of the trial slots of a single solve (stream.cuh GradRecords): 48 bytes per voxel and slot
        const int tz = G.K <= PCAMM_TZ_SMALL_K ? 32 : 16;                     // TileZ<K>
        const long long n_tiles = tile_count(G, tz), n_sub = n_tiles * GROUP_WARPS, plane = n_tiles * (TX * tz);
        const size_t words = (size_t)grad_record_words(n_sub, plane) * (size_t)m->S;          // every trial slot of every solve in flight
        int* rec = nullptr;
        cudaError_t e4 = dalloc(m, &rec, words);
        if (e4 == cudaSuccess) e4 = cudaMemsetAsync(rec, 0, sizeof(int) * words, st);
        if (e4 == cudaSuccess) e4 = cudaStreamSynchronize(st);
        if (e4 != cudaSuccess) {
            set_error(std::string("gradient records: ") + cudaGetErrorString(e4));
            cudaGetLastError();
            return fail(e4 == cudaErrorMemoryAllocation ? PCAMM_E_NOMEM : PCAMM_E_CUDA);
        }
        m->fs.grad_rec = rec;
        if (g_grad_aos) {
            float* aos = nullptr;
            e4 = dalloc(m, &aos, (size_t)V * aos_pitch(G.K));
            if (e4 == cudaSuccess) {
                k_u_to_aos<<<1184, 256, 0, st>>>(m->u, V, G.K, aos_pitch(G.K), aos);
                e4 = cudaStreamSynchronize(st);
            }
            if (e4 != cudaSuccess) {
                set_error(std::string("gradient records (u side by side): ") + cudaGetErrorString(e4));
                cudaGetLastError();
                return fail(e4 == cudaErrorMemoryAllocation ? PCAMM_E_NOMEM : PCAMM_E_CUDA);
            }
            m->fs.u_aos = aos;
        }
    }
    *out = m;
    return PCAMM_OK;
}

int pcamm_model_fields(pcamm_model* m, float* mean_dvf_out_dev, float* eig_dvf_out_dev, void* stream) {
    if (!m || !mean_dvf_out_dev || !eig_dvf_out_dev) return invalid("NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    const Geom& G = m->G;
    k_fields_to_mm<<<1184, 256, 0, st>>>(m->xbar, G.V, 3, G.hx, G.hy, G.hz, mean_dvf_out_dev);
    k_fields_to_mm<<<1184, 256, 0, st>>>(m->u, G.V, 3 * G.K, G.hx, G.hy, G.hz, eig_dvf_out_dev);
    count_launch(2);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(st));
    return PCAMM_OK;
}

int pcamm_reconstruct_batch(pcamm_model* m, int32_t B, const float* y_dev, const float* angles_rad_host,
                            const float* w_init_host, const pcamm_opts* opts, float* w_out_host, float* volumes_out_dev,
                            float* landmarks_out_host, pcamm_info* info, void* stream) {
    const int rc = solve_impl(m, B, y_dev, angles_rad_host, w_init_host, opts, w_out_host, volumes_out_dev,
                              landmarks_out_host, info, (cudaStream_t)stream);
    return (B == 1 && rc > 0) ? PCAMM_OK : rc;
}

int pcamm_reconstruct(pcamm_model* m, const float* y_dev, float angle_rad, const float* w_init_host,
                      const pcamm_opts* opts, float* w_out_host, float* volume_out_dev, float* landmarks_out_host,
                      pcamm_info* info, void* stream) {
    return solve_impl(m, 1, y_dev, &angle_rad, w_init_host, opts, w_out_host, volume_out_dev, landmarks_out_host, info,
                      (cudaStream_t)stream);
}

int pcamm_reconstruct_host(pcamm_model* m, const float* y_host, float angle_rad, const float* w_init_host,
                           const pcamm_opts* opts, float* w_out_host, float* volume_out_dev, float* landmarks_out_host,
                           pcamm_info* info, void* stream) {
    if (!m || !y_host) return invalid("NULL argument");
    float* y_stage = m->y_stage;
    CUDA_TRY(cudaMemcpyAsync(y_stage, y_host, (size_t)m->G.npix * sizeof(float), cudaMemcpyHostToDevice,
                             (cudaStream_t)stream));
    return solve_impl(m, 1, y_stage, &angle_rad, w_init_host, opts, w_out_host, volume_out_dev, landmarks_out_host, info,
                      (cudaStream_t)stream);
}

int pcamm_warp(pcamm_model* m, const float* w_host, float* volume_out_dev, void* stream) {
    if (!m || !w_host || !volume_out_dev) return invalid("NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    Seq q;
    int rc = hook_begin(m, nullptr, 0.f, w_host, 0.f, 0.f, 2, st, q);
    if (rc) return rc;
    launch_warp(q, m->G, m->fs, m->f0p, m->c.slots, 1, 0, volume_out_dev, m->G.V, nullptr, nullptr);
    if ((rc = check_seq(q, "warp"))) return rc;
    CUDA_TRY(cudaStreamSynchronize(st));
    return PCAMM_OK;
}

int pcamm_project(pcamm_model* m, const float* volume_dev, float angle_rad, float* proj_out_dev, void* stream) {
    if (!m || !volume_dev || !proj_out_dev) return invalid("NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    Seq q;
    int rc = hook_begin(m, nullptr, angle_rad, nullptr, 0.f, 0.f, 2, st, q);
    if (rc) return rc;
    launch_view_tables(q, m->G, m->c.solves, 1, m->col_hdr, m->slab_tab);
    launch_to_ray_layout(q, m->G, volume_dev, m->vol, m->occ);
    launch_project(q, m->G, m->c, 1, m->col_hdr, m->slab_tab, m->vol, m->occ, m->pseg, m->p, THEN_NONE, 0, 0, 0);
    if ((rc = check_seq(q, "project"))) return rc;
    CUDA_TRY(cudaMemcpyAsync(proj_out_dev, m->p, sizeof(float) * m->G.npix, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return PCAMM_OK;
}

int pcamm_backproject(pcamm_model* m, const float* r_dev, float angle_rad, float* volume_out_dev, void* stream) {
    if (!m || !r_dev || !volume_out_dev) return invalid("NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    Seq q;
    int rc = hook_begin(m, nullptr, angle_rad, nullptr, 0.f, 0.f, 2, st, q);
    if (rc) return rc;
    launch_resid(q, m->G, m->c.solves, m->c.in, 1, 1, m->p, r_dev, m->rL, m->utab, m->vtab, m->c.resid_part);
    if (m->G.projector == 1) backproject_rm(m, q, 1, 1, volume_out_dev, true);          // the hook wants every voxel
    else launch_backproject(q, m->G, m->c.solves, m->rL, m->utab, m->vtab, volume_out_dev);
    if ((rc = check_seq(q, "backproject"))) return rc;
    CUDA_TRY(cudaStreamSynchronize(st));
    return PCAMM_OK;
}

int pcamm_eval(pcamm_model* m, const float* y_dev, float angle_rad, const float* w_host, float a, float b, double* J_out,
               double* grad_out, double* ab_fit_out, float* proj_out_dev, void* stream) {
    if (!m || !y_dev || !w_host) return invalid("NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    const Geom& G = m->G;
    Seq q2;
    int rc = hook_begin(m, y_dev, angle_rad, w_host, a, b, 1, st, q2);
    if (rc) return rc;
    m->time_slots = 1;
    launch_ysums(q2, G, m->c, 1);
    launch_view_tables(q2, G, m->c.solves, 1, m->col_hdr, m->slab_tab);
    launch_warp(q2, G, m->fs, m->f0p, m->c.slots, 1, 1, m->vol, G.PV, m->occ, m->fs.grad_rec);
    launch_project(q2, G, m->c, 1, m->col_hdr, m->slab_tab, m->vol, m->occ, m->pseg, m->p, THEN_EVAL, 0, 0, 0);
    launch_resid(q2, G, m->c.solves, m->c.in, 1, 1, m->p, nullptr, m->rL, m->utab, m->vtab, m->c.resid_part);
    if (G.projector == 1) backproject_rm(m, q2, 1, 1, m->bvol, false);
    launch_grad(q2, G, m->fs, m->f0p, m->c, 1, m->rL, m->utab, m->vtab, m->bvol, GRAD_EVAL);
    if ((rc = check_seq(q2, "eval"))) return rc;
    if (proj_out_dev) CUDA_TRY(cudaMemcpyAsync(proj_out_dev, m->p, sizeof(float) * G.npix, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(m->h_solves, m->c.solves, sizeof(SolveState), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    const SolveState& s = m->h_solves[0];
    if (J_out) *J_out = s.J;
    if (grad_out) for (int k = 0; k < G.K; ++k) grad_out[k] = s.g[k];
    if (ab_fit_out) { ab_fit_out[0] = s.fit_a; ab_fit_out[1] = s.fit_b; }
    return PCAMM_OK;
}

int pcamm_traverse(pcamm_model* m, float angle_rad, int32_t iu, int32_t iv, int32_t cap, int32_t* ijk_out_host,
                   float* len_out_host, int32_t* n_out, void* stream) {
    if (!m || !ijk_out_host || !len_out_host || !n_out) return invalid("NULL argument");
    if (iu < 0 || iu >= m->G.nu || iv < 0 || iv >= m->G.nv || cap < 0) return invalid("pixel outside the detector");
    if (m->G.projector != 0) return invalid("pcamm_traverse lists Siddon's segments: it needs geometry.projector = 0");
    cudaStream_t st = (cudaStream_t)stream;
    Seq q;
    int rc = hook_begin(m, nullptr, angle_rad, nullptr, 0.f, 0.f, 2, st, q);
    if (rc) return rc;
    const int dcap = cap < m->trav_cap ? cap : m->trav_cap;
    launch_view_tables(q, m->G, m->c.solves, 1, m->col_hdr, m->slab_tab);
    launch_traverse(q, m->G, m->col_hdr, m->slab_tab, iu, iv, dcap, m->trav_ijk, m->trav_len, m->trav_n);
    if ((rc = check_seq(q, "traverse"))) return rc;
    int* h = m->h_trav;
    CUDA_TRY(cudaMemcpyAsync(h, m->trav_n, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(h + 1, m->trav_ijk, sizeof(int) * 3 * dcap, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(h + 1 + 3 * m->trav_cap, m->trav_len, sizeof(float) * dcap, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    const int n = h[0];
    *n_out = n;
    const int ncopy = n < dcap ? n : dcap;
    std::memcpy(ijk_out_host, h + 1, sizeof(int) * 3 * ncopy);
    std::memcpy(len_out_host, h + 1 + 3 * m->trav_cap, sizeof(float) * ncopy);
    if (n > cap) return invalid("cap too small for this ray");
    return PCAMM_OK;
}

int pcamm_localise(pcamm_model* m, const float* w_host, int32_t inv_max_iter, float inv_tol_mm, float* landmarks_out_host,
                   void* stream) {
    if (!m || !w_host || !landmarks_out_host) return invalid("NULL argument");
    if (m->M <= 0) return PCAMM_OK;
    cudaStream_t st = (cudaStream_t)stream;
    pcamm_opts o;
    pcamm_default_opts(&o);
    o.inv_max_iter = inv_max_iter; o.inv_tol_mm = inv_tol_mm;
    fill_call(m, o, 1, 1);
    SolveIn* in = h_solve_in(m);
    in[0].y = nullptr; in[0].angle = 0.f; in[0].a = in[0].b = 0.f;
    for (int k = 0; k < KMAX; ++k) in[0].w_init[k] = k < m->G.K ? w_host[k] : 0.f;
    int rc = push_call(m, 1, st);
    if (rc) return rc;
    Seq q;
    q.stream = st;
    launch_begin(q, m->G, m->c, 2);
    launch_invert(q, m->G, m->xbar, m->u, m->c, 1, m->M, m->lm0, m->lm_out);
    if ((rc = check_seq(q, "localise"))) return rc;
    CUDA_TRY(cudaMemcpyAsync(m->h_lm, m->lm_out, sizeof(double) * 3 * m->M, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    for (int i = 0; i < 3 * m->M; ++i) landmarks_out_host[i] = (float)m->h_lm[i];
    return PCAMM_OK;
}

int pcamm_tile_counts(pcamm_model* m, int32_t reset, int64_t* out, void* stream) {
    if (!m || !out) return invalid("NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long h[4] = {0ull, 0ull, 0ull, 0ull};
    CUDA_TRY(cudaMemcpyAsync(h, m->visited, sizeof(h), cudaMemcpyDeviceToHost, st));
    if (reset) CUDA_TRY(cudaMemsetAsync(m->visited, 0, sizeof(h), st));
    CUDA_TRY(cudaStreamSynchronize(st));
    const int tz = m->G.K <= PCAMM_TZ_SMALL_K ? 32 : 16;                  // TileZ<K>
    out[0] = (int64_t)h[0]; out[1] = (int64_t)h[1];
    out[2] = m->fs.use_tma ? (int64_t)tile_count(m->G, tz) : 0;
    out[3] = (int64_t)TX * tz;
    out[4] = (int64_t)h[2]; out[5] = (int64_t)h[3];
    return PCAMM_OK;
}

int pcamm_timeline(pcamm_model* m, int32_t cap, int32_t* kind_out, double* start_us_out, double* end_us_out,
                   int32_t* n_out, void* stream) {
    if (!m || !n_out || cap < 0 || (cap > 0 && (!kind_out || !start_us_out || !end_us_out))) return invalid("NULL argument");
    *n_out = 0;
    if (!m->tl) return invalid("the model was created without the timeline knob");
    std::vector<Timeline> h(1);
    CUDA_TRY(cudaMemcpyAsync(h.data(), m->tl, sizeof(Timeline), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
    const Timeline& t = h[0];
    const int n = (int)(t.n < (unsigned)TL_CAP ? t.n : (unsigned)TL_CAP);
    *n_out = n;
    for (int i = 0; i < n && i < cap; ++i) {
        kind_out[i] = t.kind[i];
        start_us_out[i] = 1e-3 * (double)(t.t0[i] - t.t0[0]);
        end_us_out[i] = 1e-3 * (double)(t.t1[i] - t.t0[0]);
    }
    return PCAMM_OK;
}

int pcamm_tune(const char* name, int32_t value) {
    if (!name) return invalid("NULL argument");
    const std::string n(name);
    if (n == "project_chunks_per_segment") { g_chunks_per_segment = value < 0 ? 0 : value; return PCAMM_OK; }
    if (n == "project_scan_slabs") { g_scan_slabs = value < 0 ? 0 : value; return PCAMM_OK; }
    if (n == "timeline") { g_timeline = value != 0; return PCAMM_OK; }
    if (n == "grad_records") { g_grad_records = value != 0; return PCAMM_OK; }
    if (n == "pdl") { g_pdl = value != 0; return PCAMM_OK; }
    if (n == "grad_aos") { g_grad_aos = value != 0; return PCAMM_OK; }
    if (n == "static_passes") {
        if (value < -1 || value > 64) return invalid("static_passes must be -1 .. 64");
        g_static_passes = value;
        return PCAMM_OK;
    }
    return invalid("unknown knob: " + n);
}

int pcamm_time_slots(pcamm_model* m, int32_t nslots, const float* w_host, void* stream) {
    if (!m || !w_host) return invalid("NULL argument");
    if (nslots < 1 || nslots > m->S) return invalid("nslots outside [1, max_batch * max_candidates]");
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<SlotState> h((size_t)nslots);
    for (int s = 0; s < nslots; ++s) {
        std::memset(&h[s], 0, sizeof(SlotState));
        for (int k = 0; k < m->G.K; ++k) h[s].w[k] = w_host[s * m->G.K + k];
        h[s].active = 1; h[s].solve = 0;
    }
    CUDA_TRY(cudaMemcpyAsync(m->c.slots, h.data(), sizeof(SlotState) * nslots, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    m->time_slots = nslots;
    return PCAMM_OK;
}

int pcamm_time_kernel(pcamm_model* m, int32_t which, int32_t reps, float* ms_out, void* stream) {
    if (!m || !ms_out || reps < 1 || which < 0 || which > 2) return invalid("invalid argument");
    cudaStream_t st = (cudaStream_t)stream;
    const Geom& G = m->G;
    Seq q;
    q.stream = st;
    CUDA_TRY(cudaEventRecord(m->ev0, st));
    for (int i = 0; i < reps; ++i) {
        if (which == 0)
            launch_warp(q, G, m->fs, m->f0p, m->c.slots, m->time_slots, 1, m->vol, G.PV, m->occ, m->fs.grad_rec);
        else if (which == 1)
            launch_project(q, G, m->c, m->time_slots, m->col_hdr, m->slab_tab, m->vol, m->occ, m->pseg, m->p, THEN_NONE, 0, 0, 0);
        else
            launch_grad(q, G, m->fs, m->f0p, m->c, 1, m->rL, m->utab, m->vtab, m->bvol, GRAD_NONE);
    }
    CUDA_TRY(cudaEventRecord(m->ev1, st));
    int rc = check_seq(q, "time_kernel");
    if (rc) return rc;
    CUDA_TRY(cudaEventSynchronize(m->ev1));
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, m->ev0, m->ev1));
    *ms_out = ms / (float)reps;
    return PCAMM_OK;
}

}  // extern "C"
