// Host-side plumbing shared by the translation units of libpcamm: the kernel sequencer (the same
// launcher code either launches on a stream or appends kernel nodes to a CUDA graph) and the
// launcher prototypes of each step of the hot path.
#pragma once

#include <cuda_runtime.h>

#include <mutex>
#include <string>
#include <vector>

#include "common.cuh"
#include "stream.cuh"

struct pcamm_model;

namespace pcamm {

void set_error(const std::string& msg);
void count_launch(long long n);
int model_K(const pcamm_model* m);   // api.cu

// Function attributes (the opt-in to more than 48 KB of dynamic shared memory) are per device:
// runs fn() the first time it is called while a given device is current (thread safe).
class DeviceOnce {
    std::mutex mu_;
    std::vector<char> done_;

  public:
    template <class F>
    cudaError_t run(F fn) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        std::lock_guard<std::mutex> lock(mu_);
        if ((int)done_.size() > dev && done_[dev]) return cudaSuccess;
        e = fn();
        if (e == cudaSuccess) {
            if ((int)done_.size() <= dev) done_.resize(dev + 1, 0);
            done_[dev] = 1;
        }
        return e;
    }
};

// A linear sequence of kernels.  stream mode: cudaLaunchKernel on `stream`.  graph mode: each
// kernel becomes a node of `graph` depending on the previous one, so the solve can be replayed
// as one graph launch with device-side while-loops (cudaGraphCondTypeWhile) around sub-sequences.
struct Seq {
    cudaStream_t stream = nullptr;
    cudaGraph_t graph = nullptr;
    cudaGraphNode_t last = nullptr;
    bool has_last = false;
    cudaError_t err = cudaSuccess;
    int n_kernels = 0;        // kernels appended so far (not counting the bodies of while-loops)
    bool pdl = false;         // graph mode: kernel -> kernel edges are programmatic (common.cuh grid_dependency_wait)
    bool last_is_kernel = false;
    bool plain_next = false;  // the next kernel takes a plain edge whatever pdl says (then reset)

    bool graph_mode() const { return graph != nullptr; }

    template <class... KArgs, class... Args>
    void launch(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, Args... args) {
        if (err != cudaSuccess) return;
        launch_impl<KArgs...>(kernel, grid, block, smem, static_cast<KArgs>(args)...);
    }

    // Appends a while-loop node; the kernels of its body go to the returned sequence.
    Seq add_while(cudaGraphConditionalHandle handle) {
        Seq body;
        body.pdl = pdl;
        if (err != cudaSuccess) { body.err = err; return body; }
        cudaGraphNodeParams p = {};
        p.type = cudaGraphNodeTypeConditional;
        p.conditional.handle = handle;
        p.conditional.type = cudaGraphCondTypeWhile;
        p.conditional.size = 1;
        cudaGraphNode_t node;
        err = cudaGraphAddNode(&node, graph, has_last ? &last : nullptr, has_last ? 1 : 0, &p);
        if (err != cudaSuccess) { body.err = err; return body; }
        last = node;
        has_last = true;
        last_is_kernel = false;
        body.graph = p.conditional.phGraph_out[0];
        return body;
    }

  private:
    template <class... KArgs>
    void launch_impl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, KArgs... args) {
        void* argv[] = {(void*)&args...};
        ++n_kernels;
        if (graph) {
            cudaKernelNodeParams kp = {};
            kp.func = (void*)kernel;
            kp.gridDim = grid;
            kp.blockDim = block;
            kp.sharedMemBytes = (unsigned)smem;
            kp.kernelParams = argv;
            cudaGraphNode_t node;
            const bool programmatic = pdl && has_last && last_is_kernel && !plain_next;
            plain_next = false;
            if (programmatic) {
                cudaGraphNodeParams np = {};
                np.type = cudaGraphNodeTypeKernel;
                np.kernel.func = kp.func;
                np.kernel.gridDim = grid;
                np.kernel.blockDim = block;
                np.kernel.sharedMemBytes = (unsigned)smem;
                np.kernel.kernelParams = argv;
                cudaGraphEdgeData ed = {};
                ed.from_port = cudaGraphKernelNodePortProgrammatic;
                ed.to_port = cudaGraphKernelNodePortDefault;
                ed.type = cudaGraphDependencyTypeProgrammatic;
                err = cudaGraphAddNode_v2(&node, graph, &last, &ed, 1, &np);
            } else {
                err = cudaGraphAddKernelNode(&node, graph, has_last ? &last : nullptr, has_last ? 1 : 0, &kp);
            }
            last = node;
            has_last = true;
            last_is_kernel = true;
        } else {
            err = cudaLaunchKernel((const void*)kernel, grid, block, argv, smem, stream);
            count_launch(1);
        }
    }
};

// ---- a-1 (warp.cu)
// f[s] = warp(f0, xbar + U w[s]) for every active slot; ray_layout: the z-fastest layout the
// projector reads (slot stride G.PV), else the standard [z][y][x] (slot stride G.V).
// occ: occupancy of the volumes written (ray layout only; common.cuh), else NULL
// rec: base of the slots' gradient records (stream.cuh GradRecords; written with the ray layout
// only) or NULL
void launch_warp(Seq& q, const Geom& G, const FieldStream& fs, const float* f0, const SlotState* slots, int nslots,
                 int ray_layout, float* vol_out, long long slot_stride, unsigned char* occ, int* rec);

// ---- a-2 (project.cu)
int project_blocks(const Geom& G);
int max_slabs(const Geom& G);
extern int g_chunks_per_segment, g_scan_slabs;     // measurement knobs (pcamm_tune): 0 = automatic
extern int g_pdl;                                  // 1: programmatic kernel -> kernel edges in the solve graphs
extern int g_timeline;                             // 1: models record the kernel timeline of their solves
bool project_fits(const Geom& G);    // the knots of one scan row set fit into shared memory (nz up to ~ 4000)
// in-plane traversal tables of the views of solves 0..B-1 (once per solve: the angle is fixed)
void launch_view_tables(Seq& q, const Geom& G, const SolveState* solves, int B, ColHdr* hdr, SlabEntry* tab);
int project_segments(const Geom& G);
// p[s] = P f[s] for every active slot (volumes in the ray layout; pseg: scratch
// [nslots][segments][nu][nv] for the per-segment partial line integrals), the a-3 partial sums
// {sum p, sum y p, sum (p - a y - b)^2}, and then the control step `then` (THEN_*, common.cuh);
// n_before: kernels of the sequence in front of this launch.
void launch_project(Seq& q, const Geom& G, const CtlBufs& c, int nslots, const ColHdr* hdr, const SlabEntry* tab,
                    const float* vol, const unsigned char* occ, float* pseg, float* p, int then,
                    cudaGraphConditionalHandle h, int use_cond, int n_before);
// the ray-marching variant (raymarch.cu; pcamm_geometry.projector = 1): p[s] and the a-3 partial sums
// (no control step: launch_project adds it), and B[b] = P^T r for the solves that need a gradient
// (force: for all), r taken from rL = r |D - S|
void launch_project_rm(Seq& q, const Geom& G, const CtlBufs& c, int nslots, const float* vol, float* p);
// rec, n_sub, cap, mask: the gradient records of the slots (stream.cuh GradRecords) and a scratch of
// record_mask_words(G) words, where the gradient of the one solve will read B at the recorded voxels
// only (the scatter then skips every other voxel); else NULL / 0
long long record_mask_words(const Geom& G);
void launch_backproject_rm(Seq& q, const Geom& G, const SolveState* solves, int B, int force, const float* rL, float* bvol,
                           int* rec, long long n_sub, int cap, unsigned* mask);
// hooks: standard layout -> ray layout; one ray of the view of solve 0
void launch_to_ray_layout(Seq& q, const Geom& G, const float* vol_std, float* vol_ray, unsigned char* occ);
void launch_traverse(Seq& q, const Geom& G, const ColHdr* hdr, const SlabEntry* tab, int iu, int iv, int cap,
                     int* ijk, float* len, int* n_out);

// ---- a-3 / a-4 (gradient.cu)
int resid_blocks(const Geom& G);
int grad_blocks(const Geom& G, const FieldStream& fs);
int grad_gather_blocks(const Geom& G, const FieldStream& fs);      // partial sums of the gather over the gradient records (one solve)
void launch_build_cellmap(cudaStream_t st, const Geom& G, const float* f0, unsigned char* cellmap);
// r = p - a y - b, rL = r * |D - S|, per-view tables, partial sums of r^2; p of solve b is read
// from its accepted slot.
// force: also for solves that are no longer running (closing pass); r_direct: take r from there.
void launch_resid(Seq& q, const Geom& G, const SolveState* solves, const SolveIn* in, int B, int force,
                  const float* p, const float* r_direct, float* rL, float4* utab, float2* vtab, double* partials);
// g = 2 U^T (df/dx) P^T r for the solves that need it (control.cuh needs_gradient), per-block partial
// sums [B][blocks][K], and then the control step `mode` (GRAD_*).
// bvol: NULL (Siddon: B_j is gathered from rL with the exact path lengths) or the backprojection
// volumes [B][V] of launch_backproject_rm
void launch_grad(Seq& q, const Geom& G, const FieldStream& fs, const float* f0, const CtlBufs& c, int B,
                 const float* rL, const float4* utab, const float2* vtab, const float* bvol, int mode);
// hook: B = P^T r as a volume for solve 0's view (rL/utab/vtab as written by launch_resid).
void launch_backproject(Seq& q, const Geom& G, const SolveState* solves, const float* rL, const float4* utab,
                        const float2* vtab, float* vol_out);

// ---- control (control.cu; the steps themselves are device functions of control.cuh)
int ysum_blocks(const Geom& G);
void launch_ysums(Seq& q, const Geom& G, const CtlBufs& c, int B);
// begin: views, w = w_init, slot 0 of every solve = w_init.  mode 0 solve, 1 eval hook.
void launch_begin(Seq& q, const Geom& G, const CtlBufs& c, int mode);
// the single-block control steps (control.cuh) behind a projection / a gradient pass; in graph mode
// the first also hands LoopFlags::loop_cond to the while-node.  n_before: kernels of the sequence
// in front of it (launch accounting)
void launch_ctl_after_project(Seq& q, const Geom& G, const CtlBufs& c, int then, cudaGraphConditionalHandle h,
                              int use_cond, int n_before);
void launch_ctl_after_grad(Seq& q, const Geom& G, const CtlBufs& c, int mode);
void launch_ctl_final(Seq& q, const Geom& G, const CtlBufs& c, SlotState* out_slots, int n_seq);
// a-6: landmarks [B][M][3]
void launch_invert(Seq& q, const Geom& G, const float* xbar, const float* u, const CtlBufs& c, int B, int M,
                   const float* r0, double* r_out);

}  // namespace pcamm
