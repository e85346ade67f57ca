// a-3 for callers that cannot allocate: the intensity fit (Eq. 4) and the cost
// (Eq. 2) of a projection pair (p, y), with every intermediate in ONE file-scope
// device array of fixed size instead of a model's cudaMalloc'ed scratch.
//
//   Sp = sum p, Sy = sum y, Syy = sum y^2, Syp = sum y p          (double, fixed order)
//   (a, b) = argmin || p - a y - b ||^2                           (control.cuh lsfit, the solve's own)
//   J = sum (p_i - a y_i - b)^2                                   (second pass, as k_resid forms it)
//
// This is the arithmetic the solve runs behind every projection (the projector's per-column partial
// sums, the control step's lsfit, k_resid's sum of r^2), as a variant of its own: block partial sums
// -> the last block to finish adds them in index order.  pcamm_eval needs a model (which allocates
// when it is created); pcamm_fit_cost_static needs nothing but its arguments.
//
// The scratch: g_fit_scratch below, FIT_SCRATCH_DOUBLES doubles = 41 216 bytes, held by every GPU
// that loads the library until the process exits.  Layout: a header of 32 doubles (two tickets, then
// a, b, status), then [FIT_MAX_BLOCKS][4] partial sums of the first pass and [FIT_MAX_BLOCKS] of the
// second.  One block takes FIT_CHUNK = 4096 pixels, so the array bounds the input at
// PCAMM_STATIC_MAX_PIXELS = 2^22 pixels (a 2048 x 2048 detector); more is rejected.
// Every call shares the array and it keeps the last call's contents: the header (the tickets must
// start at zero) is cleared on the stream at the start of every call; the partial sums a call reads
// are the ones it wrote.  Two calls that overlap on the GPU (different streams, or threads) race on
// it: callers serialise.
#include "internal.h"
#include "control.cuh"

namespace pcamm {

namespace {

constexpr int FT = 256;                    // threads of a block
constexpr int FIT_PER_THREAD = 16;
constexpr int FIT_CHUNK = FT * FIT_PER_THREAD;                                  // pixels per block
constexpr long long FIT_MAX_PIXELS = PCAMM_STATIC_MAX_PIXELS;
constexpr int FIT_MAX_BLOCKS = (int)(FIT_MAX_PIXELS / FIT_CHUNK);               // 1024
constexpr int FIT_HEADER = 32;             // doubles: [0] the two tickets (as unsigned), [2] a, [3] b, [4] status
constexpr int FIT_PART1 = FIT_HEADER, FIT_PART2 = FIT_PART1 + 4 * FIT_MAX_BLOCKS;
constexpr int FIT_SCRATCH_DOUBLES = FIT_PART2 + FIT_MAX_BLOCKS;
static_assert(FIT_MAX_PIXELS % FIT_CHUNK == 0, "whole blocks");

// In host code this name is a host-side stand-in, not a device address: the kernels get the address
// cudaGetSymbolAddress returns for the current device (fit_scratch below).
static __device__ __align__(256) double g_fit_scratch[FIT_SCRATCH_DOUBLES];

// true in the block that finishes last (its reads then see every block's partial sums)
__device__ __forceinline__ bool last_block_done(unsigned* ticket, int* s_last) {
    __syncthreads();                                   // the block's stores are ordered before thread 0's fence
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned k = atomicAdd(ticket, 1u);
        *s_last = k == gridDim.x - 1u;
        if (*s_last) __threadfence();
    }
    __syncthreads();
    return *s_last != 0;
}

// sum over the blocks' partial sums part[i * stride + q], i = 0 .. n - 1, in a fixed order
__device__ __forceinline__ double sum_partials(const double* part, int n, int stride, int q, double* red) {
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += FT) v += __ldcg(part + (long long)i * stride + q);
    return block_sum<FT>(v, red);
}

// Pass 1: the four sums; the last block fits (a, b).
__global__ void __launch_bounds__(FT)
k_fit_sums(const float* __restrict__ p, const float* __restrict__ y, long long npix, double* scratch, double* __restrict__ out) {
    __shared__ double red[FT / 32];
    __shared__ int s_last;
    double sp = 0.0, sy = 0.0, syy = 0.0, syp = 0.0;
    const long long i0 = (long long)blockIdx.x * FIT_CHUNK + threadIdx.x;
#pragma unroll 4
    for (int r = 0; r < FIT_PER_THREAD; ++r) {
        const long long i = i0 + (long long)r * FT;
        if (i < npix) {
            const double pv = (double)__ldg(p + i), yv = (double)__ldg(y + i);
            sp += pv; sy += yv; syy += yv * yv; syp += yv * pv;
        }
    }
    const double Sp = block_sum<FT>(sp, red), Sy = block_sum<FT>(sy, red);
    const double Syy = block_sum<FT>(syy, red), Syp = block_sum<FT>(syp, red);
    double* part = scratch + FIT_PART1;
    if (threadIdx.x == 0) {
        part[4 * blockIdx.x + 0] = Sp; part[4 * blockIdx.x + 1] = Sy;
        part[4 * blockIdx.x + 2] = Syy; part[4 * blockIdx.x + 3] = Syp;
    }
    if (!last_block_done(reinterpret_cast<unsigned*>(scratch), &s_last)) return;
    const double tp = sum_partials(part, gridDim.x, 4, 0, red), ty = sum_partials(part, gridDim.x, 4, 1, red);
    const double tyy = sum_partials(part, gridDim.x, 4, 2, red), typ = sum_partials(part, gridDim.x, 4, 3, red);
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        int status = PCAMM_OK;
        if (!isfinite(tp) || !isfinite(ty) || !isfinite(tyy) || !isfinite(typ)) status = PCAMM_E_NONFINITE;
        else if (!lsfit((double)npix, ty, tyy, tp, typ, &a, &b)) status = PCAMM_E_SINGULAR;      // y constant (reading A8)
        scratch[2] = a; scratch[3] = b; scratch[4] = (double)status;
        out[3] = tp; out[4] = ty; out[5] = tyy; out[6] = typ;
    }
}

// Pass 2: J at the fitted (a, b); the last block writes the results.
__global__ void __launch_bounds__(FT)
k_fit_cost(const float* __restrict__ p, const float* __restrict__ y, long long npix, double* scratch, double* __restrict__ out) {
    __shared__ double red[FT / 32];
    __shared__ int s_last;
    const double a = __ldcg(scratch + 2), b = __ldcg(scratch + 3);             // pass 1 has completed (same stream)
    double rr = 0.0;
    const long long i0 = (long long)blockIdx.x * FIT_CHUNK + threadIdx.x;
#pragma unroll 4
    for (int r = 0; r < FIT_PER_THREAD; ++r) {
        const long long i = i0 + (long long)r * FT;
        if (i < npix) {
            const double res = (double)__ldg(p + i) - a * (double)__ldg(y + i) - b;       // Eq. (2)
            rr += res * res;
        }
    }
    const double R = block_sum<FT>(rr, red);
    double* part = scratch + FIT_PART2;
    if (threadIdx.x == 0) part[blockIdx.x] = R;
    if (!last_block_done(reinterpret_cast<unsigned*>(scratch) + 1, &s_last)) return;
    const double J = sum_partials(part, gridDim.x, 1, 0, red);
    if (threadIdx.x == 0) {
        out[0] = a; out[1] = b; out[2] = J; out[7] = __ldcg(scratch + 4);
    }
}

// The device address of g_fit_scratch on the current device: looked up once per device, with that
// device current (thread safe).
cudaError_t fit_scratch(double** ptr) {
    static std::mutex mu;
    static std::vector<double*> by_device;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    if ((int)by_device.size() <= dev) by_device.resize(dev + 1, nullptr);
    if (!by_device[dev]) {
        double* d = nullptr;
        e = cudaGetSymbolAddress((void**)&d, g_fit_scratch);
        if (e != cudaSuccess) return e;
        by_device[dev] = d;
    }
    *ptr = by_device[dev];
    return cudaSuccess;
}

}  // namespace

}  // namespace pcamm

using namespace pcamm;

extern "C" int pcamm_fit_cost_static(const float* p_dev, const float* y_dev, int64_t npix, double* out_dev, void* stream) {
    if (!p_dev || !y_dev || !out_dev) { set_error("pcamm_fit_cost_static: NULL argument"); return PCAMM_E_INVALID; }
    if (npix < 1 || npix > FIT_MAX_PIXELS) {
        set_error("pcamm_fit_cost_static: npix = " + std::to_string((long long)npix) + " is outside 1 .. " +
                  std::to_string(FIT_MAX_PIXELS) + " (PCAMM_STATIC_MAX_PIXELS: the static scratch array holds no more)");
        return PCAMM_E_INVALID;
    }
    cudaStream_t st = (cudaStream_t)stream;
    double* scratch = nullptr;
    cudaError_t e = fit_scratch(&scratch);
    // the tickets must start at zero, whatever an earlier call left (no allocation: a memset node on the stream)
    if (e == cudaSuccess) e = cudaMemsetAsync(scratch, 0, sizeof(double) * FIT_HEADER, st);
    if (e == cudaSuccess) {
        const unsigned blocks = (unsigned)((npix + FIT_CHUNK - 1) / FIT_CHUNK);
        k_fit_sums<<<blocks, FT, 0, st>>>(p_dev, y_dev, (long long)npix, scratch, out_dev);
        k_fit_cost<<<blocks, FT, 0, st>>>(p_dev, y_dev, (long long)npix, scratch, out_dev);
        count_launch(2);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        set_error(std::string("pcamm_fit_cost_static: ") + cudaGetErrorString(e));
        return PCAMM_E_CUDA;
    }
    return PCAMM_OK;
}
