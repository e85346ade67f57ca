// PCA motion model from N training DVFs (include/pcamm.h, pcamm_pca_fit).
//
// PAPER.md:L63-69 (section 2.1, Eq. 1): x(t) ~ xbar + sum_k u_k w_k(t), xbar the sample mean and
// u_k the eigenvectors with the largest eigenvalues; the samples are the DVFs of
// the training phases.  Snapshot method (the samples are 3V long and there are N <= 16 of them):
//
//   k_pca_gram    one pass over the N samples: per element the mean over the samples, the
//                 centred values, and their N(N+1)/2 products summed (float per thread over a
//                 short run, double from the warp upwards, fixed order) -> the N x N scatter
//                 matrix G_ij = <D_i - xbar, D_j - xbar>.  HBM-bound: 4N bytes per element
//                 against N(N+1)/2 FMAs (45 for N = 9), so plain FMAs, not tensor cores: a 9 x 9
//                 output is too small for an MMA tile and the ALUs are idle anyway.
//   host          eigenpairs of G by cyclic Jacobi in double (N <= 16), descending; sign rule of
//                 reading A12 / B10 taken from the eigenvector's entry of the reference sample
//                 (u_k . (D_r - xbar) = sqrt(lambda_k) v_rk).
//   k_pca_fields  second pass: xbar and u_k = sum_i v_ik (D_i - xbar) / sqrt(lambda_k) written
//                 straight into the caller's planes (4N bytes read, 4(K+1) written per element).
#include <algorithm>
#include <cmath>
#include <string>
#include <vector>

#include "../../include/pcamm.h"
#include "internal.h"

namespace pcamm {
namespace {

constexpr int PCA_NT = 256;
constexpr int PCA_MAXN = PCAMM_PCA_MAX_SAMPLES;
constexpr int PCA_RUN = 32;    // items (of 1 or 4 elements) a thread sums in float before the double reduction

struct PcaCoef {
    float c[PCAMM_KMAX][PCA_MAXN];   // v_ik / sqrt(lambda_k)
};

template <int N>
__device__ __forceinline__ void centre(const float (&x)[N], float (&c)[N], float& mean) {
    float s = x[0];
#pragma unroll
    for (int i = 1; i < N; ++i) s += x[i];
    mean = s / (float)N;
#pragma unroll
    for (int i = 0; i < N; ++i) c[i] = x[i] - mean;
}

// d: N samples of n floats, `stride` floats apart.  V4: n % 4 == 0 and all rows 16 B aligned.
template <int N, bool V4>
__global__ void __launch_bounds__(PCA_NT) k_pca_gram(const float* __restrict__ d, long long n, long long stride,
                                                     double* __restrict__ partials) {
    constexpr int NP = N * (N + 1) / 2;
    constexpr int W = V4 ? 4 : 1;
    float acc[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) acc[p] = 0.f;
    const long long items = n / W;
    for (long long e = (long long)blockIdx.x * PCA_NT + threadIdx.x; e < items; e += (long long)gridDim.x * PCA_NT) {
        float x[W][N];
#pragma unroll
        for (int i = 0; i < N; ++i) {
            if (V4) {
                const float4 v = __ldcs(reinterpret_cast<const float4*>(d + i * stride) + e);
                x[0][i] = v.x; x[1 % W][i] = v.y; x[2 % W][i] = v.z; x[3 % W][i] = v.w;
            } else {
                x[0][i] = __ldcs(d + i * stride + e);
            }
        }
#pragma unroll
        for (int l = 0; l < W; ++l) {
            float c[N], mean;
            centre<N>(x[l], c, mean);
            int p = 0;
#pragma unroll
            for (int i = 0; i < N; ++i)
#pragma unroll
                for (int j = i; j < N; ++j) acc[p] = fmaf(c[i], c[j], acc[p]), ++p;
        }
    }
    __shared__ double s_part[PCA_NT / 32][NP];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const double v = warp_sum((double)acc[p]);
        if (lane == 0) s_part[wid][p] = v;
    }
    __syncthreads();
    for (int p = threadIdx.x; p < NP; p += PCA_NT) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < PCA_NT / 32; ++w) s += s_part[w][p];
        partials[(size_t)blockIdx.x * NP + p] = s;
    }
}

template <int N, bool V4>
__global__ void __launch_bounds__(PCA_NT) k_pca_fields(const float* __restrict__ d, long long n, long long stride,
                                                       PcaCoef coef, int K, float* __restrict__ mean_out,
                                                       float* __restrict__ eig_out) {
    constexpr int W = V4 ? 4 : 1;
    const long long items = n / W;
    for (long long e = (long long)blockIdx.x * PCA_NT + threadIdx.x; e < items; e += (long long)gridDim.x * PCA_NT) {
        float x[W][N];
#pragma unroll
        for (int i = 0; i < N; ++i) {
            if (V4) {
                const float4 v = __ldcs(reinterpret_cast<const float4*>(d + i * stride) + e);
                x[0][i] = v.x; x[1 % W][i] = v.y; x[2 % W][i] = v.z; x[3 % W][i] = v.w;
            } else {
                x[0][i] = __ldcs(d + i * stride + e);
            }
        }
        float c[W][N], mean[W];
#pragma unroll
        for (int l = 0; l < W; ++l) centre<N>(x[l], c[l], mean[l]);
        if (V4) reinterpret_cast<float4*>(mean_out)[e] = make_float4(mean[0], mean[1 % W], mean[2 % W], mean[3 % W]);
        else mean_out[e] = mean[0];
        for (int k = 0; k < K; ++k) {
            float u[W];
#pragma unroll
            for (int l = 0; l < W; ++l) {
                float s = 0.f;
#pragma unroll
                for (int i = 0; i < N; ++i) s = fmaf(coef.c[k][i], c[l][i], s);
                u[l] = s;
            }
            if (V4) reinterpret_cast<float4*>(eig_out + (size_t)k * n)[e] = make_float4(u[0], u[1 % W], u[2 % W], u[3 % W]);
            else eig_out[(size_t)k * n + e] = u[0];
        }
    }
}

// Eigenpairs of the symmetric n x n matrix A (row-major, destroyed) by cyclic Jacobi rotations:
// lam descending, V[i * n + k] = component i of eigenvector k.
void jacobi_eigen(int n, std::vector<double>& A, std::vector<double>& V, std::vector<double>& lam) {
    V.assign((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i) V[(size_t)i * n + i] = 1.0;
    for (int sweep = 0; sweep < 64; ++sweep) {
        double off = 0.0, diag = 0.0;
        for (int i = 0; i < n; ++i) {
            diag += A[(size_t)i * n + i] * A[(size_t)i * n + i];
            for (int j = i + 1; j < n; ++j) off += A[(size_t)i * n + j] * A[(size_t)i * n + j];
        }
        if (off <= 1e-32 * diag) break;
        for (int p = 0; p < n - 1; ++p)
            for (int q = p + 1; q < n; ++q) {
                const double apq = A[(size_t)p * n + q];
                if (apq == 0.0) continue;
                const double theta = (A[(size_t)q * n + q] - A[(size_t)p * n + p]) / (2.0 * apq);
                const double t = (theta >= 0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
                const double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
                for (int k = 0; k < n; ++k) {        // columns p, q
                    const double akp = A[(size_t)k * n + p], akq = A[(size_t)k * n + q];
                    A[(size_t)k * n + p] = c * akp - s * akq;
                    A[(size_t)k * n + q] = s * akp + c * akq;
                }
                for (int k = 0; k < n; ++k) {        // rows p, q
                    const double apk = A[(size_t)p * n + k], aqk = A[(size_t)q * n + k];
                    A[(size_t)p * n + k] = c * apk - s * aqk;
                    A[(size_t)q * n + k] = s * apk + c * aqk;
                }
                for (int k = 0; k < n; ++k) {
                    const double vkp = V[(size_t)k * n + p], vkq = V[(size_t)k * n + q];
                    V[(size_t)k * n + p] = c * vkp - s * vkq;
                    V[(size_t)k * n + q] = s * vkp + c * vkq;
                }
            }
    }
    std::vector<int> order(n);
    for (int i = 0; i < n; ++i) order[i] = i;
    std::stable_sort(order.begin(), order.end(),
                     [&](int a, int b) { return A[(size_t)a * n + a] > A[(size_t)b * n + b]; });
    std::vector<double> Vs((size_t)n * n);
    lam.resize(n);
    for (int k = 0; k < n; ++k) {
        lam[k] = A[(size_t)order[k] * n + order[k]];
        for (int i = 0; i < n; ++i) Vs[(size_t)i * n + k] = V[(size_t)i * n + order[k]];
    }
    V.swap(Vs);
}

int pca_blocks(long long items) {
    int dev = 0, n_sm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    const long long want = (items + (long long)PCA_NT * PCA_RUN - 1) / ((long long)PCA_NT * PCA_RUN);
    const long long lo = n_sm, hi = (long long)n_sm * 64;
    const long long b = std::min(std::max(want, lo), hi);
    return (int)((b + n_sm - 1) / n_sm * n_sm);      // whole waves of the SMs
}

template <int N>
cudaError_t launch_gram(const float* d, long long n, long long stride, bool v4, int blocks, double* partials,
                        cudaStream_t st) {
    if (v4) k_pca_gram<N, true><<<blocks, PCA_NT, 0, st>>>(d, n, stride, partials);
    else k_pca_gram<N, false><<<blocks, PCA_NT, 0, st>>>(d, n, stride, partials);
    count_launch(1);
    return cudaGetLastError();
}
template <int N>
cudaError_t launch_fields(const float* d, long long n, long long stride, bool v4, int blocks, const PcaCoef& coef,
                          int K, float* mean_out, float* eig_out, cudaStream_t st) {
    if (v4) k_pca_fields<N, true><<<blocks, PCA_NT, 0, st>>>(d, n, stride, coef, K, mean_out, eig_out);
    else k_pca_fields<N, false><<<blocks, PCA_NT, 0, st>>>(d, n, stride, coef, K, mean_out, eig_out);
    count_launch(1);
    return cudaGetLastError();
}

#define PCA_DISPATCH(N_, CALL)                                                                          \
    switch (N_) {                                                                                       \
        case 2: { constexpr int NN = 2; CALL; break; }   case 3: { constexpr int NN = 3; CALL; break; }   \
        case 4: { constexpr int NN = 4; CALL; break; }   case 5: { constexpr int NN = 5; CALL; break; }   \
        case 6: { constexpr int NN = 6; CALL; break; }   case 7: { constexpr int NN = 7; CALL; break; }   \
        case 8: { constexpr int NN = 8; CALL; break; }   case 9: { constexpr int NN = 9; CALL; break; }   \
        case 10: { constexpr int NN = 10; CALL; break; } case 11: { constexpr int NN = 11; CALL; break; } \
        case 12: { constexpr int NN = 12; CALL; break; } case 13: { constexpr int NN = 13; CALL; break; } \
        case 14: { constexpr int NN = 14; CALL; break; } case 15: { constexpr int NN = 15; CALL; break; } \
        case 16: { constexpr int NN = 16; CALL; break; }                                                \
        default: break;                                                                                 \
    }

int fail(int code, const std::string& msg) {
    set_error(msg);
    return code;
}
int cuda_fail(const char* what, cudaError_t e) {
    set_error(std::string(what) + ": " + cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? PCAMM_E_NOMEM : PCAMM_E_CUDA;
}

}  // namespace
}  // namespace pcamm

using namespace pcamm;

extern "C" int pcamm_pca_fit(int64_t n_per_sample, int32_t N, int32_t K, const float* dvfs_dev, int32_t sign_ref,
                             float* mean_out_dev, float* eig_out_dev, double* eigenvalues_out_host,
                             double* coeffs_out_host, float* pass_ms_out_host, void* stream) {
    if (!dvfs_dev || !mean_out_dev || !eig_out_dev) return fail(PCAMM_E_INVALID, "NULL argument");
    if (n_per_sample < 1) return fail(PCAMM_E_INVALID, "n_per_sample < 1");
    if (N < 2 || N > PCA_MAXN) return fail(PCAMM_E_INVALID, "number of samples outside [2, PCAMM_PCA_MAX_SAMPLES]");
    if (K < 1 || K > PCAMM_KMAX || K > N - 1) return fail(PCAMM_E_INVALID, "K outside [1, min(PCAMM_KMAX, N - 1)]");
    if (sign_ref < -1 || sign_ref >= N) return fail(PCAMM_E_INVALID, "sign_ref outside [-1, N)");
    if (sign_ref < 0) sign_ref = N / 2;
    cudaStream_t st = (cudaStream_t)stream;
    const long long n = n_per_sample;
    const bool v4 = n % 4 == 0 && ((uintptr_t)dvfs_dev % 16 == 0) && ((uintptr_t)mean_out_dev % 16 == 0) &&
                    ((uintptr_t)eig_out_dev % 16 == 0);
    const int blocks = pca_blocks(v4 ? n / 4 : n);
    const int NP = N * (N + 1) / 2;
    double* partials = nullptr;
    cudaError_t e = cudaMalloc(&partials, sizeof(double) * (size_t)blocks * NP);
    if (e != cudaSuccess) return cuda_fail("cudaMalloc (scatter-matrix partial sums)", e);
    cudaEvent_t ev[4] = {};
    if (pass_ms_out_host) {
        for (auto& x : ev)
            if ((e = cudaEventCreate(&x)) != cudaSuccess) { cudaFree(partials); return cuda_fail("cudaEventCreate", e); }
        cudaEventRecord(ev[0], st);
    }
    struct EventGuard {
        cudaEvent_t* ev;
        ~EventGuard() { for (int i = 0; i < 4; ++i) if (ev[i]) cudaEventDestroy(ev[i]); }
    } guard{ev};
    e = cudaErrorInvalidValue;
    PCA_DISPATCH(N, e = launch_gram<NN>(dvfs_dev, n, n, v4, blocks, partials, st));
    if (pass_ms_out_host) cudaEventRecord(ev[1], st);
    std::vector<double> hp((size_t)blocks * NP);
    if (e == cudaSuccess) e = cudaMemcpyAsync(hp.data(), partials, sizeof(double) * hp.size(), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(partials);
    if (e != cudaSuccess) return cuda_fail("scatter matrix", e);

    // the scatter matrix: blocks in index order (run-to-run reproducible)
    std::vector<double> G((size_t)N * N, 0.0), V, lam;
    {
        std::vector<double> tri(NP, 0.0);
        for (int b = 0; b < blocks; ++b)
            for (int p = 0; p < NP; ++p) tri[p] += hp[(size_t)b * NP + p];
        int p = 0;
        for (int i = 0; i < N; ++i)
            for (int j = i; j < N; ++j, ++p) {
                if (!std::isfinite(tri[p])) return fail(PCAMM_E_NONFINITE, "non-finite value in the training DVFs");
                G[(size_t)i * N + j] = G[(size_t)j * N + i] = tri[p];
            }
    }
    jacobi_eigen(N, G, V, lam);
    if (!(lam[0] > 0.0) || !(lam[K - 1] > 1e-6 * lam[0]))
        return fail(PCAMM_E_SINGULAR, "fewer than K independent modes in the training DVFs");
    PcaCoef coef = {};
    for (int k = 0; k < K; ++k) {
        // reading A12 / B10: u_k . (D_r - xbar) = sqrt(lambda_k) v_rk >= 0; if 0, the largest |v_ik| positive
        double ref = V[(size_t)sign_ref * N + k];
        if (ref == 0.0) {
            int im = 0;
            for (int i = 1; i < N; ++i)
                if (std::fabs(V[(size_t)i * N + k]) > std::fabs(V[(size_t)im * N + k])) im = i;
            ref = V[(size_t)im * N + k];
        }
        const double sgn = ref < 0.0 ? -1.0 : 1.0;
        const double rs = 1.0 / std::sqrt(lam[k]);
        for (int i = 0; i < N; ++i) {
            V[(size_t)i * N + k] *= sgn;
            coef.c[k][i] = (float)(V[(size_t)i * N + k] * rs);
            if (coeffs_out_host) coeffs_out_host[(size_t)i * K + k] = V[(size_t)i * N + k] * std::sqrt(lam[k]);
        }
    }
    if (eigenvalues_out_host)
        for (int i = 0; i < N; ++i) eigenvalues_out_host[i] = lam[i];

    if (pass_ms_out_host) cudaEventRecord(ev[2], st);
    e = cudaErrorInvalidValue;
    PCA_DISPATCH(N, e = launch_fields<NN>(dvfs_dev, n, n, v4, blocks, coef, K, mean_out_dev, eig_out_dev, st));
    if (pass_ms_out_host) cudaEventRecord(ev[3], st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail("eigenvector fields", e);
    if (pass_ms_out_host) {
        cudaEventElapsedTime(&pass_ms_out_host[0], ev[0], ev[1]);
        cudaEventElapsedTime(&pass_ms_out_host[1], ev[2], ev[3]);
    }
    return PCAMM_OK;
}
