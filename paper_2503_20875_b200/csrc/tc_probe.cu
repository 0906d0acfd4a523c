// Measured attempt at the tensor-core variant of the linear search's windowed sums (north_star:
// "any tensor-core banded-correlation variant must beat the CUDA-core version in ncu to be kept").  Not on the product
// path: cetra_tc_correlation_probe runs it on synthetic samples so that the comparison in DESIGN.md can be repeated.
//
// For one duration with K taps and a whole-sample t0 stride the sums are a banded correlation,
//     S_wmf[i] = sum_k m[k] (w f)[i + k],   S_wmm[i] = sum_k m[k]^2 w[i + k],   k in [0, K).
// As a matrix product: 16 consecutive outputs are the rows of a Toeplitz tile T[r][s] = m[s - r], eight blocks of 16
// outputs the columns of a sample tile X[s][n] = x[16 blk_n + s], and D[16 x 8] += T[16 x 8] X[8 x 8] over the K + 15
// sample columns (mma.sync.m16n8k8, TF32 operands, FP32 accumulators; the operands come straight from the staged
// sample row and tap table, nothing is materialised).  TF32 carries 10 mantissa bits, so the 1e-5 parity bar needs the
// three-product split hi*hi + hi*lo + lo*hi (3xTF32); `split = 0` runs the single product for comparison.
#include <math.h>

#include <algorithm>
#include <vector>

#include "common.cuh"
#include "cetra_diag.h"

namespace cetra {

namespace {

constexpr int kTcNt = 4;                           // n-tiles (8 blocks x 16 outputs) per warp
constexpr int kTcWarps = 4;
constexpr int kTcOutPerWarp = kTcNt * 128;
constexpr int kTcOutPerCta = kTcWarps * kTcOutPerWarp;

__device__ __forceinline__ uint32_t to_tf32(float v) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(v));
    return r;
}
__device__ __forceinline__ void split_tf32(float v, uint32_t &hi, uint32_t &lo) {
    hi = to_tf32(v);
    lo = to_tf32(v - __uint_as_float(hi));
}
__device__ __forceinline__ void mma_tf32(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// shared-memory position of sample n: four words of skew per 16 samples make the eight column blocks of a B fragment
// (16 samples apart) fall into different banks
__host__ __device__ __forceinline__ int skew(int n) { return n + 4 * (n >> 4); }

// x: (w f, w) per sample; m_pad[k + 16] = m[k], zero outside [0, K); out[i] = (S_wmf, S_wmm)
template <int SPLIT>
__global__ void __launch_bounds__(kTcWarps * 32) tc_correlation_kernel(const float2 *__restrict__ x,
                                                                     const float *__restrict__ m_pad, int K,
                                                                     float2 *__restrict__ out, long long n_out) {
    extern __shared__ float tc_smem[];
    const int S = (K + 15 + 7) & ~7;                       // sample columns of a 16-output block
    const int n_x = kTcOutPerCta + S + 16;
    float *s_wf = tc_smem;
    float *s_w = s_wf + skew(n_x) + 8;
    float *s_m = s_w + skew(n_x) + 8;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long base = static_cast<long long>(blockIdx.x) * kTcOutPerCta;
    for (int i = tid; i < n_x; i += kTcWarps * 32) {
        const float2 v = x[base + i];
        s_wf[skew(i)] = v.x;
        s_w[skew(i)] = v.y;
    }
    for (int i = tid; i < K + 48; i += kTcWarps * 32) s_m[i] = m_pad[i];
    __syncthreads();
    const int g = lane >> 2, t = lane & 3;
    float acc_f[kTcNt][4], acc_w[kTcNt][4];
#pragma unroll
    for (int nt = 0; nt < kTcNt; ++nt)
#pragma unroll
        for (int c = 0; c < 4; ++c) { acc_f[nt][c] = 0.f; acc_w[nt][c] = 0.f; }
    const int wbase = warp * kTcOutPerWarp;
    for (int s0 = 0; s0 < S; s0 += 8) {
        // Toeplitz fragment A[r][s] = m[s0 + s - r]: a0 (g, t), a1 (g + 8, t), a2 (g, t + 4), a3 (g + 8, t + 4)
        const float *mp = s_m + 16 + s0 + t - g;
        const float mv[4] = {mp[0], mp[-8], mp[4], mp[-4]};
        uint32_t ah[4], al[4], a2h[4], a2l[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            split_tf32(mv[c], ah[c], al[c]);
            split_tf32(mv[c] * mv[c], a2h[c], a2l[c]);
        }
#pragma unroll
        for (int nt = 0; nt < kTcNt; ++nt) {
            const int n0 = wbase + (nt * 8 + g) * 16 + s0 + t;      // sample of b0 (k = t, n = g); b1 is 4 further
            const float f0 = s_wf[skew(n0)], f1 = s_wf[skew(n0 + 4)];
            const float w0 = s_w[skew(n0)], w1 = s_w[skew(n0 + 4)];
            uint32_t fh0, fl0, fh1, fl1, wh0, wl0, wh1, wl1;
            split_tf32(f0, fh0, fl0); split_tf32(f1, fh1, fl1);
            split_tf32(w0, wh0, wl0); split_tf32(w1, wh1, wl1);
            mma_tf32(acc_f[nt], ah, fh0, fh1);
            mma_tf32(acc_w[nt], a2h, wh0, wh1);
            if (SPLIT) {
                mma_tf32(acc_f[nt], ah, fl0, fl1);
                mma_tf32(acc_f[nt], al, fh0, fh1);
                mma_tf32(acc_w[nt], a2h, wl0, wl1);
                mma_tf32(acc_w[nt], a2l, wh0, wh1);
            }
        }
    }
    // D[r][n]: c0 (g, 2t), c1 (g, 2t + 1), c2 (g + 8, 2t), c3 (g + 8, 2t + 1); output 16 (nt * 8 + n) + r
#pragma unroll
    for (int nt = 0; nt < kTcNt; ++nt) {
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int r = g + (c >> 1) * 8, n = 2 * t + (c & 1);
            const long long i = base + wbase + (nt * 8 + n) * 16 + r;
            if (i < n_out) out[i] = make_float2(acc_f[nt][c], acc_w[nt][c]);
        }
    }
}

// synthetic (w f, w) samples and a smooth tap table (values only need the dynamic range of real ones)
__global__ void tc_fill_kernel(float2 *x, long long n_x, float *m_pad, int K) {
    const long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x;
    if (i < n_x) {
        unsigned long long h = (static_cast<unsigned long long>(i) + 1) * 0x9E3779B97F4A7C15ull;
        h ^= h >> 29; h *= 0xBF58476D1CE4E5B9ull; h ^= h >> 32;
        const float u1 = static_cast<float>(h & 0xffffff) * (1.0f / 16777216.0f);
        const float u2 = static_cast<float>((h >> 24) & 0xffffff) * (1.0f / 16777216.0f);
        const float w = 4.0e6f * (0.5f + u1);
        x[i] = make_float2(w * (u2 - 0.5f) * 1.0e-3f, w);
    }
    if (i < K + 64) {
        const int k = static_cast<int>(i) - 16;
        m_pad[i] = (k >= 0 && k < K) ? 0.2f + 0.8f * sinf(3.14159265f * (k + 0.5f) / K) : 0.f;
    }
}

// FP64 check of every 7th output: largest |S_wmf error| / max|S_wmf| and largest relative S_wmm error
__global__ void tc_check_kernel(const float2 *x, const float *m_pad, int K, const float2 *out, long long n_out,
                                double *worst /* [3]: max |ref wf|, max abs err wf, max rel err w */) {
    const long long i = (blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x) * 7;
    double ref_f = 0.0, err_f = 0.0, err_w = 0.0;
    if (i < n_out) {
        double a = 0.0, b = 0.0;
        for (int k = 0; k < K; ++k) {
            const float m = m_pad[16 + k];
            a += static_cast<double>(m) * x[i + k].x;
            b += static_cast<double>(m * m) * x[i + k].y;
        }
        ref_f = fabs(a);
        err_f = fabs(static_cast<double>(out[i].x) - a);
        err_w = fabs(static_cast<double>(out[i].y) - b) / b;
    }
    // doubles >= 0 order like their bit patterns
    atomicMax(reinterpret_cast<unsigned long long *>(worst + 0), static_cast<unsigned long long>(__double_as_longlong(ref_f)));
    atomicMax(reinterpret_cast<unsigned long long *>(worst + 1), static_cast<unsigned long long>(__double_as_longlong(err_f)));
    atomicMax(reinterpret_cast<unsigned long long *>(worst + 2), static_cast<unsigned long long>(__double_as_longlong(err_w)));
}

size_t tc_bytes(int64_t n_out, int32_t K) {
    const size_t n_x = static_cast<size_t>(n_out) + kTcOutPerCta + K + 64;
    return align_up(n_x * sizeof(float2)) + align_up(static_cast<size_t>(n_out) * sizeof(float2)) +
           align_up((K + 64) * sizeof(float)) + align_up(4 * sizeof(double));
}

}  // namespace

}  // namespace cetra

using namespace cetra;

extern "C" {

size_t cetra_tc_correlation_probe_workspace_bytes(int64_t n_out, int32_t n_taps) {
    if (n_out < 1 || n_taps < 1 || n_taps > 8192) return 0;
    return tc_bytes(n_out, n_taps);
}

int cetra_tc_correlation_probe(int64_t n_out, int32_t n_taps, int32_t split, int32_t reps, double *ms_per_launch,
                               double *err_wmf, double *err_wmm, void *workspace_dev, size_t workspace_bytes,
                               void *cuda_stream) {
    if (n_out < 1 || n_taps < 1 || n_taps > 8192 || reps < 1) return CETRA_ERR_INVALID_ARG;
    if (!workspace_dev || (reinterpret_cast<uintptr_t>(workspace_dev) & (kAlign - 1)) != 0 ||
        workspace_bytes < tc_bytes(n_out, n_taps))
        return CETRA_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int K = n_taps;
    const long long n_x = n_out + kTcOutPerCta + K + 64;
    Carver ws(workspace_dev);
    float2 *x = ws.take<float2>(static_cast<size_t>(n_x));
    float2 *out = ws.take<float2>(static_cast<size_t>(n_out));
    float *m_pad = ws.take<float>(K + 64);
    double *worst = ws.take<double>(4);
    CETRA_CUDA_TRY(cudaMemsetAsync(worst, 0, 4 * sizeof(double), st));
    tc_fill_kernel<<<static_cast<unsigned>((n_x + 255) / 256), 256, 0, st>>>(x, n_x, m_pad, K);
    CETRA_LAUNCH_CHECK();
    const int S = (K + 15 + 7) & ~7;
    const size_t smem = (2 * (skew(kTcOutPerCta + S + 16) + 8) + K + 48) * sizeof(float);
    const unsigned grid = static_cast<unsigned>((n_out + kTcOutPerCta - 1) / kTcOutPerCta);
    auto kern = split ? tc_correlation_kernel<1> : tc_correlation_kernel<0>;
    CETRA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)));
    cudaEvent_t a, b;
    CETRA_CUDA_TRY(cudaEventCreate(&a));
    CETRA_CUDA_TRY(cudaEventCreate(&b));
    kern<<<grid, kTcWarps * 32, smem, st>>>(x, m_pad, K, out, n_out);          // warm-up
    cudaEventRecord(a, st);
    for (int r = 0; r < reps; ++r) kern<<<grid, kTcWarps * 32, smem, st>>>(x, m_pad, K, out, n_out);
    cudaEventRecord(b, st);
    g_launch_count.fetch_add(reps + 1);
    const long long checked = (n_out + 6) / 7;
    tc_check_kernel<<<static_cast<unsigned>((checked + 127) / 128), 128, 0, st>>>(x, m_pad, K, out, n_out, worst);
    double host[4] = {0, 0, 0, 0};
    float ms = 0.f;
    int rc = CETRA_OK;
    if (cudaMemcpyAsync(host, worst, sizeof(host), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess || cudaEventElapsedTime(&ms, a, b) != cudaSuccess)
        rc = CETRA_ERR_CUDA;
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    if (rc != CETRA_OK) return rc;
    if (ms_per_launch) *ms_per_launch = ms / reps;
    if (err_wmf) *err_wmf = host[0] > 0.0 ? host[1] / host[0] : 0.0;
    if (err_wmm) *err_wmm = host[2];
    return CETRA_OK;
}

}  // extern "C"
