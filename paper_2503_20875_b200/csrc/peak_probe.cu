// Unit-throughput probes behind bench.py's roofline denominators (cetra_peak_probe): the rates of the three
// instructions the two hot kernels are bound by, measured on the device the library runs on, with the same
// instruction forms the kernels use.
//
//   CETRA_PROBE_FFMA2  fma.rn.f32x2 (SASS FFMA2)  linear_search_kernel's windowed sums     -> FP32 flop
//   CETRA_PROBE_FADD2  add.rn.f32x2 (SASS FADD2)  the fold kernels' accumulation           -> FP32 flop
//   CETRA_PROBE_LDS64  ld.shared.v2.f32 at a lane stride of 11 cells (conflict-free), the fold kernels' gather
//                      -> bytes through the shared-memory crossbar
//
// One 1 024-thread CTA per SM (eight warps per scheduler).  Every CTA times itself with clock64 (SM clock domain), so the per-clock figure does not depend on the clock the
// GPU happens to run at; the per-second figure comes from CUDA events around the launch.
#include <algorithm>
#include <vector>

#include "common.cuh"
#include "cetra_diag.h"

namespace cetra {

// libcetra_diag.so is linked on its own: it keeps a launch counter of its own (the product's counts only the
// product's kernels).
std::atomic<int64_t> g_launch_count{0};

namespace {

constexpr int kProbeThreads = 1024;    // one CTA per SM (its shared-memory request excludes a second one)
constexpr int kProbeAcc = 12;          // independent accumulators per thread (covers the 4-cycle FMA latency)
constexpr int kProbeLoads = 11;        // cells per lane per iteration, as the fold kernels' full pass
constexpr size_t kProbeSmem = 160 * 1024;
constexpr int kProbeStride = 11;       // lane stride in cells (odd: no bank conflicts for 8-byte loads)

__device__ __forceinline__ float2 probe_fma2(float2 a, float2 b, float2 c) {
    float2 r;
    asm volatile("{\n\t"
                 ".reg .b64 ra, rb, rc, rd;\n\t"
                 "mov.b64 ra, {%2, %3};\n\t"
                 "mov.b64 rb, {%4, %5};\n\t"
                 "mov.b64 rc, {%6, %7};\n\t"
                 "fma.rn.f32x2 rd, ra, rb, rc;\n\t"
                 "mov.b64 {%0, %1}, rd;\n\t"
                 "}"
                 : "=f"(r.x), "=f"(r.y)
                 : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return r;
}

__device__ __forceinline__ float2 probe_add2(float2 a, float2 b) {
    float2 r;
    asm volatile("{\n\t"
                 ".reg .b64 ra, rb, rc;\n\t"
                 "mov.b64 ra, {%2, %3};\n\t"
                 "mov.b64 rb, {%4, %5};\n\t"
                 "add.rn.f32x2 rc, ra, rb;\n\t"
                 "mov.b64 {%0, %1}, rc;\n\t"
                 "}"
                 : "=f"(r.x), "=f"(r.y)
                 : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}

struct ProbeOut {
    long long cycles;
    float sink;
    int pad;
};

template <int KIND>
__global__ void __launch_bounds__(kProbeThreads, 1) peak_probe_kernel(int iters, ProbeOut *out) {
    extern __shared__ __align__(16) float2 cells[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    float2 acc[kProbeAcc];
#pragma unroll
    for (int i = 0; i < kProbeAcc; ++i) acc[i] = make_float2(1.0f + tid * 1e-6f, 0.5f + i * 1e-6f);
    uint32_t base = 0;
    if (KIND == CETRA_PROBE_LDS64) {
        const int n_cells = 32 * (kProbeThreads / 32) + 32 * kProbeStride + 4 * kProbeLoads + 4;
        for (int i = tid; i < n_cells; i += kProbeThreads) cells[i] = make_float2(1e-9f * i, 1e-9f);
        base = smem_u32(cells) + 8u * static_cast<uint32_t>(warp * 32 + lane * kProbeStride);
    }
    __syncthreads();
    const long long t0 = clock64();
    const float2 m = make_float2(0.999999f, 1.000001f);
    for (int it = 0; it < iters; ++it) {
        if (KIND == CETRA_PROBE_FFMA2) {
#pragma unroll
            for (int i = 0; i < kProbeAcc; ++i) acc[i] = probe_fma2(acc[i], m, m);
        } else if (KIND == CETRA_PROBE_FADD2) {
#pragma unroll
            for (int i = 0; i < kProbeAcc; ++i) acc[i] = probe_add2(acc[i], m);
        } else {
            float2 c[kProbeLoads];
            // Every load of an unrolled body has an address of its own (the base moves by a whole group of kProbeLoads
            // cells per trip, over a window of four groups) and is ld.volatile: ptxas may neither merge nor drop one.
            // `asm volatile` alone does not say that -- it orders the asm statements but leaves the PTX load an ordinary
            // one, and round 2's probe (base moving by ONE cell per trip, so that 30 of the 44 loads of a four-trip body
            // repeated an address) was merged down to 14 LDS.64 and reported 3.0 x the crossbar's physical rate.
            // SASS of this kernel, checked with cuobjdump: 44 LDS.64 per four-trip body.
            const uint32_t b = base + 8u * static_cast<uint32_t>(kProbeLoads * (it & 3));
#pragma unroll
            for (int i = 0; i < kProbeLoads; ++i)
                asm volatile("ld.volatile.shared.v2.f32 {%0, %1}, [%2];"
                             : "=f"(c[i].x), "=f"(c[i].y)
                             : "r"(b + 8u * i)
                             : "memory");
#pragma unroll
            for (int i = 0; i < kProbeLoads; ++i) acc[i] = probe_add2(acc[i], c[i]);
        }
    }
    const long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kProbeAcc; ++i) s += acc[i].x + acc[i].y;
    if (tid == 0) {
        out[blockIdx.x].cycles = t1 - t0;
        out[blockIdx.x].sink = s;
    }
}

template <int KIND>
int launch_probe(int grid, size_t smem, int iters, ProbeOut *out, cudaStream_t st) {
    auto k = peak_probe_kernel<KIND>;
    CETRA_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k<<<grid, kProbeThreads, smem, st>>>(iters, out);
    CETRA_LAUNCH_CHECK();
    return CETRA_OK;
}

}  // namespace

}  // namespace cetra

using namespace cetra;

extern "C" {

size_t cetra_peak_probe_workspace_bytes(void) { return align_up(sizeof(ProbeOut) * 4096); }

int cetra_peak_probe(int32_t kind, int32_t iters, double *per_clk_per_sm, double *per_second, void *workspace_dev,
                     size_t workspace_bytes, void *cuda_stream) {
    if (kind < CETRA_PROBE_FFMA2 || kind > CETRA_PROBE_LDS64 || iters < 1) return CETRA_ERR_INVALID_ARG;
    if (!workspace_dev || (reinterpret_cast<uintptr_t>(workspace_dev) & (kAlign - 1)) != 0 ||
        workspace_bytes < cetra_peak_probe_workspace_bytes())
        return CETRA_ERR_WORKSPACE;
    int dev = 0, n_sm = 0;
    CETRA_CUDA_TRY(cudaGetDevice(&dev));
    CETRA_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ProbeOut *out = static_cast<ProbeOut *>(workspace_dev);
    const int grid = std::min(n_sm, 4096);
    const size_t smem = kProbeSmem;
    cudaEvent_t a, b;
    CETRA_CUDA_TRY(cudaEventCreate(&a));
    CETRA_CUDA_TRY(cudaEventCreate(&b));
    int rc = CETRA_OK;
    for (int rep = 0; rep < 2 && rc == CETRA_OK; ++rep) {   // the first launch warms the clocks up
        if (rep) cudaEventRecord(a, st);
        switch (kind) {
            case CETRA_PROBE_FFMA2: rc = launch_probe<CETRA_PROBE_FFMA2>(grid, smem, iters, out, st); break;
            case CETRA_PROBE_FADD2: rc = launch_probe<CETRA_PROBE_FADD2>(grid, smem, iters, out, st); break;
            default: rc = launch_probe<CETRA_PROBE_LDS64>(grid, smem, iters, out, st); break;
        }
        if (rep) cudaEventRecord(b, st);
    }
    std::vector<ProbeOut> host(grid);
    float ms = 0.f;
    if (rc == CETRA_OK &&
        (cudaMemcpyAsync(host.data(), out, sizeof(ProbeOut) * grid, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
         cudaStreamSynchronize(st) != cudaSuccess || cudaEventElapsedTime(&ms, a, b) != cudaSuccess))
        rc = CETRA_ERR_CUDA;
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    if (rc != CETRA_OK) return rc;
    // work per thread and iteration: flop (2 lanes x 2 flop per FFMA2, 2 x 1 per FADD2) or bytes (8 per load)
    const double per_thread = kind == CETRA_PROBE_FFMA2   ? 4.0 * kProbeAcc
                              : kind == CETRA_PROBE_FADD2 ? 2.0 * kProbeAcc
                                                          : 8.0 * kProbeLoads;
    const double total = per_thread * kProbeThreads * static_cast<double>(iters) * grid;
    double cyc = 0.0;
    for (const ProbeOut &o : host) cyc += static_cast<double>(o.cycles);
    cyc /= grid;                                            // CTAs run side by side for the same span
    if (per_clk_per_sm) *per_clk_per_sm = total / n_sm / cyc;
    if (per_second) *per_second = total / (ms * 1e-3);
    return CETRA_OK;
}

}  // extern "C"
