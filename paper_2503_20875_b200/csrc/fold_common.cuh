// Device helpers shared by the fold kernels of the periodic search (§2.3): packed FP32 adds, shared-memory
// cell loads and the two-period register-window epoch step.
#pragma once

#include "periodic_search.cuh"

namespace cetra {

__device__ __forceinline__ float2 add2(float2 a, float2 b) {
    // packed FP32 add (FADD2 on sm_100a): one issue slot for both sufficient statistics
    float2 r;
    asm("{\n\t"
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

__device__ __forceinline__ float2 mul2(float2 a, float2 b) {
    // packed FP32 multiply (FMUL2): two independent IEEE products in one issue slot
    float2 r;
    asm("{\n\t"
        ".reg .b64 ra, rb, rc;\n\t"
        "mov.b64 ra, {%2, %3};\n\t"
        "mov.b64 rb, {%4, %5};\n\t"
        "mul.rn.f32x2 rc, ra, rb;\n\t"
        "mov.b64 {%0, %1}, rc;\n\t"
        "}"
        : "=f"(r.x), "=f"(r.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}

__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

struct GroupPeriods {
    double r[kGrpT];          // period in t0 cells, ascending
    int n_phase[kGrpT];       // R10; 0 for a period that is not searched on this row
};

__device__ __forceinline__ float2 lds_cell(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}

__device__ __forceinline__ int lds_int(uint32_t addr) {
    int v;
    asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

__device__ __forceinline__ int2 lds_int2(uint32_t addr) {
    int2 v;
    asm volatile("ld.shared.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}

__device__ __forceinline__ int4 lds_int4(uint32_t addr) {
    int4 v;
    asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}

__device__ __forceinline__ void sts_int4(uint32_t addr, int x, int y, int z, int w) {
    asm volatile("st.shared.v4.s32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}

__device__ __forceinline__ void sts_int2(uint32_t addr, int x, int y) {
    asm volatile("st.shared.v2.s32 [%0], {%1, %2};" ::"r"(addr), "r"(x), "r"(y) : "memory");
}

constexpr int kPairMaxM = 64;              // cap on the centring shift

// Centring of a pair (r0 <= r1, both searched): half of the largest offset difference, reached at the last epoch.
// Any value gives the same records (it only decides which phases a lane folds together); this one halves the
// average distance between the two periods' windows.
__device__ __forceinline__ int centring_shift(double r0, double r1, int n_t0) {
    const float e_last = static_cast<float>(n_t0 - 1) / static_cast<float>(r0);
    const float half = 0.5f * e_last * static_cast<float>(r1 - r0);
    return half < static_cast<float>(kPairMaxM) ? static_cast<int>(half + 0.5f) : kPairMaxM;
}

// One epoch of a pair whose windows are S cells apart (S < 0: the longer period's cells come first): the G + |S|
// cells from the smaller window start on are loaded once.
template <int S, int G>
__device__ __forceinline__ void fold_epoch_c(float2 (&acc)[kGrpT][G], uint32_t ptr) {
    constexpr int A = S < 0 ? -S : S;
    float2 c[G + A];
#pragma unroll
    for (int i = 0; i < G + A; ++i) c[i] = lds_cell(ptr + 8u * i);
#pragma unroll
    for (int g = 0; g < G; ++g) acc[0][g] = add2(acc[0][g], c[g + (S < 0 ? A : 0)]);
#pragma unroll
    for (int g = 0; g < G; ++g) acc[1][g] = add2(acc[1][g], c[g + (S > 0 ? A : 0)]);
}

}  // namespace cetra
