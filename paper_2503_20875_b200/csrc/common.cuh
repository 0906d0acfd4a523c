// Shared host/device helpers of the CETRA B200 library (sm_100a only).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "cetra.h"

namespace cetra {

extern std::atomic<int64_t> g_launch_count;

#define CETRA_CUDA_TRY(expr)                              \
    do {                                                  \
        cudaError_t _e = (expr);                          \
        if (_e != cudaSuccess) return CETRA_ERR_CUDA;     \
    } while (0)

#define CETRA_LAUNCH_CHECK()                              \
    do {                                                  \
        ::cetra::g_launch_count.fetch_add(1);             \
        if (cudaPeekAtLastError() != cudaSuccess) return CETRA_ERR_CUDA; \
    } while (0)

// Optional event bracketing of the two hot kernels (cetra_profile_enable / cetra_profile_read).
enum ProfiledKernel { kProfLinear = 0, kProfFold = 1 };
void profile_mark(ProfiledKernel which, bool begin, cudaStream_t st);

constexpr int kStatsPad = 512;          // zero cells after the last t0 cell of every stats row
constexpr size_t kAlign = 256;          // workspace carve-up alignment
constexpr int kMaxClasses = 256;        // residue classes of a rational off-grid t0 stride (Geometry::cls)
constexpr int kMaxClassStride = 64;     // ... and the samples between neighbouring cells of one class

inline size_t align_up(size_t x, size_t a = kAlign) { return (x + a - 1) / a * a; }
inline int64_t round_up64(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

// Bump allocator over the caller's workspace (never allocates).
struct Carver {
    char *base;
    size_t used = 0;
    explicit Carver(void *p) : base(static_cast<char *>(p)) {}
    template <typename T>
    T *take(size_t count) {
        T *p = reinterpret_cast<T *>(base + used);
        used += align_up(count * sizeof(T));
        return p;
    }
};

// Regular-grid geometry shared by the entry points (R1, R9).
struct Geometry {
    double cadence = 0.0;   // c, days
    bool on_grid = true;    // t0 grid sits on the sample grid with a whole-sample stride (R3), else R25
    int64_t n0 = 0;         // on_grid: sample index of t0 cell 0 (may be negative)
    int64_t q = 0;          // on_grid: t0 stride in samples (>= 1); rational: numerator p of stride / cadence = p / cls
    // Off the sample grid, but stride / cadence = p / cls to within 1e-6 samples at the last cell (the paper's default
    // stride on 2-min data is 18 s / 120 s = 3 / 20): the cells of one residue class i = cls a + rho then sit p whole
    // samples apart at one common sub-sample offset, and each class is an on-grid problem with its own tap tables.
    bool rational = false;
    int64_t cls = 1;        // number of residue classes (1 on the sample grid)
    double drift = 0.0;     // rational: bound on |i stride / cadence - i p / cls| over the grid, in samples
    double delta = 0.0;     // t0_start - times[0], days
    double stride = 0.0;    // t0 stride, days
};

int derive_geometry(const double *times_host, int64_t n, cetra_t0_grid grid, Geometry *g);

#ifdef __CUDACC__
// ---------------------------------------------------------------------------------------------
// mbarrier + TMA 1-D bulk copy (cp.async.bulk, SASS UBLKCP) wrappers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "CETRA_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra CETRA_DONE;\n\t"
        "bra CETRA_WAIT;\n\t"
        "CETRA_DONE:\n\t"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

// Global -> shared bulk copy; dst, src and bytes must be multiples of 16.
__device__ __forceinline__ void bulk_copy_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// Issue one logical copy as <= 32 KiB pieces (one elected thread calls this after expect_tx).
__device__ __forceinline__ void bulk_copy_g2s_chunked(void *dst_smem, const void *src_gmem, uint32_t bytes,
                                                      uint64_t *bar) {
    constexpr uint32_t kPiece = 32768;
    char *d = static_cast<char *>(dst_smem);
    const char *s = static_cast<const char *>(src_gmem);
    for (uint32_t off = 0; off < bytes; off += kPiece) {
        const uint32_t len = bytes - off < kPiece ? bytes - off : kPiece;
        bulk_copy_g2s(d + off, s + off, len, bar);
    }
}
#endif  // __CUDACC__

}  // namespace cetra
