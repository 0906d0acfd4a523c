// Steps around the two searches: light-curve resampling (§2.1.1, lines 53-61), monotransit
// search in the linear-search output and transit masking.
//
// All of them are HBM-bound streaming kernels (a few bytes of arithmetic per byte moved); every quantity
// that decides an integer (output point of an observation, in/out of a mask, the exclusion zone of an
// event) is FP64 with explicitly rounded operations, as in the searches.
#include <math.h>

#include <algorithm>
#include <mutex>
#include <vector>

#include "common.cuh"

namespace cetra {

// ------------------------------------------------------------------------------------------ resample
// Atomic-sum form, now used by cetra_resample_static only (its scratch is the fixed FP64 sums array; the fixed-order
// path below needs scratch that grows with the number of observations).
// One thread per (light curve, observation): atomically add (w, w f) to the observation's output point.
template <typename T>
__global__ void resample_accumulate_kernel(const double *__restrict__ times, const T *__restrict__ flux,
                                           const T *__restrict__ flux_err, long long n_in, long long n_lc,
                                           double t_start, double cadence, long long n_out,
                                           double2 *__restrict__ sums) {
    const long long total = n_lc * n_in;
    for (long long idx = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; idx < total;
         idx += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long lc = idx / n_in;
        const long long i = idx - lc * n_in;
        const double t = times[i];
        const double fl = static_cast<double>(flux[idx]);
        const double er = static_cast<double>(flux_err[idx]);
        if (!(isfinite(t) && isfinite(fl) && isfinite(er) && er > 0.0)) continue;      // null observation (R8)
        // nearest output point (R21)
        const double cell = floor(__dadd_rn(__ddiv_rn(__dsub_rn(t, t_start), cadence), 0.5));
        if (!(cell >= 0.0 && cell < static_cast<double>(n_out))) continue;
        const double w = __ddiv_rn(1.0, __dmul_rn(er, er));
        double2 *dst = sums + lc * n_out + static_cast<long long>(cell);
        atomicAdd(&dst->x, w);
        atomicAdd(&dst->y, __dmul_rn(w, fl));
    }
}

// One thread per output point: inverse-variance weighted mean and its formal error; null where empty.
template <typename T>
__global__ void resample_finalize_kernel(const double2 *__restrict__ sums, long long total, T *__restrict__ flux_out,
                                         T *__restrict__ err_out) {
    for (long long idx = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; idx < total;
         idx += static_cast<long long>(gridDim.x) * blockDim.x) {
        const double2 s = sums[idx];
        if (s.x > 0.0) {
            flux_out[idx] = static_cast<T>(__ddiv_rn(s.y, s.x));
            err_out[idx] = static_cast<T>(__dsqrt_rn(__ddiv_rn(1.0, s.x)));
        } else {
            flux_out[idx] = static_cast<T>(__longlong_as_double(0x7ff8000000000000LL));   // null flux
            err_out[idx] = static_cast<T>(__longlong_as_double(0x7ff0000000000000LL));    // infinite error
        }
    }
}

// ------------------------------------------------------------------- resample, fixed summation order
// cetra_resample's own path (round 3).  All light curves of a call share the timestamps, so which
// output point an observation falls on is the same for every curve: it is worked out ONCE, as a compressed list of
// observation indices per output point (count -> exclusive scan -> fill -> sort each point's few indices), and then the
// sum kernel adds each (light curve, output point)'s observations in ascending input index in FP64.  No floating-point
// atomics: the result is bit-identical from run to run and equal to a sequential loop over the input (the oracle's
// order); each flux / error value is read once and each output written once.

// Observation -> output point (R21, FP64), -1 for a non-finite or off-grid time; counts per point (integer atomics).
__global__ void resample_cells_kernel(const double *__restrict__ times, int n_in, double t_start, double cadence,
                                      int n_out, int *__restrict__ cell_of, int *__restrict__ count) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_in; i += gridDim.x * blockDim.x) {
        const double t = times[i];
        int c = -1;
        if (isfinite(t)) {
            const double cell = floor(__dadd_rn(__ddiv_rn(__dsub_rn(t, t_start), cadence), 0.5));
            if (cell >= 0.0 && cell < static_cast<double>(n_out)) c = static_cast<int>(cell);
        }
        cell_of[i] = c;
        if (c >= 0) atomicAdd(count + c, 1);
    }
}

// Exclusive scan of the counts in two launches over tiles of kScanTile points (a single CTA walking 2e5 counts was
// latency-bound at 0.3 ms, ncu r03b): first each tile's total, then every tile finds its base by adding the totals
// of the tiles before it (a few dozen numbers for a sector) and scans itself.  offsets[n_out + 1]; the counts are
// replaced by the offsets so that the fill can use them as cursors.
constexpr int kScanThreads = 256;
constexpr int kScanTile = 4 * kScanThreads;

__device__ __forceinline__ int block_sum_256(int v, int *s_warp) {          // total over the CTA, to every thread
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    __syncthreads();                                                        // s_warp may still be read from a previous use
    if (lane == 0) s_warp[warp] = v;
    __syncthreads();
    int t = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) t += s_warp[w];
    return t;
}

__global__ void __launch_bounds__(kScanThreads) resample_tile_sums_kernel(const int *__restrict__ count, int n_out,
                                                                         int *__restrict__ tile_sum) {
    __shared__ int s_warp[kScanThreads / 32];
    const int base = blockIdx.x * kScanTile + threadIdx.x * 4;
    int v = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) v += base + k < n_out ? count[base + k] : 0;
    const int t = block_sum_256(v, s_warp);
    if (threadIdx.x == 0) tile_sum[blockIdx.x] = t;
}

__global__ void __launch_bounds__(kScanThreads) resample_scan_kernel(int *__restrict__ count,
                                                                    const int *__restrict__ tile_sum,
                                                                    int *__restrict__ offsets, int n_out) {
    __shared__ int s_warp[kScanThreads / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int before = 0;
    for (int b = tid; b < static_cast<int>(blockIdx.x); b += kScanThreads) before += tile_sum[b];
    const int tile_base = block_sum_256(before, s_warp);
    const int base = blockIdx.x * kScanTile + tid * 4;
    int c[4], sum = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        c[k] = base + k < n_out ? count[base + k] : 0;
        sum += c[k];
    }
    int incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    __syncthreads();
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    int run = tile_base + incl - sum;
    for (int w = 0; w < warp; ++w) run += s_warp[w];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (base + k < n_out) {
            offsets[base + k] = run;
            count[base + k] = run;
        }
        run += c[k];
        if (base + k == n_out - 1) offsets[n_out] = run;
    }
}

__global__ void resample_fill_kernel(const int *__restrict__ cell_of, int n_in, int *__restrict__ cursor,
                                     int *__restrict__ order) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_in; i += gridDim.x * blockDim.x) {
        const int c = cell_of[i];
        if (c >= 0) order[atomicAdd(cursor + c, 1)] = i;
    }
}

// The fill leaves each point's indices in arrival order; put them in ascending order (the fixed summation order).
// One thread per output point: a point holds a handful of observations (insertion sort), heapsort beyond 16 so that
// a degenerate grid (everything in one point) costs m log m, not m^2.
__global__ void resample_sort_kernel(const int *__restrict__ offsets, int n_out, int *__restrict__ order) {
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < n_out; c += gridDim.x * blockDim.x) {
        const int lo = offsets[c], m = offsets[c + 1] - lo;
        if (m < 2) continue;
        int *a = order + lo;
        if (m <= 16) {
            for (int i = 1; i < m; ++i) {
                const int v = a[i];
                int k = i - 1;
                while (k >= 0 && a[k] > v) { a[k + 1] = a[k]; --k; }
                a[k + 1] = v;
            }
            continue;
        }
        auto sift = [a](int root, int end) {                     // max-heap on a[0 .. end)
            const int v = a[root];
            for (;;) {
                int child = 2 * root + 1;
                if (child >= end) break;
                if (child + 1 < end && a[child + 1] > a[child]) ++child;
                if (a[child] <= v) break;
                a[root] = a[child];
                root = child;
            }
            a[root] = v;
        };
        for (int i = m / 2 - 1; i >= 0; --i) sift(i, m);
        for (int end = m - 1; end > 0; --end) {
            const int t = a[0]; a[0] = a[end]; a[end] = t;
            sift(0, end);
        }
    }
}

// Inverse-variance weighted mean of an output point's valid observations, added in ascending input index; formal
// error; null (NaN, +inf) where there is none.
template <typename T>
__device__ __forceinline__ void resample_point(const T *__restrict__ fl, const T *__restrict__ er,
                                               const int *__restrict__ order, int lo, int m, T *flux_out, T *err_out) {
    double sw = 0.0, swf = 0.0;
    for (int k = lo; k < lo + m; ++k) {
        const int i = order[k];
        const double f = static_cast<double>(fl[i]), e = static_cast<double>(er[i]);
        if (!(isfinite(f) && isfinite(e) && e > 0.0)) continue;                   // null observation (R8)
        const double w = __ddiv_rn(1.0, __dmul_rn(e, e));
        sw = __dadd_rn(sw, w);
        swf = __dadd_rn(swf, __dmul_rn(w, f));
    }
    if (sw > 0.0) {
        *flux_out = static_cast<T>(__ddiv_rn(swf, sw));
        *err_out = static_cast<T>(__dsqrt_rn(__ddiv_rn(1.0, sw)));
    } else {
        *flux_out = static_cast<T>(__longlong_as_double(0x7ff8000000000000LL));
        *err_out = static_cast<T>(__longlong_as_double(0x7ff0000000000000LL));
    }
}

// One CTA per 256 output points and group of G light curves, in two phases (ncu r03c / r03d: a thread per (curve,
// point) waited on the chain offsets -> order -> flux, and one point with two observations in a warp made the other
// 31 lanes sit through its FP64 divisions and square root).
//  1. A thread per point.  No observation: null for the G curves.  Exactly one observation and float32 data -- nearly
//     every point at the native cadence -- is copied, G independent loads in flight: the FP64 sequence (w f)/w and
//     sqrt(1/w), w = 1/e^2, lands within 2^-50 of f and e, which are float32 numbers, so rounding to float32 returns
//     f and e themselves, for every finite f and every finite e > 0 (e^2 is exact in FP64 and neither overflows nor
//     vanishes).  Every other point goes on a list in shared memory.
//  2. The listed (point, curve) pairs are dealt out over all the threads, so the FP64 arithmetic runs in full warps.
// float64 data always takes the arithmetic (it is not the identity there).
template <typename T, int G>
__global__ void __launch_bounds__(256) resample_sum_kernel(const T *__restrict__ flux, const T *__restrict__ flux_err,
                                                           long long n_in, int n_lc, int n_out,
                                                           const int *__restrict__ offsets,
                                                           const int *__restrict__ order, T *__restrict__ flux_out,
                                                           T *__restrict__ err_out) {
    __shared__ int s_n;
    __shared__ int s_point[256];
    if (threadIdx.x == 0) s_n = 0;
    __syncthreads();
    const int c = blockIdx.x * 256 + threadIdx.x;
    int lo = 0, m = -1;                                           // -1: past the last point
    if (c < n_out) {
        lo = offsets[c];
        m = offsets[c + 1] - lo;
    }
    const bool copy = sizeof(T) == 4 && m == 1;
    const int first = copy ? order[lo] : 0;
    if (m > 0 && !copy) s_point[atomicAdd(&s_n, 1)] = c;
    __syncthreads();
    const int n_listed = s_n;
    const T nan_t = static_cast<T>(__longlong_as_double(0x7ff8000000000000LL));
    const T inf_t = static_cast<T>(__longlong_as_double(0x7ff0000000000000LL));
    for (int lc0 = blockIdx.y * G; lc0 < n_lc; lc0 += gridDim.y * G) {
        const int g_n = min(G, n_lc - lc0);
        const T *fl = flux + static_cast<long long>(lc0) * n_in, *er = flux_err + static_cast<long long>(lc0) * n_in;
        T *fo = flux_out + static_cast<long long>(lc0) * n_out, *eo = err_out + static_cast<long long>(lc0) * n_out;
        if (copy) {
            T f[G], e[G];
#pragma unroll
            for (int g = 0; g < G; ++g) {
                f[g] = g < g_n ? fl[g * n_in + first] : T(0);
                e[g] = g < g_n ? er[g * n_in + first] : T(0);
            }
#pragma unroll
            for (int g = 0; g < G; ++g) {
                if (g >= g_n) break;
                const bool ok = isfinite(f[g]) && isfinite(e[g]) && e[g] > T(0);
                fo[static_cast<long long>(g) * n_out + c] = ok ? f[g] : nan_t;
                eo[static_cast<long long>(g) * n_out + c] = ok ? e[g] : inf_t;
            }
        } else if (m == 0) {
            for (int g = 0; g < g_n; ++g) {
                fo[static_cast<long long>(g) * n_out + c] = nan_t;
                eo[static_cast<long long>(g) * n_out + c] = inf_t;
            }
        }
        for (int task = threadIdx.x; task < n_listed * g_n; task += 256) {
            const int g = task / n_listed, pc = s_point[task - g * n_listed];
            const int plo = offsets[pc];
            resample_point<T>(fl + g * n_in, er + g * n_in, order, plo, offsets[pc + 1] - plo,
                              fo + static_cast<long long>(g) * n_out + pc, eo + static_cast<long long>(g) * n_out + pc);
        }
    }
}

// ------------------------------------------------------------------------------------------- masking
struct MaskParams {
    const double *period, *t0, *duration;   // [n_lc] device
};

template <typename T>
__global__ void mask_transits_kernel(const double *__restrict__ times, T *__restrict__ flux, long long n,
                                     long long n_lc, MaskParams mp, double width, int *__restrict__ n_masked) {
    const long long total = n_lc * n;
    for (long long idx = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; idx < total;
         idx += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long lc = idx / n;
        const long long i = idx - lc * n;
        const double P = mp.period[lc], t0 = mp.t0[lc], D = mp.duration[lc];
        if (!(isfinite(t0) && D > 0.0)) continue;
        double d = __dsub_rn(times[i], t0);
        if (P > 0.0)                                              // distance to the nearest mid-time (R24)
            d = __dsub_rn(d, __dmul_rn(P, floor(__dadd_rn(__ddiv_rn(d, P), 0.5))));
        if (fabs(d) <= __dmul_rn(__dmul_rn(0.5, width), D)) {
            flux[idx] = static_cast<T>(__longlong_as_double(0x7ff8000000000000LL));
            if (n_masked) atomicAdd(n_masked + lc, 1);
        }
    }
}

// ---------------------------------------------------------------------------------------- monotransit
// profile(i) = max_j dlogL[j][i], ties -> smallest j; NaN / -1 where every duration is null (R23).
__global__ void monotransit_profile_kernel(const float *__restrict__ dlogL, long long n_lc, int n_dur,
                                           long long n_t0, float *__restrict__ prof_lr, int *__restrict__ prof_j) {
    const long long total = n_lc * n_t0;
    for (long long idx = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; idx < total;
         idx += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long lc = idx / n_t0;
        const long long i = idx - lc * n_t0;
        const float *col = dlogL + lc * n_dur * n_t0 + i;
        float best = -INFINITY;
        int bj = -1;
        for (int j = 0; j < n_dur; ++j) {
            const float v = col[static_cast<long long>(j) * n_t0];
            if (v > best || (bj < 0 && v == v)) { best = v; bj = j; }   // NaN compares false; -inf is a value
        }
        prof_lr[idx] = bj < 0 ? __int_as_float(0x7fc00000) : best;
        prof_j[idx] = bj;
    }
}

struct EventParams {
    double durations[CETRA_MAX_DURATIONS];
};

// One CTA per light curve: n_peaks rounds of (block argmax over the live reference times, record the event,
// retire its exclusion zone).  Key = (profile bits ordered as unsigned) << 32 | ~i: larger lr, then smaller i.
__global__ void __launch_bounds__(1024) monotransit_events_kernel(
    const float *__restrict__ depth, const float *__restrict__ var, const float *__restrict__ prof_lr,
    const int *__restrict__ prof_j, unsigned char *__restrict__ dead, int n_dur, long long n_t0, double t0_start,
    double t0_stride, const __grid_constant__ EventParams ep, int n_peaks, double excl,
    cetra_event *__restrict__ events, int *__restrict__ n_found) {
    __shared__ unsigned long long s_key[32];
    __shared__ unsigned long long s_best;
    const long long lc = blockIdx.x;
    const float *pl = prof_lr + lc * n_t0;
    const int *pj = prof_j + lc * n_t0;
    unsigned char *dd = dead + lc * n_t0;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (long long i = tid; i < n_t0; i += blockDim.x) dd[i] = pj[i] < 0 ? 1 : 0;
    __syncthreads();
    int found = 0;
    for (; found < n_peaks; ++found) {
        unsigned long long key = 0ull;
        for (long long i = tid; i < n_t0; i += blockDim.x) {
            if (dd[i]) continue;
            const unsigned int b = __float_as_uint(pl[i]);
            const unsigned int ord = (b & 0x80000000u) ? ~b : (b | 0x80000000u);    // total order of the floats
            const unsigned long long k = (static_cast<unsigned long long>(ord) << 32) |
                                         (0xffffffffu - static_cast<unsigned int>(i));
            key = k > key ? k : key;
        }
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) {
            const unsigned long long o = __shfl_xor_sync(0xffffffffu, key, s);
            key = o > key ? o : key;
        }
        if (lane == 0) s_key[warp] = key;
        __syncthreads();
        if (warp == 0) {
            key = lane < (blockDim.x >> 5) ? s_key[lane] : 0ull;
#pragma unroll
            for (int s = 16; s > 0; s >>= 1) {
                const unsigned long long o = __shfl_xor_sync(0xffffffffu, key, s);
                key = o > key ? o : key;
            }
            if (lane == 0) s_best = key;
        }
        __syncthreads();
        const unsigned long long best = s_best;
        if (best == 0ull) break;                                  // no live reference time left
        const long long bi = 0xffffffffu - static_cast<unsigned int>(best & 0xffffffffull);
        const int j = pj[bi];
        if (tid == 0) {
            cetra_event ev;
            ev.lr = pl[bi];
            ev.depth = depth[(lc * n_dur + j) * n_t0 + bi];
            ev.depth_var = var[(lc * n_dur + j) * n_t0 + bi];
            ev.t0 = static_cast<float>(__dadd_rn(t0_start, __dmul_rn(static_cast<double>(bi), t0_stride)));
            ev.i_t0 = static_cast<int>(bi);
            ev.j_dur = j;
            ev.reserved[0] = ev.reserved[1] = 0;
            events[lc * n_peaks + found] = ev;
        }
        const double reach = __dmul_rn(excl, ep.durations[j]);
        for (long long i = tid; i < n_t0; i += blockDim.x)
            if (i == bi || fabs(__dmul_rn(static_cast<double>(i - bi), t0_stride)) <= reach) dd[i] = 1;
        __syncthreads();
    }
    if (tid == 0) n_found[lc] = found;
    for (int e = found + tid; e < n_peaks; e += blockDim.x) {
        cetra_event ev;
        const float nanv = __int_as_float(0x7fc00000);
        ev.lr = nanv; ev.depth = nanv; ev.depth_var = nanv; ev.t0 = nanv;
        ev.i_t0 = -1; ev.j_dur = -1; ev.reserved[0] = ev.reserved[1] = 0;
        events[lc * n_peaks + e] = ev;
    }
}

static int stream_blocks(long long total) {
    return static_cast<int>(std::max<long long>(1, std::min<long long>((total + 255) / 256, 148LL * 16)));
}

static bool ws_ok(const void *p, size_t have, size_t need) {
    return p && (reinterpret_cast<uintptr_t>(p) & (kAlign - 1)) == 0 && have >= need;
}

static int have_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return CETRA_ERR_CUDA;
    }
    return CETRA_OK;
}

// --------------------------------------------------------------- resample with built-in scratch
// The sums of cetra_resample_static (cetra.h) live in the library image instead of a caller workspace: a fixed
// array in device global memory, one copy per GPU that loads this module, there until the process exits.
// 256-byte alignment matches what the workspace entry points require of theirs.
static __device__ __align__(256) double2 g_static_sums[CETRA_RESAMPLE_STATIC_MAX_POINTS];

// In host code `g_static_sums` is only a handle the runtime uses to find the symbol, not somewhere a kernel can
// write: handing it to a launch would fault, or on a machine where the GPU can reach host memory quietly scribble
// over the host-side shadow.  The real device address differs per GPU, so it is asked for once per device, with
// that device current, and kept here.
constexpr int kMaxStaticDevices = 64;
static std::mutex g_static_mutex;
static double2 *g_static_addr[kMaxStaticDevices] = {};

static int static_sums_on_current_device(double2 **out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return CETRA_ERR_CUDA;
    }
    if (dev < 0 || dev >= kMaxStaticDevices) return CETRA_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        double2 *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_static_sums);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return CETRA_ERR_CUDA;
        }
        g_static_addr[dev] = p;
    }
    *out = g_static_addr[dev];
    return CETRA_OK;
}

}  // namespace cetra

using namespace cetra;

extern "C" {

int cetra_median_cadence(const double *times_host, int64_t n, double *cadence) {
    if (!times_host || !cadence || n < 2) return CETRA_ERR_INVALID_ARG;
    std::vector<double> t;
    t.reserve(static_cast<size_t>(n));
    for (int64_t i = 0; i < n; ++i)
        if (std::isfinite(times_host[i])) t.push_back(times_host[i]);
    if (t.size() < 2) return CETRA_ERR_INVALID_ARG;
    std::sort(t.begin(), t.end());
    std::vector<double> d(t.size() - 1);
    for (size_t i = 0; i + 1 < t.size(); ++i) d[i] = t[i + 1] - t[i];
    std::sort(d.begin(), d.end());
    const size_t m = d.size();
    const double c = (m % 2) ? d[m / 2] : 0.5 * (d[m / 2 - 1] + d[m / 2]);     // R22
    if (!(c > 0.0)) return CETRA_ERR_INVALID_ARG;
    *cadence = c;
    return CETRA_OK;
}

int cetra_resample_template(const float *model_host, int32_t n_model, float *template_host, int32_t n_template) {
    if (!model_host || !template_host || n_model < 2 || n_template < 2) return CETRA_ERR_INVALID_ARG;
    // "resampled to a user-defined number of samples using simple linear interpolation"; both ends kept
    const double step = static_cast<double>(n_model - 1) / static_cast<double>(n_template - 1);
    for (int32_t m = 0; m < n_template; ++m) {
        const double u = static_cast<double>(m) * step;
        int32_t i0 = static_cast<int32_t>(floor(u));
        if (i0 > n_model - 2) i0 = n_model - 2;
        const double fr = u - static_cast<double>(i0);
        const double a = static_cast<double>(model_host[i0]), b = static_cast<double>(model_host[i0 + 1]);
        template_host[m] = static_cast<float>(a + (b - a) * fr);
    }
    return CETRA_OK;
}

int cetra_resample_grid(const double *times_host, int64_t n, double cadence, double pad_days, double *t_start,
                        double *cadence_out, int64_t *n_out) {
    if (!times_host || !t_start || !cadence_out || !n_out || n < 2 || !(pad_days >= 0.0) || !std::isfinite(pad_days))
        return CETRA_ERR_INVALID_ARG;
    double c = cadence;
    if (!(c > 0.0)) {
        const int rc = cetra_median_cadence(times_host, n, &c);
        if (rc != CETRA_OK) return rc;
    }
    if (!std::isfinite(c)) return CETRA_ERR_INVALID_ARG;
    double lo = INFINITY, hi = -INFINITY;
    for (int64_t i = 0; i < n; ++i) {
        if (!std::isfinite(times_host[i])) continue;
        lo = std::min(lo, times_host[i]);
        hi = std::max(hi, times_host[i]);
    }
    if (!(hi >= lo)) return CETRA_ERR_INVALID_ARG;
    const double pad_n = ceil(pad_days / c);
    const double span = floor((hi - lo) / c + 0.5) + 1.0 + 2.0 * pad_n;
    if (!(span < 2.0e9)) return CETRA_ERR_UNSUPPORTED;
    *t_start = lo - pad_n * c;
    *cadence_out = c;
    *n_out = static_cast<int64_t>(span);
    return CETRA_OK;
}

size_t cetra_resample_workspace_bytes(int64_t n_in, int32_t n_lc, int64_t n_out) {
    if (n_in < 0 || n_lc < 1 || n_out < 1 || n_in > 0x7fffffffLL || n_out > 0x7ffffffeLL) return 0;
    // output point of every observation, its slot in the per-point lists, counts / cursors, offsets, scan tile totals
    return 2 * align_up(sizeof(int) * static_cast<size_t>(std::max<int64_t>(n_in, 1))) +
           align_up(sizeof(int) * static_cast<size_t>(n_out)) + align_up(sizeof(int) * static_cast<size_t>(n_out + 1)) +
           align_up(sizeof(int) * static_cast<size_t>((n_out + kScanTile - 1) / kScanTile));
}

int cetra_resample(const double *times_dev, const void *flux_dev, const void *flux_err_dev, cetra_dtype dtype,
                   int64_t n_in, int32_t n_lc, double t_start, double cadence, int64_t n_out, void *flux_out_dev,
                   void *flux_err_out_dev, void *workspace_dev, size_t workspace_bytes, void *cuda_stream) {
    if (((!times_dev || !flux_dev || !flux_err_dev) && n_in != 0) || !flux_out_dev || !flux_err_out_dev || n_in < 0 ||
        n_lc < 1 ||
        n_out < 1 || !(cadence > 0.0) || !std::isfinite(cadence) || !std::isfinite(t_start) ||
        (dtype != CETRA_F32 && dtype != CETRA_F64))
        return CETRA_ERR_INVALID_ARG;
    if (n_in > 0x7fffffffLL || n_out > 0x7ffffffeLL) return CETRA_ERR_UNSUPPORTED;      // 32-bit indices
    if (!ws_ok(workspace_dev, workspace_bytes, cetra_resample_workspace_bytes(n_in, n_lc, n_out)))
        return CETRA_ERR_WORKSPACE;
    if (have_device() != CETRA_OK) return CETRA_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Carver ws(workspace_dev);
    int *cell_of = ws.take<int>(static_cast<size_t>(std::max<int64_t>(n_in, 1)));
    int *order = ws.take<int>(static_cast<size_t>(std::max<int64_t>(n_in, 1)));
    int *count = ws.take<int>(static_cast<size_t>(n_out));
    int *offsets = ws.take<int>(static_cast<size_t>(n_out + 1));
    int *tile_sum = ws.take<int>(static_cast<size_t>((n_out + kScanTile - 1) / kScanTile));
    const int ni = static_cast<int>(n_in), no = static_cast<int>(n_out);
    CETRA_CUDA_TRY(cudaMemsetAsync(count, 0, sizeof(int) * static_cast<size_t>(n_out), st));
    if (n_in > 0) {
        resample_cells_kernel<<<stream_blocks(n_in), 256, 0, st>>>(times_dev, ni, t_start, cadence, no, cell_of, count);
        CETRA_LAUNCH_CHECK();
    }
    const int tiles = (no + kScanTile - 1) / kScanTile;
    resample_tile_sums_kernel<<<tiles, kScanThreads, 0, st>>>(count, no, tile_sum);
    CETRA_LAUNCH_CHECK();
    resample_scan_kernel<<<tiles, kScanThreads, 0, st>>>(count, tile_sum, offsets, no);
    CETRA_LAUNCH_CHECK();
    if (n_in > 0) {
        resample_fill_kernel<<<stream_blocks(n_in), 256, 0, st>>>(cell_of, ni, count, order);
        CETRA_LAUNCH_CHECK();
        resample_sort_kernel<<<stream_blocks(n_out), 256, 0, st>>>(offsets, no, order);
        CETRA_LAUNCH_CHECK();
    }
    constexpr int kCurvesPerThread = 8;
    const dim3 grid((no + 255) / 256, std::min((n_lc + kCurvesPerThread - 1) / kCurvesPerThread, 65535));
    if (dtype == CETRA_F32)
        resample_sum_kernel<float, kCurvesPerThread><<<grid, 256, 0, st>>>(
            static_cast<const float *>(flux_dev), static_cast<const float *>(flux_err_dev), n_in, n_lc, no, offsets,
            order, static_cast<float *>(flux_out_dev), static_cast<float *>(flux_err_out_dev));
    else
        resample_sum_kernel<double, kCurvesPerThread><<<grid, 256, 0, st>>>(
            static_cast<const double *>(flux_dev), static_cast<const double *>(flux_err_dev), n_in, n_lc, no, offsets,
            order, static_cast<double *>(flux_out_dev), static_cast<double *>(flux_err_out_dev));
    CETRA_LAUNCH_CHECK();
    return CETRA_OK;
}

int64_t cetra_resample_static_max_points(void) { return CETRA_RESAMPLE_STATIC_MAX_POINTS; }

// cetra_resample for callers without a workspace to give (cetra.h has the full contract): the FP64 sums go to
// g_static_sums.  Nothing here allocates; the only set-up is the once-per-device address lookup above, done by the
// first call on each device.  The array still holds the previous call's sums, so the part this call uses is cleared
// first, on the caller's stream, ahead of the accumulation.
int cetra_resample_static(const double *times_dev, const void *flux_dev, const void *flux_err_dev, cetra_dtype dtype,
                          int64_t n_in, int32_t n_lc, double t_start, double cadence, int64_t n_out,
                          void *flux_out_dev, void *flux_err_out_dev, void *cuda_stream) {
    if (((!times_dev || !flux_dev || !flux_err_dev) && n_in != 0) || !flux_out_dev || !flux_err_out_dev || n_in < 0 ||
        n_lc < 1 || n_out < 1 || !(cadence > 0.0) || !std::isfinite(cadence) || !std::isfinite(t_start) ||
        (dtype != CETRA_F32 && dtype != CETRA_F64))
        return CETRA_ERR_INVALID_ARG;
    // n_out alone is tested first so that the product below cannot overflow
    if (n_out > CETRA_RESAMPLE_STATIC_MAX_POINTS ||
        static_cast<long long>(n_lc) * n_out > CETRA_RESAMPLE_STATIC_MAX_POINTS)
        return CETRA_ERR_STATIC_LIMIT;
    double2 *sums = nullptr;
    const int rc = static_sums_on_current_device(&sums);
    if (rc != CETRA_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const long long total_out = static_cast<long long>(n_lc) * n_out;
    CETRA_CUDA_TRY(cudaMemsetAsync(sums, 0, sizeof(double2) * static_cast<size_t>(total_out), st));
    const long long total_in = static_cast<long long>(n_lc) * n_in;
    if (total_in > 0) {
        if (dtype == CETRA_F32)
            resample_accumulate_kernel<float><<<stream_blocks(total_in), 256, 0, st>>>(
                times_dev, static_cast<const float *>(flux_dev), static_cast<const float *>(flux_err_dev), n_in, n_lc,
                t_start, cadence, n_out, sums);
        else
            resample_accumulate_kernel<double><<<stream_blocks(total_in), 256, 0, st>>>(
                times_dev, static_cast<const double *>(flux_dev), static_cast<const double *>(flux_err_dev), n_in,
                n_lc, t_start, cadence, n_out, sums);
        CETRA_LAUNCH_CHECK();
    }
    if (dtype == CETRA_F32)
        resample_finalize_kernel<float><<<stream_blocks(total_out), 256, 0, st>>>(
            sums, total_out, static_cast<float *>(flux_out_dev), static_cast<float *>(flux_err_out_dev));
    else
        resample_finalize_kernel<double><<<stream_blocks(total_out), 256, 0, st>>>(
            sums, total_out, static_cast<double *>(flux_out_dev), static_cast<double *>(flux_err_out_dev));
    CETRA_LAUNCH_CHECK();
    return CETRA_OK;
}

size_t cetra_monotransit_workspace_bytes(int32_t n_lc, int64_t n_t0) {
    if (n_lc < 1 || n_t0 < 1) return 0;
    const size_t cells = static_cast<size_t>(n_lc) * static_cast<size_t>(n_t0);
    return align_up(sizeof(float) * cells) + align_up(sizeof(int) * cells) + align_up(cells);
}

int cetra_monotransit_search(const float *depth_dev, const float *var_dev, const float *dlogL_dev, int32_t n_lc,
                             int32_t n_dur, cetra_t0_grid grid, const double *durations_host, int32_t n_peaks,
                             double excl, float *profile_lr_dev, int32_t *profile_j_dev, cetra_event *events_dev,
                             int32_t *n_found_dev, void *workspace_dev, size_t workspace_bytes, void *cuda_stream) {
    if (!depth_dev || !var_dev || !dlogL_dev || !durations_host || !events_dev || !n_found_dev || n_lc < 1 ||
        n_dur < 1 || grid.n_t0 < 1 || n_peaks < 1 || !(excl >= 0.0) || !std::isfinite(excl) ||
        !(grid.t0_stride > 0.0) || !std::isfinite(grid.t0_stride) || !std::isfinite(grid.t0_start))
        return CETRA_ERR_INVALID_ARG;
    if (n_dur > CETRA_MAX_DURATIONS || grid.n_t0 > 0xfffffffeLL) return CETRA_ERR_UNSUPPORTED;
    EventParams ep;
    for (int j = 0; j < n_dur; ++j) {
        if (!(durations_host[j] > 0.0) || !std::isfinite(durations_host[j])) return CETRA_ERR_INVALID_ARG;
        ep.durations[j] = durations_host[j];
    }
    if (!ws_ok(workspace_dev, workspace_bytes, cetra_monotransit_workspace_bytes(n_lc, grid.n_t0)))
        return CETRA_ERR_WORKSPACE;
    if (have_device() != CETRA_OK) return CETRA_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Carver ws(workspace_dev);
    const size_t cells = static_cast<size_t>(n_lc) * static_cast<size_t>(grid.n_t0);
    float *pl = ws.take<float>(cells);
    int *pj = ws.take<int>(cells);
    unsigned char *dead = ws.take<unsigned char>(cells);
    if (profile_lr_dev) pl = profile_lr_dev;
    if (profile_j_dev) pj = profile_j_dev;
    monotransit_profile_kernel<<<stream_blocks(static_cast<long long>(cells)), 256, 0, st>>>(dlogL_dev, n_lc, n_dur,
                                                                                            grid.n_t0, pl, pj);
    CETRA_LAUNCH_CHECK();
    monotransit_events_kernel<<<n_lc, 1024, 0, st>>>(depth_dev, var_dev, pl, pj, dead, n_dur, grid.n_t0, grid.t0_start,
                                                     grid.t0_stride, ep, n_peaks, excl, events_dev, n_found_dev);
    CETRA_LAUNCH_CHECK();
    return CETRA_OK;
}

size_t cetra_mask_workspace_bytes(int32_t n_lc) {
    if (n_lc < 1) return 0;
    return 3 * align_up(sizeof(double) * static_cast<size_t>(n_lc));
}

int cetra_mask_transits(const double *times_dev, void *flux_dev, cetra_dtype dtype, int64_t n, int32_t n_lc,
                        const double *period_host, const double *t0_host, const double *duration_host, double width,
                        int32_t *n_masked_dev, void *workspace_dev, size_t workspace_bytes, void *cuda_stream) {
    if (!times_dev || !flux_dev || !period_host || !t0_host || !duration_host || n < 1 || n_lc < 1 ||
        !(width >= 0.0) || !std::isfinite(width) || (dtype != CETRA_F32 && dtype != CETRA_F64))
        return CETRA_ERR_INVALID_ARG;
    if (!ws_ok(workspace_dev, workspace_bytes, cetra_mask_workspace_bytes(n_lc))) return CETRA_ERR_WORKSPACE;
    if (have_device() != CETRA_OK) return CETRA_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Carver ws(workspace_dev);
    double *per = ws.take<double>(n_lc), *t0 = ws.take<double>(n_lc), *dur = ws.take<double>(n_lc);
    CETRA_CUDA_TRY(cudaMemcpyAsync(per, period_host, sizeof(double) * n_lc, cudaMemcpyHostToDevice, st));
    CETRA_CUDA_TRY(cudaMemcpyAsync(t0, t0_host, sizeof(double) * n_lc, cudaMemcpyHostToDevice, st));
    CETRA_CUDA_TRY(cudaMemcpyAsync(dur, duration_host, sizeof(double) * n_lc, cudaMemcpyHostToDevice, st));
    if (n_masked_dev) CETRA_CUDA_TRY(cudaMemsetAsync(n_masked_dev, 0, sizeof(int32_t) * n_lc, st));
    MaskParams mp{per, t0, dur};
    const long long total = static_cast<long long>(n_lc) * n;
    if (dtype == CETRA_F32)
        mask_transits_kernel<float><<<stream_blocks(total), 256, 0, st>>>(times_dev, static_cast<float *>(flux_dev), n,
                                                                          n_lc, mp, width, n_masked_dev);
    else
        mask_transits_kernel<double><<<stream_blocks(total), 256, 0, st>>>(times_dev, static_cast<double *>(flux_dev),
                                                                           n, n_lc, mp, width, n_masked_dev);
    CETRA_LAUNCH_CHECK();
    return CETRA_OK;
}

}  // extern "C"
