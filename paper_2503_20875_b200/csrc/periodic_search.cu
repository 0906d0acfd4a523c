// Periodic search (§2.3): steps P1-P4 of DESIGN.md.
//
//   P1 epoch offsets        off_e = llrint(e * P_k / stride) in FP64, 32 epochs per warp at a time (R11)
//   P2 fold-gather-sum      SA = sum_e S_wmm[j][p + off_e], SB = sum_e S_wmf[j][p + off_e]
//   P3 combine              Z = SB/SA, var = 1/SA, LR = 1/2 SB^2/SA  (= Eq. 4 summed at Z)
//   P4 argmax               per period: max LR over (duration, phase), ties -> smallest j, then p
//
// The combined (depth, var, LR) arrays of a period are never materialised: a warp folds (period, duration)
// pairs in registers and publishes one packed 64-bit key per period with atomicMax.
// A block keeps the (S_wmm, S_wmf) row of one duration in shared memory (one TMA bulk copy per row)
// and pulls (row, period-segment) work items from a global queue; there a warp folds two neighbouring
// periods from one register window (fold_group_argmax_kernel).  Rows that do not fit in shared memory
// are gathered from global memory with coalesced read-only loads, one period per warp (fold_argmax_kernel<false>;
// neighbouring warps fold neighbouring periods, so 96 % of the sectors hit in L1).
#include "periodic_search.cuh"

#include <math.h>

#include <algorithm>

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

__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

template <bool kSmemRow>
__device__ __forceinline__ float2 load_cell(const float2 *p) {
    if (kSmemRow) return *p;
    return __ldg(p);
}

// Epoch offsets of one block of 32 epochs, as a warp holds them: lane l owns epoch eb + l.
//   oa     off_e = llrint(e * r) of the lane's epoch (FP64, R11)
//   dmask  bit l = off_{e+1} - off_e - floor(r)  (0 or 1 when `plain`)
//   plain  every in-range step is floor(r) or floor(r)+1, so the warp can walk the offsets with
//          off += floor(r) + bit: the inner loop then needs no shuffle (a SHFL costs a shared-memory
//          wavefront, the resource this kernel is bound by).  Otherwise the offsets are broadcast by SHFL.
struct EpochBlock {
    long long oa;
    int off0;           // offset of epoch eb (the same in every lane)
    unsigned dmask;
    bool plain;
};

__device__ __forceinline__ EpochBlock epoch_block(int eb, double r, long long r_floor, int n_t0, int lane) {
    EpochBlock b;
    const double e = static_cast<double>(eb + lane);
    b.oa = __double2ll_rn(__dmul_rn(e, r));
    const long long o0 = __double2ll_rn(__dmul_rn(static_cast<double>(eb), r));
    b.off0 = static_cast<int>(o0 < 0x7fffffffLL ? o0 : 0x7fffffffLL);
    const long long ob = __double2ll_rn(__dmul_rn(e + 1.0, r));
    const long long dl = ob - b.oa - r_floor;
    b.dmask = __ballot_sync(0xffffffffu, dl != 0);
    b.plain = __ballot_sync(0xffffffffu, b.oa <= n_t0 - 1 && (dl < 0 || dl > 1)) == 0u;
    return b;
}

// One pass of a warp over G*32 consecutive phases starting at p0: lane handles phases p0 + lane + 32 g.
// Cells beyond n_t0-1 are zero (row padding), so epochs that run off the end for the later phases of the
// pass add nothing; the epoch loop itself stops at the last epoch valid for p0.
template <int G, bool kSmemRow>
__device__ __forceinline__ void fold_pass(const float2 *__restrict__ row, int p0, int n_t0, int n_phase, double r,
                                          long long r_floor, const EpochBlock &b0, int lane, float &best_lr,
                                          int &best_p) {
    float2 acc[G];
#pragma unroll
    for (int g = 0; g < G; ++g) acc[g] = make_float2(0.f, 0.f);
    const long long limit = static_cast<long long>(n_t0) - 1 - p0;     // off_e <= limit  <=>  p0 + off_e <= I-1
    const float2 *base = row + p0 + lane;
    const int step = static_cast<int>(r_floor < 0x3fffffffLL ? r_floor : 0x3fffffffLL);
    EpochBlock b = b0;
    for (int eb = 0;; eb += 32) {
        if (eb > 0) b = epoch_block(eb, r, r_floor, n_t0, lane);
        const bool ok = b.oa <= limit;
        const int cnt = __popc(__ballot_sync(0xffffffffu, ok));      // offsets are monotone in e: valid ones are a prefix
        if (b.plain) {
            int off = b.off0;
            unsigned m = b.dmask;
#pragma unroll 4
            for (int t = 0; t < cnt; ++t) {
                const float2 *ptr = base + off;
#pragma unroll
                for (int g = 0; g < G; ++g) acc[g] = add2(acc[g], load_cell<kSmemRow>(ptr + 32 * g));
                off += step + static_cast<int>(m & 1u);
                m >>= 1;
            }
        } else {
            const int my_off = ok ? static_cast<int>(b.oa) : 0;
            for (int t = 0; t < cnt; ++t) {
                const float2 *ptr = base + __shfl_sync(0xffffffffu, my_off, t);
#pragma unroll
                for (int g = 0; g < G; ++g) acc[g] = add2(acc[g], load_cell<kSmemRow>(ptr + 32 * g));
            }
        }
        if (cnt < 32) break;
    }
#pragma unroll
    for (int g = 0; g < G; ++g) {
        const int p = p0 + lane + 32 * g;
        const float a = acc[g].x, bsum = acc[g].y;
        // candidate iff some epoch contributed (S_wmm > 0); selection uses an approximate reciprocal,
        // the reported values are recomputed with IEEE division by finalize_peaks_kernel
        const float lr = 0.5f * bsum * bsum * rcp_approx(a);
        if (p < n_phase && a > 0.f && lr > best_lr) { best_lr = lr; best_p = p; }
    }
}

template <bool kSmemRow>
__device__ __forceinline__ void fold_period(const float2 *__restrict__ row, int n_t0, double r, int n_phase, int lane,
                                            float &best_lr, int &best_p) {
    best_lr = -1.f;
    best_p = 0x7fffffff;
    const long long r_floor = __double2ll_rd(r);
    const EpochBlock b0 = epoch_block(0, r, r_floor, n_t0, lane);   // the first 32 epochs serve every pass
    int p0 = 0;
    for (; p0 + 32 * kFoldR <= n_phase; p0 += 32 * kFoldR)
        fold_pass<kFoldR, kSmemRow>(row, p0, n_t0, n_phase, r, r_floor, b0, lane, best_lr, best_p);
    static_assert(kFoldR == 8, "the remainder below covers 1..kFoldR groups by powers of two");
    const int groups = (n_phase - p0 + 31) >> 5;                  // the last pass: the next power of two of groups
    if (groups > 4) fold_pass<8, kSmemRow>(row, p0, n_t0, n_phase, r, r_floor, b0, lane, best_lr, best_p);
    else if (groups > 2) fold_pass<4, kSmemRow>(row, p0, n_t0, n_phase, r, r_floor, b0, lane, best_lr, best_p);
    else if (groups > 1) fold_pass<2, kSmemRow>(row, p0, n_t0, n_phase, r, r_floor, b0, lane, best_lr, best_p);
    else if (groups > 0) fold_pass<1, kSmemRow>(row, p0, n_t0, n_phase, r, r_floor, b0, lane, best_lr, best_p);
    // warp argmax: larger lr wins, ties -> smaller phase
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        const float o_lr = __shfl_xor_sync(0xffffffffu, best_lr, s);
        const int o_p = __shfl_xor_sync(0xffffffffu, best_p, s);
        if (o_lr > best_lr || (o_lr == best_lr && o_p < best_p)) { best_lr = o_lr; best_p = o_p; }
    }
}

// Persistent CTAs claim contiguous ranges of work units (unit = kWarps consecutive periods of one row, one
// period per warp) from a global counter, guided self-scheduling: a claim is 1/(2 x CTAs) of what is left,
// so a CTA loads a row a handful of times per launch and the tail still balances.
template <bool kSmemRow>
__global__ void __launch_bounds__(kFoldThreads, 1) fold_argmax_kernel(const __grid_constant__ PeriodicParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    unsigned int *s_claim = reinterpret_cast<unsigned int *>(smem_raw + 8);
    float2 *srow = reinterpret_cast<float2 *>(smem_raw + 16);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int kWarps = kFoldThreads / 32;

    if (kSmemRow && tid == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    long long cur_row = -1;
    uint32_t parity = 0;
    for (;;) {
        if (tid == 0) {
            const long long seen = *reinterpret_cast<volatile unsigned int *>(P.counter);   // may be stale: only sizes the claim
            long long want = (P.n_units - seen) / (2LL * gridDim.x);
            want = want < 1 ? 1 : (want > P.max_claim ? P.max_claim : want);
            s_claim[0] = atomicAdd(P.counter, static_cast<unsigned int>(want));
            s_claim[1] = static_cast<unsigned int>(want);
        }
        __syncthreads();
        long long u = s_claim[0];
        const long long u_end = min(u + static_cast<long long>(s_claim[1]), P.n_units);
        __syncthreads();                       // everyone has read the slot and is done with the previous claim
        if (u >= P.n_units) break;
        while (u < u_end) {
            const long long rowid = u / P.units_per_row;               // lc * n_dur + j
            const long long u_row0 = rowid * P.units_per_row;
            const long long u_stop = min(u_end, u_row0 + P.units_per_row);
            const int j = static_cast<int>(rowid % P.n_dur);
            const long long lc = rowid / P.n_dur;
            const float2 *grow = P.stats + rowid * P.stats_pitch;
            if (kSmemRow && rowid != cur_row) {
                __syncthreads();               // every warp is done with the row about to be overwritten
                if (tid == 0) {
                    const uint32_t bytes = static_cast<uint32_t>(P.stats_pitch) * 8u;
                    mbar_arrive_expect_tx(bar, bytes);
                    bulk_copy_g2s_chunked(srow, grow, bytes, bar);
                }
                mbar_wait(bar, parity);
                parity ^= 1u;
                cur_row = rowid;
            }
            const float2 *row = kSmemRow ? srow : grow;
            const double D = P.durations[j];
            const int k_end = static_cast<int>(min(static_cast<long long>(P.n_per), (u_stop - u_row0) * kWarps));
            for (int k = static_cast<int>(u - u_row0) * kWarps + warp; k < k_end; k += kWarps) {
                const double period = P.periods[k];
                if (!(D < period)) continue;                            // overlapping windows are invalid
                if (P.dur_lo && (j < P.dur_lo[k] || j >= P.dur_hi[k])) continue;
                const double r = __ddiv_rn(period, P.t0_stride);        // period in t0 cells, FP64 (R11)
                const double rc = ceil(r);
                const int n_phase = rc < static_cast<double>(P.n_t0) ? static_cast<int>(rc) : P.n_t0;   // R10
                float best_lr;
                int best_p;
                fold_period<kSmemRow>(row, P.n_t0, r, n_phase, lane, best_lr, best_p);
                if (lane == 0 && best_lr >= 0.f) {
                    const unsigned int id = static_cast<unsigned int>(j) * static_cast<unsigned int>(P.n_t0) +
                                            static_cast<unsigned int>(best_p);
                    const unsigned long long key =
                        (static_cast<unsigned long long>(__float_as_uint(best_lr)) << 32) | (0xffffffffu - id);
                    atomicMax(P.keys + lc * P.n_per + k, key);
                }
            }
            u = u_stop;
        }
    }
}

// ------------------------------------------------------------------------------- grouped fold (P1-P4)
// Neighbouring trial periods fold almost the same cells: at epoch e the offsets llrint(e r_k) of two consecutive
// periods differ by a few cells.  A warp therefore folds kGrpT = 2 periods together; a lane owns G consecutive
// phases and, per epoch, loads the G + d cells that cover both periods once (8-byte LDS at a lane stride of G
// cells: G odd => conflict-free) and adds them into the two sets of G accumulators at shift 0 and
// d = off_1(e) - off_0(e), a warp-uniform switch with one straight-line case per shift.  One load then feeds up to
// two adds, which lifts the kernel off the one-load-per-cell bound of the shared-memory crossbar (the per-period
// kernel's limit, profiles/r01c).  The per-cell arithmetic, the order of the epoch sum and the offsets (FP64, R11)
// are exactly those of the per-period kernel.  Epochs whose offsets differ by more than kGrpS cells (long
// periods) are gathered period by period in the same loop.
struct GroupPeriods {
    double r[kGrpT];          // period in t0 cells, ascending
    int n_phase[kGrpT];       // R10; 0 for a period that is not searched on this row
};

__device__ __forceinline__ float2 lds_cell(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}

__device__ __forceinline__ int2 lds_int2(uint32_t addr) {
    int2 v;
    asm volatile("ld.shared.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}

__device__ __forceinline__ void sts_int2(uint32_t addr, int x, int y) {
    asm volatile("st.shared.v2.s32 [%0], {%1, %2};" ::"r"(addr), "r"(x), "r"(y) : "memory");
}

// One epoch of a two-period group whose offsets differ by D cells: the G + D cells from the smaller offset on are
// loaded once; period 0 takes cells [0, G), period 1 cells [D, G + D).
template <int D, int G>
__device__ __forceinline__ void fold_epoch(float2 (&acc)[kGrpT][G], uint32_t ptr) {
    float2 c[G + D];
#pragma unroll
    for (int i = 0; i < G + D; ++i) c[i] = lds_cell(ptr + 8u * i);
#pragma unroll
    for (int g = 0; g < G; ++g) acc[0][g] = add2(acc[0][g], c[g]);
#pragma unroll
    for (int g = 0; g < G; ++g) acc[1][g] = add2(acc[1][g], c[g + D]);
}

// One pass of a warp over 32*G consecutive phases starting at p0; lane owns phases p0 + lane*G + g.
// ew: the warp's shared-memory slots for one block of 32 epochs: ew[e] = (off_0, off_1), the offsets of the two
// periods of the group (off_1 >= off_0 because the periods are sorted).  When off_1 - off_0 <= kGrpS the G + d
// cells from off_0 on serve both periods from one register window; otherwise each period gathers its own cells.
template <int G, bool kLastPass>
__device__ __forceinline__ void fold_group_pass(uint32_t srow, int p0, int n_t0, const GroupPeriods &gp,
                                                uint32_t ew, int lane, float (&best_lr)[kGrpT],
                                                int (&best_p)[kGrpT]) {
    static_assert(kGrpT == 2 && kGrpS == 7, "two periods per warp, one switch case per shift");
    float2 acc[kGrpT][G];
#pragma unroll
    for (int t = 0; t < kGrpT; ++t)
#pragma unroll
        for (int g = 0; g < G; ++g) acc[t][g] = make_float2(0.f, 0.f);
    const long long limit = static_cast<long long>(n_t0) - 1 - p0;   // off_e <= limit  <=>  p0 + off_e <= I-1
    const uint32_t base = srow + 8u * static_cast<uint32_t>(p0 + lane * G);
    for (int eb = 0;; eb += 32) {
        // P1: lane l derives the offsets of epoch eb + l for the two periods (FP64, R11)
        const double e = static_cast<double>(eb + lane);
        const long long o0 = __double2ll_rn(__dmul_rn(e, gp.r[0]));
        const long long o1 = __double2ll_rn(__dmul_rn(e, gp.r[1]));
        const bool ok = o0 <= limit;                                  // r ascending: o0 is the smaller
        const long long cap = 0x0fffffffLL;
        __syncwarp();                                                 // the previous block's words are consumed
        sts_int2(ew + 8u * lane, static_cast<int>(o0 < cap ? o0 : cap), static_cast<int>(o1 < cap ? o1 : cap));
        __syncwarp();
        const int cnt = __popc(__ballot_sync(0xffffffffu, ok));       // offsets are monotone in e: a prefix is valid
        for (int t = 0; t < cnt; ++t) {
            const int2 w = lds_int2(ew + 8u * t);                     // broadcast load
            const uint32_t ptr = base + 8u * static_cast<uint32_t>(w.x);
            const int d = w.y - w.x;
            // one case per shift: load the G + d cells that serve both periods, add them at shift 0 and d
            switch (d) {
                case 0: fold_epoch<0, G>(acc, ptr); break;
                case 1: fold_epoch<1, G>(acc, ptr); break;
                case 2: fold_epoch<2, G>(acc, ptr); break;
                case 3: fold_epoch<3, G>(acc, ptr); break;
                case 4: fold_epoch<4, G>(acc, ptr); break;
                case 5: fold_epoch<5, G>(acc, ptr); break;
                case 6: fold_epoch<6, G>(acc, ptr); break;
                case 7: fold_epoch<7, G>(acc, ptr); break;
                default: {
                    // offsets too far apart for one window: each period gathers its own cells
#pragma unroll
                    for (int g = 0; g < G; ++g) acc[0][g] = add2(acc[0][g], lds_cell(ptr + 8u * g));
                    if (w.y <= limit) {
                        const uint32_t pu = base + 8u * static_cast<uint32_t>(w.y);
#pragma unroll
                        for (int g = 0; g < G; ++g) acc[1][g] = add2(acc[1][g], lds_cell(pu + 8u * g));
                    }
                }
            }
        }
        if (cnt < 32) break;
    }
    // P3 + P4 within the lane: phases ascending, strict > keeps the smallest phase on ties.  A cell with no
    // contributing epoch has S_wmm = 0 (and S_wmf = 0): it is not a candidate.
#pragma unroll
    for (int t = 0; t < kGrpT; ++t) {
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const int p = p0 + lane * G + g;
            const float a = acc[t][g].x, bsum = acc[t][g].y;
            const float lr = 0.5f * bsum * bsum * rcp_approx(a);
            const bool in = kLastPass ? p < gp.n_phase[t] : true;
            if (in && a > 0.f && lr > best_lr[t]) { best_lr[t] = lr; best_p[t] = p; }
        }
    }
}

__global__ void __launch_bounds__(kGrpThreads, 1) fold_group_argmax_kernel(const __grid_constant__ PeriodicParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int kWarps = kGrpThreads / 32;
    constexpr int kUnitPeriods = kWarps * kGrpT;
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    unsigned int *s_claim = reinterpret_cast<unsigned int *>(smem_raw + 8);
    int2 *s_ew = reinterpret_cast<int2 *>(smem_raw + 16);                              // [kWarps][32]
    float2 *srow = reinterpret_cast<float2 *>(smem_raw + kGrpHeaderBytes);
    const uint32_t srow_addr = smem_u32(srow);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t ew = smem_u32(s_ew + warp * 32);

    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    long long cur_row = -1;
    uint32_t parity = 0;
    for (;;) {
        if (tid == 0) {
            const long long seen = *reinterpret_cast<volatile unsigned int *>(P.counter);   // may be stale: only sizes the claim
            long long want = (P.n_units - seen) / (2LL * gridDim.x);
            want = want < 1 ? 1 : (want > P.max_claim ? P.max_claim : want);
            s_claim[0] = atomicAdd(P.counter, static_cast<unsigned int>(want));
            s_claim[1] = static_cast<unsigned int>(want);
        }
        __syncthreads();
        long long u = s_claim[0];
        const long long u_end = min(u + static_cast<long long>(s_claim[1]), P.n_units);
        __syncthreads();                       // everyone has read the slot and is done with the previous claim
        if (u >= P.n_units) break;
        while (u < u_end) {
            const long long rowid = u / P.units_per_row;               // lc * n_dur + j
            const long long u_row0 = rowid * P.units_per_row;
            const long long u_stop = min(u_end, u_row0 + P.units_per_row);
            const int j = static_cast<int>(rowid % P.n_dur);
            const long long lc = rowid / P.n_dur;
            if (rowid != cur_row) {
                __syncthreads();               // every warp is done with the row about to be overwritten
                if (tid == 0) {
                    const uint32_t bytes = static_cast<uint32_t>(P.stats_pitch) * 8u;
                    mbar_arrive_expect_tx(bar, bytes);
                    bulk_copy_g2s_chunked(srow, P.stats + rowid * P.stats_pitch, bytes, bar);
                }
                mbar_wait(bar, parity);
                parity ^= 1u;
                cur_row = rowid;
            }
            const double D = P.durations[j];
            const int k_end = static_cast<int>(min(static_cast<long long>(P.n_per), (u_stop - u_row0) * kUnitPeriods));
            for (int k0 = static_cast<int>(u - u_row0) * kUnitPeriods + warp * kGrpT; k0 < k_end;
                 k0 += kUnitPeriods) {
                // the group's periods, sorted by ascending r (warp-uniform values)
                GroupPeriods gp;
                int kk[kGrpT];
                int n_phase_max = 0;
#pragma unroll
                for (int t = 0; t < kGrpT; ++t) {
                    const int k = min(k0 + t, P.n_per - 1);            // ragged last group: repeat the last period
                    const double period = P.periods[k];
                    bool on = k0 + t < P.n_per && D < period;          // overlapping windows are invalid
                    if (on && P.dur_lo && (j < P.dur_lo[k] || j >= P.dur_hi[k])) on = false;
                    const double r = __ddiv_rn(period, P.t0_stride);   // period in t0 cells, FP64 (R11)
                    const double rc = ceil(r);
                    const int n_phase = rc < static_cast<double>(P.n_t0) ? static_cast<int>(rc) : P.n_t0;   // R10
                    gp.r[t] = r;
                    gp.n_phase[t] = on ? n_phase : 0;
                    kk[t] = k;
                    n_phase_max = max(n_phase_max, gp.n_phase[t]);
                }
                if (n_phase_max == 0) continue;
#define CETRA_CSWAP(a, b)                                                                         \
    if (gp.r[a] > gp.r[b]) {                                                                      \
        const double tr = gp.r[a]; gp.r[a] = gp.r[b]; gp.r[b] = tr;                               \
        const int tn = gp.n_phase[a]; gp.n_phase[a] = gp.n_phase[b]; gp.n_phase[b] = tn;          \
        const int tk = kk[a]; kk[a] = kk[b]; kk[b] = tk;                                          \
    }
                CETRA_CSWAP(0, 1)
#undef CETRA_CSWAP
                int n_phase_min = 0x7fffffff;                          // over the searched periods of the group
#pragma unroll
                for (int t = 0; t < kGrpT; ++t)
                    if (gp.n_phase[t] > 0) n_phase_min = min(n_phase_min, gp.n_phase[t]);
                const bool all_on = gp.n_phase[0] > 0 && gp.n_phase[1] > 0;
                float best_lr[kGrpT];
                int best_p[kGrpT];
#pragma unroll
                for (int t = 0; t < kGrpT; ++t) { best_lr[t] = -1.f; best_p[t] = 0x7fffffff; }
                // full passes while every phase of the pass is a phase of every period of the group
                int p0 = 0;
                if (all_on)
                    for (; p0 + 32 * kGrpG <= n_phase_min; p0 += 32 * kGrpG)
                        fold_group_pass<kGrpG, false>(srow_addr, p0, P.n_t0, gp, ew, lane, best_lr, best_p);
                constexpr int kTailG = kGrpG + 2;                      // widest last pass
                for (; p0 + 32 * kTailG < n_phase_max; p0 += 32 * kGrpG)
                    fold_group_pass<kGrpG, true>(srow_addr, p0, P.n_t0, gp, ew, lane, best_lr, best_p);
                // the last pass: the narrowest odd number of phases per lane that covers what is left
                const int left = n_phase_max - p0;
                if (left > 32 * 11) fold_group_pass<13, true>(srow_addr, p0, P.n_t0, gp, ew, lane, best_lr, best_p);
                else if (left > 32 * 9) fold_group_pass<11, true>(srow_addr, p0, P.n_t0, gp, ew, lane, best_lr, best_p);
                else if (left > 32 * 7) fold_group_pass<9, true>(srow_addr, p0, P.n_t0, gp, ew, lane, best_lr, best_p);
                else if (left > 32 * 5) fold_group_pass<7, true>(srow_addr, p0, P.n_t0, gp, ew, lane, best_lr, best_p);
                else if (left > 32 * 3) fold_group_pass<5, true>(srow_addr, p0, P.n_t0, gp, ew, lane, best_lr, best_p);
                else if (left > 32) fold_group_pass<3, true>(srow_addr, p0, P.n_t0, gp, ew, lane, best_lr, best_p);
                else if (left > 0) fold_group_pass<1, true>(srow_addr, p0, P.n_t0, gp, ew, lane, best_lr, best_p);
                // P4 across the warp: larger lr wins, ties -> smaller phase; one atomicMax per period
#pragma unroll
                for (int t = 0; t < kGrpT; ++t) {
                    float lr = best_lr[t];
                    int p = best_p[t];
#pragma unroll
                    for (int s = 16; s > 0; s >>= 1) {
                        const float o_lr = __shfl_xor_sync(0xffffffffu, lr, s);
                        const int o_p = __shfl_xor_sync(0xffffffffu, p, s);
                        if (o_lr > lr || (o_lr == lr && o_p < p)) { lr = o_lr; p = o_p; }
                    }
                    if (lane == 0 && lr >= 0.f) {
                        const unsigned int id = static_cast<unsigned int>(j) * static_cast<unsigned int>(P.n_t0) +
                                                static_cast<unsigned int>(p);
                        const unsigned long long key =
                            (static_cast<unsigned long long>(__float_as_uint(lr)) << 32) | (0xffffffffu - id);
                        atomicMax(P.keys + lc * P.n_per + kk[t], key);
                    }
                }
            }
            u = u_stop;
        }
    }
}

// One thread per (light curve, period): decode the winning (j, p), redo its fold in the same order with
// IEEE division, count the contributing epochs and write the record.
__global__ void finalize_peaks_kernel(const __grid_constant__ PeriodicParams P, cetra_peak *__restrict__ peaks) {
    const long long total = static_cast<long long>(P.n_lc) * P.n_per;
    for (long long idx = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; idx < total;
         idx += static_cast<long long>(gridDim.x) * blockDim.x) {
        const unsigned long long key = P.keys[idx];
        cetra_peak out;
        const float nanv = __int_as_float(0x7fc00000);
        out.lr = nanv; out.depth = nanv; out.depth_var = nanv; out.t0 = nanv;
        out.i_t0 = -1; out.j_dur = -1; out.n_transits = 0; out.reserved = 0;
        if (key != 0ull) {
            const long long lc = idx / P.n_per;
            const int k = static_cast<int>(idx - lc * P.n_per);
            const unsigned int id = 0xffffffffu - static_cast<unsigned int>(key & 0xffffffffull);
            const int j = static_cast<int>(id / static_cast<unsigned int>(P.n_t0));
            const int p = static_cast<int>(id - static_cast<unsigned int>(j) * static_cast<unsigned int>(P.n_t0));
            const float2 *row = P.stats + (lc * P.n_dur + j) * P.stats_pitch;
            const double r = __ddiv_rn(P.periods[k], P.t0_stride);
            float sa = 0.f, sb = 0.f;
            int ntr = 0;
            for (long long e = 0;; ++e) {
                const long long cell = p + __double2ll_rn(__dmul_rn(static_cast<double>(e), r));
                if (cell > P.n_t0 - 1) break;
                const float2 ab = row[cell];
                sa += ab.x;
                sb += ab.y;
                ntr += ab.x > 0.f ? 1 : 0;
            }
            out.depth = sb / sa;                                     // common depth Z
            out.depth_var = 1.0f / sa;
            out.lr = 0.5f * sb * out.depth;
            out.t0 = static_cast<float>(P.t0_start + static_cast<double>(p) * P.t0_stride);
            out.i_t0 = p; out.j_dur = j; out.n_transits = ntr;
        }
        peaks[idx] = out;
    }
}

// (depth, var) grids -> (S_wmm, S_wmf) rows: S_wmm = 1/var, S_wmf = depth/var, null (NaN) cells -> 0.
__global__ void grids_to_stats_kernel(const float *__restrict__ depth, const float *__restrict__ var, long long n_rows,
                                      long long n_t0, long long pitch, float2 *__restrict__ stats) {
    const long long total = n_rows * pitch;
    for (long long idx = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; idx < total;
         idx += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long rowid = idx / pitch;
        const long long i = idx - rowid * pitch;
        float2 out = make_float2(0.f, 0.f);
        if (i < n_t0) {
            const float d = depth[rowid * n_t0 + i], v = var[rowid * n_t0 + i];
            if (isfinite(d) && isfinite(v) && v > 0.f) {
                const float a = 1.0f / v;
                const float b = d / v;
                if (isfinite(a) && isfinite(b)) out = make_float2(a, b);
            }
        }
        stats[idx] = out;
    }
}

// ------------------------------------------------------------------------------------------- host
int build_periodic_plan(int32_t n_lc, int32_t n_dur, cetra_t0_grid grid, const double *durations_host,
                        const double *periods_host, int32_t n_per, int smem_limit, int n_sm, PeriodicPlan *pl) {
    if (!durations_host || !periods_host || n_lc < 1 || n_dur < 1 || n_per < 1 || grid.n_t0 < 1 ||
        !(grid.t0_stride > 0.0) || !std::isfinite(grid.t0_stride) || !std::isfinite(grid.t0_start))
        return CETRA_ERR_INVALID_ARG;
    if (n_dur > CETRA_MAX_DURATIONS) return CETRA_ERR_UNSUPPORTED;
    // the packed cell id (j * n_t0 + p) must fit 32 bits, cell indices an int
    if (grid.n_t0 > 0x7fffffffLL - 4096 || static_cast<long long>(n_dur) * grid.n_t0 >= 0xffffffffLL)
        return CETRA_ERR_UNSUPPORTED;
    for (int k = 0; k < n_per; ++k)
        if (!(periods_host[k] >= grid.t0_stride) || !std::isfinite(periods_host[k])) return CETRA_ERR_INVALID_ARG;
    PeriodicParams &P = pl->P;
    for (int j = 0; j < n_dur; ++j) {
        if (!(durations_host[j] > 0.0) || !std::isfinite(durations_host[j])) return CETRA_ERR_INVALID_ARG;
        P.durations[j] = durations_host[j];
    }
    P.n_lc = n_lc; P.n_dur = n_dur; P.n_t0 = static_cast<int>(grid.n_t0); P.n_per = n_per;
    P.t0_start = grid.t0_start; P.t0_stride = grid.t0_stride;
    P.stats_pitch = cetra_stats_pitch(grid.n_t0);
    const size_t row_bytes = static_cast<size_t>(P.stats_pitch) * sizeof(float2);
    constexpr size_t kGrpHeader = kGrpHeaderBytes;
    pl->row_in_smem = row_bytes + kGrpHeader <= static_cast<size_t>(smem_limit);
    pl->smem_bytes = pl->row_in_smem ? row_bytes + kGrpHeader : 16;
    // work units: consecutive periods of one row, one period (per-period kernel) or kGrpT periods (grouped
    // kernel) per warp; see the kernels
    const long long rows = static_cast<long long>(n_lc) * n_dur;
    const int unit_periods = pl->row_in_smem ? (kGrpThreads / 32) * kGrpT : kFoldThreads / 32;
    P.units_per_row = (n_per + unit_periods - 1) / unit_periods;
    P.n_units = rows * P.units_per_row;
    if (P.n_units > 0x7fffffffLL - (1LL << 24)) return CETRA_ERR_UNSUPPORTED;   // 32-bit queue head + overshoot
    P.max_claim = std::max(1, 4 * P.units_per_row);
    const int per_sm = 1;                                     // both fold kernels fill an SM with one CTA
    pl->grid = static_cast<int>(std::min<long long>(P.n_units, static_cast<long long>(n_sm) * per_sm));
    return CETRA_OK;
}

size_t periodic_workspace_bytes(int32_t n_lc, int32_t n_per) {
    size_t b = 0;
    b += align_up(sizeof(double) * static_cast<size_t>(n_per));                           // periods
    b += 2 * align_up(sizeof(int) * static_cast<size_t>(n_per));                          // dur_lo, dur_hi
    b += align_up(sizeof(unsigned long long) * static_cast<size_t>(n_lc) * n_per + 256);  // keys + counter
    return b;
}

int run_periodic(PeriodicPlan &pl, const float2 *stats_dev, const double *periods_host, const int32_t *dur_lo_host,
                 const int32_t *dur_hi_host, bool upload, cetra_peak *peaks_dev, void *workspace_dev,
                 cudaStream_t st) {
    PeriodicParams &P = pl.P;
    Carver ws(workspace_dev);
    double *periods = ws.take<double>(P.n_per);
    int *lo = ws.take<int>(P.n_per);
    int *hi = ws.take<int>(P.n_per);
    const size_t n_keys = static_cast<size_t>(P.n_lc) * P.n_per;
    unsigned long long *keys = ws.take<unsigned long long>(n_keys + 32);
    const bool ranges = dur_lo_host && dur_hi_host;
    if (upload) {
        CETRA_CUDA_TRY(cudaMemcpyAsync(periods, periods_host, sizeof(double) * P.n_per, cudaMemcpyHostToDevice, st));
        if (ranges) {
            CETRA_CUDA_TRY(cudaMemcpyAsync(lo, dur_lo_host, sizeof(int) * P.n_per, cudaMemcpyHostToDevice, st));
            CETRA_CUDA_TRY(cudaMemcpyAsync(hi, dur_hi_host, sizeof(int) * P.n_per, cudaMemcpyHostToDevice, st));
        }
    }
    P.stats = stats_dev;
    P.periods = periods;
    P.dur_lo = ranges ? lo : nullptr;
    P.dur_hi = ranges ? hi : nullptr;
    P.keys = keys;
    P.counter = reinterpret_cast<unsigned int *>(keys + n_keys);
    CETRA_CUDA_TRY(cudaMemsetAsync(keys, 0, sizeof(unsigned long long) * (n_keys + 32), st));
    profile_mark(kProfFold, true, st);
    if (pl.row_in_smem) {
        auto k = fold_group_argmax_kernel;
        CETRA_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_bytes));
        k<<<pl.grid, kGrpThreads, pl.smem_bytes, st>>>(P);
    } else {
        fold_argmax_kernel<false><<<pl.grid, kFoldThreads, pl.smem_bytes, st>>>(P);
    }
    profile_mark(kProfFold, false, st);
    CETRA_LAUNCH_CHECK();
    {
        const long long total = static_cast<long long>(P.n_lc) * P.n_per;
        const int blocks = static_cast<int>(std::min<long long>((total + 255) / 256, 148LL * 8));
        finalize_peaks_kernel<<<blocks, 256, 0, st>>>(P, peaks_dev);
        CETRA_LAUNCH_CHECK();
    }
    return CETRA_OK;
}

int run_grids_to_stats(const float *depth_dev, const float *var_dev, int32_t n_rows, int64_t n_t0,
                       float2 *stats_dev, cudaStream_t st) {
    const long long pitch = cetra_stats_pitch(n_t0);
    const long long total = static_cast<long long>(n_rows) * pitch;
    const int blocks = static_cast<int>(std::min<long long>((total + 255) / 256, 148LL * 16));
    grids_to_stats_kernel<<<blocks, 256, 0, st>>>(depth_dev, var_dev, n_rows, n_t0, pitch, stats_dev);
    CETRA_LAUNCH_CHECK();
    return CETRA_OK;
}

}  // namespace cetra
