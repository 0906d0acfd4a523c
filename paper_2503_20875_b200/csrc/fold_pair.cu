// Periodic search, rows resident in shared memory (§2.3, steps P1-P4 of DESIGN.md): the dominant kernel.
//
//   P1 epoch offsets        off_e = llrint(e * P_k / stride) in FP64, 32 epochs per warp at a time (R11)
//   P2 fold-gather-sum      SA = sum_e S_wmm[j][p + off_e], SB = sum_e S_wmf[j][p + off_e]
//   P3 combine              Z = SB/SA, var = 1/SA, LR = 1/2 SB^2/SA  (= Eq. 4 summed at Z)
//   P4 argmax               per period: max LR over (duration, phase), ties -> smallest j, then p
//
// A CTA keeps the (S_wmm, S_wmf) row of one duration in shared memory (one TMA bulk copy per row) and claims
// (row, 40-period) work units from a global counter.  A warp folds TWO neighbouring trial periods together: a lane
// owns G consecutive phases of each, and at epoch e it loads the cells that cover both periods once (8-byte LDS at
// a lane stride of G cells, G odd => conflict-free) and adds them into the two sets of accumulators at a relative
// shift, so that one loaded cell serves up to two cells of work (the shared-memory crossbar is this kernel's bound).
//
// Two things keep the shared window narrow and the loop lean:
//  * centring: the offsets of the two periods drift apart linearly with the epoch, d(e) = off_1(e) - off_0(e) in
//    [0, d_max].  The lane's phases of the longer period are therefore taken m = d_max/2 phases EARLIER than those
//    of the shorter one (phases q-m .. q-m+G-1 against q .. q+G-1), which turns the shift into s(e) = d(e) - m in
//    [-m, m]: the window is G + |s| cells, half as wide on average.  Which phases a pass covers is bookkeeping: every
//    phase of every period is still folded exactly once, over the same cells in the same epoch order.
//  * class-sorted epochs: the shift is warp-uniform but changes from epoch to epoch (a rounding boundary may or may
//    not fall between e r_0 and e r_1), and the register window needs it at compile time.  Instead of a switch per
//    epoch, the 32 epochs of a block are grouped by shift (one MATCH.ANY) and each shift present runs its own
//    straight-line loop over its epochs (FP32 addition order within a cell then follows the class order, which
//    is as deterministic as the epoch order and covered by the same 1e-5 tolerance).
#include "fold_common.cuh"

#include <math.h>

#include <algorithm>

namespace cetra {

namespace {

#ifndef CETRA_PAIR_S
#define CETRA_PAIR_S 2
#endif
#ifndef CETRA_PAIR_TAILS
#define CETRA_PAIR_TAILS 0
#endif
constexpr int kPairS = CETRA_PAIR_S;                  // |shift| up to which the two periods share one register window
constexpr int kPairFar = 2 * kPairS + 1;   // class of the epochs whose periods gather separately
static_assert(kGrpHeaderBytes >= 16 + (kGrpThreads / 32) * 512 && kGrpHeaderBytes >= 8 * (kPairMaxM + kPairS + 1), "cells before the row start are read (and discarded)");
static_assert(kStatsPad >= 32 * (kGrpG + 2) + kPairS + 1 + kPairMaxM, "cells past the last t0 cell are read as zeros");

// The epochs `mk` (bit t = epoch eb + t) of one block, all of shift S: a straight-line loop over the set bits.
// ew holds the block's (off_0, off_1 - m) words; the next epoch's word is fetched while the current one is folded.
template <int S, int G>
__device__ __forceinline__ void class_loop(float2 (&acc)[kGrpT][G], uint32_t base, uint32_t ew, unsigned mk) {
    // word of an epoch: off_0 when period 0's cells come first in the shared window, else off_1 - m
    const uint32_t ews = ew + (S < 0 ? 4u : 0u);
    int w = lds_int(ews + 8u * static_cast<uint32_t>(__ffs(mk) - 1));
    mk &= mk - 1;
    for (;;) {
        const uint32_t ptr = base + 8u * static_cast<uint32_t>(w);
        // the next epoch's word (slot -1 when there is none: read and ignored)
        w = lds_int(ews + 8u * static_cast<uint32_t>(__ffs(mk) - 1));
        fold_epoch_c<S, G>(acc, ptr);
        if (mk == 0u) break;
        mk &= mk - 1;
    }
}

// Windows too far apart to share: each period gathers its own cells.
template <int G>
__device__ __forceinline__ void far_loop(float2 (&acc)[kGrpT][G], uint32_t base, uint32_t ew, unsigned mk, int limit) {
    while (mk) {
        const int t = __ffs(mk) - 1;
        mk &= mk - 1;
        const int2 w = lds_int2(ew + 8u * t);
        if (w.x <= limit) {
            const uint32_t ptr = base + 8u * static_cast<uint32_t>(w.x);
#pragma unroll
            for (int g = 0; g < G; ++g) acc[0][g] = add2(acc[0][g], lds_cell(ptr + 8u * g));
        }
        if (w.y <= limit) {
            const uint32_t ptr = base + 8u * static_cast<uint32_t>(w.y);
#pragma unroll
            for (int g = 0; g < G; ++g) acc[1][g] = add2(acc[1][g], lds_cell(ptr + 8u * g));
        }
    }
}

// P1 for one block of 32 epochs: lane l derives the offsets of epoch eb + l for the two periods (FP64, R11).
struct EpochWords {
    int o0;        // off_0(e)
    int o1;        // off_1(e) - m: first cell of period 1's lane window
    int cls;       // shift class s + kPairS, kPairFar when |s| > kPairS (validity is decided per pass)
};

__device__ __forceinline__ EpochWords epoch_words(int eb, int lane, const GroupPeriods &gp, int m) {
    // round-to-nearest-even conversion (= llrint for every in-range value), saturating: an offset beyond the int
    // range is beyond every row
    const double e = static_cast<double>(eb + lane);
    const int o0 = __double2int_rn(__dmul_rn(e, gp.r[0]));
    const int o1 = __double2int_rn(__dmul_rn(e, gp.r[1]));
    EpochWords w;
    w.o0 = o0 < 0x3fffffff ? o0 : 0x3fffffff;
    w.o1 = (o1 < 0x3fffffff ? o1 : 0x3fffffff) - m;
    const int s = w.o1 - w.o0;
    w.cls = s < -kPairS || s > kPairS ? kPairFar : s + kPairS;
    return w;
}

// One block of epochs of a pass: the valid epochs are grouped by shift class (MATCH.ANY), and every class present
// runs its own loop.
template <int G>
__device__ __forceinline__ int fold_block(float2 (&acc)[kGrpT][G], uint32_t base, uint32_t ew, const EpochWords &w,
                                          int limit, int lane) {
    const bool ok = min(w.o0, w.o1) <= limit;          // monotone in e: the valid epochs are a prefix
    const unsigned okm = __ballot_sync(0xffffffffu, ok);
    const int cls = ok ? w.cls : -1;
    const unsigned peers = __match_any_sync(0xffffffffu, cls);
    unsigned leaders = __ballot_sync(0xffffffffu, ok && lane == __ffs(peers) - 1);
    while (leaders) {
        const int L = __ffs(leaders) - 1;
        leaders &= leaders - 1;
        const int c = __shfl_sync(0xffffffffu, cls, L);
        const unsigned mk = __shfl_sync(0xffffffffu, peers, L);
        switch (c) {
#define CETRA_PAIR_CASE(SH) case (SH) + kPairS: class_loop<(SH), G>(acc, base, ew, mk); break;
#if CETRA_PAIR_S >= 7
            CETRA_PAIR_CASE(-7) CETRA_PAIR_CASE(-6) CETRA_PAIR_CASE(-5) CETRA_PAIR_CASE(-4)
#endif
#if CETRA_PAIR_S >= 3
            CETRA_PAIR_CASE(-3)
#endif
#if CETRA_PAIR_S >= 2
            CETRA_PAIR_CASE(-2)
#endif
            CETRA_PAIR_CASE(-1) CETRA_PAIR_CASE(0) CETRA_PAIR_CASE(1)
#if CETRA_PAIR_S >= 2
            CETRA_PAIR_CASE(2)
#endif
#if CETRA_PAIR_S >= 3
            CETRA_PAIR_CASE(3)
#endif
#if CETRA_PAIR_S >= 7
            CETRA_PAIR_CASE(4) CETRA_PAIR_CASE(5) CETRA_PAIR_CASE(6) CETRA_PAIR_CASE(7)
#endif
#undef CETRA_PAIR_CASE
            default: far_loop<G>(acc, base, ew, mk, limit); break;
        }
    }
    return __popc(okm);
}

// One pass of a warp: lane owns phases q .. q+G-1 of period 0 and q-m .. q-m+G-1 of period 1, q = p0 + lane*G.
// w0: the words of the first 32 epochs (the same for every pass of the pair, already stored at ew).
template <int G>
__device__ __forceinline__ void fold_pair_pass(uint32_t srow, int p0, int n_t0, const GroupPeriods &gp, int m, int lane,
                                               uint32_t ew, const EpochWords &w0, float (&best_lr)[kGrpT],
                                               int (&best_p)[kGrpT]) {
    static_assert(kPairS == 1 || kPairS == 2 || kPairS == 3 || kPairS == 7, "one switch case per shift");
    float2 acc[kGrpT][G];
#pragma unroll
    for (int t = 0; t < kGrpT; ++t)
#pragma unroll
        for (int g = 0; g < G; ++g) acc[t][g] = make_float2(0.f, 0.f);
    const int limit = n_t0 - 1 - p0;                  // a window starting at offset o holds a cell <= I-1 iff o <= limit
    const uint32_t base = srow + 8u * static_cast<uint32_t>(p0 + lane * G);
    EpochWords w = w0;
    uint32_t ewb = ew;
    for (int eb = 0;; eb += 32) {
        if (eb) {
            // more than 32 epochs (short periods): later blocks use the second half of the warp's word slots
            w = epoch_words(eb, lane, gp, m);
            ewb = ew + 256u;
            __syncwarp();                              // the previous block's words are consumed
            sts_int2(ewb + 8u * lane, w.o0, w.o1);
            __syncwarp();
        }
        if (fold_block<G>(acc, base, ewb, w, limit, lane) < 32) break;
    }
    // P3 + P4 within the lane: phases ascending, strict > keeps the smallest phase on ties.  A cell with no
    // contributing epoch has S_wmm = 0: not a candidate.  LR > best  <=>  SB^2 > 2 best SA: cells that cannot
    // beat the best so far are dismissed with that product (with a margin, so that none is dismissed wrongly);
    // the others take the division.  The reported values are recomputed by finalize_peaks_kernel.
#pragma unroll
    for (int t = 0; t < kGrpT; ++t) {
        const float thr0 = 1.9999981f * best_lr[t];
        bool any = false;
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const float2 pr = mul2(acc[t][g], make_float2(thr0, acc[t][g].y));   // (2 best SA, SB^2) in one issue slot
            any |= pr.y >= pr.x;
        }
        if (any) {
            const int q = p0 + lane * G - (t ? m : 0);
#pragma unroll
            for (int g = 0; g < G; ++g) {
                const float a = acc[t][g].x, bsum = acc[t][g].y;
                const int p = q + g;
                const float lr = 0.5f * bsum * bsum * rcp_approx(a);
                if (p >= 0 && p < gp.n_phase[t] && a >= 1.17549435e-38f && lr > best_lr[t]) {
                    best_lr[t] = lr;
                    best_p[t] = p;
                }
            }
        }
    }
}

}  // namespace

// Persistent CTAs claim contiguous ranges of work units (unit = 40 consecutive periods of one row, two per warp)
// from a global counter, guided self-scheduling: a claim is 1/(2 x CTAs) of what is left, so a CTA loads a row a
// handful of times per launch and the tail still balances.
__global__ void __launch_bounds__(kGrpThreads, 1) fold_pair_argmax_kernel(const __grid_constant__ PeriodicParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int kWarps = kGrpThreads / 32;
    constexpr int kUnitPeriods = kWarps * kGrpT;
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    unsigned int *s_claim = reinterpret_cast<unsigned int *>(smem_raw + 8);
    float2 *srow = reinterpret_cast<float2 *>(smem_raw + kGrpHeaderBytes);
    const uint32_t srow_addr = smem_u32(srow);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t ew = smem_u32(smem_raw + 16 + warp * 512);          // the warp's epoch words: 2 blocks x 32 x 8 B

    if (P.literal && *P.literal) return;       // a caller's likelihood-ratio grid: fold_literal_argmax_kernel searches
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
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the row was read by generic loads
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
                // the pair's periods, sorted by ascending r (warp-uniform values)
                GroupPeriods gp;
                int kk[kGrpT];
#pragma unroll
                for (int t = 0; t < kGrpT; ++t) {
                    const int k = min(k0 + t, P.n_per - 1);            // ragged last pair: repeat the last period
                    const double period = P.periods[k];
                    bool on = k0 + t < P.n_per && D < period;          // overlapping windows are invalid
                    if (on && P.dur_lo && (j < P.dur_lo[k] || j >= P.dur_hi[k])) on = false;
                    const double r = P.r_cells[k];                     // period in t0 cells: P_k / stride in FP64 (R11)
                    const double rc = ceil(r);
                    const int n_phase = rc < static_cast<double>(P.n_t0) ? static_cast<int>(rc) : P.n_t0;   // R10
                    gp.r[t] = r;
                    gp.n_phase[t] = on ? n_phase : 0;
                    kk[t] = k;
                }
                if (gp.n_phase[0] == 0 && gp.n_phase[1] == 0) continue;
                if (gp.r[0] > gp.r[1]) {
                    const double tr = gp.r[0]; gp.r[0] = gp.r[1]; gp.r[1] = tr;
                    const int tn = gp.n_phase[0]; gp.n_phase[0] = gp.n_phase[1]; gp.n_phase[1] = tn;
                    const int tk = kk[0]; kk[0] = kk[1]; kk[1] = tk;
                }
                // centring: half of the largest offset difference of the pair (reached at the last epoch)
                const int m = gp.n_phase[0] > 0 && gp.n_phase[1] > 0 ? centring_shift(gp.r[0], gp.r[1], P.n_t0) : 0;
                // phases to cover: [0, n_phase_0) of period 0 from p0 on, [0, n_phase_1) of period 1 from p0 - m on
                const int n_need = max(gp.n_phase[0], gp.n_phase[1] > 0 ? gp.n_phase[1] + m : 0);
                // The period's best so far (over the rows already folded, by any CTA) dismisses most cells without a
                // division.  It only filters: a cell that ties it still passes (bits - 1), and the packed key
                // decides ties by cell id, so the result does not depend on the order in which rows are folded.
                float best_lr[kGrpT];
                int best_p[kGrpT];
#pragma unroll
                for (int t = 0; t < kGrpT; ++t) {
                    const unsigned int hi = static_cast<unsigned int>(
                        *reinterpret_cast<volatile unsigned long long *>(P.keys + lc * P.n_per + kk[t]) >> 32);
                    best_lr[t] = hi ? __uint_as_float(hi - 1u) : -1.f;
                    best_p[t] = 0x7fffffff;
                }
                // the first 32 epochs' words are the same for every pass of the pair
                const EpochWords w0 = epoch_words(0, lane, gp, m);
                __syncwarp();                                          // the previous pair's words are consumed
                sts_int2(ew + 8u * lane, w0.o0, w0.o1);
                __syncwarp();
                // full passes of kGrpG phases per lane, then the narrowest width (of those compiled) that covers
                // what is left
                for (int p0 = 0; p0 < n_need;) {
                    const int left = n_need - p0;
#if CETRA_PAIR_TAILS == 0
                    const int G = left > 32 * (kGrpG + 2) ? kGrpG : left > 32 * 11 ? 13 : left > 32 * 7 ? 11 : left > 32 * 3 ? 7 : 3;
#elif CETRA_PAIR_TAILS == 1
                    const int G = left > 32 * (kGrpG + 2) ? kGrpG : left > 32 * 11 ? 13 : left > 32 * 5 ? 11 : 5;
#else
                    const int G = left > 32 * (kGrpG + 2) ? kGrpG : left > 32 * 11 ? 13 : left > 32 * 7 ? 11 : 7;
#endif
                    switch (G) {
                        case 13: fold_pair_pass<13>(srow_addr, p0, P.n_t0, gp, m, lane, ew, w0, best_lr, best_p); break;
                        case 11: fold_pair_pass<11>(srow_addr, p0, P.n_t0, gp, m, lane, ew, w0, best_lr, best_p); break;
#if CETRA_PAIR_TAILS == 0
                        case 7: fold_pair_pass<7>(srow_addr, p0, P.n_t0, gp, m, lane, ew, w0, best_lr, best_p); break;
                        default: fold_pair_pass<3>(srow_addr, p0, P.n_t0, gp, m, lane, ew, w0, best_lr, best_p); break;
#elif CETRA_PAIR_TAILS == 1
                        default: fold_pair_pass<5>(srow_addr, p0, P.n_t0, gp, m, lane, ew, w0, best_lr, best_p); break;
#else
                        default: fold_pair_pass<7>(srow_addr, p0, P.n_t0, gp, m, lane, ew, w0, best_lr, best_p); break;
#endif
                    }
                    p0 += 32 * G;
                }
                // P4 across the warp: larger lr wins, ties -> smaller phase; one atomicMax per period.  LR >= 0, so its
                // bit pattern orders like an unsigned integer (REDUX); most pairs end with no lane having reached the
                // period's best so far and publish nothing.
#pragma unroll
                for (int t = 0; t < kGrpT; ++t) {
                    const bool has = best_p[t] != 0x7fffffff;
                    if (__any_sync(0xffffffffu, has)) {
                        const unsigned int bits = has ? __float_as_uint(best_lr[t]) : 0u;
                        const unsigned int top = __reduce_max_sync(0xffffffffu, bits);
                        const unsigned int p = __reduce_min_sync(
                            0xffffffffu, has && bits == top ? static_cast<unsigned int>(best_p[t]) : 0x7fffffffu);
                        if (lane == 0) {
                            const unsigned int id = static_cast<unsigned int>(j) * static_cast<unsigned int>(P.n_t0) + p;
                            const unsigned long long key = (static_cast<unsigned long long>(top) << 32) | (0xffffffffu - id);
                            atomicMax(P.keys + lc * P.n_per + kk[t], key);
                        }
                    }
                }
            }
            u = u_stop;
        }
    }
}

int launch_fold_pair(const PeriodicPlan &pl, cudaStream_t st) {
    auto k = fold_pair_argmax_kernel;
    CETRA_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_bytes));
    k<<<pl.grid, kGrpThreads, pl.smem_bytes, st>>>(pl.P);
    return CETRA_OK;
}

}  // namespace cetra
