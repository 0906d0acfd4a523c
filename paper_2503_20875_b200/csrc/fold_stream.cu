// Periodic search for rows that do not fit in shared memory (§2.3, steps P1-P4 of DESIGN.md): config 4
// (256 464 cells, 2 MB per row) and every TESS sector on the paper's default t0 grid (PAPER.md:87, 1 MB per row).
//
// The row does not fit, but what one work unit touches at one epoch does.  A unit is one duration row and
// kStrUnitPeriods = 38 neighbouring trial periods (two per warp, as in fold_pair_argmax_kernel).  All warps of the
// CTA walk the unit's phase passes and epochs together: at pass p0 (32 G phases) and epoch e the 38 periods read the
// contiguous cells [p0 + off_min(e), p0 + off_max(e) + 32 G + 8), where off_min / off_max are the epoch offsets of
// the unit's shortest / longest period (R11: llrint(e P/s) is monotone in P).  A producer warp copies those windows
// from global memory (L2) into a ring of shared-memory stages with TMA bulk copies (cp.async.bulk + mbarrier
// complete_tx): a stage holds the windows of a BLOCK of up to 8 consecutive epochs (as many as fit), one copy per
// epoch issued by one lane each, all completing on the stage's "full" barrier.  The 19 consumer warps wait on that
// barrier, fold their two periods out of the block's windows epoch by epoch with the same register-window step as the
// resident-row kernel (one 8-byte LDS feeds up to two adds), and release the stage through its "empty" barrier.  One
// L2 -> shared copy therefore serves 38 periods, the gathers run at shared-memory latency, and the barrier hand-shake,
// the descriptor read and the ring bookkeeping are paid once per block instead of once per epoch.  A window wider
// than a stage (long periods, or a period array that is not sorted) is not staged: the warps gather that epoch from
// global memory directly.
//
// Centring, as in fold_pair.cu: a lane's phases of the pair's longer period are taken m phases earlier (m = half the
// pair's largest offset difference, 0 when that exceeds kStrCentreMax and the pair would rarely share a window
// anyway), so that the two windows are s = off_1 - m - off_0 in [-m, m] apart and share one register window for
// |s| <= kStrS.
//
// The per-cell arithmetic, the epoch order of every sum, the FP64 offsets (R11) and the packed argmax key (R13) are
// those of fold_pair_argmax_kernel; only the order in which a cell's epochs are added differs (epoch order here).
#include "fold_common.cuh"

#include <math.h>

#include <algorithm>

namespace cetra {

namespace {

#ifndef CETRA_STR_S
#define CETRA_STR_S 5
#endif
#ifndef CETRA_STR_CENTRE_MAX
#define CETRA_STR_CENTRE_MAX 24
#endif
constexpr int kStrS = CETRA_STR_S;                       // |shift| up to which a pair's two windows share one register window
constexpr int kStrCentreMax = CETRA_STR_CENTRE_MAX;      // pairs whose centring shift would exceed this are not centred
#ifndef CETRA_STR_BLOCK
#define CETRA_STR_BLOCK 16
#endif
constexpr int kStrBlock = CETRA_STR_BLOCK;               // epochs per stage, at most
static_assert(kStrBlock >= 1 && kStrBlock <= 31, "one producer lane per epoch of a block; the run mask needs a zero bit");
static_assert(kStrS >= 1 && kStrS <= 7, "one switch case per shift");
static_assert(kStrCentreMax <= kPairMaxM, "centring_shift caps at kPairMaxM");
static_assert(kStatsPad >= 32 * (kGrpG + 2) + 2 * kStrS + 2 + kStrCentreMax, "cells past the last t0 cell are read as zeros");
static_assert(kStrHeaderBytes >= 8 * kStrCentreMax + 8 * kStrS,
              "up to m cells before a window clamped at the row start are read (and discarded)");

constexpr int kStrWarps = kStrThreads / 32 - 1;          // consumer warps; the last warp of the CTA is the producer
static_assert(kStrUnitPeriods == kStrWarps * kGrpT && kStrUnitPeriods % 2 == 0, "two periods per consumer warp");
static_assert(kStrUnitPeriods <= 64, "the producer warp holds a unit's periods two per lane");

enum : int {
    kFirstOfPass = 1,      // the block holds epoch 0 of a pass
    kLastOfPass = 2,       // combine + per-lane argmax (P3, P4) after this block
    kFirstOfUnit = 4,      // decode the unit, load and sort the warp's periods
    kLastOfUnit = 8,       // publish the warp's two keys after this block
    kExit = 16,
    kDirect = 32           // one epoch whose window is wider than a stage: gather it from global memory
};

// What the producer tells the consumers about a stage (32 bytes + one word per epoch).
struct StageDesc {
    int p0;                // first phase of the pass
    int e0;                // first epoch of the block
    int n_ep;              // epochs in the block
    int flags;
    int unit_lo, unit_hi;  // work unit (valid with kFirstOfUnit)
    int G;                 // phases per lane of this pass (valid with kFirstOfPass)
    int pad;
    int delta[kStrBlock];  // per epoch: (cell of the stage where its window starts) - (cell of the row where it starts)
};

// the pair's centring shift in this kernel (see the header)
__device__ __forceinline__ int stream_centring(double r0, double r1, int n_t0) {
    const int m = centring_shift(r0, r1, n_t0);
    return m <= kStrCentreMax ? m : 0;
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

struct StreamSmem {
    uint64_t full[kStrStages];
    uint64_t empty[kStrStages];
    StageDesc desc[kStrStages];
};
// per-warp epoch words behind the barriers and descriptors: (kStrBlock + 1) x 16 bytes each
constexpr int kStrWordsOffset = static_cast<int>((sizeof(StreamSmem) + 1023) / 1024 * 1024);
constexpr int kStrWordsPitch = (kStrBlock + 1) * 16 + 16;
static_assert(sizeof(StreamSmem) <= kStrWordsOffset, "header");
static_assert(kStrWordsOffset + (kStrThreads / 32 - 1) * kStrWordsPitch <= kStrHeaderBytes, "header");

// ------------------------------------------------------------------------------------------ consumer
struct WarpUnit {
    GroupPeriods gp;
    int kk[kGrpT];
    long long lc;
    const float2 *grow;    // the row in global memory (direct epochs)
    int j;
    int m;                 // centring: the lane's phases of period 1 are m earlier than those of period 0
    bool active;
    float best_lr[kGrpT];
    int best_p[kGrpT];
};

template <int G>
__device__ __forceinline__ int consume_pass(StreamSmem *sm, uint32_t ring_addr, uint32_t stage_bytes, int n_t0,
                                            WarpUnit &wu, StageDesc d, uint32_t &n_stage, int lane, uint32_t ew) {
    float2 acc[kGrpT][G];
#pragma unroll
    for (int t = 0; t < kGrpT; ++t)
#pragma unroll
        for (int g = 0; g < G; ++g) acc[t][g] = make_float2(0.f, 0.f);
    const int p0 = d.p0;
    const int limit = n_t0 - 1 - p0;                  // a window starting at offset o holds a cell <= I-1 iff o <= limit
    int flags;
    for (;;) {
        const uint32_t slot = (n_stage & (kStrStages - 1));
        flags = d.flags;
        if (wu.active) {
            const bool direct = (flags & kDirect) != 0;
            // P1, one epoch per lane: lane t derives the offsets of epoch e0 + t for the two periods (FP64, R11) and
            // leaves the epoch's word in the warp's slot: (x, y) = stage cells where the lane-0 windows of period 0 and
            // of period 1 start (row cells for a direct epoch), z = which of the two still reach a cell <= I - 1.
            // Period 1's phases are m earlier (centring), so its window starts at off_1 - m.
            {
                const double e = static_cast<double>(d.e0 + lane);
                // round-to-nearest-even conversion (= llrint for every in-range value), saturating
                const int o0 = min(__double2int_rn(__dmul_rn(e, wu.gp.r[0])), 0x3fffffff);
                const int o1 = min(__double2int_rn(__dmul_rn(e, wu.gp.r[1])), 0x3fffffff) - wu.m;
                if (lane < kStrBlock) {
                    const int delta = lane < d.n_ep && !direct ? sm->desc[slot].delta[lane] : 0;
                    sts_int4(ew + 16u * lane, delta + p0 + o0, delta + p0 + o1, (o0 <= limit ? 1 : 0) | (o1 <= limit ? 2 : 0), 0);
                }
                __syncwarp();
            }
            const uint32_t stage = ring_addr + slot * stage_bytes + 8u * static_cast<uint32_t>(lane * G);
            int4 w = lds_int4(ew);
            for (int t = 0; t < d.n_ep; ++t) {
                const int4 cur = w;
                w = lds_int4(ew + 16u * (t + 1));     // the next epoch's word, fetched while this epoch is folded
                if (!(cur.z & 3)) break;              // monotone in e: the later epochs of the block are out too
                const int sh = cur.y - cur.x;         // the two windows are sh in [-m, m] cells apart
                if (!direct) {
                    if (sh >= -kStrS && sh <= kStrS) {
                        const uint32_t ptr = stage + 8u * static_cast<uint32_t>(min(cur.x, cur.y));
                        switch (sh) {
#define CETRA_STR_CASE(SH) case (SH): fold_epoch_c<(SH), G>(acc, ptr); break;
#if CETRA_STR_S >= 7
                            CETRA_STR_CASE(-7) CETRA_STR_CASE(7)
#endif
#if CETRA_STR_S >= 6
                            CETRA_STR_CASE(-6) CETRA_STR_CASE(6)
#endif
#if CETRA_STR_S >= 5
                            CETRA_STR_CASE(-5) CETRA_STR_CASE(5)
#endif
#if CETRA_STR_S >= 4
                            CETRA_STR_CASE(-4) CETRA_STR_CASE(4)
#endif
#if CETRA_STR_S >= 3
                            CETRA_STR_CASE(-3) CETRA_STR_CASE(3)
#endif
#if CETRA_STR_S >= 2
                            CETRA_STR_CASE(-2) CETRA_STR_CASE(2)
#endif
                            CETRA_STR_CASE(-1) CETRA_STR_CASE(1)
                            default: fold_epoch_c<0, G>(acc, ptr); break;
#undef CETRA_STR_CASE
                        }
                    } else {
                        // windows too far apart to share: each period gathers its own cells
                        if (cur.z & 1) {
                            const uint32_t pu = stage + 8u * static_cast<uint32_t>(cur.x);
#pragma unroll
                            for (int g = 0; g < G; ++g) acc[0][g] = add2(acc[0][g], lds_cell(pu + 8u * g));
                        }
                        if (cur.z & 2) {
                            const uint32_t pu = stage + 8u * static_cast<uint32_t>(cur.y);
#pragma unroll
                            for (int g = 0; g < G; ++g) acc[1][g] = add2(acc[1][g], lds_cell(pu + 8u * g));
                        }
                    }
                } else {
                    if (cur.z & 1) {
                        const float2 *g0 = wu.grow + cur.x + lane * G;
#pragma unroll
                        for (int g = 0; g < G; ++g) acc[0][g] = add2(acc[0][g], __ldg(g0 + g));
                    }
                    if (cur.z & 2) {
                        const int c1 = cur.y + lane * G;               // before the row for the (discarded) phases < 0
#pragma unroll
                        for (int g = 0; g < G; ++g)
                            if (c1 + g >= 0) acc[1][g] = add2(acc[1][g], __ldg(wu.grow + c1 + g));
                    }
                }
            }
        }
        // release the stage: every lane's loads have been consumed by the adds above
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm->empty[slot]);
        ++n_stage;
        if (flags & kLastOfPass) break;
        const uint32_t nslot = (n_stage & (kStrStages - 1));
        mbar_wait(&sm->full[nslot], (n_stage >> kStrStagesLog2) & 1u);
        const int4 a = *reinterpret_cast<const int4 *>(&sm->desc[nslot]);
        d.p0 = a.x; d.e0 = a.y; d.n_ep = a.z; d.flags = a.w;
    }
    // P3 + P4 within the lane: phases ascending, strict > keeps the smallest phase on ties.  LR > best  <=>
    // SB^2 > 2 best SA: cells that cannot beat the best so far are dismissed with that product (with a margin, so
    // that none is dismissed wrongly); only when some cell of the lane passes does the lane take the divisions.
    if (wu.active) {
#pragma unroll
        for (int t = 0; t < kGrpT; ++t) {
            const float thr0 = 1.9999981f * wu.best_lr[t];
            bool any = false;
#pragma unroll
            for (int g = 0; g < G; ++g) {
                const float2 pr = mul2(acc[t][g], make_float2(thr0, acc[t][g].y));   // (2 best SA, SB^2)
                any |= pr.y >= pr.x;
            }
            if (any) {
#pragma unroll
                for (int g = 0; g < G; ++g) {
                    const int p = p0 + lane * G + g - (t ? wu.m : 0);
                    const float a = acc[t][g].x, bsum = acc[t][g].y;
                    const float lr = 0.5f * bsum * bsum * rcp_approx(a);
                    if (p >= 0 && p < wu.gp.n_phase[t] && a >= 1.17549435e-38f && lr > wu.best_lr[t]) {
                        wu.best_lr[t] = lr;
                        wu.best_p[t] = p;
                    }
                }
            }
        }
    }
    return flags;
}

__device__ __forceinline__ void begin_unit(const PeriodicParams &P, long long u, int warp, WarpUnit &wu) {
    const long long rowid = u / P.units_per_row;                   // lc * n_dur + j
    const int grp = static_cast<int>(u - rowid * P.units_per_row);
    wu.j = static_cast<int>(rowid % P.n_dur);
    wu.lc = rowid / P.n_dur;
    wu.grow = P.stats + rowid * P.stats_pitch;
    const double D = P.durations[wu.j];
    const int k0 = grp * kStrUnitPeriods + warp * kGrpT;
#pragma unroll
    for (int t = 0; t < kGrpT; ++t) {
        const int k = min(k0 + t, P.n_per - 1);                    // ragged last group: repeat the last period
        const double period = P.periods[k];
        bool on = k0 + t < P.n_per && D < period;                  // overlapping windows are invalid
        if (on && P.dur_lo && (wu.j < P.dur_lo[k] || wu.j >= P.dur_hi[k])) on = false;
        const double r = P.r_cells[k];                             // period in t0 cells: P_k / stride in FP64 (R11)
        const double rc = ceil(r);
        const int n_phase = rc < static_cast<double>(P.n_t0) ? static_cast<int>(rc) : P.n_t0;   // R10
        wu.gp.r[t] = r;
        wu.gp.n_phase[t] = on ? n_phase : 0;
        wu.kk[t] = k;
        // the period's best so far (rows already folded, by any CTA) only filters: a cell that ties it still passes
        // (bits - 1) and the packed key decides ties by cell id, so the records do not depend on the fold order
        const unsigned int hi = static_cast<unsigned int>(
            *reinterpret_cast<volatile unsigned long long *>(P.keys + wu.lc * P.n_per + k) >> 32);
        wu.best_lr[t] = hi ? __uint_as_float(hi - 1u) : -1.f;
        wu.best_p[t] = 0x7fffffff;
    }
    if (wu.gp.r[0] > wu.gp.r[1]) {                                 // sorted by ascending r
        const double tr = wu.gp.r[0]; wu.gp.r[0] = wu.gp.r[1]; wu.gp.r[1] = tr;
        const int tn = wu.gp.n_phase[0]; wu.gp.n_phase[0] = wu.gp.n_phase[1]; wu.gp.n_phase[1] = tn;
        const int tk = wu.kk[0]; wu.kk[0] = wu.kk[1]; wu.kk[1] = tk;
        const float tb = wu.best_lr[0]; wu.best_lr[0] = wu.best_lr[1]; wu.best_lr[1] = tb;
    }
    wu.active = wu.gp.n_phase[0] > 0 || wu.gp.n_phase[1] > 0;
    wu.m = wu.gp.n_phase[0] > 0 && wu.gp.n_phase[1] > 0 ? stream_centring(wu.gp.r[0], wu.gp.r[1], P.n_t0) : 0;
}

__device__ __forceinline__ void end_unit(const PeriodicParams &P, WarpUnit &wu, int lane) {
    if (!wu.active) return;
    // P4 across the warp: larger lr wins, ties -> smaller phase; one atomicMax per period (LR >= 0: its bit pattern
    // orders like an unsigned integer)
#pragma unroll
    for (int t = 0; t < kGrpT; ++t) {
        const bool has = wu.best_p[t] != 0x7fffffff;
        if (__any_sync(0xffffffffu, has)) {
            const unsigned int bits = has ? __float_as_uint(wu.best_lr[t]) : 0u;
            const unsigned int top = __reduce_max_sync(0xffffffffu, bits);
            const unsigned int p = __reduce_min_sync(
                0xffffffffu, has && bits == top ? static_cast<unsigned int>(wu.best_p[t]) : 0x7fffffffu);
            if (lane == 0) {
                const unsigned int id = static_cast<unsigned int>(wu.j) * static_cast<unsigned int>(P.n_t0) + p;
                const unsigned long long key = (static_cast<unsigned long long>(top) << 32) | (0xffffffffu - id);
                atomicMax(P.keys + wu.lc * P.n_per + wu.kk[t], key);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ producer
__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, s));
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, s));
    return v;
}

}  // namespace

__global__ void __launch_bounds__(kStrThreads, 1) fold_stream_argmax_kernel(const __grid_constant__ PeriodicParams P,
                                                                            int stage_cells) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    StreamSmem *sm = reinterpret_cast<StreamSmem *>(smem_raw);
    float2 *ring = reinterpret_cast<float2 *>(smem_raw + kStrHeaderBytes);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t stage_bytes = static_cast<uint32_t>(stage_cells) * 8u;

    if (P.literal && *P.literal) return;       // a caller's likelihood-ratio grid: fold_literal_argmax_kernel searches
    if (tid == 0) {
        for (int s = 0; s < kStrStages; ++s) {
            mbar_init(&sm->full[s], 1);
            mbar_init(&sm->empty[s], kStrWarps);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp == kStrWarps) {
        // ---------------- producer warp: claims units, derives every (pass, epoch) window, fills the ring.  Lane t
        // derives the window of epoch eb + t; consecutive epochs are packed into blocks of up to kStrBlock windows
        // that fit one stage, and every lane of a block issues the copy of its own window.
        uint32_t n_stage = 0;
        for (;;) {
            long long u = 0, u_end = 0;
            if (lane == 0) {
                const long long seen = *reinterpret_cast<volatile unsigned int *>(P.counter);   // only sizes the claim
                long long want = (P.n_units - seen) / (2LL * gridDim.x);
                want = want < 1 ? 1 : (want > P.max_claim ? P.max_claim : want);
                u = atomicAdd(P.counter, static_cast<unsigned int>(want));
                u_end = min(u + want, P.n_units);
            }
            u = __shfl_sync(0xffffffffu, u, 0);
            u_end = __shfl_sync(0xffffffffu, u_end, 0);
            if (u >= P.n_units) break;
            for (; u < u_end; ++u) {
                const long long rowid = u / P.units_per_row;
                const int grp = static_cast<int>(u - rowid * P.units_per_row);
                const int j = static_cast<int>(rowid % P.n_dur);
                const double D = P.durations[j];
                const float2 *grow = P.stats + rowid * P.stats_pitch;
                // the unit's searched periods, two per lane (a pair sits in neighbouring lanes): shortest / longest r,
                // the largest centring shift, and the phases the passes must cover (a pair's longer period is folded
                // m phases later in the pass: n_phase + m)
                double r_lo = 1e300, r_hi = 0.0;
                int nph = 0, m_unit = 0;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int t = lane + 32 * h;
                    const int k = grp * kStrUnitPeriods + t;
                    const bool have = t < kStrUnitPeriods && k < P.n_per;
                    double r = 0.0;
                    int n_phase = 0;
                    if (have) {
                        bool on = D < P.periods[k];
                        if (on && P.dur_lo && (j < P.dur_lo[k] || j >= P.dur_hi[k])) on = false;
                        r = P.r_cells[k];
                        const double rc = ceil(r);
                        n_phase = on ? (rc < static_cast<double>(P.n_t0) ? static_cast<int>(rc) : P.n_t0) : 0;
                    }
                    // the pair's other period (a ragged last pair repeats the last period, unsearched)
                    const double r_p = __shfl_xor_sync(0xffffffffu, r, 1);
                    const int n_phase_p = __shfl_xor_sync(0xffffffffu, n_phase, 1);
                    if (have && (n_phase > 0 || n_phase_p > 0)) {      // a searched period brings its partner along
                        r_lo = fmin(r_lo, r);
                        r_hi = fmax(r_hi, r);
                        int m = 0;
                        if (n_phase > 0 && n_phase_p > 0) m = stream_centring(fmin(r, r_p), fmax(r, r_p), P.n_t0);
                        // the period folded m phases later is the one sorted second: the larger r (equal r: m = 0)
                        if (n_phase > 0) nph = max(nph, n_phase + (r > r_p ? m : 0));
                        m_unit = max(m_unit, m);
                    }
                }
                r_lo = warp_min(r_lo);
                r_hi = warp_max(r_hi);
#pragma unroll
                for (int s = 16; s > 0; s >>= 1) {
                    nph = max(nph, __shfl_xor_sync(0xffffffffu, nph, s));
                    m_unit = max(m_unit, __shfl_xor_sync(0xffffffffu, m_unit, s));
                }
                if (nph == 0) continue;                             // no (period, duration) pair of this unit is searched
                bool first_of_unit = true;
                for (int p0 = 0; p0 < nph;) {
                    const int left = nph - p0;
                    // full passes of kGrpG phases per lane, then the narrowest odd width that covers what is left
                    int G = kGrpG;
                    if (left <= 32 * (kGrpG + 2)) G = ((left + 31) / 32) | 1;
                    const bool last_pass = left <= 32 * (kGrpG + 2);
                    const long long limit = static_cast<long long>(P.n_t0) - 1 - p0;
                    for (int eb = 0;; eb += 32) {
                        const double e = static_cast<double>(eb + lane);
                        const long long o_lo = __double2ll_rn(__dmul_rn(e, r_lo));
                        const long long o_hi = __double2ll_rn(__dmul_rn(e, r_hi));
                        const long long o_nx = __double2ll_rn(__dmul_rn(e + 1.0, r_lo));
                        // a pair's windows start at min(off_0, off_1 - m) >= off_lo - m_unit
                        const bool ok = o_lo - m_unit <= limit;
                        const int cnt = __popc(__ballot_sync(0xffffffffu, ok));   // offsets are monotone in e
                        // this lane's window [first, end) in the row, an even number of cells from an even cell on
                        const long long first = max(0LL, p0 + o_lo - m_unit) & ~1LL;
                        long long end = p0 + min(o_hi, limit + kStrS) + 32 * G + kStrS + 1;
                        end = min((end + 1) & ~1LL, P.stats_pitch);
                        const int cells = ok ? static_cast<int>(end - first) : 0;
                        int inc = cells;                                         // inclusive prefix sum over the lanes
#pragma unroll
                        for (int s = 1; s < 32; s <<= 1) {
                            const int v = __shfl_up_sync(0xffffffffu, inc, s);
                            if (lane >= s) inc += v;
                        }
                        const bool pass_ends = __shfl_sync(0xffffffffu, o_nx - m_unit > limit ? 1 : 0, cnt - 1) != 0;
                        for (int start = 0; start < cnt;) {
                            const int before = start ? __shfl_sync(0xffffffffu, inc, start - 1) : 0;
                            const bool fits = lane >= start && lane < start + kStrBlock && lane < cnt &&
                                              inc - before <= stage_cells;
                            const unsigned run = __ballot_sync(0xffffffffu, fits) >> start;
                            int n = __ffs(~run) - 1;                             // epochs of this block
                            const bool direct = n == 0;                          // even one window is wider than a stage
                            if (direct) n = 1;
                            const bool mine = lane >= start && lane < start + n;
                            const int total = __shfl_sync(0xffffffffu, inc, start + n - 1) - before;
                            const int my_off = inc - cells - before;             // cell of the stage where my window starts
                            const bool last_epoch = start + n == cnt && pass_ends;
                            const uint32_t slot = (n_stage & (kStrStages - 1));
                            if (lane == 0) mbar_wait(&sm->empty[slot], ((n_stage >> kStrStagesLog2) & 1u) ^ 1u);
                            __syncwarp();
                            StageDesc *dsc = &sm->desc[slot];
                            if (lane == 0) {
                                dsc->p0 = p0;
                                dsc->e0 = eb + start;
                                dsc->n_ep = n;
                                dsc->flags = (eb + start == 0 ? kFirstOfPass : 0) | (last_epoch ? kLastOfPass : 0) |
                                             (first_of_unit ? kFirstOfUnit : 0) |
                                             (last_epoch && last_pass ? kLastOfUnit : 0) | (direct ? kDirect : 0);
                                dsc->unit_lo = static_cast<int>(u & 0xffffffffLL);
                                dsc->unit_hi = static_cast<int>(u >> 32);
                                dsc->G = G;
                                dsc->pad = 0;
                            }
                            if (mine) dsc->delta[lane - start] = my_off - static_cast<int>(first);
                            __syncwarp();
                            if (!direct) {
                                if (lane == 0) mbar_arrive_expect_tx(&sm->full[slot], static_cast<uint32_t>(total) * 8u);
                                __syncwarp();
                                if (mine) {
                                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the stage was read by generic loads
                                    bulk_copy_g2s_chunked(reinterpret_cast<unsigned char *>(ring) + slot * stage_bytes +
                                                              static_cast<uint32_t>(my_off) * 8u,
                                                          grow + first, static_cast<uint32_t>(cells) * 8u, &sm->full[slot]);
                                }
                            } else if (lane == 0) {
                                mbar_arrive(&sm->full[slot]);
                            }
                            ++n_stage;
                            first_of_unit = false;
                            start += n;
                        }
                        if (cnt < 32) break;
                    }
                    p0 += 32 * G;
                }
            }
        }
        if (lane == 0) {
            const uint32_t slot = (n_stage & (kStrStages - 1));
            mbar_wait(&sm->empty[slot], ((n_stage >> kStrStagesLog2) & 1u) ^ 1u);
            sm->desc[slot].n_ep = 0;
            sm->desc[slot].flags = kExit;
            mbar_arrive(&sm->full[slot]);
        }
        return;
    }

    // ---------------- consumer warps
    const uint32_t ring_addr = smem_u32(ring);
    const uint32_t ew = smem_u32(smem_raw + kStrWordsOffset + warp * kStrWordsPitch);   // this warp's epoch words
    WarpUnit wu;
    wu.active = false;
    uint32_t n_stage = 0;
    for (;;) {
        const uint32_t slot = (n_stage & (kStrStages - 1));
        mbar_wait(&sm->full[slot], (n_stage >> kStrStagesLog2) & 1u);
        const int4 a = *reinterpret_cast<const int4 *>(&sm->desc[slot]);
        const int4 b = *(reinterpret_cast<const int4 *>(&sm->desc[slot]) + 1);
        StageDesc d;
        d.p0 = a.x; d.e0 = a.y; d.n_ep = a.z; d.flags = a.w;
        d.unit_lo = b.x; d.unit_hi = b.y; d.G = b.z; d.pad = 0;
        if (d.flags & kExit) break;
        if (d.flags & kFirstOfUnit) {
            const long long u = (static_cast<long long>(d.unit_hi) << 32) | static_cast<unsigned int>(d.unit_lo);
            begin_unit(P, u, warp, wu);
        }
        int flags;
        switch (d.G) {
            case 1: flags = consume_pass<1>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane, ew); break;
            case 3: flags = consume_pass<3>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane, ew); break;
            case 5: flags = consume_pass<5>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane, ew); break;
            case 7: flags = consume_pass<7>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane, ew); break;
            case 9: flags = consume_pass<9>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane, ew); break;
            case 11: flags = consume_pass<11>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane, ew); break;
            default: flags = consume_pass<13>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane, ew); break;
        }
        if (flags & kLastOfUnit) end_unit(P, wu, lane);
    }
}

int launch_fold_stream(const PeriodicPlan &pl, cudaStream_t st) {
    auto k = fold_stream_argmax_kernel;
    CETRA_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_bytes));
    k<<<pl.grid, kStrThreads, pl.smem_bytes, st>>>(pl.P, pl.stage_cells);
    return CETRA_OK;
}

}  // namespace cetra
