// Periodic search for rows that do not fit in shared memory (§2.3, steps P1-P4 of DESIGN.md): config 4
// (256 464 cells, 2 MB per row) and every TESS sector on the paper's default t0 grid (PAPER.md:87, 1 MB per row).
//
// The row does not fit, but what one work unit touches at one epoch does.  A unit is one duration row and
// kStrUnitPeriods = 38 neighbouring trial periods (two per warp, as in fold_pair_argmax_kernel).  All warps of the
// CTA walk the unit's phase passes and epochs together: at pass p0 (32 G phases) and epoch e the 38 periods read the
// contiguous cells [p0 + off_min(e), p0 + off_max(e) + 32 G + 8), where off_min / off_max are the epoch offsets of
// the unit's shortest / longest period (R11: llrint(e P/s) is monotone in P).  A producer warp copies that window
// from global memory (L2) into a ring of shared-memory stages with one TMA bulk copy (cp.async.bulk + mbarrier
// complete_tx) per epoch; the 19 consumer warps wait on the stage's "full" barrier, fold their two periods out of
// it with the same register-window epoch step as the resident-row kernel (one 8-byte LDS feeds up to two adds), and
// release the stage through its "empty" barrier.  One L2 -> shared copy therefore serves 38 periods, and the gathers
// run at shared-memory rather than L1/L2 latency.  A window wider than a stage (long periods, or a period array that
// is not sorted) is not staged: the warps gather that epoch from global memory directly.
//
// The per-cell arithmetic, the epoch order of every sum, the FP64 offsets (R11) and the packed argmax key (R13) are
// those of fold_pair_argmax_kernel; only the order in which a cell's epochs are added differs (epoch order here).
#include "fold_common.cuh"

#include <math.h>

#include <algorithm>

namespace cetra {

namespace {

constexpr int kStrWarps = kStrThreads / 32 - 1;          // consumer warps; the last warp of the CTA is the producer
static_assert(kStrUnitPeriods == kStrWarps * kGrpT && kStrUnitPeriods % 2 == 0, "two periods per consumer warp");
static_assert(kStrUnitPeriods <= 64, "the producer warp holds a unit's periods two per lane");

enum : int {
    kFirstOfPass = 1,      // reset the accumulators
    kLastOfPass = 2,       // combine + per-lane argmax (P3, P4) after this epoch
    kFirstOfUnit = 4,      // decode the unit, load and sort the warp's periods
    kLastOfUnit = 8,       // publish the warp's two keys after this epoch
    kExit = 16,
    kDirect = 32           // window wider than a stage: gather this epoch from global memory
};

// What the producer tells the consumers about a stage (32 bytes, read with two 16-byte shared loads).
struct StageDesc {
    int origin;            // cell index (within the row) of element 0 of the stage
    int p0;                // first phase of the pass
    int e;                 // epoch
    int flags;
    int unit_lo, unit_hi;  // work unit (valid with kFirstOfUnit)
    int G;                 // phases per lane of this pass (valid with kFirstOfPass)
    int pad;
};

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

struct StreamSmem {
    uint64_t full[kStrStages];
    uint64_t empty[kStrStages];
    StageDesc desc[kStrStages];
};
static_assert(sizeof(StreamSmem) <= kStrHeaderBytes, "header");

// ------------------------------------------------------------------------------------------ consumer
struct WarpUnit {
    GroupPeriods gp;
    int kk[kGrpT];
    long long lc;
    const float2 *grow;    // the row in global memory (direct epochs)
    int j;
    bool active;
    float best_lr[kGrpT];
    int best_p[kGrpT];
};

template <int G>
__device__ __forceinline__ int consume_pass(StreamSmem *sm, uint32_t ring_addr, uint32_t stage_bytes, int n_t0,
                                            WarpUnit &wu, StageDesc d, uint32_t &n_stage, int lane) {
    float2 acc[kGrpT][G];
#pragma unroll
    for (int t = 0; t < kGrpT; ++t)
#pragma unroll
        for (int g = 0; g < G; ++g) acc[t][g] = make_float2(0.f, 0.f);
    const int p0 = d.p0;
    const int limit = n_t0 - 1 - p0;                  // off_e <= limit  <=>  p0 + off_e <= I-1
    int flags;
    for (;;) {
        const uint32_t slot = (n_stage & (kStrStages - 1));
        flags = d.flags;
        if (wu.active) {
            // P1: the epoch's offsets of the two periods (FP64, R11); warp-uniform
            const double e = static_cast<double>(d.e);
            // round-to-nearest-even conversion (= llrint for every in-range value), saturating
            const int o0 = __double2int_rn(__dmul_rn(e, wu.gp.r[0]));
            const int o1 = __double2int_rn(__dmul_rn(e, wu.gp.r[1]));
            if (o0 <= limit) {
                if (!(flags & kDirect)) {
                    const uint32_t ptr = ring_addr + slot * stage_bytes +
                                         8u * static_cast<uint32_t>(p0 + o0 - d.origin + lane * G);
                    const int dd = o1 - o0;
                    switch (dd < 8 ? dd : 8) {
                        case 0: fold_epoch<0, G>(acc, ptr); break;
                        case 1: fold_epoch<1, G>(acc, ptr); break;
                        case 2: fold_epoch<2, G>(acc, ptr); break;
                        case 3: fold_epoch<3, G>(acc, ptr); break;
                        case 4: fold_epoch<4, G>(acc, ptr); break;
                        case 5: fold_epoch<5, G>(acc, ptr); break;
                        case 6: fold_epoch<6, G>(acc, ptr); break;
                        case 7: fold_epoch<7, G>(acc, ptr); break;
                        default: {
#pragma unroll
                            for (int g = 0; g < G; ++g) acc[0][g] = add2(acc[0][g], lds_cell(ptr + 8u * g));
                            if (o1 <= limit) {
                                const uint32_t pu = ptr + 8u * static_cast<uint32_t>(dd);
#pragma unroll
                                for (int g = 0; g < G; ++g) acc[1][g] = add2(acc[1][g], lds_cell(pu + 8u * g));
                            }
                        }
                    }
                } else {
                    const float2 *g0 = wu.grow + p0 + o0 + lane * G;
#pragma unroll
                    for (int g = 0; g < G; ++g) acc[0][g] = add2(acc[0][g], __ldg(g0 + g));
                    if (o1 <= limit) {
                        const float2 *g1 = wu.grow + p0 + o1 + lane * G;
#pragma unroll
                        for (int g = 0; g < G; ++g) acc[1][g] = add2(acc[1][g], __ldg(g1 + g));
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
        d.origin = a.x; d.p0 = a.y; d.e = a.z; d.flags = a.w;
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
                    const int p = p0 + lane * G + g;
                    const float a = acc[t][g].x, bsum = acc[t][g].y;
                    const float lr = 0.5f * bsum * bsum * rcp_approx(a);
                    if (p < wu.gp.n_phase[t] && a >= 1.17549435e-38f && lr > wu.best_lr[t]) {
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
        // ---------------- producer warp: claims units, derives every (pass, epoch) window, fills the ring
        uint32_t n_stage = 0;
        auto push = [&](const StageDesc &d, const float2 *src, uint32_t cells) {    // lane 0 only
            const uint32_t slot = (n_stage & (kStrStages - 1));
            mbar_wait(&sm->empty[slot], ((n_stage >> kStrStagesLog2) & 1u) ^ 1u);
            sm->desc[slot] = d;
            if (cells) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the stage was read by generic loads
                mbar_arrive_expect_tx(&sm->full[slot], cells * 8u);
                bulk_copy_g2s_chunked(reinterpret_cast<unsigned char *>(ring) + slot * stage_bytes, src, cells * 8u,
                                      &sm->full[slot]);
            } else {
                mbar_arrive(&sm->full[slot]);
            }
        };
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
                // the unit's searched periods, two per lane: shortest / longest r and the largest phase count
                double r_lo = 1e300, r_hi = 0.0;
                int nph = 0;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int t = lane + 32 * h;
                    const int k = grp * kStrUnitPeriods + t;
                    if (t < kStrUnitPeriods && k < P.n_per) {
                        const double period = P.periods[k];
                        bool on = D < period;
                        if (on && P.dur_lo && (j < P.dur_lo[k] || j >= P.dur_hi[k])) on = false;
                        // a warp folds its two periods together: a searched period brings its partner along
                        const int kp = min(k ^ 1, P.n_per - 1);
                        const double pp = P.periods[kp];
                        bool pon = D < pp;
                        if (pon && P.dur_lo && (j < P.dur_lo[kp] || j >= P.dur_hi[kp])) pon = false;
                        if (on || pon) {
                            const double r = P.r_cells[k];
                            r_lo = fmin(r_lo, r);
                            r_hi = fmax(r_hi, r);
                            if (on) {
                                const double rc = ceil(r);
                                nph = max(nph, rc < static_cast<double>(P.n_t0) ? static_cast<int>(rc) : P.n_t0);
                            }
                        }
                    }
                }
                r_lo = warp_min(r_lo);
                r_hi = warp_max(r_hi);
#pragma unroll
                for (int s = 16; s > 0; s >>= 1) nph = max(nph, __shfl_xor_sync(0xffffffffu, nph, s));
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
                        const bool ok = o_lo <= limit;
                        const int cnt = __popc(__ballot_sync(0xffffffffu, ok));   // offsets are monotone in e
                        for (int t = 0; t < cnt; ++t) {
                            const long long a_lo = __shfl_sync(0xffffffffu, o_lo, t);
                            const long long a_hi = __shfl_sync(0xffffffffu, o_hi, t);
                            const long long a_nx = __shfl_sync(0xffffffffu, o_nx, t);
                            if (lane == 0) {
                                StageDesc d;
                                const bool last_epoch = a_nx > limit;
                                const long long first = (p0 + a_lo) & ~1LL;
                                long long end = p0 + min(a_hi, limit) + 32 * G + kGrpS + 1;
                                end = min((end + 1) & ~1LL, P.stats_pitch);
                                const long long cells = end - first;
                                d.origin = static_cast<int>(first);
                                d.p0 = p0;
                                d.e = eb + t;
                                d.flags = (eb + t == 0 ? kFirstOfPass : 0) | (last_epoch ? kLastOfPass : 0) |
                                          (first_of_unit ? kFirstOfUnit : 0) |
                                          (last_epoch && last_pass ? kLastOfUnit : 0) |
                                          (cells > stage_cells ? kDirect : 0);
                                d.unit_lo = static_cast<int>(u & 0xffffffffLL);
                                d.unit_hi = static_cast<int>(u >> 32);
                                d.G = G;
                                d.pad = 0;
                                push(d, grow + first, cells > stage_cells ? 0u : static_cast<uint32_t>(cells));
                            }
                            ++n_stage;
                            first_of_unit = false;
                        }
                        if (cnt < 32) break;
                    }
                    p0 += 32 * G;
                }
            }
        }
        if (lane == 0) {
            StageDesc d{};
            d.flags = kExit;
            push(d, nullptr, 0u);
        }
        return;
    }

    // ---------------- consumer warps
    const uint32_t ring_addr = smem_u32(ring);
    WarpUnit wu;
    wu.active = false;
    uint32_t n_stage = 0;
    for (;;) {
        const uint32_t slot = (n_stage & (kStrStages - 1));
        mbar_wait(&sm->full[slot], (n_stage >> kStrStagesLog2) & 1u);
        const int4 a = *reinterpret_cast<const int4 *>(&sm->desc[slot]);
        const int4 b = *(reinterpret_cast<const int4 *>(&sm->desc[slot]) + 1);
        StageDesc d;
        d.origin = a.x; d.p0 = a.y; d.e = a.z; d.flags = a.w;
        d.unit_lo = b.x; d.unit_hi = b.y; d.G = b.z; d.pad = 0;
        if (d.flags & kExit) break;
        if (d.flags & kFirstOfUnit) {
            const long long u = (static_cast<long long>(d.unit_hi) << 32) | static_cast<unsigned int>(d.unit_lo);
            begin_unit(P, u, warp, wu);
        }
        int flags;
        switch (d.G) {
            case 1: flags = consume_pass<1>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane); break;
            case 3: flags = consume_pass<3>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane); break;
            case 5: flags = consume_pass<5>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane); break;
            case 7: flags = consume_pass<7>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane); break;
            case 9: flags = consume_pass<9>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane); break;
            case 11: flags = consume_pass<11>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane); break;
            default: flags = consume_pass<13>(sm, ring_addr, stage_bytes, P.n_t0, wu, d, n_stage, lane); break;
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
