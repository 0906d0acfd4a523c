// Linear search (§2.2, lines 89-125): steps L0-L3 of DESIGN.md.
//
//   L0 preprocess_kernel   flux, flux_err -> (w f, w) float2, zero outside the data
//   L1 build_taps_kernel   per duration: nearest-neighbour template samples m, m^2     (R3)
//   L2 linear_search_kernel  S_wmf = sum m (w f), S_wmm = sum m^2 w for every (t_i, D_j)
//   L3 (fused epilogue)    depth = S_wmf/S_wmm, var = 1/S_wmm, dlogL = 1/2 S_wmf^2/S_wmm (Eq. 2)
//
// The windowed sums are a correlation of the sample stream with 2H_j+1 taps.  For a t0 stride of q
// samples both the taps and the samples are split into q polyphase streams (the preprocess kernel
// writes sample n_lo + q u + v to stream v, position u), so that every branch is a unit-stride
// correlation in which R consecutive outputs of one thread slide over a register window: one 8-byte
// shared-memory load feeds 2R FFMAs, and a CTA stages one (tile + taps)-long slice per branch.
#include "linear_search.cuh"

#include <math.h>

#include <algorithm>
#include <vector>

namespace cetra {

// ------------------------------------------------------------------------------------------- L0
template <typename T>
__global__ void preprocess_kernel(const T *__restrict__ flux, const T *__restrict__ flux_err, long long n,
                                  long long n_lc, float2 *__restrict__ wfw, long long ph_pitch, long long q,
                                  long long n_lo) {
    // output element (lc, v, u) holds sample n_lo + q u + v: q = 1 is the plain padded sample row
    const long long row_len = q * ph_pitch;
    const long long total = n_lc * row_len;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long lc = idx / row_len;
        const long long e = idx - lc * row_len;
        const long long v = e / ph_pitch, u = e - v * ph_pitch;
        const long long nn = n_lo + q * u + v;
        float2 out = make_float2(0.f, 0.f);
        if (nn >= 0 && nn < n) {
            const T fl = flux[lc * n + nn];
            const T er = flux_err[lc * n + nn];
            if (isfinite(fl) && isfinite(er) && er > T(0)) {      // null points carry no weight
                const T f = T(1) - fl;                            // offset from baseline, dips positive
                const T w = T(1) / (er * er);
                const float wf32 = static_cast<float>(w * f);
                const float w32 = static_cast<float>(w);
                if (isfinite(wf32) && isfinite(w32)) out = make_float2(wf32, w32);
            }
        }
        wfw[idx] = out;
    }
}

// ------------------------------------------------------------------------------------------- L1
// One thread per stored tap.  Layout per duration j: [q phases][A_j taps] float2 (m, m^2), tap (b, a) is the
// sample offset k = q*a + b - H_j from the window centre; zero beyond the window.  Every FP64 step is an
// explicitly rounded IEEE operation so that the index agrees bit for bit with a plain CPU evaluation (R3).
__global__ void build_taps_kernel(const __grid_constant__ LinearParams P, const float *__restrict__ tpl,
                                  int n_tpl, double cadence, float2 *__restrict__ taps) {
    const int j = blockIdx.y;
    tpl += static_cast<long long>(blockIdx.z) * n_tpl;          // z: template of the set
    taps += blockIdx.z * P.tset_taps;
    const int A = P.A[j], H = P.H[j], q = P.q;
    const int stored = P.tap_off[j + 1] - P.tap_off[j];
    const double D = P.durations[j];
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < stored; idx += gridDim.x * blockDim.x) {
        float m = 0.f;
        if (idx < q * A) {
            const int b = idx / A, a = idx - b * A;
            const int kk = q * a + b;
            if (kk <= 2 * H) {
                const double k = static_cast<double>(kk - H);
                const double x = __dadd_rn(__ddiv_rn(__dmul_rn(k, cadence), D), 0.5);
                if (x >= 0.0 && x <= 1.0) {
                    const double pos = __dadd_rn(__dmul_rn(x, static_cast<double>(n_tpl - 1)), 0.5);
                    m = tpl[static_cast<int>(floor(pos))];
                }
            }
        }
        taps[P.tap_off[j] + idx] = make_float2(m, m * m);
    }
}

// Exact (R25) evaluations done by the fast off-grid paths since the last reset: cetra_exact_eval_count.
__device__ unsigned long long g_exact_evals;

int exact_eval_count(int64_t *count, bool reset) {
    unsigned long long v = 0;
    CETRA_CUDA_TRY(cudaMemcpyFromSymbol(&v, g_exact_evals, sizeof(v)));
    if (count) *count = static_cast<int64_t>(v);
    if (reset) {
        v = 0;
        CETRA_CUDA_TRY(cudaMemcpyToSymbol(g_exact_evals, &v, sizeof(v)));
    }
    return CETRA_OK;
}

// R25, one (sample, cell) pair exactly as the definition reads: every FP64 step one rounded IEEE operation.
// Returns the template index, or -1 when the sample lies outside the window 0 <= x <= 1 (R2).
__device__ __forceinline__ int r25_index(long long n, double ti, double c, double D, double Mm1) {
    const double x = __dadd_rn(__ddiv_rn(__dsub_rn(__dmul_rn(static_cast<double>(n), c), ti), D), 0.5);
    if (!(x >= 0.0 && x <= 1.0)) return -1;
    return static_cast<int>(floor(__dadd_rn(__dmul_rn(x, Mm1), 0.5)));
}

// L1 for the residue classes of a rational off-grid stride.  Tap (b, a) of class rho is the sample k = q a + b - H_j
// samples after the class's anchor sample; the cell sits f_rho samples after the anchor, so the tap's position in
// the template is pos = ((k - f_rho) c / D + 1/2)(M - 1) + 1/2 for EVERY cell of the class, up to (i) the rounding
// of the definition's own FP64 sequence (R25), which depends on the cell, and (ii) the drift of the stride from
// p / cls.  Both are bounded by eps = eps_scale / D + eps_abs (see build_linear_plan).  A tap whose position is
// further than eps from every decision point (an integer, where floor() steps, or a window edge) gets the same
// template sample for every cell and goes into the table; the others are withheld (table entry 0, flag set) and
// linear_search_kernel evaluates them per cell with r25_index.
__global__ void build_class_taps_kernel(const __grid_constant__ LinearParams P, const double *__restrict__ cls_f,
                                        double eps_scale, double eps_abs, float2 *__restrict__ taps,
                                        unsigned char *__restrict__ flags) {
    const int j = blockIdx.y, tset = blockIdx.z / P.n_cls, rho = blockIdx.z - tset * P.n_cls;
    const float *tpl = P.tpl + static_cast<long long>(tset) * P.n_tpl;
    taps += tset * P.tset_taps;                                 // the flags depend on the geometry only: every template
    const int A = P.A[j], H = P.H[j], q = P.q;                   // of the set writes the same ones
    const int stored = P.tap_off[j + 1] - P.tap_off[j];
    const double D = P.durations[j], Mm1 = static_cast<double>(P.n_tpl - 1);
    const double eps = eps_scale / D + eps_abs;
    const double f = cls_f[rho];
    const long long base = static_cast<long long>(P.n_cls) * P.tap_off[j] + static_cast<long long>(rho) * stored;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < stored; idx += gridDim.x * blockDim.x) {
        float m = 0.f;
        unsigned char flag = 0;
        if (idx < q * A) {
            const int b = idx / A, a = idx - b * A;
            const int kk = q * a + b;
            if (kk <= 2 * H) {
                const double u = static_cast<double>(kk - H) - f;
                const double pos = (u * P.cadence / D + 0.5) * Mm1 + 0.5;
                const bool near_step = fabs(pos - rint(pos)) < eps;
                const bool near_edge = fabs(pos - 0.5) < eps || fabs(pos - (Mm1 + 0.5)) < eps;
                if (near_step || near_edge) {
                    flag = (pos > 0.5 - 2.0 * eps && pos < Mm1 + 0.5 + 2.0 * eps) ? 1 : 0;   // far outside: plainly 0
                } else if (pos > 0.5 && pos < Mm1 + 0.5) {
                    m = tpl[static_cast<int>(floor(pos))];
                }
            }
        }
        taps[base + idx] = make_float2(m, m * m);
        flags[base + idx] = flag;
    }
}

// One thread per (duration, class): the withheld taps of its table, as sample offsets k in table order.
__global__ void collect_withheld_taps_kernel(const __grid_constant__ LinearParams P,
                                             const unsigned char *__restrict__ flags, int *__restrict__ cnt,
                                             int *__restrict__ list) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= P.n_dur * P.n_cls) return;
    const int j = t / P.n_cls, rho = t - j * P.n_cls;
    const int A = P.A[j], H = P.H[j], q = P.q;
    const int stored = P.tap_off[j + 1] - P.tap_off[j];
    const long long base = static_cast<long long>(P.n_cls) * P.tap_off[j] + static_cast<long long>(rho) * stored;
    int n = 0;
    for (int idx = 0; idx < q * A; ++idx) {
        if (flags[base + idx]) {
            const int b = idx / A, a = idx - b * A;
            list[base + n++] = q * a + b - H;
        }
    }
    cnt[t] = n;
}

// ------------------------------------------------------------------------------------------- L2 + L3
// Packed FP32 (FFMA2 / FADD2 on sm_100a): both sufficient statistics of a cell in one issue slot.  The two
// halves are independent IEEE fp32 operations with round-to-nearest, exactly fmaf / + on each component.
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
    float2 r;
    asm("{\n\t"
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

__device__ __forceinline__ float2 add2f(float2 a, float2 b) {
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

// CLS: the cells are split into residue classes (rational off-grid stride); false on the sample grid, where the
// class decode and the exact fix-up are compiled out.
template <int R, int WARPS, bool CLS>
__global__ void __launch_bounds__(WARPS * 32)
linear_search_kernel(const __grid_constant__ LinearParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int TILE = WARPS * 32 * R;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // grid = (tiles of a row, durations, light curves): consecutive blocks share a duration's tap table
    const long long lc = blockIdx.z;
    int yy = blockIdx.y, tset = 0;                              // y = template * n_dur + duration rank
    if (P.n_tset > 1) {
        tset = yy / P.n_dur;
        yy -= tset * P.n_dur;
    }
    const int j = P.order[yy];                                  // longest durations first
    int tile = blockIdx.x, rho = 0;                             // x = tile * n_cls + class: a tile's classes run together
    const int n_cls = CLS ? P.n_cls : 1;
    if (CLS) {
        tile = blockIdx.x / static_cast<unsigned int>(n_cls);
        rho = blockIdx.x - tile * n_cls;
    }
    // cells of this class: i = n_cls a + rho < n_t0
    const long long n_cells = CLS ? (P.n_t0 - rho + n_cls - 1) / n_cls : P.n_t0;
    const int q = P.q;
    const int A = P.A[j];
    const long long i_blk = static_cast<long long>(tile) * TILE;
    const int n_tap = P.tap_off[j + 1] - P.tap_off[j];
    const int slice = (TILE + A + 2) & ~1;                       // samples of one branch (+ alignment slack)

    // element of the first tap of output 0 in the padded sample numbering; branch b starts b samples later
    const long long n0c = CLS ? static_cast<long long>(P.cls_n0[rho]) : P.n0;   // sample under (nearest to) cell 0
    const unsigned int e0 = static_cast<unsigned int>(n0c - P.H[j] - P.n_lo);   // <= h_max + q + 4, far below 2^31
    const unsigned int uq = static_cast<unsigned int>(q);

    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);      // bar[0], bar[1]: one per sample stage
    float2 *taps = reinterpret_cast<float2 *>(smem_raw + 32);
    float2 *stage0 = taps + n_tap;                               // two sample stages of `slice` elements

    // branch b reads stream v = (e0 + b) mod q from position (e0 + b) div q + i_blk on
    auto issue = [&](int b, bool with_taps) {
        const unsigned int e = e0 + static_cast<unsigned int>(b);
        const unsigned int eu = q == 1 ? e : e / uq;
        const long long v = e - eu * uq, u0 = eu + i_blk;
        const int d0 = static_cast<int>(u0 & 1);                 // bulk copies need 16-byte alignment
        const uint32_t bytes = static_cast<uint32_t>(slice) * 8u;
        const uint32_t bytes_taps = with_taps ? static_cast<uint32_t>(n_tap) * 8u : 0u;
        uint64_t *bb = bar + (b & 1);
        if (b > 1) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the stage was read by generic loads
        mbar_arrive_expect_tx(bb, bytes + bytes_taps);
        bulk_copy_g2s_chunked(stage0 + (b & 1) * slice, P.wfw + (lc * q + v) * P.ph_pitch + (u0 - d0), bytes, bb);
        if (with_taps)
            bulk_copy_g2s_chunked(taps, P.taps + tset * P.tset_taps + static_cast<long long>(n_cls) * P.tap_off[j] +
                                            static_cast<long long>(rho) * n_tap, bytes_taps, bb);
    };

    if (tid == 0) {
        mbar_init(bar, 1);
        if (q > 1) mbar_init(bar + 1, 1);
        mbar_fence_init();
        issue(0, true);
    }
    __syncthreads();
    if (P.stats && tile == P.tiles_per_row - 1 && rho == 0) {   // zero the row padding (while the fill is in flight)
        const long long prow = (static_cast<long long>(tset) * gridDim.z + lc) * P.n_dur + j;
        for (long long i = P.n_t0 + tid; i < P.stats_pitch; i += WARPS * 32)
            P.stats[prow * P.stats_pitch + i] = make_float2(0.f, 0.f);
    }
    // a warp whose 32*R cells all lie past the last t0 cell has nothing to compute (last tile of a row); with
    // several polyphase branches every warp stays for the block-wide barriers between the branches
    if (q == 1 && i_blk + static_cast<long long>(warp) * (32 * R) >= n_cells) return;

    // Two-level summation: the running FFMA accumulators are folded into a second set every kFlush tap
    // groups (and at the end of every polyphase branch), so that no FP32 sum runs over more than
    // kFlush*R terms before it is added to terms of its own size (cfg 3 has
    // windows of 2 701 points).
    constexpr int kFlush = 4;
    float2 acc[R], tot[R];                                     // (S_wmf, S_wmm) of R consecutive t0 cells
#pragma unroll
    for (int r = 0; r < R; ++r) { acc[r] = make_float2(0.f, 0.f); tot[r] = make_float2(0.f, 0.f); }

    for (int b = 0; b < q; ++b) {
        if (tid == 0 && b + 1 < q) issue(b + 1, false);          // its stage was released at the end of branch b-1
        mbar_wait(bar + (b & 1), static_cast<uint32_t>((b >> 1) & 1));
        const unsigned int eb = e0 + static_cast<unsigned int>(b);
        const int d0 = static_cast<int>(((q == 1 ? eb : eb / uq) + i_blk) & 1);
        const float2 *xb = stage0 + (b & 1) * slice + d0 + tid * R;
        const float2 *tb = taps + b * A;
        float2 win[R];
#pragma unroll
        for (int v = 0; v < R - 1; ++v) win[v] = xb[v];
        float2 nxt = xb[R - 1];
        float2 tap = tb[0];
        const float2 *xp = xb + R;
        int since_flush = 0;
        for (int a0 = 0; a0 < A; a0 += R) {
#pragma unroll
            for (int u = 0; u < R; ++u) {
                win[(u + R - 1) % R] = nxt;
                const float2 t = tap;
                nxt = xp[u];                                     // prefetch the next window element
                tap = tb[a0 + u + 1];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    // S_wmf += m * (w f),  S_wmm += m^2 * w
                    acc[r] = fma2(t, win[(u + r) % R], acc[r]);
                }
            }
            xp += R;
            if (++since_flush == kFlush || a0 + R >= A) {
                since_flush = 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    tot[r] = add2f(tot[r], acc[r]);
                    acc[r] = make_float2(0.f, 0.f);
                }
            }
        }
        if (q > 1) __syncthreads();                              // every warp is done with this stage
    }
    // The taps the class table withholds (positions within rounding of a decision point): evaluated per cell with
    // the definition's own FP64 sequence.  Rare: a handful of taps in some classes, none in most.
    if (CLS) {
        const int cnt = P.unsafe_cnt[j * n_cls + rho];
        if (cnt > 0) {
            const int *lst = P.unsafe_k + static_cast<long long>(n_cls) * P.tap_off[j] + static_cast<long long>(rho) * n_tap;
            const double D = P.durations[j], Mm1 = static_cast<double>(P.n_tpl - 1);
            unsigned int done = 0;
            for (int t = 0; t < cnt; ++t) {
                const int k = lst[t];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const long long a = i_blk + tid * R + r;
                    const long long nn = n0c + a * q + k;
                    if (a < n_cells && nn >= 0 && nn < P.n) {
                        const long long i = a * n_cls + rho;
                        const double ti = __dadd_rn(P.delta, __dmul_rn(static_cast<double>(i), P.stride));
                        const int idx = r25_index(nn, ti, P.cadence, D, Mm1);
                        ++done;
                        if (idx >= 0) {
                            const float m = __ldg(P.tpl + static_cast<long long>(tset) * P.n_tpl + idx);
                            const long long e = nn - P.n_lo;
                            const long long u = e / q, v = e - u * q;
                            const float2 sm = __ldg(P.wfw + (lc * q + v) * P.ph_pitch + u);
                            tot[r].x = fmaf(m, sm.x, tot[r].x);          // S_wmf += m * (w f)
                            tot[r].y = fmaf(m * m, sm.y, tot[r].y);      // S_wmm += m^2 * w
                        }
                    }
                }
            }
            if (done && P.exact_evals) atomicAdd(P.exact_evals, static_cast<unsigned long long>(done));
        }
    }
    // transposition buffer of the epilogue: the consumed stages when there were several branches, else its own
    float2 *stage = q > 1 ? stage0 : stage0 + slice;

    // transpose through shared memory so that the global stores are coalesced
    float2 *st = stage + warp * (32 * R);
#pragma unroll
    for (int r = 0; r < R; ++r) st[lane * R + r] = make_float2(tot[r].y, tot[r].x);   // stored as (S_wmm, S_wmf)
    __syncwarp();
    const long long row = (static_cast<long long>(tset) * gridDim.z + lc) * P.n_dur + j;
    const long long i_warp = i_blk + static_cast<long long>(warp) * (32 * R);
    const long long left_ll = n_cells - i_warp - lane;          // cell r*32 + lane of the warp exists iff r*32 < left
    const int left = left_ll > 32 * R ? 32 * R : static_cast<int>(left_ll);
    const float2 *sl = st + lane;
    const long long i_first = (i_warp + lane) * n_cls + rho;    // t0 cell of the lane's first output; 32 n_cls apart
    const int step = 32 * n_cls;
    if (P.stats) {                                               // the form the periodic search consumes: no division
        float2 *out = P.stats + row * P.stats_pitch + i_first;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (r * 32 < left) {
                const float2 ab = sl[r * 32];
                out[r * step] = ab.x > 0.f ? ab : make_float2(0.f, 0.f);   // no observation in the window: null
            }
        }
    }
    if (P.depth || P.var || P.dlogL) {
        const long long o = row * P.n_t0 + i_first;
        const float nanv = __int_as_float(0x7fc00000);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (r * 32 < left) {
                const float2 ab = sl[r * 32];
                const float a = ab.x, bsum = ab.y;
                const bool null_cell = !(a > 0.f);              // no observation in the window
                const float depth = null_cell ? nanv : bsum / a;
                if (P.depth) P.depth[o + r * step] = depth;
                if (P.var) P.var[o + r * step] = null_cell ? nanv : 1.0f / a;
                if (P.dlogL) P.dlogL[o + r * step] = null_cell ? nanv : 0.5f * bsum * depth;
            }
        }
    }
}

// ------------------------------------------------------------------------------- L2 + L3, off-grid t0
// A t0 grid off the sample grid whose stride is not a small rational multiple of the cadence (those take the residue
// classes of linear_search_kernel): the template sample of a (cell, sample) pair cannot be tabulated, so one thread
// owns one cell.  The definition (R25) derives x = (n c - t_i)/D + 1/2 and idx = floor(x (M-1) + 1/2) per pair with
// five rounded FP64 operations, one of them a division.  This kernel gets the same index from a position that is
// STEPPED: with n = n_c + k around the cell's nearest sample n_c,
//     pos(k) = x(M-1) + 1/2 = k alpha + beta,   alpha = c (M-1)/D,   beta = (n_c c - t_i)(M-1)/D + (M-1)/2 + 1/2,
// beta from one exact FMA per cell, pos re-anchored in FP64 every 64 samples and advanced in 32.32 fixed point in
// between (two integer adds per sample).  pos differs from the position the definition's rounded sequence produces by
// at most eps (host: build_linear_plan), so floor(pos) is the definition's index unless pos lies within eps of an
// integer; the kernel tracks the smallest distance of a block's positions from an integer (one IMNMX per sample, on a
// representation shifted by eps so that the distance is the low word) and recomputes a block with the exact sequence
// (r25_index) when that distance is below 2 eps.  The window edges (x = 0, x = 1) are decided the same way: from pos
// when it is further than eps from the edge, exactly otherwise.
// Neighbouring lanes read the same samples (the stride is far below the cadence), so those loads broadcast; the
// template (m, m^2) pairs are gathered from shared memory.
constexpr int kGenThreads = 128;          // 256 threads, 64 threads and deeper unrolling measured the same or slower
constexpr int kGenBlock = 64;            // samples between FP64 re-anchorings of the position (and per FP32 partial sum)

template <bool TPL_SMEM>
__global__ void __launch_bounds__(kGenThreads) linear_general_kernel(const __grid_constant__ GeneralParams P) {
    extern __shared__ __align__(16) float2 s_tpl2[];   // (m, m^2) per template sample, one spare entry
    if (TPL_SMEM) {
        for (int t = threadIdx.x; t <= P.n_tpl; t += kGenThreads) {
            const float m = t < P.n_tpl ? P.tpl[t] : 0.f;
            s_tpl2[t] = make_float2(m, m * m);
        }
        __syncthreads();
    }
    const long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x;
    const int j = blockIdx.y;
    const long long lc = blockIdx.z;
    const long long row = P.row0 + lc * P.n_dur + j;
    if (i >= P.n_t0) {
        if (P.stats && i < P.stats_pitch) P.stats[row * P.stats_pitch + i] = make_float2(0.f, 0.f);   // row padding
        return;
    }
    const double D = P.durations[j], c = P.cadence;
    const double Mm1 = static_cast<double>(P.n_tpl - 1);
    const double ti = __dadd_rn(P.delta, __dmul_rn(static_cast<double>(i), P.stride));   // t_i - times[0], as R25 forms it
    // nearest sample and the stepped position
    const long long nc = __double2ll_rn(ti / c);
    const double d0 = fma(static_cast<double>(nc), c, -ti);                 // n_c c - t_i, one rounding
    const double g = Mm1 / D;
    const double alpha = c * g;
    const double beta = fma(d0, g, 0.5 * Mm1 + 0.5);
    const double eps = P.eps_scale / D + P.eps_abs;
    // window: samples with 1/2 <= pos <= M - 1/2 (x in [0, 1], both edges included, R2), clipped to the data
    const double inv_alpha = 1.0 / alpha;
    long long kf = static_cast<long long>(ceil((0.5 - beta) * inv_alpha));
    long long kl = static_cast<long long>(floor((Mm1 + 0.5 - beta) * inv_alpha));
    {
        // an edge is decided by the stepped position when that is further than eps from it, exactly otherwise
        const double pf0 = fma(static_cast<double>(kf - 1), alpha, beta), pf1 = fma(static_cast<double>(kf), alpha, beta);
        if (!(pf0 < 0.5 - eps && pf1 > 0.5 + eps)) {
            long long k = kf - 2;
            for (; k <= kf + 2; ++k)
                if (r25_index(nc + k, ti, c, D, Mm1) >= 0) break;
            kf = k;                                                          // kf + 3 when none: an empty window
        }
        const double pl0 = fma(static_cast<double>(kl), alpha, beta), pl1 = fma(static_cast<double>(kl + 1), alpha, beta);
        if (!(pl0 < Mm1 + 0.5 - eps && pl1 > Mm1 + 0.5 + eps)) {
            long long k = kl + 2;
            for (; k >= kl - 2; --k)
                if (r25_index(nc + k, ti, c, D, Mm1) >= 0) break;
            kl = k;
        }
    }
    kf = kf < -nc ? -nc : kf;
    kl = kl > P.n - 1 - nc ? P.n - 1 - nc : kl;
    // fixed point: 32.32, positions shifted up by eps (then "within eps of an integer" reads "low word < 2 eps")
    const double two32 = 4294967296.0;
    const unsigned long long alpha_fx = static_cast<unsigned long long>(__double2ll_rn(alpha * two32));
    const double eps_c = eps < 0.24 ? eps : 0.24;
    const unsigned int two_eps_fx = static_cast<unsigned int>(2.0 * eps_c * two32) + 2u;
    const bool all_exact = !(eps < 0.24) || !(alpha < 1.0e9);               // no usable margin: every block exactly
    const float2 *x_row = P.wfw + lc * P.lc_pitch + nc;
    float s_mf = 0.f, s_mm = 0.f;                       // two-level FP32 sums, as in linear_search_kernel
    unsigned int n_exact = 0;
    for (long long kb = kf; kb <= kl; kb += kGenBlock) {
        const int cnt = static_cast<int>(kl - kb + 1 < kGenBlock ? kl - kb + 1 : kGenBlock);
        const float2 *xp = x_row + kb;
        float a_mf = 0.f, a_mm = 0.f;
        unsigned int nearest = 0xffffffffu;
        if (!all_exact) {
            const double pos0 = fma(static_cast<double>(kb), alpha, beta) + eps_c;
            unsigned long long fx = static_cast<unsigned long long>(__double2ll_rn(pos0 * two32));
#pragma unroll 4
            for (int t = 0; t < cnt; ++t) {
                const unsigned int idx = static_cast<unsigned int>(fx >> 32);
                nearest = min(nearest, static_cast<unsigned int>(fx));
                const float2 s = __ldg(xp + t);
                float2 m2;
                if (TPL_SMEM) {
                    m2 = s_tpl2[idx];
                } else {
                    const float m = __ldg(P.tpl + (idx < static_cast<unsigned int>(P.n_tpl) ? idx : P.n_tpl - 1));
                    m2 = make_float2(m, m * m);
                }
                a_mf = fmaf(m2.x, s.x, a_mf);            // S_wmf += m * (w f)
                a_mm = fmaf(m2.y, s.y, a_mm);            // S_wmm += m^2 * w
                fx += alpha_fx;
            }
        }
        if (all_exact || nearest < two_eps_fx) {
            // some position of the block is within rounding of an index step: the definition's own sequence
            a_mf = 0.f; a_mm = 0.f;
            for (int t = 0; t < cnt; ++t) {
                const int idx = r25_index(nc + kb + t, ti, c, D, Mm1);
                if (idx >= 0) {
                    const float m = __ldg(P.tpl + idx);
                    const float2 s = __ldg(xp + t);
                    a_mf = fmaf(m, s.x, a_mf);
                    a_mm = fmaf(m * m, s.y, a_mm);
                }
            }
            n_exact += cnt;
        }
        s_mf += a_mf;
        s_mm += a_mm;
    }
    if (n_exact && P.exact_evals) atomicAdd(P.exact_evals, static_cast<unsigned long long>(n_exact));
    const bool null_cell = !(s_mm > 0.f);               // no observation in the window
    const float nanv = __int_as_float(0x7fc00000);
    const float depth = null_cell ? nanv : s_mf / s_mm;
    if (P.depth) P.depth[row * P.n_t0 + i] = depth;
    if (P.var) P.var[row * P.n_t0 + i] = null_cell ? nanv : 1.0f / s_mm;
    if (P.dlogL) P.dlogL[row * P.n_t0 + i] = null_cell ? nanv : 0.5f * s_mf * depth;
    if (P.stats) P.stats[row * P.stats_pitch + i] = null_cell ? make_float2(0.f, 0.f) : make_float2(s_mm, s_mf);
}

// ------------------------------------------------------------------------------------------- host
static size_t linear_smem_bytes(const LinearPlan &pl, int R, int warps) {
    // barriers, the duration's tap table (all branches), then either two sample stages (several branches; the
    // epilogue's transposition buffer aliases them) or one stage and the transposition buffer (one branch)
    const int tile = warps * 32 * R;
    size_t worst = 0;
    for (int j = 0; j < pl.P.n_dur; ++j) {
        const size_t slice = (static_cast<size_t>(tile + pl.P.A[j] + 2)) & ~size_t(1);
        const size_t n_tap = pl.P.tap_off[j + 1] - pl.P.tap_off[j];
        worst = std::max(worst, 32 + (n_tap + (pl.P.q > 1 ? 2 * slice : slice + tile)) * 8);
    }
    return worst;
}

int build_linear_plan(const double *times_host, int64_t n, int32_t n_lc, const double *durations_host,
                      int32_t n_dur, cetra_t0_grid grid, int32_t n_template, int smem_limit, int n_sm,
                      LinearPlan *pl, int32_t n_templates) {
    if (!times_host || !durations_host || n < 2 || n_lc < 1 || n_dur < 1 || grid.n_t0 < 1 || n_template < 2 ||
        n_templates < 1)
        return CETRA_ERR_INVALID_ARG;
    if (static_cast<long long>(n_templates) * n_dur > 65535) return CETRA_ERR_UNSUPPORTED;   // grid y dimension
    pl->n_templates = n_templates;
    if (n_dur > CETRA_MAX_DURATIONS) return CETRA_ERR_UNSUPPORTED;
    int rc = derive_geometry(times_host, n, grid, &pl->geo);
    if (rc != CETRA_OK) return rc;
    const bool classes = !pl->geo.on_grid && pl->geo.rational;
    if (!pl->geo.on_grid && !classes) {
        // R25: per-cell evaluation; the (w f, w) row is the plain sample array, no tap tables
        if (n_lc > 65535) return CETRA_ERR_UNSUPPORTED;
        GeneralParams &G = pl->G;
        G.n = n; G.n_t0 = grid.n_t0; G.n_dur = n_dur; G.n_tpl = n_template;
        G.cadence = pl->geo.cadence; G.delta = pl->geo.delta; G.stride = pl->geo.stride;
        G.lc_pitch = round_up64(n, 4);
        G.stats_pitch = cetra_stats_pitch(grid.n_t0);
        for (int j = 0; j < n_dur; ++j) {
            if (!(durations_host[j] > 0.0) || !std::isfinite(durations_host[j])) return CETRA_ERR_INVALID_ARG;
            G.durations[j] = durations_host[j];
        }
        // How far the stepped position (see linear_general_kernel) can lie from the one the definition's rounded FP64
        // sequence produces, in template samples: the sequence itself (3 T 2^-53 (M-1)/D + 4 M 2^-53, T the largest
        // time magnitude), the stepping (FMA anchor, alpha's rounding over <= 64 steps, the 32.32 conversion and 64
        // fixed-point steps: < 2^-26); doubled.
        {
            double t_max = std::max(fabs(pl->geo.delta), fabs(pl->geo.delta + static_cast<double>(grid.n_t0) * pl->geo.stride));
            t_max = std::max(t_max, static_cast<double>(n) * pl->geo.cadence);
            const double ulp = 1.1102230246251565e-16;
            G.eps_scale = 2.0 * 6.0 * t_max * ulp * static_cast<double>(n_template - 1);
            G.eps_abs = 2.0 * (64.0 * static_cast<double>(n_template) * ulp + 1.4901161193847656e-08);
        }
        pl->P.lc_pitch = G.lc_pitch;
        pl->P.n_lo = 0;
        pl->taps_total = 0;
        return CETRA_OK;
    }
    if (pl->geo.q > (1 << 20)) return CETRA_ERR_UNSUPPORTED;
    LinearParams &P = pl->P;
    constexpr int R = kLinearR;
    P.q = static_cast<int>(pl->geo.q);
    P.n0 = pl->geo.n0;
    P.n_t0 = grid.n_t0;
    P.n_dur = n_dur;
    P.n_cls = static_cast<int>(pl->geo.cls);
    P.n_tpl = n_template;
    P.n = n;
    P.cadence = pl->geo.cadence; P.delta = pl->geo.delta; P.stride = pl->geo.stride;
    long long n0_min = pl->geo.n0, n0_max = pl->geo.n0;
    if (classes) {
        // class rho: its cell 0 is t0 cell rho, at phi = (delta + rho stride) / c samples = anchor sample + f
        pl->cls_n0.resize(P.n_cls);
        pl->cls_f.resize(P.n_cls);
        for (int rho = 0; rho < P.n_cls; ++rho) {
            const double phi = (pl->geo.delta + static_cast<double>(rho) * pl->geo.stride) / pl->geo.cadence;
            if (!(fabs(phi) < 1e9)) return CETRA_ERR_UNSUPPORTED;
            const long long nn = llrint(phi);
            pl->cls_n0[rho] = static_cast<int>(nn);
            pl->cls_f[rho] = phi - static_cast<double>(nn);
            if (rho == 0) n0_min = n0_max = nn;
            n0_min = std::min(n0_min, nn);
            n0_max = std::max(n0_max, nn);
        }
        // How far the position of a tap in the template, computed once per class, can lie from the position the
        // definition's rounded FP64 sequence (R25) produces for one of the class's cells, in template samples:
        // (6 T 2^-53 + drift c) (M - 1) / D for the time arithmetic (T: largest time magnitude, drift: Geometry),
        // 32 M 2^-53 for the last two operations; doubled.
        double t_max = std::max(fabs(pl->geo.delta), fabs(pl->geo.delta + static_cast<double>(grid.n_t0) * pl->geo.stride));
        t_max = std::max(t_max, static_cast<double>(n) * pl->geo.cadence);
        const double ulp = 1.1102230246251565e-16;
        pl->eps_scale = 2.0 * (6.0 * t_max * ulp + pl->geo.drift * pl->geo.cadence) * static_cast<double>(n_template - 1);
        pl->eps_abs = 2.0 * 32.0 * static_cast<double>(n_template) * ulp + 1e-12;
    }
    const long long cells_cls0 = (grid.n_t0 + P.n_cls - 1) / P.n_cls;     // class 0 has the most cells
    int h_max = 0, a_max = 0;
    P.tap_off[0] = 0;
    for (int j = 0; j < n_dur; ++j) {
        const double D = durations_host[j];
        if (!(D > 0.0) || !std::isfinite(D)) return CETRA_ERR_INVALID_ARG;
        // window half-reach in samples (R2): floor(D / 2c), one more where the taps' own rounded arithmetic
        // (build_taps_kernel) still places sample h + 1 inside 0 <= x <= 1
        double h = floor(D / (2.0 * pl->geo.cadence));
        if (classes) {
            h = floor(D / (2.0 * pl->geo.cadence) + 0.5) + 1.0;         // |k - f| c <= D / 2 with |f| <= 1/2, and one spare
        } else {
            const volatile double kc = (h + 1.0) * pl->geo.cadence;
            const volatile double xr = kc / D;
            const volatile double x_hi = xr + 0.5, x_lo = -xr + 0.5;
            if (x_hi <= 1.0 || x_lo >= 0.0) h += 1.0;
        }
        if (h > 4.0e6) return CETRA_ERR_UNSUPPORTED;
        P.H[j] = static_cast<int>(h);
        const int ntap = 2 * P.H[j] + 1;
        const int per_phase = (ntap + P.q - 1) / P.q;
        P.A[j] = (per_phase + R - 1) / R * R;
        P.durations[j] = D;
        const long long stored = (static_cast<long long>(P.q) * P.A[j] + 2 + 1) & ~1LL;   // +2: prefetch overrun
        if (P.tap_off[j] + stored > 0x7fffffffLL) return CETRA_ERR_UNSUPPORTED;
        P.tap_off[j + 1] = static_cast<int>(P.tap_off[j] + stored);
        h_max = std::max(h_max, P.H[j]);
        a_max = std::max(a_max, P.A[j]);
    }
    pl->taps_total = static_cast<long long>(P.tap_off[n_dur]) * P.n_cls;
    if (pl->taps_total * n_templates > 0x7fffffffLL) return CETRA_ERR_UNSUPPORTED;
    P.n_tset = n_templates;
    P.tset_taps = pl->taps_total;
    // durations by decreasing cost, so that the heavy blocks are scheduled first
    std::vector<int> ord(n_dur);
    for (int j = 0; j < n_dur; ++j) ord[j] = j;
    std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) { return P.A[a] > P.A[b]; });
    for (int j = 0; j < n_dur; ++j) P.order[j] = static_cast<unsigned char>(ord[j]);

    // tile shape: as many warps per block as shared memory allows, fewer when the grid would not fill the chip
    // (picking the width that wastes the fewest cells in a row's last tile measured slower: 0.496 vs 0.465 ms)
    int warps = 4;
    for (;;) {
        const int tile = warps * 32 * R;
        const long long tiles = (cells_cls0 + tile - 1) / tile;
        const long long blocks = tiles * n_dur * n_lc * P.n_cls * n_templates;
        const bool fits = linear_smem_bytes(*pl, R, warps) <= static_cast<size_t>(smem_limit);
        if (warps == 1 || (fits && blocks >= 2LL * n_sm)) {
            if (!fits) return CETRA_ERR_UNSUPPORTED;
            break;
        }
        warps /= 2;
    }
    pl->warps = warps;
    pl->tile = warps * 32 * R;
    P.tiles_per_row = static_cast<int>((cells_cls0 + pl->tile - 1) / pl->tile);
    if (n_lc > 65535) return CETRA_ERR_UNSUPPORTED;          // light curves are the grid's z dimension
    if (static_cast<long long>(P.tiles_per_row) * P.n_cls > 0x7fffffffLL) return CETRA_ERR_UNSUPPORTED;
    pl->smem_bytes = linear_smem_bytes(*pl, R, warps);

    // padded (w f, w) samples in q polyphase streams: element u of stream v is sample n_lo + q u + v
    P.n_lo = n0_min - h_max - 2;
    const long long u_hi = (n0_max - n0_min + h_max + 2 + P.q) / P.q + static_cast<long long>(P.tiles_per_row) * pl->tile + a_max + 8;
    P.ph_pitch = round_up64(u_hi, 4);
    P.lc_pitch = P.ph_pitch * P.q;
    P.stats_pitch = cetra_stats_pitch(grid.n_t0);
    return CETRA_OK;
}

size_t linear_workspace_bytes(const LinearPlan &pl, int32_t n_lc, int32_t n_template) {
    size_t b = 0;
    b += align_up(sizeof(float2) * static_cast<size_t>(pl.P.lc_pitch) * n_lc);   // (w f, w)
    b += align_up(sizeof(float2) * static_cast<size_t>(pl.taps_total) * pl.n_templates);   // taps
    b += align_up(sizeof(float) * static_cast<size_t>(n_template) * pl.n_templates);       // template(s)
    if (!pl.geo.on_grid && pl.geo.rational) {                                    // residue classes: see run_linear
        b += align_up(sizeof(int) * static_cast<size_t>(pl.P.n_cls));
        b += align_up(sizeof(double) * static_cast<size_t>(pl.P.n_cls));
        b += align_up(sizeof(int) * static_cast<size_t>(pl.P.n_cls) * pl.P.n_dur);
        b += align_up(sizeof(int) * static_cast<size_t>(pl.taps_total));
        b += align_up(static_cast<size_t>(pl.taps_total));
    }
    return b;
}

template <int R, int WARPS, bool CLS>
static int launch_linear(const LinearPlan &pl, const LinearParams &P, int32_t n_lc, cudaStream_t st) {
    auto k = linear_search_kernel<R, WARPS, CLS>;
    CETRA_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_bytes));
    const dim3 grid(static_cast<unsigned>(P.tiles_per_row) * static_cast<unsigned>(P.n_cls),
                    static_cast<unsigned>(P.n_dur) * static_cast<unsigned>(P.n_tset), static_cast<unsigned>(n_lc));
    k<<<grid, WARPS * 32, pl.smem_bytes, st>>>(P);
    CETRA_LAUNCH_CHECK();
    return CETRA_OK;
}

int run_linear(LinearPlan &pl, const void *flux_dev, const void *flux_err_dev, cetra_dtype dtype, int64_t n,
               int32_t n_lc, const float *template_host, int32_t n_template, bool template_on_device,
               float *depth_dev, float *var_dev, float *dlogL_dev, float *stats_dev, void *workspace_dev,
               cudaStream_t st) {
    // the tap tables come first: their place must not depend on n_lc, because the batched search builds
    // them once and then runs ragged last chunks with fewer light curves in the same workspace
    Carver ws(workspace_dev);
    const int T = pl.n_templates;                             // template_host holds T templates of n_template samples
    float2 *taps = ws.take<float2>(static_cast<size_t>(pl.taps_total) * T);
    float *tpl = ws.take<float>(static_cast<size_t>(n_template) * T);
    unsigned long long *exact_evals = nullptr;                // diagnostics counter (a device variable of the library)
    CETRA_CUDA_TRY(cudaGetSymbolAddress(reinterpret_cast<void **>(&exact_evals), g_exact_evals));
    LinearParams &P = pl.P;
    const bool classes = pl.geo.on_grid ? false : pl.geo.rational;
    int *cls_n0 = nullptr, *unsafe_cnt = nullptr, *unsafe_k = nullptr;
    double *cls_f = nullptr;
    unsigned char *flags = nullptr;
    if (classes) {
        cls_n0 = ws.take<int>(P.n_cls);
        cls_f = ws.take<double>(P.n_cls);
        unsafe_cnt = ws.take<int>(static_cast<size_t>(P.n_cls) * P.n_dur);
        unsafe_k = ws.take<int>(static_cast<size_t>(pl.taps_total));
        flags = ws.take<unsigned char>(static_cast<size_t>(pl.taps_total));
    }
    float2 *wfw = ws.take<float2>(static_cast<size_t>(pl.P.lc_pitch) * n_lc);
    P.cls_n0 = cls_n0; P.unsafe_cnt = unsafe_cnt; P.unsafe_k = unsafe_k;
    P.tpl = tpl;
    P.exact_evals = exact_evals;
    pl.G.exact_evals = exact_evals;
    P.wfw = wfw;
    P.taps = taps;
    P.depth = depth_dev; P.var = var_dev; P.dlogL = dlogL_dev;
    P.stats = reinterpret_cast<float2 *>(stats_dev);

    if (!pl.geo.on_grid && !classes && !pl.taps_ready) {
        CETRA_CUDA_TRY(cudaMemcpyAsync(tpl, template_host, sizeof(float) * n_template * T,
                                       template_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
        pl.taps_ready = true;
    }
    if (classes && !pl.taps_ready) {
        // the per-class anchors (small host arrays of the plan: copied before cudaMemcpyAsync returns), then the
        // class tap tables and the lists of the taps they withhold
        CETRA_CUDA_TRY(cudaMemcpyAsync(tpl, template_host, sizeof(float) * n_template * T,
                                       template_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
        CETRA_CUDA_TRY(cudaMemcpyAsync(cls_n0, pl.cls_n0.data(), sizeof(int) * P.n_cls, cudaMemcpyHostToDevice, st));
        CETRA_CUDA_TRY(cudaMemcpyAsync(cls_f, pl.cls_f.data(), sizeof(double) * P.n_cls, cudaMemcpyHostToDevice, st));
        int max_stored = 0;
        for (int j = 0; j < P.n_dur; ++j) max_stored = std::max(max_stored, P.tap_off[j + 1] - P.tap_off[j]);
        dim3 g((max_stored + 255) / 256, P.n_dur, P.n_cls * T);
        build_class_taps_kernel<<<g, 256, 0, st>>>(P, cls_f, pl.eps_scale, pl.eps_abs, taps, flags);
        CETRA_LAUNCH_CHECK();
        const int pairs = P.n_dur * P.n_cls;
        collect_withheld_taps_kernel<<<(pairs + 63) / 64, 64, 0, st>>>(P, flags, unsafe_cnt, unsafe_k);
        CETRA_LAUNCH_CHECK();
        pl.taps_ready = true;
    }
    if (!pl.taps_ready) {
        CETRA_CUDA_TRY(cudaMemcpyAsync(tpl, template_host, sizeof(float) * n_template * T,
                                       template_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
        int max_stored = 0;
        for (int j = 0; j < P.n_dur; ++j) max_stored = std::max(max_stored, P.tap_off[j + 1] - P.tap_off[j]);
        dim3 g((max_stored + 255) / 256, P.n_dur, T);
        build_taps_kernel<<<g, 256, 0, st>>>(P, tpl, n_template, pl.geo.cadence, taps);
        CETRA_LAUNCH_CHECK();
        pl.taps_ready = true;
    }
    {
        const long long total = static_cast<long long>(n_lc) * P.lc_pitch;
        // off-grid plans keep the plain sample row (one stream)
        const bool streams = pl.geo.on_grid || classes;
        const long long ph_q = streams ? P.q : 1, ph_pitch = streams ? P.ph_pitch : P.lc_pitch;
        const int blocks = static_cast<int>(std::min<long long>((total + 255) / 256, 148LL * 16));
        if (dtype == CETRA_F32)
            preprocess_kernel<float><<<blocks, 256, 0, st>>>(static_cast<const float *>(flux_dev),
                                                            static_cast<const float *>(flux_err_dev), n, n_lc, wfw,
                                                            ph_pitch, ph_q, P.n_lo);
        else
            preprocess_kernel<double><<<blocks, 256, 0, st>>>(static_cast<const double *>(flux_dev),
                                                             static_cast<const double *>(flux_err_dev), n, n_lc, wfw,
                                                             ph_pitch, ph_q, P.n_lo);
        CETRA_LAUNCH_CHECK();
    }
    if (!pl.geo.on_grid && !classes) {
        GeneralParams &G = pl.G;
        G.wfw = wfw;
        G.depth = depth_dev; G.var = var_dev; G.dlogL = dlogL_dev;
        G.stats = reinterpret_cast<float2 *>(stats_dev);
        const long long cells = stats_dev ? G.stats_pitch : G.n_t0;
        const dim3 g(static_cast<unsigned>((cells + kGenThreads - 1) / kGenThreads), static_cast<unsigned>(G.n_dur),
                     static_cast<unsigned>(n_lc));
        profile_mark(kProfLinear, true, st);
        for (int t = 0; t < T; ++t) {                           // one launch per template of the set
            G.tpl = tpl + static_cast<size_t>(t) * n_template;
            G.row0 = static_cast<long long>(t) * n_lc * G.n_dur;
            const size_t tpl_bytes = sizeof(float2) * (static_cast<size_t>(n_template) + 1);
            if (tpl_bytes <= 96 * 1024) {                       // (m, m^2) table in shared memory
                auto k = linear_general_kernel<true>;
                CETRA_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
                k<<<g, kGenThreads, tpl_bytes, st>>>(G);
            } else {
                linear_general_kernel<false><<<g, kGenThreads, 0, st>>>(G);
            }
            CETRA_LAUNCH_CHECK();
        }
        profile_mark(kProfLinear, false, st);
        return CETRA_OK;
    }
    constexpr int R = kLinearR;
    profile_mark(kProfLinear, true, st);
    int rc;
    switch (pl.warps * 2 + (classes ? 1 : 0)) {
        case 8: rc = launch_linear<R, 4, false>(pl, P, n_lc, st); break;
        case 9: rc = launch_linear<R, 4, true>(pl, P, n_lc, st); break;
        case 4: rc = launch_linear<R, 2, false>(pl, P, n_lc, st); break;
        case 5: rc = launch_linear<R, 2, true>(pl, P, n_lc, st); break;
        case 2: rc = launch_linear<R, 1, false>(pl, P, n_lc, st); break;
        default: rc = launch_linear<R, 1, true>(pl, P, n_lc, st); break;
    }
    profile_mark(kProfLinear, false, st);
    return rc;
}

}  // namespace cetra
