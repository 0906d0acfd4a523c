/*
 * cetra_diag.h -- measurement probes of the CETRA B200 build, NOT part of the product ABI.
 *
 * These live in a library of their own (libcetra_diag.so, built by paper_2503_20875_b200/build.py from
 * csrc/peak_probe.cu and csrc/tc_probe.cu) that only bench.py loads: libcetra_b200.so exports no probe.
 * Conventions as in cetra.h (status codes, caller-owned 256-byte aligned workspace, stream as void*).
 */
#ifndef CETRA_DIAG_H_
#define CETRA_DIAG_H_

#include "cetra.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Unit-throughput probes (diagnostic, for bench.py's roofline denominators): the measured rate of the instruction
 * that bounds each hot kernel, in the form the kernel issues it.  Runs a short self-timed kernel on `cuda_stream`
 * with one 1 024-thread CTA per SM and SYNCHRONISES the stream.
 *   CETRA_PROBE_FFMA2  packed FP32 fused multiply-add (linear search)      unit: FP32 flop
 *   CETRA_PROBE_FADD2  packed FP32 add (fold accumulation)                  unit: FP32 flop
 *   CETRA_PROBE_LDS64  conflict-free 8-byte shared-memory loads (fold gather)             unit: bytes
 *  iters            loop trips per thread (>= 1; 20 000 gives a few milliseconds)
 *  per_clk_per_sm   optional out: units per SM clock per SM (from clock64 inside the kernel)
 *  per_second       optional out: units per second over the whole GPU (CUDA events around the launch)
 *  workspace_dev    cetra_peak_probe_workspace_bytes() bytes of device memory, 256-byte aligned
 * Returns CETRA_ERR_INVALID_ARG / CETRA_ERR_WORKSPACE / CETRA_ERR_CUDA as the other entry points. */
typedef enum { CETRA_PROBE_FFMA2 = 0, CETRA_PROBE_FADD2 = 1, CETRA_PROBE_LDS64 = 2 } cetra_probe_kind;
size_t cetra_peak_probe_workspace_bytes(void);
int cetra_peak_probe(int32_t kind, int32_t iters, double *per_clk_per_sm, double *per_second,
                     void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Diagnostic, not on the search path: the measured tensor-core variant of the linear search's windowed sums
 * (north_star: "must beat the CUDA-core version in ncu to be kept"; DESIGN.md §7 has the outcome).
 * Runs the banded correlation S_wmf[i] = sum_k m[k] (w f)[i + k], S_wmm[i] = sum_k m[k]^2 w[i + k] over n_taps taps
 * for n_out consecutive outputs on synthetic device-generated samples as Toeplitz x sample-tile products on
 * mma.sync.m16n8k8 TF32 (split != 0: the 3xTF32 product that the 1e-5 parity bar needs; 0: one TF32 product),
 * `reps` times, and returns the mean launch time (CUDA events) and the largest errors against an FP64 evaluation
 * of every 7th output (err_wmf relative to the largest |S_wmf|, err_wmm relative per output).  Synchronises. */
size_t cetra_tc_correlation_probe_workspace_bytes(int64_t n_out, int32_t n_taps);
int cetra_tc_correlation_probe(int64_t n_out, int32_t n_taps, int32_t split, int32_t reps, double *ms_per_launch,
                               double *err_wmf, double *err_wmm, void *workspace_dev, size_t workspace_bytes,
                               void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* CETRA_DIAG_H_ */
