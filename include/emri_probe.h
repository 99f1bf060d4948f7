/* emri_probe.h -- measurement helpers of bench.py (libemri_probe.so): peak probes on the current CUDA device, so that
 * the roofline denominators DESIGN.md section 7 quotes are re-measured in the run that reports a fraction of them.
 * NOT part of the boundary: the hot path of the paper is include/emri.h; nothing there calls these.
 * All return 0 on success, < 0 on error; `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream);
 * each call synchronises on its own events. */
#ifndef EMRI_PROBE_H
#define EMRI_PROBE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { EMRI_PROBE_EINVAL = -1, EMRI_PROBE_ENOMEM = -2, EMRI_PROBE_ECUDA = -3 };

/* TFLOP/s (FMA = 2) of a kernel of independent DFMA chains with a constant operand: the FP64 issue peak. */
int emri_probe_fp64_peak(double* tflops, void* cuda_stream);
/* The same with three fresh vector-register operands per DFMA (no constant, uniform-register or reused operand):
 * what register-bound FP64 code can reach (on B200 2/3 of the figure above). */
int emri_probe_fp64_peak3(double* tflops, void* cuda_stream);
/* GB/s of one streaming read of `bytes` (>= 1 MiB) of device memory. */
int emri_probe_hbm_read(int64_t bytes, double* gbs, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* EMRI_PROBE_H */
