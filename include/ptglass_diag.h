/*
 * ptglass_diag.h -- test and measurement probes of libptglass.so.  NOT part of the method's interface (include/ptglass.h):
 * nothing here computes a step of the path of arXiv 2003.04621; the parity tests, the roofline measurement of bench.py and
 * the build checks use them.  Same conventions as ptglass.h (return codes, pt_last_error, host / device pointers).
 */
#ifndef PTGLASS_DIAG_H
#define PTGLASS_DIAG_H

#include "ptglass.h"

#ifdef __cplusplus
extern "C" {
#endif

/* force = -1 leaves the choice between the word-parallel kernels (L a power of two >= 8) and the general-L kernels to
 * the library (pt_get_path reports it), 0 forces the general path.  After pt_bind, before pt_init. */
int pt_force_general_path(int force);
/* Philox4x32-10 evaluated by the device code for n counters (HOST arrays ctr[n][4], out[n][4]); test hook. */
int pt_philox_selftest(const uint32_t key[2], const uint32_t *ctr, uint32_t *out, int n);
/* THR(x) = min(2^32-1, floor(2^32 exp(x))) evaluated by the DEVICE double exp for n arguments (HOST arrays): the rare exact
 * decisions of the fixed-point model use it where the +-J model uses host tables (R34); test hook that lets a harness count
 * how often it differs from the host libm's value. */
int pt_threshold_selftest(const double *x, uint32_t *out, int n);
/* INT32 issue-rate microbenchmark, the roofline denominator of the sweep kernel:
 * kind 0 = IMAD.WIDE.U32, 1 = LOP3, 2 = IADD3 carry pair, 3 = IMAD.WIDE+LOP3 mix, 4 = whole Philox4x32-10 blocks
 * (40 ops each).  Launches 256-thread CTAs, ctas_per_sm per SM, on cuda_stream; device_scratch: >= 4 bytes of
 * DEVICE memory.  Returns sustained thread-operations per ns (best of 3 after a warm-up) and the kernel time. */
int pt_microbench(int kind, int ctas_per_sm, int iters, void *device_scratch, void *cuda_stream,
                  double *thread_ops_per_ns, double *ms_out);
/* 1 if this libptglass.so is a development build (PTG_DEV_LATTICE: kernels of one lattice dimension only; pt_init then
 * refuses the other dimension with PT_ERR_ARG), 0 for the full library.  Benchmarks and tests assert 0. */
int pt_is_dev_build(void);

#ifdef __cplusplus
}
#endif
#endif
