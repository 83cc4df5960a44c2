/*
 * rpa_probes.h -- C ABI of librpa_probes.so: issue-rate probes of the two tensor pipes the rank-K update (Eq. 17 /
 * Eq. 20) can run on.  MEASUREMENT helpers for bench.py, not part of the product library
 * (librpa_chi0.so, include/rpa_chi0.h): they have no handle and no workspace, and each call allocates and frees its own
 * small device buffer.  MEASURED_PEAKS.json has neither an FP64 nor an int8 entry; these probes supply the measured
 * denominators of the `roofline` objects bench.py prints ("Roofline denominators").
 *
 * All calls block until the probe kernels have finished.  Return 0 on success or a negative code; rpa_probe_last_error()
 * holds a thread-local message.
 */
#ifndef RPA_PROBES_H
#define RPA_PROBES_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RPA_PROBE_OK 0
#define RPA_PROBE_ERR_INVALID_ARG (-1)
#define RPA_PROBE_ERR_CUDA (-4)

/* Register-only DMMA issue-rate probe: every warp of a 16-warp CTA per SM runs dependent-free mma.sync.m8n8k4.f64
 * (DMMA.8x8x4, the only native FP64 MMA of sm_100a) and *tflops receives the achieved FP64 tensor TFLOP/s: the measured
 * roofline denominator of rank_k3m_kernel.  cuda_stream: a cudaStream_t (NULL = default); tflops: host.  Allocates and
 * frees 64 bytes of device memory. */
int rpa_probe_fp64_tensor_peak(void *cuda_stream, double *tflops);

/* tcgen05 int8 issue-rate probe (denominator of the opt-in int8-sliced rank-K arm): on every SM one thread
 * issues 20000 accumulating tcgen05.mma.kind::i8 of 128 x 256 x 32 (operands in shared memory, s32 accumulator in TMEM);
 * *tops = achieved int8 Top/s.  The first MMA of CTA 0 is read back from TMEM and compared with the host product of the
 * same seeded operands: *mismatches = number of wrong elements of 32768 (0 on a working path).  Allocates and frees
 * 140 KB of device memory. */
int rpa_probe_int8_tensor_peak(void *cuda_stream, double *tops, int32_t *mismatches);

/* Thread-local message of the last probe error on this thread (static storage, never NULL). */
const char *rpa_probe_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* RPA_PROBES_H */
