/* gsvox_probe.h — bench-only companion of gsvox.h: the ALU microbenchmarks bench.py uses as roofline
 * denominators.  Built into its own shared object (paper_2503_22139_b200/libgsvox_probe.so), NOT into the
 * product library libgsvox.so: nothing on the hot path needs it.                                     */
#ifndef GSVOX_PROBE_H
#define GSVOX_PROBE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* Live ALU rooflines of the device the calling thread has current (the hot path is
 * FP32-issue / MUFU bound, and MEASURED_PEAKS.json holds no FP32 figure).  Runs three register-only
 * microbenchmarks on `stream` and SYNCHRONISES: scalar FFMA chains (fp32_tflops, 2 flops per lane
 * instruction), packed fma.rn.f32x2 chains (fp32x2_tflops, 4 flops per lane instruction) and
 * ex2.approx chains (ex2_tera_per_s, 1e12 results/s).  `scratch` = at least 4 bytes of DEVICE
 * memory (never written in practice).  Any output pointer may be NULL.  HOST output pointers.  */
int gsvox_probe_peaks(void* scratch, double* fp32_tflops, double* fp32x2_tflops,
                      double* ex2_tera_per_s, int32_t* sm_count, void* stream);

#ifdef __cplusplus
}
#endif
#endif
