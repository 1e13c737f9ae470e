/*
 * apd_probe.h -- C ABI of libapd_probe.so: FP32 microbenchmarks for bench.py.
 * A measurement tool, NOT part of the method and not part of libapd_b200.so (include/apd.h): MEASURED_PEAKS.json
 * holds no FP32 CUDA-core figure, so the FP32 roofline denominator is measured here.
 */
#ifndef APD_PROBE_H
#define APD_PROBE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { APD_PROBE_OK = 0, APD_PROBE_E_ARG = -1, APD_PROBE_E_CUDA = -2, APD_PROBE_E_ARCH = -3 };

/* Runs a register-only FP32 loop on CUDA device `device` (compute capability 10.x) and returns the achieved rate in
 * *ops_per_s (HOST out): variant 0 = scalar FFMA (2 flop each), 1 = packed fma.rn.f32x2 (4 flop each), 2 = 3-input
 * min.f32, 3 = the ROWPOLY inner-loop mix (3 f32x2 FMA + 2 three-input min per 4 voxel-seed pairs).  *ops_per_s counts
 * FMA lanes (variants 0, 1), min instructions x 32 lanes (2) or voxel-seed pairs (3).  *sm_clock_mhz (HOST out, may be
 * NULL): SM clock during the loop (clock64 / globaltimer).  Synchronous.  Returns APD_PROBE_OK or a negative code. */
int apd_fp32_probe(int32_t device, int32_t variant, double* ops_per_s, double* sm_clock_mhz);

#ifdef __cplusplus
}
#endif
#endif /* APD_PROBE_H */
