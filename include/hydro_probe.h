/*
 * hydro_probe.h -- C ABI of libhydro_probe_b200: a measurement aid, NOT part of the hydro path and not part
 * of libhydro_b200.  bench.py loads it to measure the plain FP64 pipe of the device, the second roofline
 * of DESIGN.md sec. 5 (MEASURED_PEAKS.json carries no FP64 figure; SURVEY.md sec. 8(d) asks for a
 * dependent-free FMA loop and a non-FMA add/mul loop).
 */
#ifndef HYDRO_PROBE_B200_H
#define HYDRO_PROBE_B200_H

#ifdef __cplusplus
extern "C" {
#endif

/* Times three small kernels on the current device (default stream, synchronous; allocates and frees
 * 2.4 MB of device memory) and writes FP64 thread-instructions per second (x2 = FLOP/s for an FMA) into
 * rates_host[3] (HOST memory): [0] independent DFMA chains, [1] DADD/DMUL chains (no FMA), [2] DFMA chains
 * with one independent integer multiply-add between consecutive DFMAs (counts the DFMAs only).
 * Returns 0, or -1 (null pointer), -2 (allocation failed), -3 (kernel failed). */
int hydro_probe_fp64(double *rates_host);

#ifdef __cplusplus
}
#endif
#endif /* HYDRO_PROBE_B200_H */
