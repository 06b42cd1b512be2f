/*
 * ds_dev.h -- development and measurement hooks of libds.so.  NOT part of the product boundary (include/ds.h): tests
 * use them to force launch shapes through every code path, bench.py to measure the roofline denominators and to count
 * launches.  Same conventions as ds.h (extern "C", plain pointers, int return codes).
 */
#ifndef DS_DEV_H_
#define DS_DEV_H_

#include "ds.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Launch-shape override for tuning and tests: number of row tiles (CTAs) per system; 0 = library
 * heuristic.  Values below ceil(ceil(N/4)/512) or above ceil(N/4) are clamped; the step modes also
 * clamp to the SM count (their CTAs meet at a barrier every stage and must be co-resident).      */
int ds_set_tuning(ds_system *s, int32_t n_tiles);

/* Development instrumentation: device_buffer (DEVICE pointer, 16 int64 per CTA of the largest launch,
 * or NULL to switch off) receives clock64() samples of the last stage of every hot-kernel launch.  */
int ds_set_probe(ds_system *s, void *device_buffer);

/* Number of kernels launched by this system since creation (bench.py's gpu_launches claim). */
int64_t ds_launch_count(const ds_system *s);

/* Measurement aid for the roofline denominators (bench.py): runs an FMA-chain microbenchmark on
 * `device` (packed FP32 FMA for DS_F32, DFMA for DS_F64) and writes the best achieved FLOP/s
 * (FMA = 2) to *flops_per_s (HOST pointer).  Synchronous; uses the legacy default stream.       */
int ds_peak_probe(int32_t precision, int32_t device, double *flops_per_s);

/* Step-kernel choice for ds_step / ds_batch_step: -1 = library heuristic (default), 0 = always the one-pass kernel
 * (mobility.cuh), 1 = the pipelined two-pass kernel (pipeline.cuh) whenever the launch shape allows it (several CTAs per
 * system, each half of a CTA's rows at most 16 quads, streams resident in shared memory).  Both kernels advance the same
 * equations; they differ in the order of the split-beta sums, i.e. in the last bits.
 * Ensembles (n_batch >= 2) whose systems can each take one thread-block cluster (cluster.cuh: all clusters resident at once
 * and filling at least 3/4 of the SMs) use the cluster kernel unless mode is 0.
 * Systems with short pair loops (17 <= S up to about 200 in FP32, 130 in FP64: at most 3 iterations per warp, 4 in ensembles)
 * whose clusters of 2 ... 16 CTAs are all resident at once use the latency variant cluster_lat_kernel unless mode is 0 or 1.
 * ds_pipeline_active: the kernel the next ds_step / ds_batch_step would use: 0 = one-pass (or, for small S, the
 * warp-per-system kernel), 1 = pipelined two-pass, 2 = cluster kernel, 3 = its latency variant.
 * Modes 2 and 3 (tests, measurements): the cluster kernel / its latency variant for every shape they can run, whatever the
 * heuristic says.                                                                                                       */
int ds_set_pipeline(ds_system *s, int32_t mode);
int ds_pipeline_active(const ds_system *s);

#ifdef __cplusplus
}
#endif
#endif /* DS_DEV_H_ */
