/* mlens_bench.h -- C ABI of libmlens_bench: micro-benchmarks that measure the roofline denominators of the hot
 * path on the device at hand ("the FP64 and atomic ceilings must be measured by micro-benchmarks
 * in the same run").  A separate shared library: nothing in libmlens depends on it, bench.py alone loads it.
 *
 * Every call runs on the CURRENT device, enqueues on `stream` (void* cudaStream_t, NULL = default stream),
 * synchronises it, returns 0 on success and a negative cudaError_t otherwise; outputs are HOST pointers. */
#ifndef MLENS_BENCH_H
#define MLENS_BENCH_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Sustained FP64 fused multiply-add rate [FLOP/s]: eight independent DFMA chains per thread, all SMs. */
int mlens_bench_dfma(double *flops_per_s, void *stream);

/* Rate [adds/s] of 64-bit atomic adds (use_u64 = 1: unsigned integers, the type the map accumulators use;
 * 0: doubles) at uniformly random slots of a buffer of n_slots 8-byte slots -- L2-resident or HBM-resident
 * according to its size. */
int mlens_bench_atomics(int64_t n_slots, int32_t use_u64, double *adds_per_s, void *stream);

/* Rate [adds/s] of 64-bit atomic adds at uniformly random slots of a 64 KB tile of SHARED memory per block (as many
 * blocks per SM as fit): what a per-tile shared-memory accumulator could absorb.  On a B200 it equals the rate of
 * L2-resident global adds. */
int mlens_bench_shared_atomics(double *adds_per_s, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* MLENS_BENCH_H */
