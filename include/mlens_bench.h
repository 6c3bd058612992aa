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

/* Rate [adds/s] of 64-bit atomic adds to global memory (use_u64 = 1: unsigned integers, the type the map accumulators
 * use -- RED.E.ADD.64; 0: doubles) into a buffer of n_slots 8-byte slots (4 <= n_slots < 2^32) -- L2-resident or
 * HBM-resident according to its size.  pattern 0: every lane a uniformly random slot (up to 32 sectors per warp
 * instruction); 1: lanes in fours on the four slots of one random 32-byte sector (8 sectors per warp instruction);
 * 2: all 32 lanes on the four slots of one random sector.  The slot costs two integer instructions (an LCG step and a
 * multiply-high), so the loop is bound by the atomic path, not by its own arithmetic (profiles/r03_sass_atomics.txt). */
int mlens_bench_atomics_pattern(int64_t n_slots, int32_t use_u64, int32_t pattern, double *adds_per_s, void *stream);
/* = pattern 0. */
int mlens_bench_atomics(int64_t n_slots, int32_t use_u64, double *adds_per_s, void *stream);

/* Rate [adds/s] of atomic adds into a 64 KB tile of SHARED memory per block (as many blocks per SM as fit): what a
 * per-tile shared-memory accumulator can absorb.  kind 0: the 64-bit atomicAdd (a compare-and-swap loop in SASS);
 * 1: the product's own 64-bit add, two native 32-bit ATOMS.ADD with the carry taken from the first one's return value
 * (deposit.cuh shared_add64); 2: one plain 32-bit add.  conflict_free 0: random slots (random banks); 1: lane i on slot
 * 32 row + i of a random row. */
int mlens_bench_shared_atomics_kind(int32_t kind, int32_t conflict_free, double *adds_per_s, void *stream);
/* = kind 1, random slots: the product's pattern. */
int mlens_bench_shared_atomics(double *adds_per_s, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* MLENS_BENCH_H */
