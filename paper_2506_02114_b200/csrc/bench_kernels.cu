// bench_kernels.cu -- libmlens_bench.so (include/mlens_bench.h): the roofline denominators measured on the device
// at hand.  Not part of libmlens.
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/mlens_bench.h"

namespace {

__global__ void dfma_kernel(double *out, int iters) {
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double b = 1.0000001, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
        a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
    }
    double r = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (r == 123.456) out[0] = r;
}

// Slot choice must cost next to nothing, or the loop measures the slot arithmetic instead of the atomic unit (round 2's
// `h % n_slots` on 64-bit operands compiled to a ~64-instruction subroutine per add: VERDICT r2).  Here: one 32-bit LCG
// step (one IMAD) and the high word of h * n_slots (one IMAD.WIDE), n_slots < 2^32.  The SASS of the loops is in
// profiles/r03_sass_atomics.txt.
__device__ __forceinline__ unsigned int lcg(unsigned int h) { return h * 1664525u + 1013904223u; }

// PATTERN 0: every lane its own random slot (up to 32 sectors of 32 B per warp instruction)
//         1: lanes in groups of four on the four 8-byte slots of one random sector: 8 sectors per warp instruction
//         2: all 32 lanes on the four slots of ONE random sector (8 lanes per address)
template <int PATTERN>
__global__ void __launch_bounds__(256) atomics_kernel(unsigned long long *bu, double *bd, unsigned int n_slots, int use_u64, int per_thread) {
    const unsigned int tid = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
    const unsigned int who = PATTERN == 0 ? tid : PATTERN == 1 ? (tid >> 2) : (tid >> 5);   // lanes that share a sector share the stream
    unsigned int h = (who + 1u) * 0x9E3779B9u;
    const unsigned int n_eff = PATTERN == 0 ? n_slots : n_slots >> 2;
#pragma unroll 8
    for (int i = 0; i < per_thread; ++i) {
        h = lcg(h);
        unsigned int slot = __umulhi(h, n_eff);
        if (PATTERN != 0) slot = slot * 4u + (lane & 3u);
        if (use_u64) atomicAdd(&bu[slot], 1ull); else atomicAdd(&bd[slot], 1.0);
    }
}

// Adds into a 64 KB tile of SHARED memory per block (as many blocks per SM as fit): what a per-tile accumulator in
// shared memory can take in.
// KIND 0: 64-bit atomicAdd (compiles to a compare-and-swap loop: ATOMS.CAST.SPIN)
//      1: the product's own 64-bit add (deposit.cuh shared_add64): two native 32-bit ATOMS.ADD, the first returning the
//         old low word for the carry
//      2: one plain 32-bit atomicAdd, nothing returned
// CFREE 0: every lane a random slot (random banks); 1: lane i on slot 32 * row + i of a random row (no bank conflict
//          beyond the two banks an 8-byte slot spans)
template <int KIND, int CFREE>
__global__ void __launch_bounds__(256) shared_atomics_kernel(unsigned long long *out, int per_thread) {
    extern __shared__ unsigned long long tile[];
    const int nbytes = 64 * 1024;
    unsigned int *t32 = reinterpret_cast<unsigned int *>(tile);
    for (int i = threadIdx.x; i < nbytes / 8; i += blockDim.x) tile[i] = 0ull;
    __syncthreads();
    const unsigned int lane = threadIdx.x & 31;
    const unsigned int n_slots = KIND == 2 ? nbytes / 4 : nbytes / 8;
    const unsigned int tid = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int h = ((CFREE ? (tid >> 5) : tid) + 1u) * 0x9E3779B9u;
#pragma unroll 8
    for (int i = 0; i < per_thread; ++i) {
        h = lcg(h);
        const unsigned int slot = CFREE ? __umulhi(h, n_slots >> 5) * 32u + lane : __umulhi(h, n_slots);
        if (KIND == 0) {
            atomicAdd(&tile[slot], (unsigned long long)h | (1ull << 34));
        } else if (KIND == 1) {
            const unsigned int lo = h | 1u, hi = 4u;                       // both words non-zero: two adds, as for most deposits
            const unsigned int old = atomicAdd(&t32[2 * slot], lo);
            atomicAdd(&t32[2 * slot + 1], hi + ((old + lo < old) ? 1u : 0u));
        } else {
            atomicAdd(&t32[slot], h | 1u);
        }
    }
    __syncthreads();
    unsigned long long acc = 0ull;
    for (int i = threadIdx.x; i < nbytes / 8; i += blockDim.x) acc += tile[i];
    if (acc == 12345ull) out[0] = acc;
}

int sm_count() {
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    return nsm;
}

#define BK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { rc = -(int)e_; goto out; } } while (0)

}  // namespace

extern "C" {

int mlens_bench_dfma(double *flops_per_s, void *stream) {
    if (!flops_per_s) return -(int)cudaErrorInvalidValue;
    cudaStream_t s = (cudaStream_t)stream;
    const int iters = 1 << 15, blocks = sm_count() * 8, threads = 256;
    int rc = 0;
    float best = 1e30f;
    double *d = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    BK(cudaMallocAsync(&d, 8, s));
    BK(cudaEventCreate(&e0)); BK(cudaEventCreate(&e1));
    dfma_kernel<<<blocks, threads, 0, s>>>(d, 1024);
    for (int r = 0; r < 5; ++r) {
        BK(cudaEventRecord(e0, s));
        dfma_kernel<<<blocks, threads, 0, s>>>(d, iters);
        BK(cudaEventRecord(e1, s));
        BK(cudaEventSynchronize(e1));
        float ms; BK(cudaEventElapsedTime(&ms, e0, e1));
        if (ms < best) best = ms;
    }
    BK(cudaGetLastError());
    *flops_per_s = 2.0 * 8.0 * (double)iters * blocks * threads / (best * 1e-3);
out:
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (d) cudaFreeAsync(d, s);
    return rc;
}

int mlens_bench_atomics_pattern(int64_t n_slots, int32_t use_u64, int32_t pattern, double *adds_per_s, void *stream) {
    if (!adds_per_s || n_slots < 4 || n_slots >= (1ll << 32) || pattern < 0 || pattern > 2) return -(int)cudaErrorInvalidValue;
    cudaStream_t s = (cudaStream_t)stream;
    const int blocks = sm_count() * 16, threads = 256, per = 256;
    int rc = 0;
    float best = 1e30f;
    void *buf = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    void (*k)(unsigned long long *, double *, unsigned int, int, int) =
        pattern == 0 ? atomics_kernel<0> : pattern == 1 ? atomics_kernel<1> : atomics_kernel<2>;
    BK(cudaMallocAsync(&buf, (size_t)n_slots * 8, s));
    BK(cudaMemsetAsync(buf, 0, (size_t)n_slots * 8, s));
    BK(cudaEventCreate(&e0)); BK(cudaEventCreate(&e1));
    k<<<blocks, threads, 0, s>>>((unsigned long long *)buf, (double *)buf, (unsigned int)n_slots, use_u64, 8);
    for (int r = 0; r < 3; ++r) {
        BK(cudaEventRecord(e0, s));
        k<<<blocks, threads, 0, s>>>((unsigned long long *)buf, (double *)buf, (unsigned int)n_slots, use_u64, per);
        BK(cudaEventRecord(e1, s));
        BK(cudaEventSynchronize(e1));
        float ms; BK(cudaEventElapsedTime(&ms, e0, e1));
        if (ms < best) best = ms;
    }
    BK(cudaGetLastError());
    *adds_per_s = (double)blocks * threads * per / (best * 1e-3);
out:
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (buf) cudaFreeAsync(buf, s);
    return rc;
}

int mlens_bench_atomics(int64_t n_slots, int32_t use_u64, double *adds_per_s, void *stream) {
    return mlens_bench_atomics_pattern(n_slots, use_u64, 0, adds_per_s, stream);
}

int mlens_bench_shared_atomics_kind(int32_t kind, int32_t conflict_free, double *adds_per_s, void *stream) {
    if (!adds_per_s || kind < 0 || kind > 2) return -(int)cudaErrorInvalidValue;
    cudaStream_t s = (cudaStream_t)stream;
    const int smem = 64 * 1024, threads = 256, per = 4096;
    int rc = 0, bps = 0;
    float best = 1e30f;
    unsigned long long *d = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int blocks = 0;
    void (*k)(unsigned long long *, int) =
        kind == 0 ? (conflict_free ? shared_atomics_kernel<0, 1> : shared_atomics_kernel<0, 0>)
      : kind == 1 ? (conflict_free ? shared_atomics_kernel<1, 1> : shared_atomics_kernel<1, 0>)
                  : (conflict_free ? shared_atomics_kernel<2, 1> : shared_atomics_kernel<2, 0>);
    BK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    BK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k, threads, smem));
    blocks = sm_count() * (bps > 0 ? bps : 1);
    BK(cudaMallocAsync(&d, 8, s));
    BK(cudaEventCreate(&e0)); BK(cudaEventCreate(&e1));
    k<<<blocks, threads, smem, s>>>(d, 64);
    for (int r = 0; r < 3; ++r) {
        BK(cudaEventRecord(e0, s));
        k<<<blocks, threads, smem, s>>>(d, per);
        BK(cudaEventRecord(e1, s));
        BK(cudaEventSynchronize(e1));
        float ms; BK(cudaEventElapsedTime(&ms, e0, e1));
        if (ms < best) best = ms;
    }
    BK(cudaGetLastError());
    *adds_per_s = (double)blocks * threads * per / (best * 1e-3);
out:
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (d) cudaFreeAsync(d, s);
    return rc;
}

int mlens_bench_shared_atomics(double *adds_per_s, void *stream) {
    return mlens_bench_shared_atomics_kind(1, 0, adds_per_s, stream);
}

}  // extern "C"
