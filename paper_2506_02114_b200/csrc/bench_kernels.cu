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

__global__ void atomics_kernel(unsigned long long *bu, double *bd, long long n_slots, int use_u64, int per_thread) {
    unsigned long long h = (blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x + 1) * 0x9E3779B97F4A7C15ull;
    for (int i = 0; i < per_thread; ++i) {
        h ^= h >> 29; h *= 0xBF58476D1CE4E5B9ull; h ^= h >> 32;
        long long slot = (long long)(h % (unsigned long long)n_slots);
        if (use_u64) atomicAdd(&bu[slot], 1ull); else atomicAdd(&bd[slot], 1.0);
    }
}

// random 64-bit adds into a 64 KB tile of SHARED memory per block (three blocks per SM): what a per-tile accumulator
// in shared memory could take in
__global__ void __launch_bounds__(256) shared_atomics_kernel(unsigned long long *out, int nslots, int per_thread) {
    extern __shared__ unsigned long long tile[];
    for (int i = threadIdx.x; i < nslots; i += blockDim.x) tile[i] = 0ull;
    __syncthreads();
    unsigned long long h = (blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x + 1) * 0x9E3779B97F4A7C15ull;
    for (int i = 0; i < per_thread; ++i) {
        h ^= h >> 29; h *= 0xBF58476D1CE4E5B9ull; h ^= h >> 32;
        atomicAdd(&tile[(int)(h % (unsigned long long)nslots)], (h >> 20) | (1ull << 34));
    }
    __syncthreads();
    unsigned long long acc = 0ull;
    for (int i = threadIdx.x; i < nslots; i += blockDim.x) acc += tile[i];
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

int mlens_bench_atomics(int64_t n_slots, int32_t use_u64, double *adds_per_s, void *stream) {
    if (!adds_per_s || n_slots <= 0) return -(int)cudaErrorInvalidValue;
    cudaStream_t s = (cudaStream_t)stream;
    const int blocks = sm_count() * 16, threads = 256, per = 256;
    int rc = 0;
    float best = 1e30f;
    void *buf = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    BK(cudaMallocAsync(&buf, (size_t)n_slots * 8, s));
    BK(cudaMemsetAsync(buf, 0, (size_t)n_slots * 8, s));
    BK(cudaEventCreate(&e0)); BK(cudaEventCreate(&e1));
    atomics_kernel<<<blocks, threads, 0, s>>>((unsigned long long *)buf, (double *)buf, n_slots, use_u64, 8);
    for (int r = 0; r < 3; ++r) {
        BK(cudaEventRecord(e0, s));
        atomics_kernel<<<blocks, threads, 0, s>>>((unsigned long long *)buf, (double *)buf, n_slots, use_u64, per);
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

int mlens_bench_shared_atomics(double *adds_per_s, void *stream) {
    if (!adds_per_s) return -(int)cudaErrorInvalidValue;
    cudaStream_t s = (cudaStream_t)stream;
    const int smem = 64 * 1024, nslots = smem / 8, threads = 256, per = 4096;
    int rc = 0, bps = 0;
    float best = 1e30f;
    unsigned long long *d = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int blocks = 0;
    BK(cudaFuncSetAttribute(shared_atomics_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    BK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, shared_atomics_kernel, threads, smem));
    blocks = sm_count() * (bps > 0 ? bps : 1);
    BK(cudaMallocAsync(&d, 8, s));
    BK(cudaEventCreate(&e0)); BK(cudaEventCreate(&e1));
    shared_atomics_kernel<<<blocks, threads, smem, s>>>(d, nslots, 64);
    for (int r = 0; r < 3; ++r) {
        BK(cudaEventRecord(e0, s));
        shared_atomics_kernel<<<blocks, threads, smem, s>>>(d, nslots, per);
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

}  // extern "C"
