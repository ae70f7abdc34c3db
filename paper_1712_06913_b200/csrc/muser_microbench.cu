// Microbenchmarks of the three device limits the gridding roofline discussion refers to:
// FP32 FMA issue rate (plain and packed FFMA2), native 32-bit shared-memory integer adds (what the owner gridder
// merges with), fp32 shared-memory adds (compare-and-swap loops), and fp32 global reductions (what the generic
// gridders flush with).  Each call runs one kernel `reps` times on stream 0 and returns the best rate.
#include "../../include/muser.h"

#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__global__ void __launch_bounds__(256) k_mb_fma(float* out, int iters) {
    float a0 = threadIdx.x * 1e-3f, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f, a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f, a7 = a0 + 7.f;
    const float b = 1.000001f, c = 1e-7f;
    for (int i = 0; i < iters; ++i) {
        a0 = fmaf(a0, b, c); a1 = fmaf(a1, b, c); a2 = fmaf(a2, b, c); a3 = fmaf(a3, b, c);
        a4 = fmaf(a4, b, c); a5 = fmaf(a5, b, c); a6 = fmaf(a6, b, c); a7 = fmaf(a7, b, c);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
}

__device__ __forceinline__ unsigned long long mb_fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__global__ void __launch_bounds__(256) k_mb_fma2(unsigned long long* out, int iters) {
    unsigned long long a[8];
    for (int j = 0; j < 8; ++j) a[j] = 0x3f8000003f800000ull + (unsigned long long)(threadIdx.x + j);
    const unsigned long long b = 0x3f8000013f800001ull, c = 0x33d6bf9533d6bf95ull;
    for (int i = 0; i < iters; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = mb_fma2(a[j], b, c);
    unsigned long long s = 0;
    for (int j = 0; j < 8; ++j) s ^= a[j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// kind 0: native integer shared add, 1: fp32 shared add (CAS loop); addresses spread over 4096 words, conflict-free per warp
template <int KIND>
__global__ void __launch_bounds__(256) k_mb_shared(float* out, int iters) {
    __shared__ int s_i[4096];
    float* s_f = reinterpret_cast<float*>(s_i);
    for (int i = threadIdx.x; i < 4096; i += 256) s_i[i] = 0;
    __syncthreads();
    int idx = threadIdx.x;
    for (int i = 0; i < iters; ++i) {
        if (KIND == 0) atomicAdd(&s_i[idx], 1); else atomicAdd(&s_f[idx], 1.0f);
        idx = (idx + 256) & 4095;
    }
    __syncthreads();
    out[blockIdx.x * blockDim.x + threadIdx.x] = (float)s_i[threadIdx.x];
}

// fp32 global reductions spread over `span` floats (coalesced within a warp)
__global__ void __launch_bounds__(256) k_mb_red(float* buf, size_t span, int iters) {
    size_t idx = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) % span;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int i = 0; i < iters; ++i) {
        atomicAdd(buf + idx, 1.0f);
        idx += stride;
        if (idx >= span) idx -= span;
    }
}

template <typename F>
double best_ms(F launch, int reps) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int r = 0; r < reps + 1; ++r) {
        cudaEventRecord(e0, 0);
        launch();
        cudaEventRecord(e1, 0);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return best;
}

}  // namespace

extern "C" int muser_microbench(int kind, double* rate_out) {
    if (!rate_out || kind < 0 || kind > 4) return MUSER_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return MUSER_ECUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = sms * 8, iters = 4096;
    void* buf = nullptr;
    const size_t span = (size_t)64 << 20;                             // 256 MB of floats for the global reductions
    if (cudaMalloc(&buf, kind == 4 ? span * sizeof(float) : (size_t)blocks * 256 * 8) != cudaSuccess) return MUSER_ENOMEM;
    if (kind == 4) cudaMemset(buf, 0, span * sizeof(float));
    double ms = 0, ops = 0;
    switch (kind) {
        case 0: ms = best_ms([&] { k_mb_fma<<<blocks, 256>>>((float*)buf, iters); }, 5); ops = 2.0 * 8 * iters * blocks * 256.0; break;            // flop
        case 1: ms = best_ms([&] { k_mb_fma2<<<blocks, 256>>>((unsigned long long*)buf, iters); }, 5); ops = 4.0 * 8 * iters * blocks * 256.0; break;  // flop
        case 2: ms = best_ms([&] { k_mb_shared<0><<<blocks, 256>>>((float*)buf, iters); }, 5); ops = (double)iters * blocks * 256.0; break;        // adds
        case 3: ms = best_ms([&] { k_mb_shared<1><<<blocks, 256>>>((float*)buf, iters / 4); }, 5); ops = (double)(iters / 4) * blocks * 256.0; break;
        case 4: ms = best_ms([&] { k_mb_red<<<blocks, 256>>>((float*)buf, span, 256); }, 5); ops = 256.0 * blocks * 256.0; break;
    }
    cudaError_t e = cudaDeviceSynchronize();
    cudaFree(buf);
    if (e != cudaSuccess) return MUSER_ECUDA;
    *rate_out = ops / (ms * 1e-3);
    return MUSER_OK;
}
