// muser_histogram_static: the own-range histogram of NEXT-4 ("the data from a dirty image is divided into 2000
// ranges") for callers that must not allocate device memory.
//
// Who that is: a monitoring loop that images every 3 ms frame cannot take cudaMalloc / cudaFree in its
// steady state -- both synchronise the whole device and stall the imaging streams -- and a process that shares the GPU with
// a framework whose caching allocator has already reserved the HBM may find that cudaMalloc simply fails.  The handle-based
// muser_histogram needs a muser_imager (whose creation allocates grids, tables and the per-grid minimum / maximum slots it
// reads its range from).  This file gives such callers the same histogram with NO handle and NO allocation: the per-grid
// minimum / maximum slots -- the only scratch the histogram kernel needs -- live in a file-scope __device__ array that is
// part of the library image.  Every GPU that loads libmuser.so holds that array (16 KB) until the process exits.
//
// Rules that follow from the shared array (also in include/muser.h):
//   - at most MUSER_STATIC_MAX_GRIDS images per call; more is refused with MUSER_EINVAL, nothing is enqueued;
//   - every call on a device uses the SAME slots.  A call clears the slots it is about to use (they keep the previous call's
//     minimum / maximum otherwise), so calls in one stream are safe back to back; two calls that can overlap on the GPU
//     (different streams, no event between them) race on the slots and give wrong histograms;
//   - the first call on each device looks up the array's device address (cudaGetSymbolAddress, which also makes the runtime
//     load this module on that device).  Make that first call during start-up, outside any stream capture; later calls on
//     that device only enqueue a memset and two kernels.
// The existing muser_histogram path is untouched; tests/test_zz_no_alloc.py checks this entry point against it bin by bin.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/muser.h"
#include "muser_internal.h"

namespace {

using muser::PeakSlot;
using muser::peak_ordered;
using muser::peak_unordered;

// The scratch.  In HOST code this name is only a stand-in the runtime maps to the real array: it is never passed to a
// kernel or to cudaMemsetAsync.  Host code uses the pointer that cudaGetSymbolAddress returned for the current device.
static __device__ __align__(256) PeakSlot g_static_slots[MUSER_STATIC_MAX_GRIDS];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
PeakSlot* g_slots_addr[kMaxDevices] = {};           // per device: device address of g_static_slots, nullptr = not set up yet

// Minimum and maximum of one image (blockIdx.y) into its slot; non-finite pixels are ignored.  Same keys as the imaging
// epilogue (PeakSlot): maxkey = ordered(value) << 32 | ~index, minkey = ~ordered(value), both combined with atomicMax.
__global__ void __launch_bounds__(256) k_static_minmax(const float* __restrict__ image, const size_t npix, PeakSlot* __restrict__ slots) {
    const int gi = blockIdx.y;
    const float* img = image + (size_t)gi * npix;
    unsigned long long best = 0ull;
    unsigned int lo = 0u;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < npix; i += (size_t)gridDim.x * 256) {
        const float v = img[i];
        if (isfinite(v)) {
            const unsigned int ord = peak_ordered(v);
            const unsigned long long key = ((unsigned long long)ord << 32) | (unsigned long long)(~(unsigned int)i);
            best = key > best ? key : best;
            lo = max(lo, ~ord);
        }
    }
#pragma unroll
    for (int d = 16; d; d >>= 1) {
        const unsigned long long ob = __shfl_xor_sync(0xFFFFFFFFu, best, d);
        best = ob > best ? ob : best;
        lo = max(lo, __shfl_xor_sync(0xFFFFFFFFu, lo, d));
    }
    __shared__ unsigned long long s_best[8];
    __shared__ unsigned int s_lo[8];
    if ((threadIdx.x & 31) == 0) { s_best[threadIdx.x >> 5] = best; s_lo[threadIdx.x >> 5] = lo; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { best = s_best[w] > best ? s_best[w] : best; lo = max(lo, s_lo[w]); }
        if (best) { atomicMax(&slots[gi].maxkey, best); atomicMax(&slots[gi].minkey, lo); }
    }
}

// The variant of k_histogram (muser_kernels.cu) that takes its range from the static slots: bin = floor((v - lo) * (nbins /
// (hi - lo))) in fp32 without contraction, hi itself in the last bin (reading R23).  An image without a finite pixel gives
// an empty histogram; a constant image puts every pixel into bin 0.
__global__ void __launch_bounds__(256) k_static_histogram(const float* __restrict__ image, const size_t npix, const int nbins,
                                                          const PeakSlot* __restrict__ slots, unsigned int* __restrict__ hist) {
    extern __shared__ unsigned int s_h[];
    const int gi = blockIdx.y;
    const PeakSlot slot = slots[gi];
    if (slot.maxkey == 0ull) return;                                     // no finite pixel (uniform over the CTA)
    for (int i = threadIdx.x; i < nbins; i += 256) s_h[i] = 0u;
    const float hi = peak_unordered((unsigned int)(slot.maxkey >> 32));
    const float lo = peak_unordered(~slot.minkey);
    const bool flat = !(lo < hi);
    const float scale = flat ? 0.0f : __fdiv_rn((float)nbins, __fsub_rn(hi, lo));
    __syncthreads();
    const float* img = image + (size_t)gi * npix;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < npix; i += (size_t)gridDim.x * 256) {
        const float v = img[i];
        if (v >= lo && v <= hi) {
            const int b = flat ? 0 : min((int)floorf(__fmul_rn(__fsub_rn(v, lo), scale)), nbins - 1);
            atomicAdd(&s_h[b], 1u);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nbins; i += 256)
        if (s_h[i]) atomicAdd(&hist[(size_t)gi * nbins + i], s_h[i]);
}

int refuse(char* err_out, int err_cap, int code, const char* what, const char* detail = "") {
    if (err_out && err_cap > 0) std::snprintf(err_out, (size_t)err_cap, "muser_histogram_static: %s%s", what, detail);
    return code;
}

// Once per device, with that device current: the device address of g_static_slots.
int slots_for_current_device(PeakSlot** out, char* err_out, int err_cap) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return refuse(err_out, err_cap, MUSER_ECUDA, "cudaGetDevice: ", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return refuse(err_out, err_cap, MUSER_EUNSUPPORTED, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_slots_addr[dev]) {
        PeakSlot* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_static_slots);
        if (e != cudaSuccess || !p)
            return refuse(err_out, err_cap, MUSER_ECUDA, "cudaGetSymbolAddress(g_static_slots): ", cudaGetErrorString(e));
        g_slots_addr[dev] = p;
    }
    *out = g_slots_addr[dev];
    return MUSER_OK;
}

}  // namespace

extern "C" int muser_histogram_static(const float* image, long long npix, int ngrids, int nbins, unsigned int* hist_out,
                                      muser_stream sv, char* err_out, int err_cap) {
    if (err_out && err_cap > 0) err_out[0] = '\0';
    if (!image || !hist_out) return refuse(err_out, err_cap, MUSER_EINVAL, "null pointer");
    if (npix < 1) return refuse(err_out, err_cap, MUSER_EINVAL, "npix must be >= 1");
    if (nbins < 1 || nbins > 8192) return refuse(err_out, err_cap, MUSER_EINVAL, "nbins must be in [1, 8192]");
    if (ngrids < 1) return refuse(err_out, err_cap, MUSER_EINVAL, "ngrids must be >= 1");
    if (ngrids > MUSER_STATIC_MAX_GRIDS) {
        char detail[96];
        std::snprintf(detail, sizeof detail, "%d images in one call, the static scratch holds MUSER_STATIC_MAX_GRIDS = %d; split the call",
                      ngrids, MUSER_STATIC_MAX_GRIDS);
        return refuse(err_out, err_cap, MUSER_EINVAL, detail);
    }
    PeakSlot* slots = nullptr;
    const int rc = slots_for_current_device(&slots, err_out, err_cap);
    if (rc != MUSER_OK) return rc;
    cudaStream_t s = (cudaStream_t)sv;
    // the slots keep the last call's minimum / maximum: clear the ones this call uses, in stream order
    cudaError_t e = cudaMemsetAsync(slots, 0, (size_t)ngrids * sizeof(PeakSlot), s);
    if (e == cudaSuccess) e = cudaMemsetAsync(hist_out, 0, (size_t)ngrids * (size_t)nbins * sizeof(unsigned int), s);
    if (e != cudaSuccess) return refuse(err_out, err_cap, MUSER_ECUDA, "cudaMemsetAsync: ", cudaGetErrorString(e));
    size_t bx = ((size_t)npix + 256 * 16 - 1) / (256 * 16);
    if (bx > 592) bx = 592;
    const dim3 grid((unsigned)bx, (unsigned)ngrids);
    k_static_minmax<<<grid, 256, 0, s>>>(image, (size_t)npix, slots);
    k_static_histogram<<<grid, 256, (size_t)nbins * sizeof(unsigned int), s>>>(image, (size_t)npix, nbins, slots, hist_out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return refuse(err_out, err_cap, MUSER_ECUDA, "kernel launch: ", cudaGetErrorString(e));
    return MUSER_OK;
}
