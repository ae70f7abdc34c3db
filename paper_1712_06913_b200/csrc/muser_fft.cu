// A5 (second half) + A6 fused: column pass of the 2-D inverse transform with the fftshift / checkerboard sign /
// grid correction / real-imaginary split in its epilogue.  The row pass (contiguous 1-D transforms along x) is
// cuFFT's; this kernel transforms the columns and writes the dirty image and the beam directly, so the transformed
// grid is never written back and k_correct never runs (16 B per cell instead of 32).
//   F[ky][x] = sum_y F1[y][x] * exp(+2 pi i ky y / ny)               (unnormalised inverse, Alg. 1 l.19)
//   dirty[yo][xo] = (-1)^(xo+yo) * Re F[(yo+ny/2)%ny][(xo+nx/2)%nx] * icx[xo] * icy[yo];  beam from Im F / alpha
// Stockham autosort FFT, radix 16 or 8 (registers, straight from global memory) followed by radix-4 stages in shared
// memory: ny = 16 * 4^m (256, 1024) or 8 * 4^m (512), one CTA of ny/2 threads per strip of 8 columns, a thread owns one butterfly of 4
// columns (one twiddle serves them).  Shared layout: float4 s[c/2][pad(i)] = (column c, column c+1), pad(i) = i + i/16,
// pitch = 2 (mod 8) float4: the 8-byte stores of the first stage and the 16-byte accesses of the radix-4 stages are
// bank-conflict free.
#include "muser_internal.h"

#include <cuda.h>

#include <algorithm>
#include <cstring>

namespace muser {

// columns per CTA: 8 (ny <= 1024: 64-byte row segments) or 4 (ny = 2048, 4096: the strip has to fit shared memory)
__host__ __device__ constexpr int fft_cols_per_cta(int N) { return N <= 1024 ? 8 : 4; }

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// 4-point inverse DFT (kernel exp(+2 pi i nk/4)): in place on (a, b, c, d) -> (X0, X1, X2, X3)
__device__ __forceinline__ void idft4(float2& a, float2& b, float2& c, float2& d) {
    const float2 s0 = make_float2(a.x + c.x, a.y + c.y), s1 = make_float2(a.x - c.x, a.y - c.y);
    const float2 s2 = make_float2(b.x + d.x, b.y + d.y), s3 = make_float2(b.x - d.x, b.y - d.y);   // i*s3 = (-s3.y, s3.x)
    a = make_float2(s0.x + s2.x, s0.y + s2.y);
    c = make_float2(s0.x - s2.x, s0.y - s2.y);
    b = make_float2(s1.x - s3.y, s1.y + s3.x);
    d = make_float2(s1.x + s3.y, s1.y - s3.x);
}

// 16-point inverse DFT in registers: in v[i] = x[i], out v[4 b + c] = X[b + 4 c]
__device__ __forceinline__ void idft16(float2 (&v)[16]) {
#pragma unroll
    for (int a = 0; a < 4; ++a) idft4(v[a], v[a + 4], v[a + 8], v[a + 12]);              // -> u[a][b] at v[a + 4 b]
    const float c1 = 0.92387953251128674f, s1 = 0.38268343236508977f, h = 0.70710678118654752f;
    v[1 + 4 * 1] = cmul(v[1 + 4 * 1], make_float2(c1, s1));
    v[2 + 4 * 1] = cmul(v[2 + 4 * 1], make_float2(h, h));
    v[3 + 4 * 1] = cmul(v[3 + 4 * 1], make_float2(s1, c1));
    v[1 + 4 * 2] = cmul(v[1 + 4 * 2], make_float2(h, h));
    v[2 + 4 * 2] = make_float2(-v[2 + 4 * 2].y, v[2 + 4 * 2].x);
    v[3 + 4 * 2] = cmul(v[3 + 4 * 2], make_float2(-h, h));
    v[1 + 4 * 3] = cmul(v[1 + 4 * 3], make_float2(s1, c1));
    v[2 + 4 * 3] = cmul(v[2 + 4 * 3], make_float2(-h, h));
    v[3 + 4 * 3] = cmul(v[3 + 4 * 3], make_float2(-c1, -s1));
#pragma unroll
    for (int b = 0; b < 4; ++b) idft4(v[4 * b], v[4 * b + 1], v[4 * b + 2], v[4 * b + 3]);
}
// 8-point inverse DFT in registers: in v[i] = x[i], out X[b] = v[2 b] + v[2 b + 1], X[b + 4] = v[2 b] - v[2 b + 1]
__device__ __forceinline__ void idft8_half(float2 (&v)[8]) {
    idft4(v[0], v[2], v[4], v[6]);
    idft4(v[1], v[3], v[5], v[7]);
    const float h = 0.70710678118654752f;
    v[3] = cmul(v[3], make_float2(h, h));
    v[5] = make_float2(-v[5].y, v[5].x);
    v[7] = cmul(v[7], make_float2(-h, h));
}

// ---- TMA staging of the column strip (TMA = 1): the strip of 8 columns x N rows (64 bytes per row) is fetched by N / 256
// cp.async.bulk.tensor.2d copies (box 8 columns x 256 rows) into a dense [N][8] float2 tile that ALIASES the stage
// buffers: every thread takes its first-stage inputs from it into registers, a barrier, then the stage-1 outputs
// overwrite it.  The load side then issues no per-lane global requests at all (the 64-byte row segments cost one L1
// request per 4 rows otherwise).
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t phase) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(phase) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}

// R8 (ny = 512, 1024): after the first stage the remaining factor 64 is done as TWO radix-8 stages instead of three radix-4
// ones -- one shared-memory round trip less (the kernel is bound by its shared-memory traffic); a thread then owns one radix-8
// butterfly of one column pair; tw8[(7 stage + i - 1) (N/8) + j] = exp(+2 pi i * i * (j mod Ns) / (8 Ns)).
template <int N, int TMA, int R8>
__global__ void __launch_bounds__((N / 4) * (fft_cols_per_cta(N) / 4), N >= 4096 ? 1 : (N >= 1024 ? 2 : (N == 512 ? 4 : 8))) k_fft_cols_correct(const __grid_constant__ CUtensorMap tmap,
                                                                               const int nx, const float2* __restrict__ F1,
                                                                               const float2* __restrict__ tw,
                                                                               const float* __restrict__ icx,
                                                                               const float* __restrict__ icy,
                                                                               const Stats* __restrict__ stats,
                                                                               float* __restrict__ dirty, float* __restrict__ psf,
                                                                               PeakSlot* __restrict__ peaks, const int grid0) {
    constexpr int T = N / 4;                   // butterflies per column and stage
    constexpr int kFftC = fft_cols_per_cta(N), NH = kFftC / 4, CS = kFftC == 8 ? 3 : 2;
    constexpr int NT = T * NH;                 // threads: thread (j, half) owns butterfly j of columns 4 half .. 4 half + 3
    constexpr int PITCH = N + N / 16 + 2;      // float4 per column pair, = 2 (mod 8)
    extern __shared__ __align__(128) float4 sm[];
    const int tid = threadIdx.x;
    const int sx0 = blockIdx.x * kFftC;        // source columns sx0 .. sx0 + 7
    const int gi = grid0 + (int)blockIdx.y;
    const size_t gbase = (size_t)gi * N * nx;
    auto pad = [](int i) { return i + (i >> 4); };

    constexpr int R1 = (N == 256 || N == 1024 || N == 4096) ? 16 : 8;                      // radix of the first stage
    if constexpr (TMA != 0) {
        __shared__ __align__(8) uint64_t bar;
        constexpr int TPT = (N / R1) * kFftC / NT;                                         // first-stage tasks per thread (1 or 2)
        if (tid == 0) {
            mbar_init(&bar, 1);
            mbar_expect_tx(&bar, (uint32_t)(N * kFftC * sizeof(float2)));
#pragma unroll
            for (int b = 0; b < N / 256; ++b)
                tma_load_2d(reinterpret_cast<float2*>(sm) + b * 256 * kFftC, &tmap, 2 * sx0, gi * N + b * 256, &bar);
        }
        __syncthreads();                                                                   // the barrier is initialised
        mbar_wait(&bar, 0);
        const float2* raw = reinterpret_cast<const float2*>(sm);                           // [N][8]
        float2 v[TPT][R1];
#pragma unroll
        for (int t = 0; t < TPT; ++t) {
            const int task = tid + t * NT, c = task & (kFftC - 1), j = task >> CS;
#pragma unroll
            for (int i = 0; i < R1; ++i) v[t][i] = raw[(j + i * (N / R1)) * kFftC + c];
        }
        __syncthreads();                                                                   // everyone holds its inputs: the tile may be overwritten
#pragma unroll
        for (int t = 0; t < TPT; ++t) {
            const int task = tid + t * NT, c = task & (kFftC - 1), j = task >> CS;
            float2* dst = reinterpret_cast<float2*>(sm + (c >> 1) * PITCH) + (c & 1);
            if constexpr (R1 == 16) {
                idft16(v[t]);
#pragma unroll
                for (int b = 0; b < 4; ++b)
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) dst[2 * pad(16 * j + b + 4 * cc)] = v[t][4 * b + cc];
            } else {
                idft8_half(v[t]);
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const float2 p0 = v[t][2 * b], p1 = v[t][2 * b + 1];
                    dst[2 * pad(8 * j + b)] = make_float2(p0.x + p1.x, p0.y + p1.y);
                    dst[2 * pad(8 * j + b + 4)] = make_float2(p0.x - p1.x, p0.y - p1.y);
                }
            }
        }
    } else if (R1 == 8) {
        // ---- stage 1: radix 8, Ns = 1, straight from global memory; outputs y[8 j + i]
        for (int task = tid; task < (N / 8) * kFftC; task += NT) {
            const int c = task & (kFftC - 1), j = task >> CS;
            float2 v[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = __ldg(F1 + gbase + (size_t)(j + i * (N / 8)) * nx + sx0 + c);
            // n = a + 2 m (a = 0..1, m = 0..3), k = b + 4 c' (b = 0..3, c' = 0..1): X[b + 4 c'] = sum_a W2^{a c'} W8^{a b} sum_m x[a + 2 m] W4^{m b}
            idft4(v[0], v[2], v[4], v[6]);                                                // a = 0: u[0][b] at v[2 b]
            idft4(v[1], v[3], v[5], v[7]);                                                // a = 1: u[1][b] at v[2 b + 1]
            const float h = 0.70710678118654752f;
            v[3] = cmul(v[3], make_float2(h, h));                                         // W8^1
            v[5] = make_float2(-v[5].y, v[5].x);                                          // W8^2 = i
            v[7] = cmul(v[7], make_float2(-h, h));                                        // W8^3
            float2* dst = reinterpret_cast<float2*>(sm + (c >> 1) * PITCH) + (c & 1);
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const float2 p0 = v[2 * b], p1 = v[2 * b + 1];
                dst[2 * pad(8 * j + b)] = make_float2(p0.x + p1.x, p0.y + p1.y);
                dst[2 * pad(8 * j + b + 4)] = make_float2(p0.x - p1.x, p0.y - p1.y);
            }
        }
    } else
    // ---- stage 1: radix 16, Ns = 1, straight from global memory; outputs y[16 j + i]
    for (int task = tid; task < (N / 16) * kFftC; task += NT) {
        const int c = task & (kFftC - 1), j = task >> CS;
        float2 v[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = __ldg(F1 + gbase + (size_t)(j + i * (N / 16)) * nx + sx0 + c);
        // n = a + 4 m: inner DFTs over m for every a
#pragma unroll
        for (int a = 0; a < 4; ++a) idft4(v[a], v[a + 4], v[a + 8], v[a + 12]);          // -> u[a][b] at v[a + 4 b]
        // twiddle u[a][b] *= exp(+2 pi i a b / 16)
        const float c1 = 0.92387953251128674f, s1 = 0.38268343236508977f, h = 0.70710678118654752f;
        v[1 + 4 * 1] = cmul(v[1 + 4 * 1], make_float2(c1, s1));
        v[2 + 4 * 1] = cmul(v[2 + 4 * 1], make_float2(h, h));
        v[3 + 4 * 1] = cmul(v[3 + 4 * 1], make_float2(s1, c1));
        v[1 + 4 * 2] = cmul(v[1 + 4 * 2], make_float2(h, h));
        v[2 + 4 * 2] = make_float2(-v[2 + 4 * 2].y, v[2 + 4 * 2].x);                     // * i
        v[3 + 4 * 2] = cmul(v[3 + 4 * 2], make_float2(-h, h));
        v[1 + 4 * 3] = cmul(v[1 + 4 * 3], make_float2(s1, c1));
        v[2 + 4 * 3] = cmul(v[2 + 4 * 3], make_float2(-h, h));
        v[3 + 4 * 3] = cmul(v[3 + 4 * 3], make_float2(-c1, -s1));                        // exp(2 pi i 9/16)
        // outer DFTs over a for every b: X[b + 4 c'] = sum_a W4^{a c'} u[a][b]
#pragma unroll
        for (int b = 0; b < 4; ++b) idft4(v[4 * b], v[4 * b + 1], v[4 * b + 2], v[4 * b + 3]);   // -> X[b + 4 c'] at v[4 b + c']
        float2* dst = reinterpret_cast<float2*>(sm + (c >> 1) * PITCH) + (c & 1);
#pragma unroll
        for (int b = 0; b < 4; ++b)
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) dst[2 * pad(16 * j + b + 4 * cc)] = v[4 * b + cc];
    }
    __syncthreads();

    if constexpr (R8 != 0) {
        constexpr int T8 = N / 8;
        const int j = tid >> 2, cp = tid & 3;                                              // butterfly j of column pair cp
        float4* col = sm + cp * PITCH;
        const float2* twp = tw + j;
        float2 a[8], b[8];                                                                 // the two columns of the pair
#pragma unroll 1
        for (int Ns = R1; Ns < N; Ns *= 8, twp += 7 * T8) {
            const int k = j & (Ns - 1);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float4 q = col[pad(j + i * T8)];
                a[i] = make_float2(q.x, q.y); b[i] = make_float2(q.z, q.w);
            }
#pragma unroll
            for (int i = 1; i < 8; ++i) {
                const float2 w = __ldg(twp + (i - 1) * T8);
                a[i] = cmul(a[i], w); b[i] = cmul(b[i], w);
            }
            idft8_half(a); idft8_half(b);                                                  // X[m] = v[2m] + v[2m+1], X[m+4] = v[2m] - v[2m+1]
            if (Ns * 8 == N) break;                                                        // results stay in registers
            __syncthreads();
            const int o = (j - k) * 8 + k;
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                col[pad(o + m * Ns)] = make_float4(a[2 * m].x + a[2 * m + 1].x, a[2 * m].y + a[2 * m + 1].y,
                                                   b[2 * m].x + b[2 * m + 1].x, b[2 * m].y + b[2 * m + 1].y);
                col[pad(o + (m + 4) * Ns)] = make_float4(a[2 * m].x - a[2 * m + 1].x, a[2 * m].y - a[2 * m + 1].y,
                                                         b[2 * m].x - b[2 * m + 1].x, b[2 * m].y - b[2 * m + 1].y);
            }
            __syncthreads();
        }
        // epilogue: F[ky = j + m T8][sx0 + 2 cp + {0, 1}]; the four lanes of a butterfly write one 32-byte sector per row
        const int x0 = (sx0 + (nx >> 1)) % nx + 2 * cp;
        const float2 cx = *reinterpret_cast<const float2*>(icx + x0);
        const float ia = stats->inv_alpha;
        const size_t obase = (size_t)gi * N * nx;
        unsigned long long best = 0ull;
        unsigned int lowest = 0u;
#pragma unroll
        for (int m = 0; m < 8; ++m) {
            const int h2 = m & 3;
            const float2 fa = m < 4 ? make_float2(a[2 * h2].x + a[2 * h2 + 1].x, a[2 * h2].y + a[2 * h2 + 1].y)
                                    : make_float2(a[2 * h2].x - a[2 * h2 + 1].x, a[2 * h2].y - a[2 * h2 + 1].y);
            const float2 fb = m < 4 ? make_float2(b[2 * h2].x + b[2 * h2 + 1].x, b[2 * h2].y + b[2 * h2 + 1].y)
                                    : make_float2(b[2 * h2].x - b[2 * h2 + 1].x, b[2 * h2].y - b[2 * h2 + 1].y);
            const int ky = j + m * T8, y = (ky + N / 2) & (N - 1);
            const float cy = (y & 1) ? -icy[y] : icy[y];                                   // x0 is even: sign = (-1)^y * (+, -)
            const float m0 = cx.x * cy, m1 = -cx.y * cy;
            const size_t o = obase + (size_t)y * nx + x0;
            if (dirty) {
                const float2 d = make_float2(fa.x * m0, fb.x * m1);
                *reinterpret_cast<float2*>(dirty + o) = d;
                if (peaks) {
                    const unsigned int base = (unsigned int)(y * nx + x0);
                    const float dv[2] = {d.x, d.y};
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const unsigned int ord = peak_ordered(dv[c]);
                        const unsigned long long key = ((unsigned long long)ord << 32) | (unsigned long long)(~(base + c));
                        best = key > best ? key : best;
                        lowest = max(lowest, ~ord);
                    }
                }
            }
            if (psf) *reinterpret_cast<float2*>(psf + o) = make_float2(fa.y * m0 * ia, fb.y * m1 * ia);
        }
        if (dirty && peaks) {
            for (int o = 16; o > 0; o >>= 1) {
                const unsigned long long ob = __shfl_xor_sync(0xffffffffu, best, o);
                best = ob > best ? ob : best;
                lowest = max(lowest, __shfl_xor_sync(0xffffffffu, lowest, o));
            }
            if ((tid & 31) == 0) { atomicMax(&peaks[gi].maxkey, best); atomicMax(&peaks[gi].minkey, lowest); }
        }
        return;
    }

    // ---- radix-4 stages in shared memory: Ns = 16, 64, ... ; the last one (Ns = N/4) ends in registers.
    // tw[(3 stage + i - 1) T + j] = exp(+2 pi i * i * (j mod Ns) / (4 Ns)): per-stage tables in butterfly order.
    const int j = tid / NH, half = tid - j * NH;
    float2 v[4][4];
    const float2* twp = tw + j;
    float4* colp = sm + 2 * half * PITCH;      // this thread's two column pairs
#pragma unroll 1
    for (int Ns = R1; Ns < N; Ns *= 4, twp += 3 * T) {
        const int k = j & (Ns - 1);
        const float2 w1 = __ldg(twp), w2 = __ldg(twp + T), w3 = __ldg(twp + 2 * T);
#pragma unroll
        for (int cp = 0; cp < 2; ++cp) {
            const float4* src = colp + cp * PITCH;
            const float4 q0 = src[pad(j)], q1 = src[pad(j + T)], q2 = src[pad(j + 2 * T)], q3 = src[pad(j + 3 * T)];
            v[2 * cp][0] = make_float2(q0.x, q0.y); v[2 * cp + 1][0] = make_float2(q0.z, q0.w);
            v[2 * cp][1] = cmul(make_float2(q1.x, q1.y), w1); v[2 * cp + 1][1] = cmul(make_float2(q1.z, q1.w), w1);
            v[2 * cp][2] = cmul(make_float2(q2.x, q2.y), w2); v[2 * cp + 1][2] = cmul(make_float2(q2.z, q2.w), w2);
            v[2 * cp][3] = cmul(make_float2(q3.x, q3.y), w3); v[2 * cp + 1][3] = cmul(make_float2(q3.z, q3.w), w3);
            idft4(v[2 * cp][0], v[2 * cp][1], v[2 * cp][2], v[2 * cp][3]);
            idft4(v[2 * cp + 1][0], v[2 * cp + 1][1], v[2 * cp + 1][2], v[2 * cp + 1][3]);
        }
        if (Ns * 4 == N) break;                                                           // results stay in registers
        __syncthreads();
        const int o = (j - k) * 4 + k;
#pragma unroll
        for (int cp = 0; cp < 2; ++cp) {
            float4* dst = colp + cp * PITCH;
#pragma unroll
            for (int i = 0; i < 4; ++i)
                dst[pad(o + i * Ns)] = make_float4(v[2 * cp][i].x, v[2 * cp][i].y, v[2 * cp + 1][i].x, v[2 * cp + 1][i].y);
        }
        __syncthreads();
    }

    // ---- epilogue: v[c][i] = F[ky = j + i T][sx0 + 4 half + c].  The two lanes of a pair (same j) write the two
    // 16-byte halves of one 32-byte sector of each output row.
    const int x0 = (sx0 + (nx >> 1)) % nx + 4 * half;                                      // output columns x0 .. x0 + 3
    const float4 cx = *reinterpret_cast<const float4*>(icx + x0);
    const float ia = stats->inv_alpha;
    const size_t obase = (size_t)gi * N * nx;
    unsigned long long best = 0ull;                                                        // NEXT-4 peak search (see PeakSlot)
    unsigned int lowest = 0u;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int ky = j + i * T, y = (ky + N / 2) & (N - 1);
        const float cy = (y & 1) ? -icy[y] : icy[y];                                       // x0 is a multiple of 4: sign = (-1)^y * (+,-,+,-)
        const float m0 = cx.x * cy, m1 = -cx.y * cy, m2 = cx.z * cy, m3 = -cx.w * cy;
        const size_t o = obase + (size_t)y * nx + x0;
        if (dirty) {
            const float4 d = make_float4(v[0][i].x * m0, v[1][i].x * m1, v[2][i].x * m2, v[3][i].x * m3);
            *reinterpret_cast<float4*>(dirty + o) = d;
            if (peaks) {
                const unsigned int base = (unsigned int)(y * nx + x0);
                const float dv[4] = {d.x, d.y, d.z, d.w};
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const unsigned int ord = peak_ordered(dv[c]);
                    const unsigned long long key = ((unsigned long long)ord << 32) | (unsigned long long)(~(base + c));
                    best = key > best ? key : best;
                    lowest = max(lowest, ~ord);
                }
            }
        }
        if (psf) *reinterpret_cast<float4*>(psf + o) = make_float4(v[0][i].y * m0 * ia, v[1][i].y * m1 * ia, v[2][i].y * m2 * ia, v[3][i].y * m3 * ia);
    }
    if (dirty && peaks) {                                                                  // one atomic pair per warp
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long ob = __shfl_xor_sync(0xffffffffu, best, o);
            best = ob > best ? ob : best;
            lowest = max(lowest, __shfl_xor_sync(0xffffffffu, lowest, o));
        }
        if ((tid & 31) == 0) { atomicMax(&peaks[gi].maxkey, best); atomicMax(&peaks[gi].minkey, lowest); }
    }
}

// ------------------------------------------------------------------------------------------------- row pass
// A5 (first half) on the STORED HALF-PLANE.  G and Gw are Hermitian about the centre cell [ny/2][nx/2] (every
// visibility is gridded with its conjugate; "half the grid (as the data is Hermitian)"), and the owner
// gridder stores rows ny/2 .. ny-1 only.  For a stored row iy the row transforms
//     a[kx] = sum_ix G [iy][ix] exp(+2 pi i ix kx / nx),      b[kx] = alpha * sum_ix Gw[iy][ix] exp(+2 pi i ix kx / nx)
// give BOTH rows of the column pass's input Z = rowIFFT(G + i alpha Gw):
//     Z[iy][kx] = a + i b,        Z[ny - iy][kx] = conj(a) + i conj(b)          (row 0 has no mirror and is zero),
// because G[ny-iy][nx-ix] = conj G[iy][ix] (column 0 and row 0 are empty by the drop rule R5).  So the lower half-plane
// is never read (nor written by the gridder), and H = G + i alpha Gw is never materialised.  In 2-D mode Gw is real:
// two rows are packed into one complex transform, P = FFT(alpha (B1 + i B2)), and separated with
// b1 = (P[k] + conj P[-k]) / 2, b2 = (P[k] - conj P[-k]) / (2i): 3 transforms per 2 stored rows.
// Same Stockham scheme as the column pass: radix-16 / radix-8 first stage in registers straight from global memory,
// radix-4 stages in shared memory on float4 = two sequences (padded, conflict-free), last stage ends in registers.
template <int N, int WMODE>
struct RowCfg {
    static constexpr int ROWS = WMODE ? (N <= 2048 ? 2 : 1) : (N <= 1024 ? 4 : 2);   // stored rows per CTA pass
    static constexpr int NSEQ = WMODE ? 2 * ROWS : ROWS + ROWS / 2;                 // complex sequences transformed
    static constexpr int NP = (NSEQ + 1) / 2;                                       // float4 pairs
    static constexpr int T = N / 4;                                                 // threads = radix-4 butterflies
    static constexpr int PITCH = N + N / 16 + 2;
    static constexpr int R1 = (N == 64 || N == 256 || N == 1024 || N == 4096) ? 16 : 8;
    static constexpr size_t SMEM = (size_t)NP * PITCH * sizeof(float4);
};

// predicated read-only loads (no branch: the 8 or 16 loads of a first-stage butterfly stay in flight together)
__device__ __forceinline__ float2 ldg_f2_if(const float2* p, const bool ok) {
    float2 v;
    asm("{\n.reg .pred q;\nsetp.ne.s32 q, %3, 0;\nmov.f32 %0, 0f00000000;\nmov.f32 %1, 0f00000000;\n@q ld.global.nc.v2.f32 {%0, %1}, [%2];\n}"
        : "=f"(v.x), "=f"(v.y) : "l"(p), "r"((int)ok));
    return v;
}
__device__ __forceinline__ float ldg_f_if(const float* p, const bool ok) {
    float v;
    asm("{\n.reg .pred q;\nsetp.ne.s32 q, %2, 0;\nmov.f32 %0, 0f00000000;\n@q ld.global.nc.f32 %0, [%1];\n}" : "=f"(v) : "l"(p), "r"((int)ok));
    return v;
}

template <int N, int WMODE, int UNIFORM>
__global__ void __launch_bounds__(N / 4, N == 1024 ? 3 : (N == 512 ? 6 : 1)) k_fft_rows_half(const int ny, const int grp0, const int ngroups, const float2* __restrict__ G,
                                                         const float* __restrict__ Gw, const int* __restrict__ cnt,
                                                         const float2* __restrict__ tw, Stats* __restrict__ stats,
                                                         float2* __restrict__ Z, const uint32_t* __restrict__ valid,
                                                         const int otx) {
    using C = RowCfg<N, WMODE>;
    constexpr int T = C::T, PITCH = C::PITCH, R1 = C::R1, ROWS = C::ROWS, NSEQ = C::NSEQ, NP = C::NP;
    extern __shared__ __align__(16) float4 sm[];
    const int tid = threadIdx.x;
    auto pad = [](int i) { return i + (i >> 4); };
    // alpha balances G against Gw in the packed transform (power of two: exact); same rule as k_pack
    float al = 1.0f;
    {
        const double v2 = stats->sum_val2, w2 = stats->sum_wt2;
        if (v2 > 0.0 && w2 > 0.0) al = exp2f(rintf(0.5f * log2f((float)(v2 / w2))));
        al = fminf(fmaxf(al, 9.5367431640625e-07f), 1048576.0f);
        if (blockIdx.x == 0 && tid == 0) { stats->alpha = al; stats->inv_alpha = 1.0f / al; }
    }
    const int hy = ny >> 1, gpg = hy / ROWS;                       // row groups per grid
    // tile flags of a group's row of tiles, one per lane and word of 32 tiles (fetched one group ahead)
    uint32_t nflag[3] = {0u, 0u, 0u};
    auto load_flags = [&](const int grp) {
        if (grp >= ngroups) return;
        const int gi = grp / gpg, ty = ((grp - gi * gpg) * ROWS) / kTile;
        const uint32_t* vrow = valid + ((size_t)gi * (size_t)((hy + kTile - 1) / kTile) + ty) * otx;
#pragma unroll
        for (int w = 0; w < 3; ++w) {
            const int t = 32 * w + (tid & 31);
            nflag[w] = t < otx ? __ldg(vrow + t) : 0u;
        }
    };
    if (valid) load_flags(grp0 + (int)blockIdx.x);
    for (int grp = grp0 + (int)blockIdx.x; grp < ngroups; grp += gridDim.x) {       // groups [grp0, ngroups): the grids of this sub-batch
        const int gi = grp / gpg, iy0 = hy + (grp - gi * gpg) * ROWS;
        const size_t gbase = (size_t)gi * ny * N;
        // tile flags of this row of 64 x 32 tiles (the rows of a group lie in one tile row): a tile that has not been written
        // since the last reset stands for zeros and is not loaded (`valid` == nullptr: the grids are dense)
        uint32_t vm[3] = {0xffffffffu, 0xffffffffu, 0xffffffffu};
        if (valid) {
#pragma unroll
            for (int w = 0; w < 3; ++w) vm[w] = __ballot_sync(__activemask(), nflag[w] != 0u);   // (N = 64: a CTA of 16 threads)
            load_flags(grp + (int)gridDim.x);                      // the next group's flags: in flight during this group
        }
        if (valid && (vm[0] | vm[1] | vm[2]) == 0u) {              // no tile of this row of tiles has been written: zeros
            for (int r = 0; r < ROWS; ++r) {
                const int iy = iy0 + r;
                for (int kx = tid; kx < N; kx += T) {
                    Z[gbase + (size_t)iy * N + kx] = make_float2(0.f, 0.f);
                    Z[gbase + (size_t)(iy == hy ? 0 : ny - iy) * N + kx] = make_float2(0.f, 0.f);
                }
            }
            continue;
        }
        auto live = [&](int x) -> bool {                           // column x lies in a written tile
            const int t = (x + kOwTileW / 2) / kOwTileW;
            return ((t < 32 ? vm[0] : (t < 64 ? vm[1] : vm[2])) >> (t & 31)) & 1u;
        };
        __syncthreads();                                           // the previous group is done with the shared buffers
        // ---- stage 1: radix R1 straight from global memory; sequence s, butterfly j -> y_s[R1 j + i]
        for (int task = tid; task < NSEQ * (N / R1); task += T) {
            const int s = task / (N / R1), j = task - s * (N / R1);
            float2 v[R1];
            // wgtGrid_kernel (Alg. 1 l.1-16) in uniform mode: a cell is multiplied by 1 / count where
            // count != 0, here as the cell is loaded
            auto wgt = [&](size_t cell) -> float {
                if constexpr (UNIFORM == 0) return 1.0f;
                const int c = __ldg(cnt + cell);
                return c ? 1.0f / (float)c : 1.0f;
            };
            if (WMODE) {
                const size_t row = gbase + (size_t)(iy0 + (s >> 1)) * N;
                if (s & 1) {
                    const float2* src = reinterpret_cast<const float2*>(Gw) + row;
#pragma unroll
                    for (int i = 0; i < R1; ++i) {
                        const float2 q = ldg_f2_if(src + j + i * (N / R1), live(j + i * (N / R1)));
                        const float u = al * wgt(row + j + i * (N / R1));
                        v[i] = make_float2(u * q.x, u * q.y);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < R1; ++i) {
                        const float2 q = ldg_f2_if(G + row + j + i * (N / R1), live(j + i * (N / R1)));
                        const float u = wgt(row + j + i * (N / R1));
                        v[i] = make_float2(u * q.x, u * q.y);
                    }
                }
            } else if (s < ROWS) {
                const size_t row = gbase + (size_t)(iy0 + s) * N;
#pragma unroll
                for (int i = 0; i < R1; ++i) {
                    const float2 q = ldg_f2_if(G + row + j + i * (N / R1), live(j + i * (N / R1)));
                    const float u = wgt(row + j + i * (N / R1));
                    v[i] = make_float2(u * q.x, u * q.y);
                }
            } else {
                const size_t row = gbase + (size_t)(iy0 + 2 * (s - ROWS)) * N;
#pragma unroll
                for (int i = 0; i < R1; ++i) {
                    const size_t c0 = row + j + i * (N / R1);
                    const bool ok = live(j + i * (N / R1));
                    v[i] = make_float2(al * wgt(c0) * ldg_f_if(Gw + c0, ok), al * wgt(c0 + N) * ldg_f_if(Gw + c0 + N, ok));
                }
            }
            float2* dst = reinterpret_cast<float2*>(sm + (s >> 1) * PITCH) + (s & 1);
            if constexpr (R1 == 16) {
                idft16(v);
#pragma unroll
                for (int b = 0; b < 4; ++b)
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) dst[2 * pad(16 * j + b + 4 * cc)] = v[4 * b + cc];
            } else {
                idft8_half(v);
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const float2 p0 = v[2 * b], p1 = v[2 * b + 1];
                    dst[2 * pad(8 * j + b)] = make_float2(p0.x + p1.x, p0.y + p1.y);
                    dst[2 * pad(8 * j + b + 4)] = make_float2(p0.x - p1.x, p0.y - p1.y);
                }
            }
        }
        __syncthreads();
        // ---- radix-4 stages in shared memory; the last one ends in registers: v[s][i] = X_s[j + i T]
        const int j = tid;
        float2 v[2 * NP][4];
        const float2* twp = tw + j;
#pragma unroll 1
        for (int Ns = R1; Ns < N; Ns *= 4, twp += 3 * T) {
            const int k = j & (Ns - 1);
            const float2 w1 = __ldg(twp), w2 = __ldg(twp + T), w3 = __ldg(twp + 2 * T);
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                const float4* src = sm + p * PITCH;
                const float4 q0 = src[pad(j)], q1 = src[pad(j + T)], q2 = src[pad(j + 2 * T)], q3 = src[pad(j + 3 * T)];
                v[2 * p][0] = make_float2(q0.x, q0.y); v[2 * p + 1][0] = make_float2(q0.z, q0.w);
                v[2 * p][1] = cmul(make_float2(q1.x, q1.y), w1); v[2 * p + 1][1] = cmul(make_float2(q1.z, q1.w), w1);
                v[2 * p][2] = cmul(make_float2(q2.x, q2.y), w2); v[2 * p + 1][2] = cmul(make_float2(q2.z, q2.w), w2);
                v[2 * p][3] = cmul(make_float2(q3.x, q3.y), w3); v[2 * p + 1][3] = cmul(make_float2(q3.z, q3.w), w3);
                idft4(v[2 * p][0], v[2 * p][1], v[2 * p][2], v[2 * p][3]);
                idft4(v[2 * p + 1][0], v[2 * p + 1][1], v[2 * p + 1][2], v[2 * p + 1][3]);
            }
            if (Ns * 4 == N) break;
            __syncthreads();
            const int o = (j - k) * 4 + k;
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                float4* dst = sm + p * PITCH;
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    dst[pad(o + i * Ns)] = make_float4(v[2 * p][i].x, v[2 * p][i].y, v[2 * p + 1][i].x, v[2 * p + 1][i].y);
            }
            __syncthreads();
        }
        // ---- epilogue: both rows of Z per stored row
        if (!WMODE) {
            // the packed weight transforms go through shared memory once more: every thread needs P[N - kx]
            __syncthreads();
            float4* pp = sm + (NP - 1) * PITCH;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float2 p0 = v[ROWS][i], p1 = (ROWS == 4) ? v[ROWS + 1][i] : make_float2(0.f, 0.f);
                pp[pad(j + i * T)] = make_float4(p0.x, p0.y, p1.x, p1.y);
            }
            __syncthreads();
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int kx = j + i * T;
            float2 b[ROWS];
            if (WMODE) {
#pragma unroll
                for (int r = 0; r < ROWS; ++r) b[r] = v[2 * r + 1][i];
            } else {
                const float4 pm = sm[(NP - 1) * PITCH + pad((N - kx) & (N - 1))];
#pragma unroll
                for (int q = 0; q < ROWS / 2; ++q) {
                    const float2 P = v[ROWS + q][i];
                    const float2 Pc = q ? make_float2(pm.z, -pm.w) : make_float2(pm.x, -pm.y);      // conj P[-k]
                    b[2 * q] = make_float2(0.5f * (P.x + Pc.x), 0.5f * (P.y + Pc.y));
                    b[2 * q + 1] = make_float2(0.5f * (P.y - Pc.y), -0.5f * (P.x - Pc.x));         // (P - Pc) / (2i)
                }
            }
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const float2 a = WMODE ? v[2 * r][i] : v[r][i];
                const int iy = iy0 + r;
                Z[gbase + (size_t)iy * N + kx] = make_float2(a.x - b[r].y, a.y + b[r].x);
                const float2 lo = (iy == hy) ? make_float2(0.f, 0.f) : make_float2(a.x + b[r].y, b[r].x - a.y);
                Z[gbase + (size_t)(iy == hy ? 0 : ny - iy) * N + kx] = lo;
            }
        }
    }
}

static size_t fft_smem_bytes(int N) { return (size_t)(fft_cols_per_cta(N) / 2) * (N + N / 16 + 2) * sizeof(float4); }

bool fft_cols_supported(int nx, int ny) { return (ny == 256 || ny == 512 || ny == 1024 || ny == 2048 || ny == 4096) && (nx % 16) == 0; }
int fft_cols_first_radix(int ny) { return (ny == 256 || ny == 1024 || ny == 4096) ? 16 : 8; }

cudaError_t fft_cols_setup() {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<256, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(256)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<512, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(512)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<1024, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(1024)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<256, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(256)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<512, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(512)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<1024, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(1024)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<2048, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(2048)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<2048, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(2048)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<4096, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(4096)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<4096, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(4096)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<512, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(512)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<1024, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(1024)))) return e;
    return cudaSuccess;
}

// Tensor map of the column pass's input F1 [ngrids * ny][nx] float2 seen as fp32 [rows][2 nx], box = 16 floats (8 columns)
// x 256 rows, no swizzle.  `map128` = 128 bytes, 64-byte aligned.  The driver entry point is looked up at run time (the
// library does not link libcuda).  Returns false when the map cannot be made (the per-lane load path is used then).
bool fft_cols_make_tmap(void* map128, const float2* F1, int nx, int ny, int ngrids) {
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
            qres != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            return false;
        }
        encode = reinterpret_cast<EncodeFn>(fn);
    }
    const unsigned long long rows = (unsigned long long)ngrids * ny;
    if (ny % 256 != 0 || rows >= (1ull << 32)) return false;
    const cuuint64_t dims[2] = {(cuuint64_t)2 * nx, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)nx * sizeof(float2)};
    const cuuint32_t box[2] = {(cuuint32_t)(2 * fft_cols_per_cta(ny)), 256};
    const cuuint32_t estr[2] = {1, 1};
    return encode(reinterpret_cast<CUtensorMap*>(map128), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float2*>(F1), dims, strides,
                  box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int N, int WMODE>
static cudaError_t launch_rows_t(const Geom& g, const float2* G, const float* Gw, const int* cnt, const float2* tw, Stats* stats,
                                 float2* Z, const uint32_t* valid, int grid_begin, int grid_count, int num_sms, cudaStream_t s) {
    using C = RowCfg<N, WMODE>;
    const int gpg = (g.ny / 2) / C::ROWS;
    const int grp0 = grid_begin * gpg, ngroups = (grid_begin + grid_count) * gpg, mine = grid_count * gpg;
    int per_sm = (int)(200 * 1024 / (C::SMEM + 1024));
    per_sm = per_sm < 1 ? 1 : (per_sm > 2048 / C::T ? 2048 / C::T : per_sm);
    const int blocks = mine < num_sms * per_sm ? mine : num_sms * per_sm;
    if (g.uniform && cnt) k_fft_rows_half<N, WMODE, 1><<<blocks, C::T, C::SMEM, s>>>(g.ny, grp0, ngroups, G, Gw, cnt, tw, stats, Z, valid, g.otx);
    else k_fft_rows_half<N, WMODE, 0><<<blocks, C::T, C::SMEM, s>>>(g.ny, grp0, ngroups, G, Gw, nullptr, tw, stats, Z, valid, g.otx);
    return cudaGetLastError();
}

template <int N>
static cudaError_t rows_setup_t() {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(k_fft_rows_half<N, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<N, 0>::SMEM))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_rows_half<N, 0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<N, 0>::SMEM))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_rows_half<N, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<N, 1>::SMEM))) return e;
    return cudaFuncSetAttribute(k_fft_rows_half<N, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<N, 1>::SMEM);
}

int fft_rows_first_radix(int nx) { return (nx == 64 || nx == 256 || nx == 1024 || nx == 4096) ? 16 : 8; }
int fft_rows_group(int nx, int wmode) { return wmode ? (nx <= 2048 ? 2 : 1) : (nx <= 1024 ? 4 : 2); }
bool fft_rows_supported(int nx, int ny, int wmode) {
    const bool pow2 = nx >= 64 && nx <= 4096 && (nx & (nx - 1)) == 0;
    return pow2 && ((ny / 2) % fft_rows_group(nx, wmode)) == 0;
}

cudaError_t fft_rows_setup() {
    cudaError_t e;
    if ((e = rows_setup_t<64>())) return e;
    if ((e = rows_setup_t<128>())) return e;
    if ((e = rows_setup_t<256>())) return e;
    if ((e = rows_setup_t<512>())) return e;
    if ((e = rows_setup_t<1024>())) return e;
    if ((e = rows_setup_t<2048>())) return e;
    return rows_setup_t<4096>();
}

cudaError_t launch_fft_rows_half(const Geom& g, const float2* G, const float* Gw, const int* cnt, const float2* tw,
                                 Stats* stats, float2* Z, const uint32_t* valid, int grid_begin, int grid_count, int num_sms,
                                 cudaStream_t s) {
    if (g.otx > 96) valid = nullptr;                                     // (image_impl made the grids dense: its rows_take_flags needs otx <= 96)
#define MUSER_ROWS_CASE(NN)                                                                                     \
    case NN:                                                                                                    \
        return g.wmode ? launch_rows_t<NN, 1>(g, G, Gw, cnt, tw, stats, Z, valid, grid_begin, grid_count, num_sms, s) \
                       : launch_rows_t<NN, 0>(g, G, Gw, cnt, tw, stats, Z, valid, grid_begin, grid_count, num_sms, s);
    switch (g.nx) {
        MUSER_ROWS_CASE(64) MUSER_ROWS_CASE(128) MUSER_ROWS_CASE(256) MUSER_ROWS_CASE(512) MUSER_ROWS_CASE(1024)
        MUSER_ROWS_CASE(2048) MUSER_ROWS_CASE(4096)
        default: return cudaErrorInvalidValue;
    }
#undef MUSER_ROWS_CASE
}

bool fft_cols_radix8(int ny) { return ny == 512 || ny == 1024; }

cudaError_t launch_fft_cols_correct(const Geom& g, const float2* F1, const float2* tw, const float2* tw8, const float* icx,
                                    const float* icy, const Stats* stats, float* dirty, float* psf, PeakSlot* peaks,
                                    const void* tmap128, int grid_begin, int grid_count, cudaStream_t s) {
    CUtensorMap map;
    memset(&map, 0, sizeof(map));
    if (tmap128) memcpy(&map, tmap128, sizeof(map));
    const int grid_end = grid_begin + grid_count;                        // the grids of this sub-batch
    for (int grid0 = grid_begin; grid0 < grid_end; grid0 += 65535) {     // gridDim.y holds at most 65535 grids
        const dim3 blocks((unsigned)(g.nx / fft_cols_per_cta(g.ny)), (unsigned)std::min(65535, grid_end - grid0));
#define MUSER_COLS_CASE(NN)                                                                                                   \
        if (tmap128) k_fft_cols_correct<NN, 1, 0><<<blocks, (NN / 4) * (fft_cols_per_cta(NN) / 4), fft_smem_bytes(NN), s>>>(map, g.nx, F1, tw, icx, icy, stats, dirty, psf, peaks, grid0); \
        else k_fft_cols_correct<NN, 0, 0><<<blocks, (NN / 4) * (fft_cols_per_cta(NN) / 4), fft_smem_bytes(NN), s>>>(map, g.nx, F1, tw, icx, icy, stats, dirty, psf, peaks, grid0);
        if (tmap128 && tw8 && g.ny == 512) {
            k_fft_cols_correct<512, 1, 1><<<blocks, 256, fft_smem_bytes(512), s>>>(map, g.nx, F1, tw8, icx, icy, stats, dirty, psf, peaks, grid0);
            continue;
        }
        if (tmap128 && tw8 && g.ny == 1024) {
            k_fft_cols_correct<1024, 1, 1><<<blocks, 512, fft_smem_bytes(1024), s>>>(map, g.nx, F1, tw8, icx, icy, stats, dirty, psf, peaks, grid0);
            continue;
        }
        if (g.ny == 256) { MUSER_COLS_CASE(256) }
        else if (g.ny == 512) { MUSER_COLS_CASE(512) }
        else if (g.ny == 1024) { MUSER_COLS_CASE(1024) }
        else if (g.ny == 2048) { MUSER_COLS_CASE(2048) }
        else { MUSER_COLS_CASE(4096) }
#undef MUSER_COLS_CASE
    }
    return cudaGetLastError();
}

}  // namespace muser
