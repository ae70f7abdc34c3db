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

namespace muser {

constexpr int kFftC = 8;                       // columns per CTA

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

template <int N>
__global__ void __launch_bounds__(N / 2, N == 1024 ? 2 : (N == 512 ? 4 : 8)) k_fft_cols_correct(const int nx, const float2* __restrict__ F1,
                                                                               const float2* __restrict__ tw,
                                                                               const float* __restrict__ icx,
                                                                               const float* __restrict__ icy,
                                                                               const Stats* __restrict__ stats,
                                                                               float* __restrict__ dirty, float* __restrict__ psf) {
    constexpr int T = N / 4;                   // butterflies per column and stage
    constexpr int NT = N / 2;                  // threads: thread (j, half) owns butterfly j of columns 4 half .. 4 half + 3
    constexpr int PITCH = N + N / 16 + 2;      // float4 per column pair, = 2 (mod 8)
    extern __shared__ __align__(16) float4 sm[];
    const int tid = threadIdx.x;
    const int sx0 = blockIdx.x * kFftC;        // source columns sx0 .. sx0 + 7
    const size_t gbase = (size_t)blockIdx.y * N * nx;
    auto pad = [](int i) { return i + (i >> 4); };

    constexpr int R1 = (N == 256 || N == 1024) ? 16 : 8;                                   // radix of the first stage
    if (R1 == 8) {
        // ---- stage 1: radix 8, Ns = 1, straight from global memory; outputs y[8 j + i]
        for (int task = tid; task < (N / 8) * kFftC; task += NT) {
            const int c = task & (kFftC - 1), j = task >> 3;
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
        const int c = task & (kFftC - 1), j = task >> 3;
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

    // ---- radix-4 stages in shared memory: Ns = 16, 64, ... ; the last one (Ns = N/4) ends in registers.
    // tw[(3 stage + i - 1) T + j] = exp(+2 pi i * i * (j mod Ns) / (4 Ns)): per-stage tables in butterfly order.
    const int j = tid >> 1, half = tid & 1;
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
    const size_t obase = (size_t)blockIdx.y * N * nx;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int ky = j + i * T, y = (ky + N / 2) & (N - 1);
        const float cy = (y & 1) ? -icy[y] : icy[y];                                       // x0 is a multiple of 4: sign = (-1)^y * (+,-,+,-)
        const float m0 = cx.x * cy, m1 = -cx.y * cy, m2 = cx.z * cy, m3 = -cx.w * cy;
        const size_t o = obase + (size_t)y * nx + x0;
        if (dirty) *reinterpret_cast<float4*>(dirty + o) = make_float4(v[0][i].x * m0, v[1][i].x * m1, v[2][i].x * m2, v[3][i].x * m3);
        if (psf) *reinterpret_cast<float4*>(psf + o) = make_float4(v[0][i].y * m0 * ia, v[1][i].y * m1 * ia, v[2][i].y * m2 * ia, v[3][i].y * m3 * ia);
    }
}

static size_t fft_smem_bytes(int N) { return (size_t)(kFftC / 2) * (N + N / 16 + 2) * sizeof(float4); }

bool fft_cols_supported(int nx, int ny) { return (ny == 256 || ny == 512 || ny == 1024) && (nx % 16) == 0; }
int fft_cols_first_radix(int ny) { return (ny == 256 || ny == 1024) ? 16 : 8; }

cudaError_t fft_cols_setup() {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(256)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(512)))) return e;
    if ((e = cudaFuncSetAttribute(k_fft_cols_correct<1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes(1024)))) return e;
    return cudaSuccess;
}

cudaError_t launch_fft_cols_correct(const Geom& g, const float2* F1, const float2* tw, const float* icx, const float* icy,
                                    const Stats* stats, float* dirty, float* psf, cudaStream_t s) {
    const dim3 blocks((unsigned)(g.nx / kFftC), (unsigned)g.ngrids);
    if (g.ny == 256)
        k_fft_cols_correct<256><<<blocks, 128, fft_smem_bytes(256), s>>>(g.nx, F1, tw, icx, icy, stats, dirty, psf);
    else if (g.ny == 512)
        k_fft_cols_correct<512><<<blocks, 256, fft_smem_bytes(512), s>>>(g.nx, F1, tw, icx, icy, stats, dirty, psf);
    else
        k_fft_cols_correct<1024><<<blocks, 512, fft_smem_bytes(1024), s>>>(g.nx, F1, tw, icx, icy, stats, dirty, psf);
    return cudaGetLastError();
}

}  // namespace muser
