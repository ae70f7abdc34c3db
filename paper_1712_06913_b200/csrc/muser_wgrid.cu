// W-projection gridder (A3: per-plane complex separable kernels, supports 1..31), sm_100a; also the 2-D gridder for supports
// other than 7 (one plane with a real table: the imaginary halves of the packed FMAs then carry zeros).
//
//   Kw1 k_wtile_items   work items: <= 4096 consecutive records of one 32x32 tile (bins are ordered tile-major,
//                       plane-minor, so an item is a sequence of plane segments)
//   Kw2 k_wgrid<SHP>    one kernel per window SHAPE (a range of supports; each has its own register budget and shared
//                       memory footprint); a kernel handles the plane segments of its supports.  Persistent CTAs pull
//                       items from a device counter.  Per item the CTA accumulates the tile plus its halo in 32-bit
//                       fixed-point shared memory (one region for all its plane segments of the item) and adds the
//                       touched cells of the stored half-plane to G and Gw once.  Per plane segment:
//                       the plane's complex table is staged in shared memory; the records are
//                       counting-sorted by 2x2-aligned window and conjugate flag; every warp streams an equal share
//                       of the sorted order and keeps the (S+1) x (S+1) window of a run of equal key in REGISTERS
//                       (lane = row slot x column strip, packed fp32x2 FMAs: 4 per cell and record, the row factor
//                       ky * (wt V) hoisted per lane); a run is merged into the region with native integer adds.
//                       Shapes: S <= 7, 9, 11, 13-15, 17, 19, 21-23 (2 to 18 cells per lane) and S = 25..31 (lane =
//                       footprint column, shared adds per cell: 0.7 % of cfg 5's work).
// Passages: PAPER.md:126 (w-projection), Alg. 1 l.18 PAPER.md:251 (gridding of the visibilities), :222 (half the grid).
// The kernels follow DESIGN.md R15 only through the tables they are given (muser_set_wplanes).
#include "muser_internal.h"

#include <cstring>

namespace muser {

namespace {

constexpr unsigned kAll = 0xffffffffu;
constexpr int kWgChunk = 4096;                   // records per item and per in-CTA sort (12-bit index + flag in 16 bits)
constexpr int kWgKeys = 512;                     // conjugate flag << 8 | (ly >> 1) << 4 | lx >> 1

// Window shapes.  SMIN..SMAX: supports handled; LR x CW x RP: lane layout of wg_stream; HMAX = (SMAX - 1) / 2; RR x PR:
// rows and pitch of the shared region: tile + halo + the whole lane layout of a window at the far corner (31 + HMAX +
// rows resp. columns of the layout), so that a run is merged without bounds tests; PT: table row pitch in entries
// (>= max(rows, columns) of the lane layout + 2); MINB: CTAs per SM the register budget is set for; MINSEG: plane
// segments with fewer records go to the direct kernel (shape 7: lane = footprint column, any support <= 31, tables read
// through L1, no per-segment set-up), which also takes every segment of supports 25..31; SUB: records of the shape per
// work-list entry -- an item with more of them is listed nsub times and each entry takes the k-th part of every segment
// (the big windows cost ~10x more per record than the small ones: equal-time work units).
constexpr int kWgShapes = 8;
template <int SHP> struct WgShape;
template <> struct WgShape<0> { static constexpr int SMIN = 1, SMAX = 7, LR = 4, CW = 2, RP = 1, SPLIT = 1, RR = 42, PR = 44, PT = 10, MINB = 4, MINSEG = 192, SUB = 4096; };
template <> struct WgShape<1> { static constexpr int SMIN = 9, SMAX = 9, LR = 6, CW = 2, RP = 2, SPLIT = 1, RR = 42, PR = 44, PT = 14, MINB = 3, MINSEG = 128, SUB = 4096; };
template <> struct WgShape<2> { static constexpr int SMIN = 11, SMAX = 11, LR = 4, CW = 3, RP = 2, SPLIT = 0, RR = 46, PR = 44, PT = 18, MINB = 3, MINSEG = 96, SUB = 2048; };
template <> struct WgShape<3> { static constexpr int SMIN = 13, SMAX = 15, LR = 4, CW = 4, RP = 2, SPLIT = 0, RR = 48, PR = 52, PT = 18, MINB = 3, MINSEG = 48, SUB = 1024; };
template <> struct WgShape<4> { static constexpr int SMIN = 17, SMAX = 17, LR = 5, CW = 4, RP = 3, SPLIT = 0, RR = 48, PR = 52, PT = 22, MINB = 2, MINSEG = 24, SUB = 1024; };
template <> struct WgShape<5> { static constexpr int SMIN = 19, SMAX = 19, LR = 4, CW = 5, RP = 3, SPLIT = 0, RR = 54, PR = 52, PT = 26, MINB = 2, MINSEG = 16, SUB = 512; };
template <> struct WgShape<6> { static constexpr int SMIN = 21, SMAX = 23, LR = 4, CW = 6, RP = 3, SPLIT = 0, RR = 56, PR = 60, PT = 26, MINB = 2, MINSEG = 8, SUB = 512; };
template <> struct WgShape<7> { static constexpr int SMIN = 1, SMAX = 31, LR = 0, CW = 0, RP = 0, SPLIT = 0, RR = 64, PR = 64, PT = 0, MINB = 3, MINSEG = 0, SUB = 256; };

__host__ __device__ __forceinline__ int wg_shape(int S) {
    return S <= 7 ? 0 : S == 9 ? 1 : S == 11 ? 2 : S <= 15 ? 3 : S == 17 ? 4 : S == 19 ? 5 : S <= 23 ? 6 : 7;
}
// the kernel (shape) that grids a plane segment of n records with support S
__host__ __device__ __forceinline__ int wg_route(int S, uint32_t n) {
    const int shp = wg_shape(S);
    const uint32_t minseg = shp == 0 ? WgShape<0>::MINSEG : shp == 1 ? WgShape<1>::MINSEG : shp == 2 ? WgShape<2>::MINSEG
                          : shp == 3 ? WgShape<3>::MINSEG : shp == 4 ? WgShape<4>::MINSEG : shp == 5 ? WgShape<5>::MINSEG
                          : shp == 6 ? WgShape<6>::MINSEG : 0u;
    return n < minseg ? 7 : shp;
}
__host__ __device__ __forceinline__ uint32_t wg_sub(int shp) {
    return shp == 0 ? WgShape<0>::SUB : shp == 1 ? WgShape<1>::SUB : shp == 2 ? WgShape<2>::SUB : shp == 3 ? WgShape<3>::SUB
         : shp == 4 ? WgShape<4>::SUB : shp == 5 ? WgShape<5>::SUB : shp == 6 ? WgShape<6>::SUB : WgShape<7>::SUB;
}

__device__ __forceinline__ unsigned long long wg_pack(float x, float y) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
    return r;
}
__device__ __forceinline__ float2 wg_unpack(unsigned long long v) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
__device__ __forceinline__ unsigned long long wg_fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long wg_mul2(unsigned long long a, unsigned long long b) {
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

__device__ __forceinline__ uint32_t wg_key(uint32_t w) {
    return ((w >> 28) & 1u) << 8 | ((w >> 6) & 15u) << 4 | ((w >> 1) & 15u);
}

// Staged record: values in fixed-point units (conjugate samples enter as conj V: the run's sum is conjugated when it
// is merged), table entry indices of the window's first column / row: x = rx * PT + 1 - (lx & 1), likewise y.
template <int PT>
__device__ __forceinline__ uint4 wg_stage(const uint4 rec, const float sv, const float sw) {
    const uint32_t w = rec.w;
    uint4 st;
    const float im = __uint_as_float(rec.y) * sv;
    st.x = __float_as_uint(__uint_as_float(rec.x) * sv);
    st.y = __float_as_uint(((w >> 28) & 1u) ? -im : im);
    st.z = __float_as_uint(__uint_as_float(rec.z) * sw);
    const uint32_t xo = ((w >> 10) & 511u) * (uint32_t)PT + 1u - (w & 1u);
    const uint32_t yo = ((w >> 19) & 511u) * (uint32_t)PT + 1u - ((w >> 5) & 1u);
    st.w = xo | (yo << 16);
    return st;
}

// One warp streams records [p0, e) of the segment's sorted order.  The 32 lanes tile the window as RS = 32 / LR row
// slots x LR column groups (lanes beyond RS * LR idle); a lane holds the RP rows slot + k * RS and the CW consecutive
// columns of its group: RP * CW cells (re, im of G and of Gw as packed fp32 pairs), RP + CW table loads per record.
// FFMA2 takes a scalar operand broadcast to both halves: acc += kx.re * t + kx.im * rot(t), rot(a, b) = (-b, a).
// SPLIT (small windows): the two terms are accumulated separately, Ga += kx.re * t and Gb += kx.im * t, and the
// rotation is applied once per run when the window is merged (it is linear) -- 4 FFMA2 per cell and record and nothing
// else; otherwise rot(t) is formed per row and record.
template <int LR, int CW, int RP, int SPLIT, int PR, int PL, int PT>
__device__ __forceinline__ void wg_stream(const uint4* __restrict__ src, const int n, const unsigned short* __restrict__ sI,
                                          uint4* __restrict__ wb, const float2* __restrict__ sTab, const int dh,
                                          int* __restrict__ sReg, const float sv, const float sw, const int lane,
                                          const int warp) {
    constexpr int RS = 32 / LR;
    const int rs0 = lane / LR, c = lane - rs0 * LR;
    const bool active = rs0 < RS;
    const int rs = active ? rs0 : 0;
    const float2* tabx = sTab + c * CW;
    const float2* taby = sTab + rs;
    unsigned long long Ga[RP][CW], Wa[RP][CW], Gb[SPLIT ? RP : 1][SPLIT ? CW : 1], Wb[SPLIT ? RP : 1][SPLIT ? CW : 1];
    int off = 0;
    uint32_t kc = 0;

    const int per = (n + 7) >> 3;
    const int e = min(n, (warp + 1) * per);
    int p = warp * per;
    uint4 nxt = make_uint4(0, 0, 0, 0);
    uint32_t nidx = 0;
    if (p + lane < e) { nidx = sI[p + lane]; nxt = __ldg(src + (nidx & 0xFFFu)); }
    int buf = 0;
    bool open = false;
    while (p < e) {
        const int m = min(32, e - p);
        wb[buf * 32 + lane] = wg_stage<PT>(nxt, sv, sw);
        const uint32_t mykey = wg_key(nxt.w);
        uint32_t ends = __ballot_sync(kAll, lane < m && ((nidx >> 15) != 0u || (p + 32 >= e && lane == m - 1)));
        __syncwarp();
        if (p + 32 + lane < e) { nidx = sI[p + 32 + lane]; nxt = __ldg(src + (nidx & 0xFFFu)); }
        const uint4* __restrict__ q = wb + buf * 32;
        int j = 0;
        uint4 st = q[0];
        while (j < m) {
            const bool closes = ends != 0u;
            const int len = closes ? __ffs(ends) : m - j;
            if (!open) {
                const uint32_t key = __shfl_sync(kAll, mykey, j);
                kc = key >> 8;
                off = (2 * (int)((key >> 4) & 15u) + dh + rs) * PR + 2 * (int)(key & 15u) + dh + c * CW;
#pragma unroll
                for (int k = 0; k < RP; ++k)
#pragma unroll
                    for (int i = 0; i < CW; ++i) {
                        Ga[k][i] = Wa[k][i] = 0ull;
                        if (SPLIT) Gb[k][i] = Wb[k][i] = 0ull;
                    }
            }
            j += len;
            for (int t = len; t > 0; --t) {
                const float2* px = tabx + (st.w & 0xFFFFu);
                const float2* py = taby + (st.w >> 16);
                float2 kx[CW], ky[RP];
#pragma unroll
                for (int k = 0; k < RP; ++k) ky[k] = py[k * RS];
#pragma unroll
                for (int i = 0; i < CW; ++i) kx[i] = px[i];
                const float re = __uint_as_float(st.x), im = __uint_as_float(st.y), wt = __uint_as_float(st.z);
                st = q[min(j - t + 1, 31)];                            // the next record (of this or the next run)
                const unsigned long long v = wg_pack(re, im), vr = wg_pack(-im, re);
#pragma unroll
                for (int k = 0; k < RP; ++k) {
                    // row factors: t = ky * V, tw = ky * wt
                    const unsigned long long tt = wg_fma2(wg_pack(ky[k].y, ky[k].y), vr, wg_mul2(wg_pack(ky[k].x, ky[k].x), v));
                    const unsigned long long tw = wg_mul2(wg_pack(ky[k].x, ky[k].y), wg_pack(wt, wt));
                    if (SPLIT) {
#pragma unroll
                        for (int i = 0; i < CW; ++i) {
                            const unsigned long long kr = wg_pack(kx[i].x, kx[i].x), ki = wg_pack(kx[i].y, kx[i].y);
                            Ga[k][i] = wg_fma2(kr, tt, Ga[k][i]);
                            Gb[k][i] = wg_fma2(ki, tt, Gb[k][i]);
                            Wa[k][i] = wg_fma2(kr, tw, Wa[k][i]);
                            Wb[k][i] = wg_fma2(ki, tw, Wb[k][i]);
                        }
                    } else {
                        const float2 tf = wg_unpack(tt), wf = wg_unpack(tw);
                        const unsigned long long tr = wg_pack(-tf.y, tf.x), twx = wg_pack(-wf.y, wf.x);
#pragma unroll
                        for (int i = 0; i < CW; ++i) {
                            const unsigned long long kr = wg_pack(kx[i].x, kx[i].x), ki = wg_pack(kx[i].y, kx[i].y);
                            Ga[k][i] = wg_fma2(ki, tr, wg_fma2(kr, tt, Ga[k][i]));
                            Wa[k][i] = wg_fma2(ki, twx, wg_fma2(kr, tw, Wa[k][i]));
                        }
                    }
                }
            }
            if (closes && active) {
                // merge the run: cells beyond the window hold exact zeros (zero table entries) and land inside the region
                const float sg = kc ? -1.0f : 1.0f;                    // conjugate-kernel samples: conj of the run's sum
#pragma unroll
                for (int k = 0; k < RP; ++k)
#pragma unroll
                    for (int i = 0; i < CW; ++i) {
                        float2 gv = wg_unpack(Ga[k][i]), wv = wg_unpack(Wa[k][i]);
                        if (SPLIT) {
                            const float2 gb = wg_unpack(Gb[k][i]), wb2 = wg_unpack(Wb[k][i]);
                            gv.x -= gb.y; gv.y += gb.x; wv.x -= wb2.y; wv.y += wb2.x;
                        }
                        int* cell = sReg + off + k * RS * PR + i;
                        atomicAdd(cell, __float2int_rn(gv.x));
                        atomicAdd(cell + PL, __float2int_rn(gv.y * sg));
                        atomicAdd(cell + 2 * PL, __float2int_rn(wv.x));
                        atomicAdd(cell + 3 * PL, __float2int_rn(wv.y * sg));
                    }
            }
            open = !closes;
            ends = len < 32 ? ends >> len : 0u;
        }
        buf ^= 1;
        p += 32;
    }
}

// shape 7 (direct): S lanes per record, lane = footprint column, floor(32 / S) records per warp pass; loop over the rows;
// the row factors ky * (wt V), ky * wt are formed once per row; table TT[r][j] (pitch tp) read through L1
template <int PR, int PL>
__device__ __forceinline__ void wg_direct(const uint4* __restrict__ src, const int n, const float* __restrict__ tabf, const bool cplx,
                                          const int tp, const int S, const int dh, int* __restrict__ sReg, const float sv,
                                          const float sw, const int lane, const int warp) {
    // entry i of the plane's table: complex (w mode) or real (2-D mode, any support)
    auto entry = [&](const int i) -> float2 {
        return cplx ? __ldg(reinterpret_cast<const float2*>(tabf) + i) : make_float2(__ldg(tabf + i), 0.f);
    };
    const int per = 32 / S, sub = lane / S, jx = lane - sub * S;
    if (sub >= per) return;
    for (int i = warp * per + sub; i < n; i += 8 * per) {
        const uint4 a = __ldg(src + i);
        const uint32_t w = a.w;
        const float cs = ((w >> 28) & 1u) ? -1.0f : 1.0f;
        const float re = __uint_as_float(a.x) * sv, im = __uint_as_float(a.y) * sv, wt = __uint_as_float(a.z) * sw;
        const int lx = (int)(w & 31u), ly = (int)((w >> 5) & 31u);
        const int rx = (int)((w >> 10) & 511u), ry = (int)((w >> 19) & 511u);
        const float2 kx2 = entry(rx * tp + jx);
        const float kxr = kx2.x, kxi = kx2.y * cs;
        const int kyb = ry * tp;
        int* cell = sReg + (ly + dh) * PR + lx + dh + jx;
        for (int jy = 0; jy < S; ++jy, cell += PR) {
            const float2 ky2 = entry(kyb + jy);
            const float kyr = ky2.x, kyi = ky2.y * cs;
            const float tr = kyr * re - kyi * im, ti = kyr * im + kyi * re;
            const float ur = kyr * wt, ui = kyi * wt;
            atomicAdd(cell, __float2int_rn(kxr * tr - kxi * ti));
            atomicAdd(cell + PL, __float2int_rn(kxr * ti + kxi * tr));
            atomicAdd(cell + 2 * PL, __float2int_rn(kxr * ur - kxi * ui));
            atomicAdd(cell + 3 * PL, __float2int_rn(kxr * ui + kxi * ur));
        }
    }
}

template <int SHP>
__global__ void __launch_bounds__(256, WgShape<SHP>::MINB) k_wgrid(const Geom g, const Sample* __restrict__ sorted,
                                                                    const Item* __restrict__ items,
                                                                    const uint32_t* __restrict__ list, uint32_t* __restrict__ ctl,
                                                                    const uint32_t* __restrict__ bin_offset,
                                                                    const PlaneMeta* __restrict__ planes,
                                                                    const float* __restrict__ tables, GridPtrs grids,
                                                                    const float kbmax) {
    using C = WgShape<SHP>;
    constexpr int RR = C::RR, PR = C::PR, PT = C::PT > 0 ? C::PT : 1, PL = RR * PR, HMAX = (C::SMAX - 1) / 2;
    extern __shared__ __align__(16) unsigned char smem[];
    int* sReg = reinterpret_cast<int*>(smem);
    uint32_t* sH = reinterpret_cast<uint32_t*>(smem + 16 * PL);
    unsigned short* sP = reinterpret_cast<unsigned short*>(sH + kWgKeys + 8);
    unsigned short* sI = sP + kWgChunk;
    float2* sTab = reinterpret_cast<float2*>(sI + kWgChunk);
    __shared__ uint32_t sW[8];
    __shared__ float sSum[8][2];
    __shared__ uint32_t sWork;
    __shared__ int sSup[kMaxPlanes];
    __shared__ int sSegP[kMaxPlanes], sNSeg;
    __shared__ uint32_t sSegA[kMaxPlanes], sSegB[kMaxPlanes];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int P = g.nplanes;
    for (int p = tid; p < P; p += 256) sSup[p] = planes[p].support;
    const uint32_t n_items = ctl[kWgShapes + SHP];                   // items that hold records of this shape
    int cached = -1;

    for (;;) {
        __syncthreads();
        if (tid == 0) sWork = atomicAdd(&ctl[SHP], 1u);
        __syncthreads();
        const uint32_t wi = sWork;
        if (wi >= n_items) break;
        const uint32_t entry = list[wi];                              // item | part << 24 | log2(parts) << 28
        const uint32_t part = (entry >> 24) & 15u, lparts = entry >> 28;
        const Item item = items[entry & 0xFFFFFFu];
        const uint32_t T = item.bin, lo = item.start, hi = lo + item.count;
        if (warp == 0) {   // this entry's plane segments: the part-th of 2^lparts equal pieces of every segment routed to this kernel
            const uint32_t* __restrict__ off = bin_offset + (size_t)T * P;
            int cnt = 0;
            for (int base = 0; base < P; base += 32) {
                const int p = base + lane;
                uint32_t a = 0, b = 0;
                if (p < P) {
                    a = max(off[p], lo); b = min(off[p + 1], hi);
                    if (a < b && wg_route(sSup[p], b - a) == SHP) {
                        const uint32_t len = b - a;
                        b = a + ((len * (part + 1u)) >> lparts);
                        a += (len * part) >> lparts;
                    } else {
                        b = a;
                    }
                }
                const unsigned m = __ballot_sync(kAll, a < b);
                if (a < b) {
                    const int at = cnt + __popc(m & ((1u << lane) - 1u));
                    sSegP[at] = p; sSegA[at] = a; sSegB[at] = b;
                }
                cnt += __popc(m);
            }
            if (lane == 0) sNSeg = cnt;
        }
        __syncthreads();
        const int nseg = sNSeg;
        if (nseg == 0) continue;
        // fixed-point scales from the entry's records (one region for all its plane segments)
        float mv = 0.f, mw = 0.f;
        for (int q = 0; q < nseg; ++q) {
            const uint32_t b = sSegB[q];
            for (uint32_t i = sSegA[q] + tid; i < b; i += 256) {
                const uint4 v = __ldg(reinterpret_cast<const uint4*>(sorted + i));
                mv += fabsf(__uint_as_float(v.x)) + fabsf(__uint_as_float(v.y));
                mw += __uint_as_float(v.z);
            }
        }
        const uint32_t gi = T / (uint32_t)g.ntiles, tile = T - gi * (uint32_t)g.ntiles;
        const int ty = (int)(tile / (uint32_t)g.ntx), tx = (int)(tile - (uint32_t)ty * (uint32_t)g.ntx);
        {   // zero the region
            int4* z = reinterpret_cast<int4*>(sReg);
            for (int i = tid; i < PL; i += 256) z[i] = make_int4(0, 0, 0, 0);
        }
        for (int o = 16; o > 0; o >>= 1) { mv += __shfl_xor_sync(kAll, mv, o); mw += __shfl_xor_sync(kAll, mw, o); }
        if (lane == 0) { sSum[warp][0] = mv; sSum[warp][1] = mw; }
        __syncthreads();
        mv = 0.f; mw = 0.f;
        for (int w = 0; w < 8; ++w) { mv += sSum[w][0]; mw += sSum[w][1]; }
        const float sv = 2104533975.0f / fmaxf(mv * kbmax, 1e-30f), sw = 2104533975.0f / fmaxf(mw * kbmax, 1e-30f);

        for (int q = 0; q < nseg; ++q) {
            const int p = sSegP[q], S = sSup[p];
            const uint32_t a = sSegA[q], b = sSegB[q];
            const int n = (int)(b - a), dh = HMAX - ((S - 1) >> 1);
            const uint4* __restrict__ src = reinterpret_cast<const uint4*>(sorted + a);
            if constexpr (C::LR == 0) {                               // direct: no per-segment state in shared memory
                const PlaneMeta pm = planes[p];
                wg_direct<PR, PL>(src, n, tables + (size_t)pm.offset * (g.wmode ? 2 : 1), g.wmode != 0, pm.pitch, S, dh, sReg, sv, sw, lane, warp);
                continue;
            }
            __syncthreads();                                          // the previous segment is done with sH / sP / the table
            if (cached != p) {                                        // stage the plane's table: entry e = footprint index + 1
                const PlaneMeta pm = planes[p];
                const float2* tc = reinterpret_cast<const float2*>(tables) + pm.offset;   // w mode: complex entries
                const float* tr = tables + pm.offset;                                       // 2-D mode: real entries
                for (int i = tid; i < (g.Q + 1) * PT; i += 256) {
                    const int r = i / PT, e = i - r * PT, j = e - 1;
                    float2 v = make_float2(0.f, 0.f);
                    if (j >= 0 && j < S) v = g.wmode ? __ldg(tc + r * pm.pitch + j) : make_float2(__ldg(tr + r * pm.pitch + j), 0.f);
                    sTab[i] = v;
                }
                cached = p;
            }
            if constexpr (C::LR != 0) {
                for (int i = tid; i < kWgKeys + 8; i += 256) sH[i] = 0;
                __syncthreads();
                for (int i = tid; i < n; i += 256) sP[i] = (unsigned short)atomicAdd(&sH[wg_key(__ldg(&src[i].w))], 1u);
                __syncthreads();
                {   // exclusive scan of the 512 keys, two per thread
                    const uint32_t h0 = sH[2 * tid], h1 = sH[2 * tid + 1], tot = h0 + h1;
                    uint32_t inc = tot;
                    for (int o = 1; o < 32; o <<= 1) {
                        const uint32_t t = __shfl_up_sync(kAll, inc, o);
                        if (lane >= o) inc += t;
                    }
                    if (lane == 31) sW[warp] = inc;
                    __syncthreads();
                    uint32_t ex = inc - tot;
                    for (int w = 0; w < warp; ++w) ex += sW[w];
                    sH[2 * tid] = ex; sH[2 * tid + 1] = ex + h0;
                    if (tid == 255) sH[kWgKeys] = ex + tot;
                }
                __syncthreads();
                for (int i = tid; i < n; i += 256) {
                    const uint32_t k = wg_key(__ldg(&src[i].w)), pos = sH[k] + sP[i];
                    sI[pos] = (unsigned short)((uint32_t)i | ((pos + 1u == sH[k + 1u]) ? 0x8000u : 0u));
                }
                __syncthreads();
                uint4* wb = reinterpret_cast<uint4*>(sP) + warp * 64;  // sP is free now: 8 warps x 2 x 32 staged records
                wg_stream<C::LR, C::CW, C::RP, C::SPLIT, PR, PL, PT>(src, n, sI, wb, sTab, dh, sReg, sv, sw, lane, warp);
            }
        }
        __syncthreads();
        // add the touched cells of the stored half-plane to the grids
        const float iv = 1.0f / sv, iw = 1.0f / sw;
        const int x0 = tx * kTile - kTile / 2 - HMAX, y0 = ty * kTile - kTile / 2 - HMAX;
        const size_t gbase = (size_t)gi * g.ny * g.nx;
        float2* __restrict__ Gw2 = reinterpret_cast<float2*>(grids.Gw);
        for (int i = tid; i < PL; i += 256) {
            const int y = i / PR, x = i - y * PR;
            const int gx = x0 + x, gy = y0 + y;
            if (gx < 0 || gx >= g.nx || gy < (g.ny >> 1) || gy >= g.ny) continue;
            const int vr = sReg[i], vi = sReg[PL + i], wr = sReg[2 * PL + i], wim = sReg[3 * PL + i];
            const size_t idx = gbase + (size_t)gy * g.nx + gx;
            if (vr | vi) atomicAdd(&grids.G[idx], make_float2((float)vr * iv, (float)vi * iv));
            if (g.wmode) { if (wr | wim) atomicAdd(&Gw2[idx], make_float2((float)wr * iw, (float)wim * iw)); }
            else if (wr) atomicAdd(&grids.Gw[idx], (float)wr * iw);                         // 2-D mode: the weight grid is real
        }
    }
}

// Kw1: one warp per tile; items of <= kWgChunk consecutive records (they may span planes), and per window shape the list
// of the items that hold records of it.  ctl[0..7]: work counters, ctl[8..15]: list lengths.
__global__ void __launch_bounds__(256) k_wtile_items(const uint32_t ntiles_total, const int P, const uint32_t list_cap,
                                                     const uint32_t* __restrict__ bin_offset,
                                                     const PlaneMeta* __restrict__ planes, Item* __restrict__ items,
                                                     uint32_t* __restrict__ lists, uint32_t* __restrict__ nitems,
                                                     uint32_t* __restrict__ ctl) {
    const uint32_t t = (blockIdx.x * 256u + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (t >= ntiles_total) return;
    const uint32_t* __restrict__ off = bin_offset + (size_t)t * P;
    const uint32_t a = off[0], b = off[P];
    if (a == b) return;
    const uint32_t cnt = b - a, n = (cnt + kWgChunk - 1) / kWgChunk;
    uint32_t slot = 0;
    if (lane == 0) slot = atomicAdd(nitems, n);
    slot = __shfl_sync(kAll, slot, 0);
    for (uint32_t q = lane; q < n; q += 32) {
        Item it;
        it.bin = t; it.start = a + q * kWgChunk; it.count = min((uint32_t)kWgChunk, cnt - q * kWgChunk);
        items[slot + q] = it;
        uint32_t nrec[kWgShapes] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
        for (int p = 0; p < P; ++p) {
            const uint32_t sa = max(off[p], it.start), sb = min(off[p + 1], it.start + it.count);
            if (sa >= sb) continue;
            const int r = wg_route(planes[p].support, sb - sa);
#pragma unroll
            for (int sh = 0; sh < kWgShapes; ++sh) nrec[sh] += r == sh ? sb - sa : 0u;
        }
#pragma unroll
        for (int sh = 0; sh < kWgShapes; ++sh) {
            if (!nrec[sh]) continue;
            uint32_t lparts = 0;                                      // parts = 2^lparts <= 16 (SUB >= 256, <= 4096 records)
            while (lparts < 4u && (nrec[sh] >> lparts) > wg_sub(sh)) ++lparts;
            const uint32_t parts = 1u << lparts, at = atomicAdd(&ctl[kWgShapes + sh], parts);
            for (uint32_t k = 0; k < parts; ++k) lists[(size_t)sh * list_cap + at + k] = (slot + q) | k << 24 | lparts << 28;
        }
    }
}

template <int SHP>
size_t wg_smem_bytes(int Q) {
    using C = WgShape<SHP>;
    if (C::LR == 0) return (size_t)16 * C::RR * C::PR;
    return (size_t)16 * C::RR * C::PR + (size_t)(kWgKeys + 8) * 4 + (size_t)2 * kWgChunk * 2 + (size_t)(Q + 1) * C::PT * 8;
}

template <int SHP>
bool wg_fits(int Q, int max_smem_bytes) { return wg_smem_bytes<SHP>(Q) + 2048 <= (size_t)max_smem_bytes; }   // + static shared memory

template <int SHP>
cudaError_t wg_setup(int max_smem_bytes) {
    return cudaFuncSetAttribute(k_wgrid<SHP>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes - 2048);
}

template <int SHP>
void wg_launch(const Geom& g, const Sample* sorted, const Item* items, const uint32_t* lists, uint32_t list_cap, uint32_t* ctl,
               const uint32_t* bin_offset, const PlaneMeta* planes, const float* tables, GridPtrs grids, float kbmax, int num_sms,
               cudaStream_t s) {
    const size_t smem = wg_smem_bytes<SHP>(g.Q);
    int per_sm = (int)((size_t)227 * 1024 / (smem + 1024));
    per_sm = per_sm < 1 ? 1 : (per_sm > WgShape<SHP>::MINB ? WgShape<SHP>::MINB : per_sm);
    k_wgrid<SHP><<<num_sms * per_sm, 256, smem, s>>>(g, sorted, items, lists + (size_t)SHP * list_cap, ctl, bin_offset, planes, tables,
                                                     grids, kbmax);
}

}  // namespace

bool wgrid_supported(const PlaneMeta* planes_host, int P, int Q, int max_smem_bytes) {
    if (P < 1 || P > kMaxPlanes) return false;
    const bool fits[kWgShapes] = {wg_fits<0>(Q, max_smem_bytes), wg_fits<1>(Q, max_smem_bytes), wg_fits<2>(Q, max_smem_bytes),
                                  wg_fits<3>(Q, max_smem_bytes), wg_fits<4>(Q, max_smem_bytes), wg_fits<5>(Q, max_smem_bytes),
                                  wg_fits<6>(Q, max_smem_bytes), wg_fits<7>(Q, max_smem_bytes)};
    for (int p = 0; p < P; ++p) {
        const int S = planes_host[p].support;
        if (S > 31 || !fits[wg_shape(S)]) return false;
    }
    return true;
}

cudaError_t wgrid_kernel_setup(int max_smem_bytes) {
    cudaError_t e;
    if ((e = wg_setup<0>(max_smem_bytes)) || (e = wg_setup<1>(max_smem_bytes)) || (e = wg_setup<2>(max_smem_bytes)) ||
        (e = wg_setup<3>(max_smem_bytes)) || (e = wg_setup<4>(max_smem_bytes)) || (e = wg_setup<5>(max_smem_bytes)) ||
        (e = wg_setup<6>(max_smem_bytes)) || (e = wg_setup<7>(max_smem_bytes)))
        return e;
    return cudaSuccess;
}

// items, per-shape item lists (8 x list_cap entries), work counters and list lengths ctl[0..15] (zeroed here, on the stream)
cudaError_t launch_wtile_items(const Geom& g, const uint32_t* bin_offset, const PlaneMeta* planes, Item* items, uint32_t* lists,
                               uint32_t list_cap, uint32_t* nitems, uint32_t* ctl, cudaStream_t s) {
    cudaError_t e;
    if ((e = cudaMemsetAsync(nitems, 0, sizeof(uint32_t), s))) return e;
    if ((e = cudaMemsetAsync(ctl, 0, 2 * kWgShapes * sizeof(uint32_t), s))) return e;
    const uint32_t nt = (uint32_t)g.ngrids * (uint32_t)g.ntiles;
    k_wtile_items<<<(nt * 32u + 255u) / 256u, 256, 0, s>>>(nt, g.nplanes, list_cap, bin_offset, planes, items, lists, nitems, ctl);
    return cudaGetLastError();
}

// entries per shape list: an item is listed at most 16 times (items < 2^24 by the 2^30 bound on visibilities per call)
size_t wgrid_list_cap(const Geom& g, size_t nsamples) { return 16 * ((size_t)g.ngrids * g.ntiles + nsamples / kWgChunk + 2); }

// One launch per window shape that occurs.  side != nullptr: 7 side streams and 8 events (ev[0] forks, ev[1..7] join): the
// kernels are persistent and of very different length, so they are enqueued on separate streams (longest first) and
// the CTAs of the next one start as those of the previous one run out of work; all of them add into the grids atomically.
int launch_wgrid(const Geom& g, const Sample* sorted, const Item* items, const uint32_t* lists, uint32_t list_cap, uint32_t* ctl,
                 const uint32_t* bin_offset, const PlaneMeta* planes, const PlaneMeta* planes_host, const float* tables,
                 GridPtrs grids, int num_sms, cudaStream_t s, const cudaStream_t* side, const cudaEvent_t* ev, cudaError_t* err) {
    bool present[kWgShapes] = {false};
    present[7] = true;                                                // small segments of any support
    float kbmax = 1.0f;
    for (int p = 0; p < g.nplanes; ++p) {
        present[wg_shape(planes_host[p].support)] = true;
        float kb;
        memcpy(&kb, &planes_host[p].pad, sizeof(float));
        kbmax = kb > kbmax ? kb : kbmax;
    }
    int launches = 0;
    *err = cudaSuccess;
    if (side && (*err = cudaEventRecord(ev[0], s)) != cudaSuccess) return 0;
    int nside = 0;
    auto stream_for = [&](void) -> cudaStream_t {
        if (!side || launches == 0) return s;                         // the first (longest) kernel stays on the caller's stream
        cudaStream_t t = side[nside];
        if (*err == cudaSuccess) *err = cudaStreamWaitEvent(t, ev[0], 0);
        return t;
    };
    auto joined = [&](cudaStream_t t) {
        if (t == s) return;
        if (*err == cudaSuccess) *err = cudaEventRecord(ev[1 + nside], t);
        if (*err == cudaSuccess) *err = cudaStreamWaitEvent(s, ev[1 + nside], 0);
        ++nside;
    };
#define WG_LAUNCH(SHP)                                                                                                  \
    if (present[SHP]) {                                                                                                 \
        cudaStream_t t = stream_for();                                                                                  \
        wg_launch<SHP>(g, sorted, items, lists, list_cap, ctl, bin_offset, planes, tables, grids, kbmax, num_sms, t);  \
        ++launches;                                                                                                     \
        joined(t);                                                                                                      \
    }
    WG_LAUNCH(0) WG_LAUNCH(3) WG_LAUNCH(1) WG_LAUNCH(2) WG_LAUNCH(7) WG_LAUNCH(4) WG_LAUNCH(6) WG_LAUNCH(5)
#undef WG_LAUNCH
    if (*err == cudaSuccess) *err = cudaGetLastError();
    return launches;
}

}  // namespace muser
