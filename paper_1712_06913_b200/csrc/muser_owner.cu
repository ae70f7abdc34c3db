// Owner-tile gridding path (2-D mode, support 7), sm_100a.
//
//   O1  k_owner_count      A1: fp64 coordinates (O1 order), keep/drop, statistics; stores the integer
//                              result per visibility (16 B) and histograms the tiles each sample's 7x7 footprint
//                              touches (1, 2 or 4) in a CTA-private shared histogram (one global atomic per touched
//                              tile per CTA)
//   O2  k_owner_scan_*     A1: multi-CTA exclusive scan of the histogram (one chained launch): sample offsets, chunk
//                              items of heavy tiles (> item_size samples), work list of light non-empty tiles
//   O3  k_owner_scatter    A1: reads O1's integer result and writes one 16-byte record per (sample, touched tile)
//   O4a (tile flags)       A2: a tile that has not been written since the last reset has its flag in `valid` at 0: it is
//                              never zero-filled -- the gridder stores instead of adding, the row transform skips its
//                              loads, and k_owner_fill_invalid zeroes such tiles for the consumers of the dense grids
//   O4  k_grid_owner_s7    A2/A4: persistent kernel, 4 CTAs per SM pulling work units (chunks of heavy tiles first,
//                              then the light non-empty 64x32 tiles) from a device counter.  Per unit: counting sort of
//                              <= 4096 records by 8x8 window (shared histogram, 2-byte positions); every warp then streams an equal share
//                              of the sorted order through a private 2 x 32-record buffer (gather loads one batch
//                              ahead, records staged in fixed-point units with table row offsets); a run of equal
//                              window is accumulated in registers (lane = row r, column pair c; three packed FFMA2 per
//                              sample; kernel table in shared memory) and merged into the 32-bit fixed-point shared
//                              tile with native integer adds.  The tile is written to G and Gw with plain coalesced
//                              stores: no memset, no global atomics.  Chunks of a heavy tile publish partial tiles,
//                              which are added up in two levels, always in chunk order (no CTA waits for another).
// Passages: PAPER.md:78 (gridding = convolution onto a regular grid), :136-138 (spheroidal GCF), :216-228 (float2
// grid, row-major, Hermitian), :249-256 (DIRTY_IMAGE).  The binning and tiling are this build's design.
#include "muser_internal.h"

namespace muser {

static constexpr double kC = 299792458.0;   // m/s
static constexpr unsigned kFull = 0xffffffffu;

// Owner tiles are kOwTW cells wide (x) and kTile = 32 cells tall (y): tile (tx, ty) covers cells
// [kOwTW*tx - kOwTW/2, ...) x [32*ty - 16, ...), so the uv origin sits in the middle of a tile.  Wider tiles mean fewer
// records listed twice (halo duplication 1.33 -> 1.19 on MUSER frames) and half as many tiles to set up and store.
constexpr int kOwTW = kOwTileW, kOwTWS = kOwTW == 64 ? 6 : 5;
constexpr int kOwNKX = (kOwTW + 6) / 2;          // 8-wide windows per tile row incl. halo: 19 (32-wide) or 35 (64-wide)
constexpr int kOwKXB = kOwTWS;                   // bits of the window column index in a record
constexpr uint32_t kOwKeyMask = (1u << (5 + kOwKXB)) - 1u;

// ------------------------------------------------------------------------------------------------- coordinates
// O1 for one axis (same operation order and the same fp64 roundings as the oracle; _rn intrinsics forbid FMA
// contraction).  xs = c_lambda * scale already rounded (the conjugate sample negates it: exact).  The two floors and the
// conversions to int are done in the FP64 add pipe with the 1.5 * 2^52 constant (x + M rounds x to the nearest integer,
// whose two's complement sits in the low word; one compare turns nearest into floor) instead of FRND.F64 / F2I.F64,
// which are conversion-unit instructions at a fraction of the FP64 rate.  Exact for |x| < 2^31 (callers test |xs| < 1e9).
struct OwAxes { double hx, hy, Qd; };
__device__ __forceinline__ OwAxes ow_axes(const Geom& g) { return {(double)(g.nx / 2), (double)(g.ny / 2), (double)g.Q}; }
__device__ __forceinline__ void ow_cell_phase(const double xs, const double half, const double Qd, int& i0, int& r) {
    constexpr double M = 6755399441055744.0;
    const double p = __dadd_rn(xs, half);
    const double t = __dadd_rn(p, 0.5);
    const double tm = __dadd_rn(t, M);
    double fl = __dadd_rn(tm, -M);
    int i = __double2loint(tm);
    if (fl > t) { fl = __dadd_rn(fl, -1.0); --i; }                    // i0 = floor(p + 0.5)
    const double fr = __dsub_rn(p, fl);
    const double u = __dadd_rn(__dmul_rn(fr, Qd), 0.5);
    const double um = __dadd_rn(u, M);
    int q = __double2loint(um);
    if (__dadd_rn(um, -M) > u) --q;                                   // r = floor(fr * Q + 0.5)
    i0 = i; r = q;
}
__device__ __noinline__ double ow_freq_over_c(const double f) { return __ddiv_rn(f, kC); }

struct OwLoc {
    int state;                 // 0 none (k >= nvis), 1 flagged, 2 dropped, 3 kept
    float re, im, wt;          // wt*Re V, wt*Im V (primary sample; the conjugate negates im), wt
    int cu[2], cv[2], rx[2], ry[2];
    int gid;
};

// `f_cache`/`il_cache`: the division f/c is repeated only when the frequency differs from the thread's previous
// visibility (a thread's visibilities are 256 apart: almost always the same channel).
struct OwIn { float um, vm, wm, wt; double f; float2 V; int gid; };   // one visibility's inputs
__device__ __forceinline__ OwIn ow_load(const float* __restrict__ uvw, const double* __restrict__ freq,
                                        const float2* __restrict__ vis, const float* __restrict__ weight,
                                        const int* __restrict__ grid_id, const long long k, const long long nvis) {
    OwIn in = {0.f, 0.f, 0.f, 0.f, 0.0, make_float2(0.f, 0.f), 0};
    if (k < nvis) {
        in.um = __ldg(uvw + 3 * k); in.vm = __ldg(uvw + 3 * k + 1); in.wm = __ldg(uvw + 3 * k + 2);
        in.f = __ldg(freq + k);
        if (vis) in.V = __ldg(vis + k);
        in.wt = __ldg(weight + k);
        if (grid_id) in.gid = __ldg(grid_id + k);
    }
    return in;
}
__device__ __forceinline__ void ow_locate(const Geom& g, const OwIn& in, long long k, long long nvis, OwLoc& L,
                                          float2& Vraw, double& f_cache, double& il_cache, const OwAxes& ax) {
    L.state = 0;
    if (k >= nvis) return;
    const float um = in.um, vm = in.vm, wm = in.wm;
    const double f = in.f;
    const float2 V = in.V;
    const float wt = in.wt;
    const int gid = in.gid;
    Vraw = V;
    if (f != f_cache) { il_cache = ow_freq_over_c(f); f_cache = f; }   // a call: taken once per channel and thread
    const double il = il_cache;
    const double ul = __dmul_rn((double)um, il), vl = __dmul_rn((double)vm, il), wl = __dmul_rn((double)wm, il);
    const bool ok = isfinite(ul) && isfinite(vl) && isfinite(wl) && isfinite(wt) && isfinite(V.x) && isfinite(V.y) &&
                    isfinite(f) && wt > 0.0f && gid >= 0 && gid < g.ngrids;
    if (!ok) { L.state = 1; return; }
    const int h = (g.S - 1) >> 1;
    const double xu = __dmul_rn(ul, g.su), xv = __dmul_rn(vl, g.sv);
    bool inside = fabs(xu) < 1.0e9 && fabs(xv) < 1.0e9;               // beyond: off any grid, and outside the int range
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        int iu, iv, ru, rv;
        ow_cell_phase(s ? -xu : xu, ax.hx, ax.Qd, iu, ru);
        ow_cell_phase(s ? -xv : xv, ax.hy, ax.Qd, iv, rv);
        inside = inside && iu >= h + 1 && iu <= g.nx - 1 - h && iv >= h + 1 && iv <= g.ny - 1 - h;
        L.cu[s] = iu; L.cv[s] = iv;
        L.rx[s] = g.Q / 2 - ru; L.ry[s] = g.Q / 2 - rv;
    }
    if (!inside) { L.state = 2; return; }
    L.state = 3;
    L.re = wt * V.x; L.im = wt * V.y; L.wt = wt; L.gid = gid;
}

// Bin of the q-th tile (q = qx | qy << 1) touched by the footprint of a sample at nearest cell (cu, cv), or kNoBin.
__device__ __forceinline__ uint32_t ow_bin(const Geom& g, int gid, int cu, int cv, int q, int& tx, int& ty) {
    const int h = (g.S - 1) >> 1, hy = g.ny >> 1;
    if (cv + h < hy) return kNoBin;                                   // footprint entirely in the lower half-plane
    const int tx0 = (cu - h + kOwTW / 2) >> kOwTWS, tx1 = (cu + h + kOwTW / 2) >> kOwTWS;
    const int ty0 = max(cv - h - hy, 0) >> kTileShift, ty1 = (cv + h - hy) >> kTileShift;
    if (((q & 1) && tx1 == tx0) || ((q & 2) && ty1 == ty0)) return kNoBin;
    tx = (q & 1) ? tx1 : tx0;
    ty = (q & 2) ? ty1 : ty0;
    return (uint32_t)gid * (uint32_t)g.ontiles + (uint32_t)(ty * g.otx + tx);
}

// Warp-aggregated counter increment: lanes with the same bin issue one atomicAdd; returns the lane's rank.
// Every lane of the warp must call it (bin == kNoBin: no increment).
__device__ __forceinline__ uint32_t ow_agg_inc(uint32_t* __restrict__ cnt, uint32_t bin, int lane) {
    const unsigned m = __match_any_sync(kFull, bin);
    const int leader = __ffs(m) - 1;
    uint32_t base = 0;
    if (bin != kNoBin && lane == leader) base = atomicAdd(&cnt[bin], (uint32_t)__popc(m));
    base = __shfl_sync(kFull, base, leader);
    return base + (uint32_t)__popc(m & ((1u << lane) - 1u));
}

// CTA-level aggregation for the two binning kernels: when every visibility of the CTA belongs to one grid and that
// grid's tile count fits the shared histogram, the CTA counts in shared memory and issues ONE global atomic per
// touched tile (MUSER's central tile takes a third of all samples: per-sample global atomics serialise on it).
constexpr int kBinThreads = 256;
constexpr int kBinSmemTiles = 4096;      // two u32 arrays of this many tiles must fit the default 48 KB

// The (at most 2 x 2) tiles a 7x7 footprint at nearest cell (cu, cv) touches: first tile (tx0, ty0) and whether the
// footprint also reaches the next tile in x / in y.
struct OwTiles { int tx0, ty0, t00; bool mx, my, up; };
__device__ __forceinline__ OwTiles ow_tiles(const Geom& g, int cu, int cv) {
    const int h = (g.S - 1) >> 1, hy = g.ny >> 1;
    OwTiles t;
    t.up = cv + h >= hy;                                              // touches the stored (upper) half-plane
    t.tx0 = (cu - h + kOwTW / 2) >> kOwTWS;
    t.ty0 = max(cv - h - hy, 0) >> kTileShift;
    t.mx = ((cu + h + kOwTW / 2) >> kOwTWS) != t.tx0;
    t.my = t.up && ((cv + h - hy) >> kTileShift) != t.ty0;
    t.t00 = t.ty0 * g.otx + t.tx0;
    return t;
}

// ------------------------------------------------------------------------------------------------- O1 count
// packed tiles of one sample: first tile t00 | reaches the next tile in x << 29 | in y << 30 | touches the stored
// half-plane << 31 (0 = the sample has no record)
__device__ __forceinline__ uint32_t ow_tiles_packed(const Geom& g, int cu, int cv) {
    const OwTiles t = ow_tiles(g, cu, cv);
    return t.up ? ((uint32_t)t.t00 | (t.mx ? 1u << 29 : 0u) | (t.my ? 1u << 30 : 0u) | 1u << 31) : 0u;
}

// A CTA handles kBinThreads * iters consecutive visibilities in a loop (thread: k, k + 256, ...): the per-CTA work --
// histogram zeroing and flush, statistics reduction -- is shared by `iters` visibilities per thread at no cost in
// registers.  Records of the CTA's reference grid (that of its first visibility; every record when the call has one grid)
// are counted in the shared histogram, ONE global atomic per touched tile per CTA (MUSER's central tile takes a third of
// all samples: per-sample global atomics would serialise on it); records of other grids, and every record when the
// grid's tiles do not fit the shared histogram, take warp-aggregated global atomics straight away.  The CTA's shared
// histogram is also saved (cta_hist) so that k_owner_scatter does not have to count again.
__global__ void __launch_bounds__(kBinThreads, 4) k_owner_count(const Geom g, const float* __restrict__ uvw,
                                                             const double* __restrict__ freq, const float2* __restrict__ vis,
                                                             const float* __restrict__ weight, const int* __restrict__ grid_id,
                                                             const long long nvis, const int iters,
                                                             uint32_t* __restrict__ bin_count, uint32_t* __restrict__ cta_hist,
                                                             Stats* __restrict__ stats, uint4* __restrict__ loc) {
    extern __shared__ uint32_t s_hist[];
    const long long base = (long long)blockIdx.x * kBinThreads * iters;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool fits = g.ontiles <= kBinSmemTiles;
    if (fits)
        for (int i = threadIdx.x; i < g.ontiles; i += kBinThreads) s_hist[i] = 0;
    const int ref = grid_id ? grid_id[base] : 0;                      // base < nvis by the launch geometry
    __syncthreads();
    int kept = 0, dropped = 0, flagged = 0;
    double wsum = 0.0, v2sum = 0.0, w2sum = 0.0, f_cache = 0.0, il_cache = 0.0;
    const OwAxes ax = ow_axes(g);
    float w2f = 0.f, v2f = 0.f;
    for (int it = 0; it < iters; ++it) {
        const long long k = base + (long long)it * kBinThreads + threadIdx.x;
        const OwIn cur = ow_load(uvw, freq, vis, weight, grid_id, k, nvis);
        OwLoc L;
        float2 V;
        ow_locate(g, cur, k, nvis, L, V, f_cache, il_cache, ax);
        uint32_t tp[2] = {0u, 0u};
        if (k < nvis) {                                               // integer result of O1 for k_owner_scatter
            uint4 o = make_uint4(0u, 0u, (uint32_t)L.state << 30, 0u);
            if (L.state == 3) {
                o.x = (uint32_t)L.cu[0] | ((uint32_t)L.cv[0] << 16);
                o.y = (uint32_t)L.cu[1] | ((uint32_t)L.cv[1] << 16);
                o.z |= (uint32_t)L.rx[0] | ((uint32_t)L.ry[0] << 9) | ((uint32_t)L.rx[1] << 18);
                o.w = (uint32_t)L.ry[1];
                tp[0] = ow_tiles_packed(g, L.cu[0], L.cv[0]);
                tp[1] = ow_tiles_packed(g, L.cu[1], L.cv[1]);
                ++kept;
                wsum += 2.0 * (double)L.wt;
                const float w2 = L.wt * L.wt;                          // feed alpha only (a power of two): fp32 per thread
                w2f += w2;
                v2f += w2 * (V.x * V.x + V.y * V.y);
            }
            dropped += L.state == 2;
            flagged += L.state == 1;
            loc[k] = o;
        }
        const bool local = fits && L.state == 3 && L.gid == ref;
        if (local) {
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const uint32_t t = tp[s];
                if (!(t >> 31)) continue;
                const uint32_t t00 = t & 0x1FFFFFFFu;
                const bool mx = (t >> 29) & 1u, my = (t >> 30) & 1u;
                atomicAdd(&s_hist[t00], 1u);
                if (mx) atomicAdd(&s_hist[t00 + 1], 1u);
                if (my) atomicAdd(&s_hist[t00 + g.otx], 1u);
                if (mx && my) atomicAdd(&s_hist[t00 + g.otx + 1], 1u);
            }
        }
        if (__any_sync(kFull, L.state == 3 && !local)) {              // other grids / huge grids: global atomics now
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t t = tp[s];
                    const bool on = L.state == 3 && !local && (t >> 31) && (!(q & 1) || ((t >> 29) & 1u)) &&
                                    (!(q & 2) || ((t >> 30) & 1u));
                    const uint32_t bin = on ? (uint32_t)L.gid * (uint32_t)g.ontiles + (t & 0x1FFFFFFFu) + (q & 1) +
                                                  ((q & 2) ? (uint32_t)g.otx : 0u)
                                            : kNoBin;
                    if (__any_sync(kFull, on)) ow_agg_inc(bin_count, bin, lane);
                }
        }
    }
    v2sum = (double)v2f; w2sum = (double)w2f;
    __syncthreads();
    if (fits) {
        const bool ok = ref >= 0 && ref < g.ngrids;
        const uint32_t gbase = ok ? (uint32_t)ref * (uint32_t)g.ontiles : 0u;
        uint32_t* mine = cta_hist + (size_t)blockIdx.x * g.ontiles;
        for (int i = threadIdx.x; i < g.ontiles; i += kBinThreads) {
            const uint32_t n = s_hist[i];
            mine[i] = n;
            if (n && ok) atomicAdd(&bin_count[gbase + i], n);
        }
    }
    // block reduction of the counters, one atomic set per block
    __shared__ int s_cnt[3][8];
    __shared__ double s_w[3][8];
    const int c0 = __reduce_add_sync(kFull, kept), c1 = __reduce_add_sync(kFull, dropped), c2 = __reduce_add_sync(kFull, flagged);
    for (int o = 16; o > 0; o >>= 1) {
        wsum += __shfl_xor_sync(kFull, wsum, o);
        v2sum += __shfl_xor_sync(kFull, v2sum, o);
        w2sum += __shfl_xor_sync(kFull, w2sum, o);
    }
    if (lane == 0) { s_cnt[0][warp] = c0; s_cnt[1][warp] = c1; s_cnt[2][warp] = c2; s_w[0][warp] = wsum; s_w[1][warp] = v2sum; s_w[2][warp] = w2sum; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int t0 = 0, t1 = 0, t2 = 0;
        double tw = 0.0, tv2 = 0.0, tw2 = 0.0;
        for (int w = 0; w < kBinThreads / 32; ++w) {
            t0 += s_cnt[0][w]; t1 += s_cnt[1][w]; t2 += s_cnt[2][w];
            tw += s_w[0][w]; tv2 += s_w[1][w]; tw2 += s_w[2][w];
        }
        if (t0) {
            atomicAdd(&stats->n_gridded, (unsigned long long)t0);
            atomicAdd(&stats->sum_weights, tw);
            atomicAdd(&stats->sum_val2, tv2);
            atomicAdd(&stats->sum_wt2, tw2);
        }
        if (t1) atomicAdd(&stats->n_dropped, (unsigned long long)t1);
        if (t2) atomicAdd(&stats->n_flagged, (unsigned long long)t2);
    }
}

// ------------------------------------------------------------------------------------------------- O2 scan
// Three small launches over the tile histogram, 4096 bins per CTA (4 per thread):
//   k_owner_scan_reduce   per-CTA totals of (samples, chunk items of heavy tiles, light non-empty tiles)
//   k_owner_scan_tops     one CTA: exclusive scan of the per-CTA totals, grand totals, work counter reset
//   k_owner_scan_write    per-CTA local scan + base: sample offsets, chunk items of the heavy tiles (more than
//                         item_size samples), the work list of light non-empty tiles; re-zeroes the histogram (for
//                         the next call's O1) and the scatter cursor (for this call's O3)
struct OwScan3 { uint32_t c, m, l; };

__device__ __forceinline__ OwScan3 ow_block_scan3(OwScan3 v, OwScan3& total, uint32_t (*s_w)[32]) {
    // exclusive block scan of three counters over 1024 threads; `total` = block sum
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    OwScan3 inc = v;
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t xc = __shfl_up_sync(kFull, inc.c, o), xm = __shfl_up_sync(kFull, inc.m, o), xl = __shfl_up_sync(kFull, inc.l, o);
        if (lane >= o) { inc.c += xc; inc.m += xm; inc.l += xl; }
    }
    if (lane == 31) { s_w[0][warp] = inc.c; s_w[1][warp] = inc.m; s_w[2][warp] = inc.l; }
    __syncthreads();
    if (warp == 0) {
        uint32_t wc = s_w[0][lane], wm = s_w[1][lane], wl = s_w[2][lane];
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t xc = __shfl_up_sync(kFull, wc, o), xm = __shfl_up_sync(kFull, wm, o), xl = __shfl_up_sync(kFull, wl, o);
            if (lane >= o) { wc += xc; wm += xm; wl += xl; }
        }
        s_w[0][lane] = wc; s_w[1][lane] = wm; s_w[2][lane] = wl;
    }
    __syncthreads();
    OwScan3 ex;
    ex.c = (warp ? s_w[0][warp - 1] : 0u) + inc.c - v.c;
    ex.m = (warp ? s_w[1][warp - 1] : 0u) + inc.m - v.m;
    ex.l = (warp ? s_w[2][warp - 1] : 0u) + inc.l - v.l;
    total.c = s_w[0][31]; total.m = s_w[1][31]; total.l = s_w[2][31];
    __syncthreads();
    return ex;
}

__device__ __forceinline__ OwScan3 ow_load4(const Geom& g, const uint32_t* __restrict__ bin_count, uint32_t b0,
                                            uint32_t item_size, uint32_t c[4], uint32_t m[4]) {
    c[0] = c[1] = c[2] = c[3] = 0;
    if (b0 < g.onbins) {                                                // bin_count is padded to a multiple of 4
        const uint4 v = *reinterpret_cast<const uint4*>(bin_count + b0);
        c[0] = v.x; c[1] = v.y; c[2] = v.z; c[3] = v.w;
    }
    OwScan3 t = {0u, 0u, 0u};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        m[j] = c[j] > item_size ? (c[j] + item_size - 1) / item_size : 0u;
        t.c += c[j]; t.m += m[j]; t.l += (c[j] != 0u && m[j] == 0u);
    }
    return t;
}

__global__ void __launch_bounds__(1024) k_owner_scan_reduce(const Geom g, const uint32_t* __restrict__ bin_count,
                                                            const uint32_t item_size, uint32_t* __restrict__ tops) {
    __shared__ uint32_t s_w[3][32];
    uint32_t c[4], m[4];
    const OwScan3 t = ow_load4(g, bin_count, blockIdx.x * 4096u + 4u * threadIdx.x, item_size, c, m);
    OwScan3 total;
    ow_block_scan3(t, total, s_w);
    if (threadIdx.x == 0) { tops[3 * blockIdx.x] = total.c; tops[3 * blockIdx.x + 1] = total.m; tops[3 * blockIdx.x + 2] = total.l; }
}

__global__ void __launch_bounds__(1024) k_owner_scan_tops(const Geom g, const uint32_t nblocks, uint32_t* __restrict__ tops,
                                                          uint32_t* __restrict__ bin_offset, uint32_t* __restrict__ nitems,
                                                          uint32_t* __restrict__ ctl) {
    __shared__ uint32_t s_w[3][32];
    OwScan3 carry = {0u, 0u, 0u};
    for (uint32_t base = 0; base < nblocks; base += 1024) {
        const uint32_t b = base + threadIdx.x;
        OwScan3 v = {0u, 0u, 0u};
        if (b < nblocks) { v.c = tops[3 * b]; v.m = tops[3 * b + 1]; v.l = tops[3 * b + 2]; }
        OwScan3 total;
        const OwScan3 ex = ow_block_scan3(v, total, s_w);
        if (b < nblocks) { tops[3 * b] = carry.c + ex.c; tops[3 * b + 1] = carry.m + ex.m; tops[3 * b + 2] = carry.l + ex.l; }
        carry.c += total.c; carry.m += total.m; carry.l += total.l;
    }
    if (threadIdx.x == 0) { bin_offset[g.onbins] = carry.c; *nitems = carry.m; ctl[0] = carry.l; ctl[1] = 0; }
}

// SINGLE = 1: the whole histogram fits one CTA (<= 4096 bins): no reduce / tops launches, this kernel also writes the totals.
// SINGLE = 2: chained scan in ONE launch for up to 1024 CTAs: a CTA publishes its totals (tops[4 b + 0..2], then the flag
// tops[4 b + 3]), waits for the flags of the CTAs before it and adds their totals up.  b is the CTA's arrival ticket
// (tops[4 nblocks + 1]), so a CTA only ever waits for CTAs that are already running; the last CTA to have read
// its predecessors clears the flags for the next launch (tops[4 nblocks] counts them), so there is no state to reset.
template <int SINGLE>
__global__ void __launch_bounds__(1024) k_owner_scan_write(const Geom g, uint32_t* __restrict__ bin_count,
                                                           uint32_t* __restrict__ cursor,
                                                           const uint32_t item_size, uint32_t* tops,
                                                           uint32_t* __restrict__ bin_offset, OwItem* __restrict__ items,
                                                           uint4* __restrict__ work, uint32_t* __restrict__ nitems,
                                                           uint32_t* __restrict__ ctl, uint32_t* __restrict__ valid_reset) {
    __shared__ uint32_t s_w[3][32];
    __shared__ uint32_t s_me;
    uint32_t blk = blockIdx.x;
    if (SINGLE == 2) {                                                // block index = arrival ticket: a CTA only waits for CTAs that run
        if (threadIdx.x == 0) s_me = atomicAdd(&tops[4 * gridDim.x + 1], 1u);
        __syncthreads();
        blk = s_me;
    }
    const uint32_t b0 = blk * 4096u + 4u * threadIdx.x;
    uint32_t c[4], m[4];
    const OwScan3 t = ow_load4(g, bin_count, b0, item_size, c, m);
    if (t.c) *reinterpret_cast<uint4*>(bin_count + b0) = make_uint4(0, 0, 0, 0);      // ready for the next call's O1
    if (b0 < g.onbins) *reinterpret_cast<uint4*>(cursor + b0) = make_uint4(0, 0, 0, 0);   // ready for this call's O3
    if (valid_reset && b0 < g.onbins) *reinterpret_cast<uint4*>(valid_reset + b0) = make_uint4(0, 0, 0, 0);   // first call after a reset
    OwScan3 total;
    const OwScan3 ex = ow_block_scan3(t, total, s_w);
    uint32_t off = ex.c, slot = ex.m, wpos = ex.l;
    if (SINGLE == 1) {
        if (threadIdx.x == 0) { bin_offset[g.onbins] = total.c; *nitems = total.m; ctl[0] = total.l; ctl[1] = 0; }
    } else if (SINGLE == 2) {
        __shared__ uint32_t s_base[3];
        volatile uint32_t* vt = tops;
        const uint32_t me = blk, nb = gridDim.x;
        if (threadIdx.x == 0) {
            vt[4 * me] = total.c; vt[4 * me + 1] = total.m; vt[4 * me + 2] = total.l;
            __threadfence();
            vt[4 * me + 3] = 1u;
        }
        OwScan3 pre = {0u, 0u, 0u};
        if (threadIdx.x < me) {                                       // predecessor threadIdx.x (me < 1024)
            while (vt[4 * threadIdx.x + 3] == 0u) {}
            __threadfence();
            pre.c = vt[4 * threadIdx.x]; pre.m = vt[4 * threadIdx.x + 1]; pre.l = vt[4 * threadIdx.x + 2];
        }
        OwScan3 sum;
        ow_block_scan3(pre, sum, s_w);                                // (only the block sum is used)
        if (threadIdx.x == 0) {
            s_base[0] = sum.c; s_base[1] = sum.m; s_base[2] = sum.l;
            if (me == nb - 1u) { bin_offset[g.onbins] = sum.c + total.c; *nitems = sum.m + total.m; ctl[0] = sum.l + total.l; ctl[1] = 0; }
            if (atomicAdd(&tops[4 * nb], 1u) == nb - 1u) {            // everybody has read its predecessors: re-arm
                for (uint32_t i = 0; i < nb; ++i) vt[4 * i + 3] = 0u;
                vt[4 * nb] = 0u; vt[4 * nb + 1] = 0u;
            }
        }
        __syncthreads();
        off += s_base[0]; slot += s_base[1]; wpos += s_base[2];
    } else {
        off += tops[3 * blockIdx.x]; slot += tops[3 * blockIdx.x + 1]; wpos += tops[3 * blockIdx.x + 2];
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t b = b0 + j;
        if (b < g.onbins) {
            bin_offset[b] = off;
            if (c[j] != 0u && m[j] == 0u) {                            // light non-empty tile: one work unit
                const uint32_t gi = b / (uint32_t)g.ontiles, tile = b - gi * (uint32_t)g.ontiles;
                const uint32_t ty = tile / (uint32_t)g.otx;
                work[wpos++] = make_uint4(off, gi, (ty << 16) | (tile - ty * (uint32_t)g.otx), c[j]);
            }
            for (uint32_t q = 0; q < m[j]; ++q) {
                OwItem it;
                it.bin = b; it.start = off + q * item_size; it.count = min(item_size, c[j] - q * item_size);
                it.first_slot = slot; it.nchunks = m[j]; it.chunk = q;
                items[slot + q] = it;
            }
        }
        off += c[j]; slot += m[j];
    }
}

// ------------------------------------------------------------------------------------------------- O3 scatter
// Record: {wt*Re, +-wt*Im, wt, key | X << 10 | Y << 20}.  (ox, oy) = first footprint cell relative to the tile
// origin, plus 6, in [0, 38); key = (oy >> 1) << 5 | ox >> 1 names the 8 x 8 register window (rows 2*(oy>>1) - 6 ...
// + 7, columns 2*(ox>>1) - 6 ... + 7 of the tile) that holds the 7 x 7 footprint; (ox & 1, oy & 1) is the
// footprint's offset inside it; X = (ox&1)*(Q+1) + rx and Y = (oy&1)*(Q+1) + ry select the rows of the two-parity
// table TT2 (rx = Q/2 - ru, ry = Q/2 - rv in [0, Q]).
__device__ __forceinline__ void ow_write_record(const Geom& g, const OwLoc& L, int s, int tx, int ty, uint4* dst) {
    const int h = (g.S - 1) >> 1;
    const int ox = L.cu[s] - (tx * kOwTW - kOwTW / 2) + h;
    const int oy = L.cv[s] - ((g.ny >> 1) + ty * kTile) + h;
    uint4 o;
    o.x = __float_as_uint(L.re);
    o.y = __float_as_uint(s ? -L.im : L.im);
    o.z = __float_as_uint(L.wt);
    const uint32_t X = (uint32_t)((ox & 1) * (g.Q + 1) + L.rx[s]);
    const uint32_t Y = (uint32_t)((oy & 1) * (g.Q + 1) + L.ry[s]);
    o.w = (uint32_t)((oy >> 1) << kOwKXB | ox >> 1) | (X << (5 + kOwKXB)) | (Y << (15 + kOwKXB));
    *dst = o;
}

// Same CTA -> visibility mapping as k_owner_count.  The CTA's per-tile counts of its reference grid come from cta_hist:
// it reserves a run in each touched tile (one global atomic per tile), then hands out the positions inside the runs with
// the shared counters; records of other grids take warp-aggregated global cursors.
__global__ void __launch_bounds__(kBinThreads, 4) k_owner_scatter(const Geom g, const uint4* __restrict__ loc,
                                                               const float* __restrict__ uvw, const double* __restrict__ freq,
                                                               const float2* __restrict__ vis,
                                                               const float* __restrict__ weight, const int* __restrict__ grid_id,
                                                               const long long nvis, const int iters,
                                                               const uint32_t* __restrict__ bin_offset,
                                                               const uint32_t* __restrict__ cta_hist,
                                                               uint32_t* __restrict__ cursor, uint4* __restrict__ sorted,
                                                               int* __restrict__ cnt) {
    extern __shared__ uint32_t s_hist[];
    const long long base = (long long)blockIdx.x * kBinThreads * iters;
    const int lane = threadIdx.x & 31;
    const bool fits = g.ontiles <= kBinSmemTiles;
    const int ref = grid_id ? grid_id[base] : 0;
    uint32_t* s_base = s_hist + g.ontiles;                             // global position of this CTA's run in each tile
    if (fits) {
        const bool ok = ref >= 0 && ref < g.ngrids;
        const uint32_t gbase = ok ? (uint32_t)ref * (uint32_t)g.ontiles : 0u;
        const uint32_t* mine = cta_hist + (size_t)blockIdx.x * g.ontiles;
        for (int i = threadIdx.x; i < g.ontiles; i += kBinThreads) {
            const uint32_t n = mine[i];
            s_hist[i] = 0;
            if (n && ok) s_base[i] = bin_offset[gbase + i] + atomicAdd(&cursor[gbase + i], n);
        }
    }
    __syncthreads();
    // the loads of a visibility do not depend on one another (flagged visibilities are rare: vis / weight are read
    // unconditionally) and are issued one iteration ahead
    struct ScIn { uint4 o; float2 V; float wt; int gid; };
    auto load = [&](const long long k) {
        ScIn r;
        r.o = make_uint4(0u, 0u, 0u, 0u); r.V = make_float2(0.f, 0.f); r.wt = 0.f; r.gid = 0;
        if (k < nvis) {
            r.o = __ldg(loc + k);
            if (vis) r.V = __ldg(vis + k);
            r.wt = __ldg(weight + k);
            if (grid_id) r.gid = __ldg(grid_id + k);
        }
        return r;
    };
    ScIn nxt = load(base + threadIdx.x);
    for (int it = 0; it < iters; ++it) {
        const long long k = base + (long long)it * kBinThreads + threadIdx.x;
        const ScIn cur = nxt;
        if (it + 1 < iters) nxt = load(k + kBinThreads);
        OwLoc L;
        L.state = 0;
        if (k < nvis) {                                               // k_owner_count's integer decisions
            const uint4 o = cur.o;
            L.state = (int)(o.z >> 30);
            if (L.state == 3) {
                L.cu[0] = (int)(o.x & 0xFFFFu); L.cv[0] = (int)(o.x >> 16);
                L.cu[1] = (int)(o.y & 0xFFFFu); L.cv[1] = (int)(o.y >> 16);
                L.rx[0] = (int)(o.z & 511u); L.ry[0] = (int)((o.z >> 9) & 511u); L.rx[1] = (int)((o.z >> 18) & 511u);
                L.ry[1] = (int)(o.w & 511u);
                float2 V = cur.V;
                if (g.phase_on) V = phase_rotate(g, uvw[3 * k], uvw[3 * k + 1], freq[k], V);
                const float wt = cur.wt;
                L.re = wt * V.x; L.im = wt * V.y; L.wt = wt; L.gid = cur.gid;
                if (cnt) {                                            // NEXT-2: one hit per sample at its nearest cell (stored half-plane)
#pragma unroll
                    for (int s = 0; s < 2; ++s)
                        if (L.cv[s] >= (g.ny >> 1))
                            atomicAdd(cnt + ((size_t)L.gid * g.ny + L.cv[s]) * g.nx + L.cu[s], 1);
                }
            }
        }
        const bool kept = L.state == 3;
        const bool local = fits && kept && L.gid == ref;
        if (local) {
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const OwTiles t = ow_tiles(g, L.cu[s], L.cv[s]);
                if (!t.up) continue;
                ow_write_record(g, L, s, t.tx0, t.ty0, sorted + s_base[t.t00] + atomicAdd(&s_hist[t.t00], 1u));
                if (t.mx) ow_write_record(g, L, s, t.tx0 + 1, t.ty0, sorted + s_base[t.t00 + 1] + atomicAdd(&s_hist[t.t00 + 1], 1u));
                if (t.my)
                    ow_write_record(g, L, s, t.tx0, t.ty0 + 1,
                                    sorted + s_base[t.t00 + g.otx] + atomicAdd(&s_hist[t.t00 + g.otx], 1u));
                if (t.mx && t.my)
                    ow_write_record(g, L, s, t.tx0 + 1, t.ty0 + 1,
                                    sorted + s_base[t.t00 + g.otx + 1] + atomicAdd(&s_hist[t.t00 + g.otx + 1], 1u));
            }
        }
        if (__any_sync(kFull, kept && !local)) {
#pragma unroll
            for (int s = 0; s < 2; ++s) {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    int tx = 0, ty = 0;
                    const uint32_t bin = (kept && !local) ? ow_bin(g, L.gid, L.cu[s], L.cv[s], q, tx, ty) : kNoBin;
                    if (!__any_sync(kFull, bin != kNoBin)) continue;
                    const uint32_t rank = ow_agg_inc(cursor, bin, lane);
                    if (bin != kNoBin) ow_write_record(g, L, s, tx, ty, sorted + bin_offset[bin] + rank);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------- O1r / O3r rows
// NEXT-1, the channelised entry point (a 3 ms frame is 16 channels x 2 polarisations of the SAME baselines):
//   uvw_m [ntime][nrow][3], freq_hz [nchan], vis / weight [ntime][npol][nchan][nrow], 12.4 bytes per visibility.
// An ELEMENT is (t, po, c, r): one baseline at one channel.  Its O1 coordinates are computed once -- f/c once per channel
// and CTA -- and shared by the polarisations of the element: in SUM mode (npo = 1, npi = npol) they all go onto one
// grid, so their weighted visibilities and weights are added up BEFORE gridding and the element becomes one record
// per sample instead of npol (identical cells and kernel weights; only the order of the fp32 sums changes); in SPLIT mode
// (npo = npol, npi = 1) every polarisation has its own grid.  From the records on, the path is the flat one.
struct RowsShape { int ntime, npo, npi, nchan, nrow; };

// the polarisations p = po + pi of one element: flag, drop or keep each; sums over the kept ones
struct RowsSum { int kept, flagged; float re, im, wt; double wsum, v2sum, w2sum; };
__device__ __forceinline__ RowsSum rows_sum_pols(const Geom& g, const RowsShape& sh, const float2* __restrict__ vis,
                                                 const float* __restrict__ weight, const int t, const int po, const int c,
                                                 const int r, const bool geom_ok, const bool inside, const float um,
                                                 const float vm, const double f) {
    RowsSum o = {0, 0, 0.f, 0.f, 0.f, 0.0, 0.0, 0.0};
    const int npol = sh.npo * sh.npi;
#pragma unroll 2
    for (int pi = 0; pi < sh.npi; ++pi) {
        const size_t k = (((size_t)t * npol + (po + pi)) * sh.nchan + c) * sh.nrow + r;
        float2 V = vis ? vis[k] : make_float2(0.f, 0.f);
        const float wt = weight[k];
        if (!(geom_ok && isfinite(wt) && isfinite(V.x) && isfinite(V.y) && wt > 0.0f)) { ++o.flagged; continue; }
        if (!inside) continue;
        ++o.kept;
        o.wsum += 2.0 * (double)wt;
        const double w2 = (double)wt * (double)wt;
        o.w2sum += w2;
        o.v2sum += w2 * ((double)V.x * (double)V.x + (double)V.y * (double)V.y);
        if (g.phase_on) V = phase_rotate(g, um, vm, f, V);
        o.re += wt * V.x; o.im += wt * V.y; o.wt += wt;
    }
    return o;
}

// element -> (t, po, c, r), coordinates and keep/drop of its two samples (same arithmetic as ow_locate)
// A CTA handles 256 rows of ONE (t, po) and a GROUP of `cpc` consecutive channels, looping over them: blockIdx.y =
// (t * npo + po) * ncg + channel group (folded over gridDim.y, gridDim.z), blockIdx.x = block of rows.  The per-CTA work
// (histogram zeroing and flush, statistics reduction) is shared by the channels of the group.
struct RowsElem { int t, po, c, r, gid; bool geom_ok, inside; float um, vm; double f; OwLoc L; };
__device__ __forceinline__ void rows_block(const RowsShape& sh, const int cpc, int& t, int& po, int& c0) {
    const unsigned ncg = (unsigned)((sh.nchan + cpc - 1) / cpc);
    const unsigned tpc = blockIdx.y + blockIdx.z * gridDim.y;
    c0 = (int)(tpc % ncg) * cpc;
    const unsigned tp = tpc / ncg;
    po = (int)(tp % (unsigned)sh.npo);
    t = (int)(tp / (unsigned)sh.npo);
}
__device__ __forceinline__ size_t rows_cta(void) { return blockIdx.x + (size_t)gridDim.x * (blockIdx.y + (size_t)gridDim.y * blockIdx.z); }
__device__ __forceinline__ void rows_locate(const Geom& g, const RowsShape& sh, const float* __restrict__ uvw,
                                            const double f, const double il, const int gid, const int t, const int po,
                                            const int c, const int r, const OwAxes& ax, RowsElem& E) {
    E.t = t; E.po = po; E.c = c; E.r = r;
    const size_t ub = ((size_t)E.t * sh.nrow + E.r) * 3;
    const float um = uvw[ub], vm = uvw[ub + 1], wm = uvw[ub + 2];
    E.um = um; E.vm = vm; E.f = f;
    E.gid = gid;
    const double ul = __dmul_rn((double)um, il), vl = __dmul_rn((double)vm, il), wl = __dmul_rn((double)wm, il);
    E.geom_ok = isfinite(ul) && isfinite(vl) && isfinite(wl) && isfinite(E.f) && E.gid >= 0 && E.gid < g.ngrids;
    E.inside = false;
    if (!E.geom_ok) return;
    const int h = (g.S - 1) >> 1;
    const double xu = __dmul_rn(ul, g.su), xv = __dmul_rn(vl, g.sv);
    bool inside = fabs(xu) < 1.0e9 && fabs(xv) < 1.0e9;
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        int iu, iv, ru, rv;
        ow_cell_phase(s ? -xu : xu, ax.hx, ax.Qd, iu, ru);
        ow_cell_phase(s ? -xv : xv, ax.hy, ax.Qd, iv, rv);
        inside = inside && iu >= h + 1 && iu <= g.nx - 1 - h && iv >= h + 1 && iv <= g.ny - 1 - h;
        E.L.cu[s] = iu; E.L.cv[s] = iv;
        E.L.rx[s] = g.Q / 2 - ru; E.L.ry[s] = g.Q / 2 - rv;
    }
    E.inside = inside;
}

constexpr int kRowsMaxChan = 65535;

constexpr int kRowsMaxCpc = 32;                                       // channels a CTA loops over

__global__ void __launch_bounds__(kBinThreads, 4) k_rows_count(const Geom g, const RowsShape sh, const int cpc,
                                                               const float* __restrict__ uvw, const double* __restrict__ freq,
                                                               const float2* __restrict__ vis, const float* __restrict__ weight,
                                                               const int* __restrict__ grid_id, uint32_t* __restrict__ bin_count,
                                                               uint32_t* __restrict__ cta_hist, Stats* __restrict__ stats,
                                                               uint4* __restrict__ loc) {
    extern __shared__ uint32_t s_hist[];
    __shared__ double s_il[kRowsMaxCpc];
    int t, po, c0;
    rows_block(sh, cpc, t, po, c0);
    if (t >= sh.ntime) return;                                        // padding of the folded launch grid (whole CTA)
    const int r = blockIdx.x * kBinThreads + threadIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool fits = g.ontiles <= kBinSmemTiles;
    if (fits)
        for (int i = threadIdx.x; i < g.ontiles; i += kBinThreads) s_hist[i] = 0;
    const int nc = min(cpc, sh.nchan - c0);
    if (threadIdx.x < nc) s_il[threadIdx.x] = __ddiv_rn(freq[c0 + threadIdx.x], kC);   // f / c once per channel and CTA
    const int* gids = grid_id ? grid_id + ((size_t)t * sh.npo + po) * sh.nchan : nullptr;
    const int ref = gids ? gids[c0] : 0;
    __syncthreads();
    int kept = 0, dropped = 0, flagged = 0;
    double wsum = 0.0, v2sum = 0.0, w2sum = 0.0;
    const OwAxes ax = ow_axes(g);
    for (int ci = 0; ci < nc; ++ci) {
        const int c = c0 + ci;
        const int gid = gids ? gids[c] : 0;
        uint32_t tp[2] = {0u, 0u};
        if (r < sh.nrow) {
            RowsElem E;
            rows_locate(g, sh, uvw, freq[c], s_il[ci], gid, t, po, c, r, ax, E);
            const RowsSum S = rows_sum_pols(g, sh, vis, weight, E.t, E.po, E.c, E.r, E.geom_ok, E.inside, E.um, E.vm, E.f);
            kept += S.kept; flagged += S.flagged; dropped += sh.npi - S.kept - S.flagged;
            wsum += S.wsum; v2sum += S.v2sum; w2sum += S.w2sum;
            uint4 o = make_uint4(0u, 0u, (S.kept ? 3u : 0u) << 30, 0u);
            if (S.kept) {
                o.x = (uint32_t)E.L.cu[0] | ((uint32_t)E.L.cv[0] << 16);
                o.y = (uint32_t)E.L.cu[1] | ((uint32_t)E.L.cv[1] << 16);
                o.z |= (uint32_t)E.L.rx[0] | ((uint32_t)E.L.ry[0] << 9) | ((uint32_t)E.L.rx[1] << 18);
                o.w = (uint32_t)E.L.ry[1];
                tp[0] = ow_tiles_packed(g, E.L.cu[0], E.L.cv[0]);
                tp[1] = ow_tiles_packed(g, E.L.cu[1], E.L.cv[1]);
            }
            loc[(((size_t)t * sh.npo + po) * sh.nchan + c) * sh.nrow + r] = o;
        }
        const bool local = fits && gid == ref;                        // uniform over the CTA
        if (local) {
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const uint32_t tt = tp[s];
                if (!(tt >> 31)) continue;
                const uint32_t t00 = tt & 0x1FFFFFFFu;
                const bool mx = (tt >> 29) & 1u, my = (tt >> 30) & 1u;
                atomicAdd(&s_hist[t00], 1u);
                if (mx) atomicAdd(&s_hist[t00 + 1], 1u);
                if (my) atomicAdd(&s_hist[t00 + g.otx], 1u);
                if (mx && my) atomicAdd(&s_hist[t00 + g.otx + 1], 1u);
            }
        } else {
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t tt = tp[s];
                    const bool on = (tt >> 31) && (!(q & 1) || ((tt >> 29) & 1u)) && (!(q & 2) || ((tt >> 30) & 1u));
                    const uint32_t bin = on ? (uint32_t)gid * (uint32_t)g.ontiles + (tt & 0x1FFFFFFFu) + (q & 1) +
                                                  ((q & 2) ? (uint32_t)g.otx : 0u)
                                            : kNoBin;
                    if (__any_sync(kFull, on)) ow_agg_inc(bin_count, bin, lane);
                }
        }
    }
    __syncthreads();
    if (fits) {
        const bool ok = ref >= 0 && ref < g.ngrids;
        const uint32_t gbase = ok ? (uint32_t)ref * (uint32_t)g.ontiles : 0u;
        uint32_t* mine = cta_hist + rows_cta() * g.ontiles;
        for (int i = threadIdx.x; i < g.ontiles; i += kBinThreads) {
            const uint32_t n = s_hist[i];
            mine[i] = n;
            if (n && ok) atomicAdd(&bin_count[gbase + i], n);
        }
    }
    __shared__ int s_cnt[3][8];
    __shared__ double s_w[3][8];
    const int q0 = __reduce_add_sync(kFull, kept), q1 = __reduce_add_sync(kFull, dropped), q2 = __reduce_add_sync(kFull, flagged);
    for (int o = 16; o > 0; o >>= 1) {
        wsum += __shfl_xor_sync(kFull, wsum, o);
        v2sum += __shfl_xor_sync(kFull, v2sum, o);
        w2sum += __shfl_xor_sync(kFull, w2sum, o);
    }
    if (lane == 0) { s_cnt[0][warp] = q0; s_cnt[1][warp] = q1; s_cnt[2][warp] = q2; s_w[0][warp] = wsum; s_w[1][warp] = v2sum; s_w[2][warp] = w2sum; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int t0 = 0, t1 = 0, t2 = 0;
        double tw = 0.0, tv2 = 0.0, tw2 = 0.0;
        for (int w = 0; w < kBinThreads / 32; ++w) {
            t0 += s_cnt[0][w]; t1 += s_cnt[1][w]; t2 += s_cnt[2][w];
            tw += s_w[0][w]; tv2 += s_w[1][w]; tw2 += s_w[2][w];
        }
        if (t0) {
            atomicAdd(&stats->n_gridded, (unsigned long long)t0);
            atomicAdd(&stats->sum_weights, tw);
            atomicAdd(&stats->sum_val2, tv2);
            atomicAdd(&stats->sum_wt2, tw2);
        }
        if (t1) atomicAdd(&stats->n_dropped, (unsigned long long)t1);
        if (t2) atomicAdd(&stats->n_flagged, (unsigned long long)t2);
    }
}

__global__ void __launch_bounds__(kBinThreads, 5) k_rows_scatter(const Geom g, const RowsShape sh, const int cpc,
                                                                 const uint4* __restrict__ loc, const float* __restrict__ uvw,
                                                                 const double* __restrict__ freq, const float2* __restrict__ vis,
                                                                 const float* __restrict__ weight, const int* __restrict__ grid_id,
                                                                 const uint32_t* __restrict__ bin_offset,
                                                                 const uint32_t* __restrict__ cta_hist,
                                                                 uint32_t* __restrict__ cursor, uint4* __restrict__ sorted,
                                                                 int* __restrict__ cnt) {
    extern __shared__ uint32_t s_hist[];
    int t, po, c0;
    rows_block(sh, cpc, t, po, c0);
    if (t >= sh.ntime) return;
    const int r = blockIdx.x * kBinThreads + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool fits = g.ontiles <= kBinSmemTiles;
    const int nc = min(cpc, sh.nchan - c0);
    const int* gids = grid_id ? grid_id + ((size_t)t * sh.npo + po) * sh.nchan : nullptr;
    const int ref = gids ? gids[c0] : 0;
    uint32_t* s_base = s_hist + g.ontiles;
    if (fits) {
        const bool ok = ref >= 0 && ref < g.ngrids;
        const uint32_t gbase = ok ? (uint32_t)ref * (uint32_t)g.ontiles : 0u;
        const uint32_t* mine = cta_hist + rows_cta() * g.ontiles;
        for (int i = threadIdx.x; i < g.ontiles; i += kBinThreads) {
            const uint32_t n = mine[i];
            s_hist[i] = 0;
            if (n && ok) s_base[i] = bin_offset[gbase + i] + atomicAdd(&cursor[gbase + i], n);
        }
    }
    __syncthreads();
    for (int ci = 0; ci < nc; ++ci) {
        const int c = c0 + ci;
        const int gid = gids ? gids[c] : 0;
        OwLoc L;
        L.state = 0;
        if (r < sh.nrow) {
            const uint4 o = __ldg(loc + (((size_t)t * sh.npo + po) * sh.nchan + c) * sh.nrow + r);
            L.state = (int)(o.z >> 30);
            if (L.state == 3) {
                L.cu[0] = (int)(o.x & 0xFFFFu); L.cv[0] = (int)(o.x >> 16);
                L.cu[1] = (int)(o.y & 0xFFFFu); L.cv[1] = (int)(o.y >> 16);
                L.rx[0] = (int)(o.z & 511u); L.ry[0] = (int)((o.z >> 9) & 511u); L.rx[1] = (int)((o.z >> 18) & 511u);
                L.ry[1] = (int)(o.w & 511u);
                L.gid = gid;
                const size_t ub = ((size_t)t * sh.nrow + r) * 3;
                const RowsSum S = rows_sum_pols(g, sh, vis, weight, t, po, c, r, true, true, uvw[ub], uvw[ub + 1], freq[c]);
                L.re = S.re; L.im = S.im; L.wt = S.wt;
                if (cnt) {                                            // NEXT-2: one hit per visibility and sample
#pragma unroll
                    for (int s = 0; s < 2; ++s)
                        if (L.cv[s] >= (g.ny >> 1)) atomicAdd(cnt + ((size_t)L.gid * g.ny + L.cv[s]) * g.nx + L.cu[s], S.kept);
                }
            }
        }
        const bool kept = L.state == 3;
        if (fits && gid == ref) {                                     // uniform over the CTA
            if (kept) {
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    const OwTiles tt = ow_tiles(g, L.cu[s], L.cv[s]);
                    if (!tt.up) continue;
                    ow_write_record(g, L, s, tt.tx0, tt.ty0, sorted + s_base[tt.t00] + atomicAdd(&s_hist[tt.t00], 1u));
                    if (tt.mx) ow_write_record(g, L, s, tt.tx0 + 1, tt.ty0, sorted + s_base[tt.t00 + 1] + atomicAdd(&s_hist[tt.t00 + 1], 1u));
                    if (tt.my)
                        ow_write_record(g, L, s, tt.tx0, tt.ty0 + 1,
                                        sorted + s_base[tt.t00 + g.otx] + atomicAdd(&s_hist[tt.t00 + g.otx], 1u));
                    if (tt.mx && tt.my)
                        ow_write_record(g, L, s, tt.tx0 + 1, tt.ty0 + 1,
                                        sorted + s_base[tt.t00 + g.otx + 1] + atomicAdd(&s_hist[tt.t00 + g.otx + 1], 1u));
                }
            }
        } else if (__any_sync(kFull, kept)) {
#pragma unroll
            for (int s = 0; s < 2; ++s) {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    int tx = 0, ty = 0;
                    const uint32_t bin = kept ? ow_bin(g, L.gid, L.cu[s], L.cv[s], q, tx, ty) : kNoBin;
                    if (!__any_sync(kFull, bin != kNoBin)) continue;
                    const uint32_t rank = ow_agg_inc(cursor, bin, lane);
                    if (bin != kNoBin) ow_write_record(g, L, s, tx, ty, sorted + bin_offset[bin] + rank);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------- O4 gridding
__device__ __forceinline__ unsigned long long ow_pack(float x, float y) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
    return r;
}
__device__ __forceinline__ float2 ow_unpack(unsigned long long v) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
__device__ __forceinline__ unsigned long long ow_fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
constexpr int kOwPitch = kOwTW + 8; // cells per row of the shared tile (8 pad)
constexpr int kOwKPT = (19 * kOwNKX + 1 + 255) / 256;   // window keys per thread in the scan (2 or 3)
constexpr int kOwKeys = 256 * kOwKPT;                   // 19 x kOwNKX windows (+1 end marker), padded
constexpr int kOwDirect = 32;     // tiles with at most this many samples skip the shared-memory sort
constexpr int kOwUnit = 4096;     // samples counting-sorted together

// shared-memory layout (bytes); the table region is sized by Q at launch
constexpr int kOwOffA = 0;                                  // int2 [32][kOwPitch]  fixed-point (re, im)
constexpr int kOwOffB = kOwOffA + 32 * kOwPitch * 8;        // int  [32][kOwPitch]  fixed-point weight
constexpr int kOwOffH = kOwOffB + 32 * kOwPitch * 4;        // u32  [kOwKeys]       window histogram / run starts
constexpr int kOwOffP = kOwOffH + kOwKeys * 4;              // u16  [kOwUnit] ranks, later 8 warps x 2 x 32 records
constexpr int kOwOffI = kOwOffP + kOwUnit * 2;              // u16  [kOwUnit] record index by sorted position
constexpr int kOwOffT = kOwOffI + kOwUnit * 2;              // f32  [2(Q+1)][8]     two-parity table
static size_t owner_smem_bytes(int Q) { return (size_t)kOwOffT + (size_t)2 * (Q + 1) * 8 * sizeof(float); }

// The shared tile is accumulated in 32-bit FIXED POINT: integer shared-memory adds are native single instructions,
// fp32 adds are compare-and-swap loops.  Per work unit the scale maps the largest possible cell sum (sum of
// |wt*Re V|, |wt*Im V| resp. wt over the unit's records; the kernel never exceeds 1) to 0.98 * 2^31, so a run's
// fp32 register sum is rounded once, by at most 2^-32 of that bound, when it is merged into the tile (the 2 %
// margin covers the fp32 rounding of the bound itself and the half-unit roundings of up to 4096 merges).
struct OwScale {
    float v, w;                    // fixed-point units per unit of value / of weight
};

struct OwWarpAcc {
    unsigned long long a0, a1, b;  // (re, im) of the lane's two cells; (wt, wt') of the two cells
    int off;                       // cell index of the lane's first cell in the shared tile, -1 outside the tile
};

// Point the warp's 8 x 8 register window at window `key`; lane (r, c) holds row r, columns 2c and 2c + 1.
__device__ __forceinline__ void ow_window(OwWarpAcc& A, const uint32_t key, const int r, const int c) {
    const int row = 2 * (int)(key >> kOwKXB) - 6 + r, col0 = 2 * (int)(key & ((1u << kOwKXB) - 1u)) - 6 + 2 * c;
    A.off = (((unsigned)row < 32u) && ((unsigned)col0 < (unsigned)kOwTW)) ? row * kOwPitch + col0 : -1;
    A.a0 = A.a1 = A.b = 0ull;
}

// Merge the window into the shared tile.  The accumulators are already in fixed-point units (ow_stage scales the
// values once per record), so this is six conversions and six native integer adds.
__device__ __forceinline__ void ow_flush(const OwWarpAcc& A, int* sA, int* sB) {
    if (A.off >= 0) {
        const float2 c0 = ow_unpack(A.a0), c1 = ow_unpack(A.a1), w = ow_unpack(A.b);
        int* pa = sA + 2 * A.off;
        atomicAdd(pa + 0, __float2int_rn(c0.x));
        atomicAdd(pa + 1, __float2int_rn(c0.y));
        atomicAdd(pa + 2, __float2int_rn(c1.x));
        atomicAdd(pa + 3, __float2int_rn(c1.y));
        atomicAdd(sB + A.off, __float2int_rn(w.x));
        atomicAdd(sB + A.off + 1, __float2int_rn(w.y));
    }
}

// Staged form of a record, built once by the lane that loads it: values in fixed-point units, table row byte
// offsets (X * 32 | Y * 32 << 16) instead of the packed word.
__device__ __forceinline__ uint4 ow_stage(const uint4 rec, const OwScale sc) {
    uint4 st;
    st.x = __float_as_uint(__uint_as_float(rec.x) * sc.v);
    st.y = __float_as_uint(__uint_as_float(rec.y) * sc.v);
    st.z = __float_as_uint(__uint_as_float(rec.z) * sc.w);
    st.w = ((rec.w >> kOwKXB) & 0x7FE0u) | (((rec.w >> (10 + kOwKXB)) & 0x7FE0u) << 16);
    return st;
}

// One staged sample into the register window.  tbx = table + 2c floats, tby = table + r floats (shared memory).
__device__ __forceinline__ void ow_add(OwWarpAcc& A, const uint4 st, const char* tbx, const char* tby) {
    const float2 kx = *reinterpret_cast<const float2*>(tbx + (st.w & 0xFFFFu));
    const float ky = *reinterpret_cast<const float*>(tby + (st.w >> 16));
    const float k0 = kx.x * ky, k1 = kx.y * ky;
    const unsigned long long v = ow_pack(__uint_as_float(st.x), __uint_as_float(st.y));
    const float wt = __uint_as_float(st.z);
    A.a0 = ow_fma2(ow_pack(k0, k0), v, A.a0);
    A.a1 = ow_fma2(ow_pack(k1, k1), v, A.a1);
    A.b = ow_fma2(ow_pack(k0, k1), ow_pack(wt, wt), A.b);
}

__device__ __forceinline__ uint32_t ow_sortkey(uint32_t w) {
    return ((w >> kOwKXB) & 31u) * (uint32_t)kOwNKX + (w & ((1u << kOwKXB) - 1u));
}

__device__ __forceinline__ float3 ow_warp_sum3(float3 a) {
    for (int o = 16; o > 0; o >>= 1) {
        a.x += __shfl_xor_sync(kFull, a.x, o);
        a.y += __shfl_xor_sync(kFull, a.y, o);
        a.z += __shfl_xor_sync(kFull, a.z, o);
    }
    return a;
}
__device__ __forceinline__ OwScale ow_scale_from(float3 s) {
    OwScale sc;
    sc.v = 2104533975.0f / fmaxf(fmaxf(s.x, s.y), 1e-30f);           // 0.98 * 2^31
    sc.w = 2104533975.0f / fmaxf(s.z, 1e-30f);
    return sc;
}

// Persistent kernel: 4 CTAs per SM pull work units from a device-side counter.  Units [0, nitems) are the chunk items
// of heavy tiles (started first), units [nitems, nitems + nlight) the light non-empty tiles listed by k_owner_scan.
// Empty tiles are not touched: their flag in `valid` stays 0 and every consumer takes them as zeros.
// FIRST: the first call after a reset (the scan has just cleared every flag): every tile is stored
template <int FIRST>
__global__ void __launch_bounds__(256, 4) k_grid_owner_s7(const Geom g, const uint4* __restrict__ sorted,
                                                          const uint32_t* __restrict__ bin_offset,
                                                          const OwItem* __restrict__ items,
                                                          const uint32_t* __restrict__ nitems,
                                                          const uint4* __restrict__ work, uint32_t* __restrict__ ctl,
                                                          const float* __restrict__ tt2, GridPtrs grids,
                                                          float* __restrict__ scratch, uint32_t* __restrict__ tickets,
                                                          uint32_t* __restrict__ valid) {
    extern __shared__ __align__(16) unsigned char smem[];
    int* sA = reinterpret_cast<int*>(smem + kOwOffA);
    int* sB = reinterpret_cast<int*>(smem + kOwOffB);
    uint32_t* sH = reinterpret_cast<uint32_t*>(smem + kOwOffH);
    unsigned short* sP = reinterpret_cast<unsigned short*>(smem + kOwOffP);
    unsigned short* sI = reinterpret_cast<unsigned short*>(smem + kOwOffI);
    float* sT = reinterpret_cast<float*>(smem + kOwOffT);
    __shared__ uint32_t sW[8];
    __shared__ float sSum[8][3];
    __shared__ float sScale[4];                                       // {scale v, scale w, 1/scale v, 1/scale w}
    __shared__ int sLast;
    __shared__ uint32_t sWork;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    {   // stage the two-parity table once per CTA
        const float4* src = reinterpret_cast<const float4*>(tt2);
        float4* dst = reinterpret_cast<float4*>(sT);
        for (int i = tid; i < 2 * (g.Q + 1) * 2; i += 256) dst[i] = __ldg(src + i);
    }
    const int r = lane >> 2, c = lane & 3;
    const char* tbx = reinterpret_cast<const char*>(sT + 2 * c);
    const char* tby = reinterpret_cast<const char*>(sT + r);
    // Work units: [0, n_items) chunks of heavy tiles, then the n_light light non-empty tiles.
    const uint32_t n_items = *nitems, n_light = ctl[0];
    const uint32_t n_work = n_items + n_light;

  for (;;) {
    __syncthreads();                                                  // the previous unit is done with the shared tile
    if (tid == 0) sWork = atomicAdd(&ctl[1], 1u);
    __syncthreads();
    const uint32_t wi = sWork;
    if (wi >= n_work) break;
    uint32_t gi, start, cnt, first_slot = 0, nchunks = 0, chunk = 0;
    int tx, ty;
    const bool heavy = wi < n_items;
    const uint32_t li = wi - n_items;                                 // index into the light-tile list
    if (heavy) {
        const OwItem it = items[wi];
        start = it.start; cnt = it.count; first_slot = it.first_slot; nchunks = it.nchunks; chunk = it.chunk;
        gi = it.bin / (uint32_t)g.ontiles;
        const uint32_t tile = it.bin - gi * (uint32_t)g.ontiles;
        ty = (int)(tile / (uint32_t)g.otx); tx = (int)(tile - (uint32_t)ty * (uint32_t)g.otx);
    } else {
        const uint4 wk = __ldg(work + li);                           // {start, grid, ty << 16 | tx, count}
        start = wk.x; gi = wk.y; ty = (int)(wk.z >> 16); tx = (int)(wk.z & 0xFFFFu); cnt = wk.w;
    }
    // `valid` = 0: the tile has not been written since the last reset -- its cells in G, Gw hold garbage that stands for
    // zeros (nobody zero-fills empty tiles; the row transform skips them): the tile is stored, else added to.  One writer
    // per tile and launch (for a heavy tile: the last chunk to arrive), which also sets the flag.
    uint32_t* vflag = valid + (size_t)gi * g.ontiles + (size_t)ty * g.otx + tx;
    const bool STORE = FIRST ? true : (*vflag == 0u);
    const int x0 = tx * kOwTW - kOwTW / 2, y0 = (g.ny >> 1) + ty * kTile;
    float2* __restrict__ Gt = grids.G + (size_t)gi * g.ny * g.nx;
    float* __restrict__ Wt = grids.Gw + (size_t)gi * g.ny * g.nx;
    {   // zero the fixed-point tile
        int4* za = reinterpret_cast<int4*>(smem + kOwOffA);
        for (int i = tid; i < (kOwOffH - kOwOffA) / 16; i += 256) za[i] = make_int4(0, 0, 0, 0);
    }
    const uint4* __restrict__ recs = sorted + start;
    OwWarpAcc A;
    OwScale sc;

    if (cnt <= (uint32_t)kOwDirect) {
        // every warp derives the scale from all (<= 32) records, then takes every 8th record as a run of one
        float3 s = make_float3(0.f, 0.f, 0.f);
        if ((uint32_t)lane < cnt) {
            const uint4 q = __ldg(recs + lane);
            s = make_float3(fabsf(__uint_as_float(q.x)), fabsf(__uint_as_float(q.y)), __uint_as_float(q.z));
        }
        sc = ow_scale_from(ow_warp_sum3(s));
        if (tid == 0) { sScale[2] = 1.0f / sc.v; sScale[3] = 1.0f / sc.w; }
        __syncthreads();
        for (uint32_t i = warp; i < cnt; i += 8) {
            const uint4 rec = __ldg(recs + i);
            ow_window(A, rec.w & kOwKeyMask, r, c);
            ow_add(A, ow_stage(rec, sc), tbx, tby);
            ow_flush(A, sA, sB);
        }
        __syncthreads();
    } else {
        float3 s = make_float3(0.f, 0.f, 0.f);
        if (cnt > (uint32_t)kOwUnit) {                                // several units: bound over all of them first
            for (uint32_t i = tid; i < cnt; i += 256) {
                const uint4 q = __ldg(recs + i);
                s.x += fabsf(__uint_as_float(q.x)); s.y += fabsf(__uint_as_float(q.y)); s.z += __uint_as_float(q.z);
            }
        }
        for (uint32_t ubase = 0; ubase < cnt; ubase += kOwUnit) {
            const uint32_t n = min((uint32_t)kOwUnit, cnt - ubase);
            const uint4* __restrict__ src = recs + ubase;
            for (int i = tid; i < kOwKeys; i += 256) sH[i] = 0;
            __syncthreads();
            // (1) counting sort of the unit by window (row-major): rank of every record inside its window
            for (uint32_t i = tid; i < n; i += 256) {
                const uint4 q = __ldg(src + i);
                sP[i] = (unsigned short)atomicAdd(&sH[ow_sortkey(q.w)], 1u);
                if (cnt <= (uint32_t)kOwUnit) {
                    s.x += fabsf(__uint_as_float(q.x)); s.y += fabsf(__uint_as_float(q.y)); s.z += __uint_as_float(q.z);
                }
            }
            if (ubase == 0) {
                const float3 t = ow_warp_sum3(s);
                if (lane == 0) { sSum[warp][0] = t.x; sSum[warp][1] = t.y; sSum[warp][2] = t.z; }
            }
            __syncthreads();
            if (ubase == 0 && tid == 0) {
                float3 t = make_float3(0.f, 0.f, 0.f);
                for (int w = 0; w < 8; ++w) { t.x += sSum[w][0]; t.y += sSum[w][1]; t.z += sSum[w][2]; }
                const OwScale q = ow_scale_from(t);
                sScale[0] = q.v; sScale[1] = q.w; sScale[2] = 1.0f / q.v; sScale[3] = 1.0f / q.w;
            }
            {
                uint32_t hk[kOwKPT], tot = 0;
#pragma unroll
                for (int j = 0; j < kOwKPT; ++j) { hk[j] = sH[kOwKPT * tid + j]; tot += hk[j]; }
                uint32_t inc = tot;
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t t = __shfl_up_sync(kFull, inc, o);
                    if (lane >= o) inc += t;
                }
                if (lane == 31) sW[warp] = inc;
                __syncthreads();
                uint32_t ex = inc - tot;
                for (int w = 0; w < warp; ++w) ex += sW[w];
#pragma unroll
                for (int j = 0; j < kOwKPT; ++j) { sH[kOwKPT * tid + j] = ex; ex += hk[j]; }
            }
            __syncthreads();
            sc.v = sScale[0]; sc.w = sScale[1];
            for (uint32_t i = tid; i < n; i += 256) {                  // bit 15: last record of its window
                const uint32_t k = ow_sortkey(__ldg(&src[i].w)), pos = sH[k] + sP[i];
                sI[pos] = (unsigned short)(i | ((pos + 1u == sH[k + 1u]) ? 0x8000u : 0u));
            }
            __syncthreads();
            // (2) every warp streams an equal share of the sorted order through its private 2 x 32-record buffer
            //     (gather loads one batch ahead); runs of equal window stay in registers across batches
            {
                uint4* wb = reinterpret_cast<uint4*>(smem + kOwOffP) + warp * 64;
                const int per = ((int)n + 7) >> 3;
                const int e = min((int)n, (warp + 1) * per);
                int p = warp * per;
                uint4 nxt = make_uint4(0, 0, 0, 0);
                uint32_t nidx = 0;
                if (p + lane < e) { nidx = sI[p + lane]; nxt = __ldg(src + (nidx & 0xFFFu)); }
                int buf = 0;
                bool open = false;                                    // the window in registers continues from the last batch
                while (p < e) {
                    const int m = min(32, e - p);
                    wb[buf * 32 + lane] = ow_stage(nxt, sc);
                    const uint32_t mykey = nxt.w & kOwKeyMask;
                    // a run ends at the last record of its window and at the end of the warp's share; a run that
                    // reaches the end of a batch without either stays in registers for the next batch
                    uint32_t ends = __ballot_sync(kFull, lane < m && ((nidx >> 15) != 0u || (p + 32 >= e && lane == m - 1)));
                    __syncwarp();
                    if (p + 32 + lane < e) { nidx = sI[p + 32 + lane]; nxt = __ldg(src + (nidx & 0xFFFu)); }
                    const uint4* __restrict__ q = wb + buf * 32;
                    int j = 0;
                    uint4 st = q[0];
                    while (j < m) {
                        const bool closes = ends != 0u;
                        const int len = closes ? __ffs(ends) : m - j;  // records j .. j + len - 1 share one window
                        if (!open) ow_window(A, __shfl_sync(kFull, mykey, j), r, c);
                        j += len;
#pragma unroll 2
                        for (int t = len; t > 0; --t) {                // the next record is fetched before this one's FMAs
                            const uint4 cur = st;
                            st = q[min(j - t + 1, 31)];
                            ow_add(A, cur, tbx, tby);
                        }
                        if (closes) ow_flush(A, sA, sB);
                        open = !closes;
                        ends = len < 32 ? ends >> len : 0u;
                    }
                    buf ^= 1;
                    p += 32;
                }
            }
            __syncthreads();
        }
    }

    // (3) output: fixed point -> fp32
    const float iv = sScale[2], iw = sScale[3];
    float4* part = nullptr;
    if (heavy) part = reinterpret_cast<float4*>(scratch + (size_t)(first_slot + chunk) * kOwTileFloats);
    constexpr int kG4 = kOwTW / 2, kW4 = kOwTW / 4;                   // float4 per tile row of G / H and of Gw
    if (!heavy) {
        // a thread owns one 16-byte column chunk and walks down the rows: addresses advance by constants
        {
            constexpr int kStep = 256 / kG4;
            const int c2 = tid % kG4, r0 = tid / kG4, gx = x0 + 2 * c2;
            if ((unsigned)gx < (unsigned)g.nx) {
                const int* pa = sA + 2 * (r0 * kOwPitch + 2 * c2);
                const long long goff = (long long)(y0 + r0) * g.nx + gx;   // before the grid for gy < 0: not dereferenced
                float4* gd = reinterpret_cast<float4*>(Gt + goff);
                const size_t gstep = (size_t)kStep * (g.nx >> 1);
#pragma unroll
                for (int k = 0; k < 32 / kStep; ++k) {
                    if ((unsigned)(y0 + r0 + k * kStep) < (unsigned)g.ny) {
                        const int4 a = *reinterpret_cast<const int4*>(pa + 2 * k * kStep * kOwPitch);
                        float4 v = make_float4((float)a.x * iv, (float)a.y * iv, (float)a.z * iv, (float)a.w * iv);
                        if (!STORE) { const float4 o = gd[k * gstep]; v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w; }
                        gd[k * gstep] = v;
                    }
                }
            }
        }
        {
            constexpr int kStep = 256 / kW4;
            const int c4 = tid % kW4, r0 = tid / kW4, gx = x0 + 4 * c4;
            if ((unsigned)gx < (unsigned)g.nx) {
                const int* pb = sB + r0 * kOwPitch + 4 * c4;
                float4* wd = reinterpret_cast<float4*>(Wt + ((long long)(y0 + r0) * g.nx + gx));
                const size_t wstep = (size_t)kStep * (g.nx >> 2);
#pragma unroll
                for (int k = 0; k < 32 / kStep; ++k) {
                    if ((unsigned)(y0 + r0 + k * kStep) < (unsigned)g.ny) {
                        const int4 a = *reinterpret_cast<const int4*>(pb + k * kStep * kOwPitch);
                        float4 v = make_float4((float)a.x * iw, (float)a.y * iw, (float)a.z * iw, (float)a.w * iw);
                        if (!STORE) { const float4 o = wd[k * wstep]; v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w; }
                        wd[k * wstep] = v;
                    }
                }
            }
        }
        if (tid == 0) *vflag = 1u;
        continue;
    }
    for (int i = tid; i < 32 * kG4; i += 256) {                       // heavy chunk: publish the partial tile
        const int row = i / kG4, c2 = i % kG4;
        const int4 a = *reinterpret_cast<const int4*>(sA + 2 * (row * kOwPitch + 2 * c2));
        __stcg(part + i, make_float4((float)a.x * iv, (float)a.y * iv, (float)a.z * iv, (float)a.w * iv));
    }
    for (int i = tid; i < 32 * kW4; i += 256) {
        const int row = i / kW4, c4 = i % kW4;
        const int4 a = *reinterpret_cast<const int4*>(sB + row * kOwPitch + 4 * c4);
        __stcg(part + 32 * kG4 + i, make_float4((float)a.x * iw, (float)a.y * iw, (float)a.z * iw, (float)a.w * iw));
    }
    // heavy tile: the partial tiles are added up in two levels, always in chunk order.  The chunks form groups of G
    // (G^2 >= nchunks); the last chunk of a GROUP to arrive sums its group into the group's first slot, the last group to
    // finish sums the group sums and writes the tile.  One CTA reading all nchunks x 24 KB (37 chunks for the central tile
    // of a single MUSER-II frame) was the critical path of a single frame; no CTA ever waits for another.
    uint32_t G = 2;
    while (G * G < nchunks) ++G;
    const uint32_t ngroups = (nchunks + G - 1u) / G, g0 = (chunk / G) * G, gn = min(G, nchunks - g0);
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        const uint32_t t = atomicAdd(&tickets[first_slot + g0], 1u);   // group counters sit at the groups' first slots
        sLast = (t == gn - 1u);
    }
    __syncthreads();
    if (!sLast) continue;
    __threadfence();
    float4* parts = reinterpret_cast<float4*>(scratch + (size_t)first_slot * kOwTileFloats);
    auto sum_slots = [&](const int i, const uint32_t first, const uint32_t count, const uint32_t stride) -> float4 {
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        for (uint32_t q = 0; q < count; ++q) {
            const float4 p = __ldcg(parts + (size_t)(first + q * stride) * (kOwTileFloats / 4) + i);
            v.x += p.x; v.y += p.y; v.z += p.z; v.w += p.w;
        }
        return v;
    };
    if (ngroups > 1u) {
        for (int i = tid; i < kOwTileFloats / 4; i += 256) __stcg(parts + (size_t)g0 * (kOwTileFloats / 4) + i, sum_slots(i, g0, gn, 1u));
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            const uint32_t t = atomicAdd(&tickets[first_slot + 1u], 1u);   // tile counter (slot 1 is never a group's first: G >= 2)
            sLast = (t == ngroups - 1u);
        }
        __syncthreads();
        if (!sLast) continue;
        __threadfence();
    }
    const uint32_t nsl = ngroups > 1u ? ngroups : nchunks, stride = ngroups > 1u ? G : 1u;
    for (int j = tid; j < 32 * kW4; j += 256) {                       // weights first
        float4 v = sum_slots(32 * kG4 + j, 0u, nsl, stride);
        const int gx = x0 + 4 * (j % kW4), gy = y0 + (j / kW4);
        if ((unsigned)gx < (unsigned)g.nx && (unsigned)gy < (unsigned)g.ny) {
            float4* dst = reinterpret_cast<float4*>(Wt + (size_t)gy * g.nx + gx);
            if (!STORE) { const float4 o = *dst; v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w; }
            *dst = v;
        }
    }
    for (int i = tid; i < 32 * kG4; i += 256) {
        float4 v = sum_slots(i, 0u, nsl, stride);
        const int gx = x0 + 2 * (i % kG4), gy = y0 + (i / kG4);
        if ((unsigned)gx < (unsigned)g.nx && (unsigned)gy < (unsigned)g.ny) {
            float4* dst = reinterpret_cast<float4*>(Gt + (size_t)gy * g.nx + gx);
            if (!STORE) { const float4 o = *dst; v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w; }
            *dst = v;
        }
    }
    for (uint32_t q = tid; q < ngroups; q += 256) tickets[first_slot + q * G] = 0;
    if (tid == 0) tickets[first_slot + 1u] = 0;
    if (tid == 0) *vflag = 1u;
  }
}

// ------------------------------------------------------------------------------------------------- launchers
static size_t bin_smem_bytes(const Geom& g) { return g.ontiles <= kBinSmemTiles ? (size_t)2 * g.ontiles * sizeof(uint32_t) : 0; }

// visibilities per thread of the binning kernels (MUSER_TUNE_BIN_ITERS): a CTA loops over `iters` blocks of 256
int owner_bin_iters(long long nvis, int forced) {
    if (forced >= 1 && forced <= 64) return forced;
    // enough CTAs to fill the machine a few times over, else one block per CTA (a single small frame)
    int it = 8;
    while (it > 1 && nvis / (kBinThreads * it) < 148 * 8) it >>= 1;
    return it;
}
size_t owner_bin_ctas(long long nvis, int iters) { return (size_t)((nvis + (long long)kBinThreads * iters - 1) / ((long long)kBinThreads * iters)); }

cudaError_t launch_owner_count(const Geom& g, const float* uvw, const double* freq, const float2* vis, const float* wt,
                               const int* grid_id, long long nvis, uint32_t* bin_count, uint32_t* cta_hist, Stats* stats,
                               uint4* loc, int iters, cudaStream_t s) {
    k_owner_count<<<(unsigned)owner_bin_ctas(nvis, iters), kBinThreads, bin_smem_bytes(g), s>>>(
        g, uvw, freq, vis, wt, grid_id, nvis, iters, bin_count, cta_hist, stats, loc);
    return cudaGetLastError();
}

cudaError_t launch_owner_scatter(const Geom& g, const uint4* loc, const float* uvw, const double* freq, const float2* vis,
                                 const float* wt, const int* grid_id, long long nvis, const uint32_t* bin_offset,
                                 const uint32_t* cta_hist, uint32_t* cursor, uint4* sorted, int* cnt, int iters,
                                 cudaStream_t s) {
    k_owner_scatter<<<(unsigned)owner_bin_ctas(nvis, iters), kBinThreads, bin_smem_bytes(g), s>>>(
        g, loc, uvw, freq, vis, wt, grid_id, nvis, iters, bin_offset, cta_hist, cursor, sorted, cnt);
    return cudaGetLastError();
}

// channels per CTA of the rows kernels: enough CTAs to fill the machine a few times over
int rows_cpc(int ntime, int npo, int nchan, int nrow) {
    int cpc = nchan < kRowsMaxCpc ? nchan : kRowsMaxCpc;
    const long long rb = (nrow + kBinThreads - 1) / kBinThreads;
    while (cpc > 1 && rb * ntime * npo * ((nchan + cpc - 1) / cpc) < 148LL * 8) cpc = (cpc + 1) / 2;
    return cpc;
}
static dim3 rows_grid(const RowsShape& sh, int cpc) {
    // x: blocks of 256 rows; (t, po, channel group) folded over y (<= 32768) and z
    const unsigned tpc = (unsigned)sh.ntime * (unsigned)sh.npo * (unsigned)((sh.nchan + cpc - 1) / cpc);
    const unsigned gy = tpc < 32768u ? tpc : 32768u;
    return dim3((unsigned)((sh.nrow + kBinThreads - 1) / kBinThreads), gy, (tpc + gy - 1) / gy);
}
size_t rows_ctas(int ntime, int npol, int nchan, int nrow, int pols_split, int cpc) {
    const RowsShape sh = {ntime, pols_split ? npol : 1, pols_split ? 1 : npol, nchan, nrow};
    const dim3 d = rows_grid(sh, cpc);
    return (size_t)d.x * d.y * d.z;
}

cudaError_t launch_rows_count(const Geom& g, int ntime, int npol, int nchan, int nrow, int pols_split, int cpc, const float* uvw,
                              const double* freq, const float2* vis, const float* wt, const int* grid_id, uint32_t* bin_count,
                              uint32_t* cta_hist, Stats* stats, uint4* loc, cudaStream_t s) {
    const RowsShape sh = {ntime, pols_split ? npol : 1, pols_split ? 1 : npol, nchan, nrow};
    k_rows_count<<<rows_grid(sh, cpc), kBinThreads, bin_smem_bytes(g), s>>>(g, sh, cpc, uvw, freq, vis, wt, grid_id, bin_count,
                                                                           cta_hist, stats, loc);
    return cudaGetLastError();
}

cudaError_t launch_rows_scatter(const Geom& g, int ntime, int npol, int nchan, int nrow, int pols_split, int cpc,
                                const uint4* loc, const float* uvw, const double* freq, const float2* vis, const float* wt,
                                const int* grid_id, const uint32_t* bin_offset, const uint32_t* cta_hist, uint32_t* cursor,
                                uint4* sorted, int* cnt, cudaStream_t s) {
    const RowsShape sh = {ntime, pols_split ? npol : 1, pols_split ? 1 : npol, nchan, nrow};
    k_rows_scatter<<<rows_grid(sh, cpc), kBinThreads, bin_smem_bytes(g), s>>>(g, sh, cpc, loc, uvw, freq, vis, wt, grid_id, bin_offset,
                                                                             cta_hist, cursor, sorted, cnt);
    return cudaGetLastError();
}

int rows_max_channels() { return kRowsMaxChan; }

cudaError_t launch_owner_scan(const Geom& g, uint32_t* bin_count, uint32_t* cursor, uint32_t* bin_offset, OwItem* items,
                              uint32_t* nitems, uint32_t item_size, uint4* work, uint32_t* ctl, uint32_t* tops,
                              uint32_t* valid_reset, cudaStream_t s) {
    const uint32_t nblocks = (g.onbins + 4095u) / 4096u;
    if (nblocks == 1) {
        k_owner_scan_write<1><<<1, 1024, 0, s>>>(g, bin_count, cursor, item_size, tops, bin_offset, items, work, nitems, ctl, valid_reset);
        return cudaGetLastError();
    }
    if (nblocks <= 1024u) {                                           // (tops: 4 (nblocks + 1) words, zero when idle)
        k_owner_scan_write<2><<<nblocks, 1024, 0, s>>>(g, bin_count, cursor, item_size, tops, bin_offset, items, work, nitems, ctl, valid_reset);
        return cudaGetLastError();
    }
    k_owner_scan_reduce<<<nblocks, 1024, 0, s>>>(g, bin_count, item_size, tops);
    k_owner_scan_tops<<<1, 1024, 0, s>>>(g, nblocks, tops, bin_offset, nitems, ctl);
    k_owner_scan_write<0><<<nblocks, 1024, 0, s>>>(g, bin_count, cursor, item_size, tops, bin_offset, items, work, nitems, ctl, valid_reset);
    return cudaGetLastError();
}

cudaError_t owner_kernel_setup(int max_smem_bytes) {
    cudaError_t e = cudaFuncSetAttribute(k_grid_owner_s7<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes - 1024);
    if (e) return e;
    return cudaFuncSetAttribute(k_grid_owner_s7<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes - 1024);
}

cudaError_t launch_owner_grid(const Geom& g, const uint4* sorted, const uint32_t* bin_offset,
                              const OwItem* items, const uint32_t* nitems, const uint4* work, uint32_t* ctl,
                              const float* tt2, GridPtrs grids, float* scratch, uint32_t* tickets, uint32_t* valid,
                              int first, int num_sms, cudaStream_t s) {
    const size_t smem = owner_smem_bytes(g.Q);
    const unsigned blocks = (unsigned)num_sms * 4u;
    if (first) k_grid_owner_s7<1><<<blocks, 256, smem, s>>>(g, sorted, bin_offset, items, nitems, work, ctl, tt2, grids, scratch, tickets, valid);
    else k_grid_owner_s7<0><<<blocks, 256, smem, s>>>(g, sorted, bin_offset, items, nitems, work, ctl, tt2, grids, scratch, tickets, valid);
    return cudaGetLastError();
}

// zero the tiles of the stored half-plane that have not been written since the last reset and flag them (consumers of the
// dense grids call this first): one CTA per (grid, tile)
__global__ void __launch_bounds__(256) k_owner_fill_invalid(const Geom g, GridPtrs grids, uint32_t* __restrict__ valid) {
    const uint32_t b = blockIdx.x;
    if (valid[b] != 0u) return;
    const uint32_t gi = b / (uint32_t)g.ontiles, tile = b - gi * (uint32_t)g.ontiles;
    const int ty = (int)(tile / (uint32_t)g.otx), tx = (int)(tile - (uint32_t)ty * (uint32_t)g.otx);
    const int x0 = tx * kOwTW - kOwTW / 2, y0 = (g.ny >> 1) + ty * kTile;
    float2* __restrict__ Gt = grids.G + (size_t)gi * g.ny * g.nx;
    float* __restrict__ Wt = grids.Gw + (size_t)gi * g.ny * g.nx;
    for (int i = threadIdx.x; i < kTile * kOwTW; i += 256) {
        const int x = x0 + (i & (kOwTW - 1)), y = y0 + (i >> kOwTWS);
        if ((unsigned)x < (unsigned)g.nx && y < g.ny) {
            Gt[(size_t)y * g.nx + x] = make_float2(0.f, 0.f);
            Wt[(size_t)y * g.nx + x] = 0.f;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) valid[b] = 1u;
}

cudaError_t launch_owner_fill_invalid(const Geom& g, GridPtrs grids, uint32_t* valid, cudaStream_t s) {
    k_owner_fill_invalid<<<g.onbins, 256, 0, s>>>(g, grids, valid);
    return cudaGetLastError();
}

}  // namespace muser
