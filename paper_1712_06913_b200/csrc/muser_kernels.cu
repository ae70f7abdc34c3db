// Device kernels of the MUSER dirty-imaging hot path, sm_100a.
//   K1 k_coords       A1: fp64 coordinates, keep/drop, Hermitian conjugate sample, tile histogram + rank
//   K2 k_scan_items   A1: exclusive scan of the tile histogram, work items of <= chunk samples
//   K3 k_scatter      A1: counting-sort scatter into 16-byte tile-local samples
//   K4 k_grid_tiled_* A2/A3/A4: convolutional gridding, generic strategy (tiled shared-memory accumulators + global reductions)
//   Kp k_pack         H = G + i*Gw, the single FFT input that yields dirty image and beam together
//   K5 k_correct      A6: fused fftshift (index roll + checkerboard sign) + grid correction + real/imag part
// Passages: PAPER.md:78 (gridding = convolution onto a regular grid), :136-138 (spheroidal GCF, inverse FFT),
// :216-228 (float2 grid, row-major iv*nu+iu, Hermitian), :249-256 (DIRTY_IMAGE).  Arithmetic order of the
// coordinates follows DESIGN.md O1 exactly (fp64, no FMA contraction) so that every integer decision
// (cell, oversample phase, plane, keep/drop) is the oracle's decision.
#include "muser_internal.h"

#include <math_constants.h>

#include <algorithm>

namespace muser {

static constexpr double kC = 299792458.0;   // m/s

// ------------------------------------------------------------------------------------------------- K1
// O1 for one axis: p = xs + n/2 (xs = c_lambda * scale, already rounded); i0 = floor(p + 0.5); r = floor((p - i0)*Q + 0.5).
// Explicit _rn intrinsics keep nvcc from contracting mul+add into an FMA (the oracle has none).  The two floors and the
// conversions to int run in the FP64 add pipe with the 1.5 * 2^52 constant (x + M rounds x to the nearest integer, whose
// two's complement sits in the low word; one compare turns nearest into floor): exact for |xs| < 2^31 (callers test 1e9).
__device__ __forceinline__ void cell_phase(const double xs, const double half, const double Qd, int& i0, int& r) {
    constexpr double M = 6755399441055744.0;
    const double p = __dadd_rn(xs, half);
    const double t = __dadd_rn(p, 0.5);
    const double tm = __dadd_rn(t, M);
    double fl = __dadd_rn(tm, -M);
    int i = __double2loint(tm);
    if (fl > t) { fl = __dadd_rn(fl, -1.0); --i; }
    const double fr = __dsub_rn(p, fl);
    const double u = __dadd_rn(__dmul_rn(fr, Qd), 0.5);
    const double um = __dadd_rn(u, M);
    int q = __double2loint(um);
    if (__dadd_rn(um, -M) > u) --q;
    i0 = i; r = q;
}

// A CTA loops over `iters` blocks of 256 visibilities (statistics reduced once per CTA).  wstep > 0: the plane centres
// are the ladder wc[p] = p * wstep (checked on the host), so the nearest centre is looked for among the three around
// floor(|w| / wstep + 1/2) with the same fp64 comparisons as the full scan (identical result); else all planes are scanned.
// A sample that is not gridded (flagged, dropped, footprint below the stored half-plane) only writes its bin word.
// Histogram: a third of a MUSER frame lands in the few bins around the uv origin, and atomics on one address serialise
// in L2, so the CTA first counts in a shared-memory hash table (1024 slots keyed by bin, two probes; a sample that finds
// both taken falls back to a warp-aggregated global atomic at once) and hands out CTA-local ranks; after the loop every
// occupied slot reserves its run with ONE global atomic and the threads add the slot's base to the ranks they hold.
// ROWS (NEXT-1, the channelised call): the unit of work is an ELEMENT (t, po, c, r) -- one baseline at one
// channel -- in the order of the flat layout; uvw_m [ntime][nrow][3], freq_hz [nchan], vis / weight [ntime][npol][nchan][nrow],
// grid_id [ntime][npo][nchan].  Its npi polarisations po + pi share the coordinates; they are flagged / dropped / kept one
// by one (counters per visibility, as in the flat call) and the kept ones are added up BEFORE gridding (npo = 1: all the
// polarisations of a channel go onto one grid) -- same cells and kernel values, only the order of the fp32 sums differs.
constexpr int kHashSlots = 1024;
template <int ROWS>
__global__ void __launch_bounds__(256) k_coords(const Geom g, const RowsShapeG sh, const float* __restrict__ uvw,
                                                const double* __restrict__ freq, const float2* __restrict__ vis,
                                                const float* __restrict__ weight, const int* __restrict__ grid_id,
                                                const long long nvis, const int iters, const double wstep,
                                                const PlaneMeta* __restrict__ planes,
                                                Staged* __restrict__ staged, uint32_t* __restrict__ bin_count,
                                                Stats* __restrict__ stats, int* __restrict__ cnt) {
    __shared__ double s_wc[kMaxPlanes];
    __shared__ int s_sup[kMaxPlanes];
    __shared__ uint32_t s_tag[kHashSlots], s_num[kHashSlots];
    const int P = g.wmode ? g.nplanes : 1;
    for (int p = threadIdx.x; p < P; p += 256) { s_wc[p] = planes[p].wc; s_sup[p] = planes[p].support; }
    for (int i = threadIdx.x; i < kHashSlots; i += 256) { s_tag[i] = kNoBin; s_num[i] = 0u; }
    uint32_t held[8];                                              // per sample of this thread: slot << 16 | local rank, or ~0
    __syncthreads();
    const long long base = (long long)blockIdx.x * 256 * iters;
    const double hx = (double)(g.nx / 2), hy = (double)(g.ny / 2), Qd = (double)g.Q;
    const double inv_wstep = wstep > 0.0 ? 1.0 / wstep : 0.0;
    int flagged = 0, dropped = 0, kept = 0;
    double wsum = 0.0, v2sum = 0.0, w2sum = 0.0;
    for (int it = 0; it < iters; ++it) {
        const long long k = base + (long long)it * 256 + threadIdx.x;
        Staged s0, s1;
        s0.bin = s1.bin = kNoBin;
        s0.rank = s1.rank = 0u;
        if (k < nvis) {
            float um, vm, wm;
            double f;
            int gid, npi = 1;
            size_t k0 = (size_t)k, kstep = 0;                         // index of the first polarisation's value, stride to the next
            if (ROWS) {
                const int r = (int)(k % sh.nrow);
                const long long q = k / sh.nrow;
                const int c = (int)(q % sh.nchan);
                const long long tp = q / sh.nchan;
                const int po = (int)(tp % sh.npo), t = (int)(tp / sh.npo);
                const size_t ub = ((size_t)t * sh.nrow + r) * 3;
                um = uvw[ub]; vm = uvw[ub + 1]; wm = uvw[ub + 2];
                f = freq[c];
                gid = grid_id ? grid_id[((size_t)t * sh.npo + po) * sh.nchan + c] : 0;
                npi = sh.npi;
                kstep = (size_t)sh.nchan * sh.nrow;
                k0 = (((size_t)t * sh.npo * sh.npi + po) * sh.nchan + c) * sh.nrow + r;
            } else {
                um = uvw[3 * k + 0]; vm = uvw[3 * k + 1]; wm = uvw[3 * k + 2];
                f = freq[k];
                gid = grid_id ? grid_id[k] : 0;
            }
            const double il = __ddiv_rn(f, kC);
            const double ul = __dmul_rn((double)um, il), vl = __dmul_rn((double)vm, il), wl = __dmul_rn((double)wm, il);
            const bool geom_ok = isfinite(ul) && isfinite(vl) && isfinite(wl) && isfinite(f) && gid >= 0 && gid < g.ngrids;
            // the polarisations of the element (one in the flat call): flag each, add the others up
            float2 V = make_float2(0.f, 0.f);                        // sum of wt * V (phase-rotated) over the unflagged ones
            float wt = 0.f;                                           // sum of their weights
            int nok = 0;
            double e_wsum = 0.0, e_w2 = 0.0, e_v2 = 0.0;
            for (int pi = 0; pi < npi; ++pi) {
                const size_t kk = k0 + pi * kstep;
                float2 Vp = vis ? vis[kk] : make_float2(0.f, 0.f);
                const float wp = weight[kk];
                if (!(geom_ok && isfinite(wp) && isfinite(Vp.x) && isfinite(Vp.y) && wp > 0.0f)) { ++flagged; continue; }
                ++nok;
                e_wsum += 2.0 * (double)wp;
                const double w2 = (double)wp * (double)wp;
                e_w2 += w2;
                e_v2 += w2 * ((double)Vp.x * (double)Vp.x + (double)Vp.y * (double)Vp.y);
                if (g.phase_on) Vp = phase_rotate(g, um, vm, f, Vp);
                if (ROWS) { V.x += wp * Vp.x; V.y += wp * Vp.y; wt += wp; }
                else { V = make_float2(wp * Vp.x, wp * Vp.y); wt = wp; }
            }
            if (nok) {
                int p = 0;
                if (g.wmode) {                                   // O6: nearest plane centre in |w|, tie -> lower p
                    const double aw = fabs(wl);
                    int lo = 0, hi = g.nplanes - 1;
                    if (wstep > 0.0) {
                        const int q0 = __double2int_rz(fmin(__dadd_rn(__dmul_rn(aw, inv_wstep), 0.5), (double)(g.nplanes - 1)));
                        lo = max(q0 - 1, 0); hi = min(q0 + 1, g.nplanes - 1);
                    }
                    p = lo;
                    double best = fabs(__dsub_rn(aw, s_wc[lo]));
                    for (int q = lo + 1; q <= hi; ++q) {
                        const double d = fabs(__dsub_rn(aw, s_wc[q]));
                        if (d < best) { best = d; p = q; }
                    }
                }
                const int S = s_sup[p], h = (S - 1) >> 1;
                const double xu = __dmul_rn(ul, g.su), xv = __dmul_rn(vl, g.sv);
                int iu[2], iv[2], ru[2], rv[2];
                bool inside = fabs(xu) < 1.0e9 && fabs(xv) < 1.0e9;   // beyond: off any grid, and outside the int range
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    cell_phase(s ? -xu : xu, hx, Qd, iu[s], ru[s]);
                    cell_phase(s ? -xv : xv, hy, Qd, iv[s], rv[s]);
                    inside = inside && iu[s] >= h + 1 && iu[s] <= g.nx - 1 - h && iv[s] >= h + 1 && iv[s] <= g.ny - 1 - h;
                }
                if (!inside) {
                    dropped += nok;
                } else {
                    kept += nok;
                    wsum += e_wsum; w2sum += e_w2; v2sum += e_v2;
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        Staged& o = s ? s1 : s0;
                        const int cu = iu[s], cv = iv[s];
                        const int rx = g.Q / 2 - ru[s], ry = g.Q / 2 - rv[s];
                        const int kconj = g.wmode && ((s ? -wl : wl) < 0.0);
                        o.re = V.x;
                        o.im = s ? -V.y : V.y;
                        o.wt = wt;
                        o.cell = (uint32_t)cu | ((uint32_t)cv << 16);
                        o.phase = (uint32_t)rx | ((uint32_t)ry << 9) | ((uint32_t)kconj << 18);
                        o.gp = (uint32_t)gid | ((uint32_t)p << 24);
                        // the grids are Hermitian: only rows >= ny/2 are computed and stored ("half the grid"); a
                        // sample whose footprint stays below them is not gridded (its partner covers the mirror cells)
                        if (cv + h >= (g.ny >> 1)) {
                            const int tx = (cu + kTile / 2) >> kTileShift, ty = (cv + kTile / 2) >> kTileShift;
                            o.bin = g.wtile ? (uint32_t)((((long long)gid * g.nty + ty) * g.ntx + tx) * P + p)
                                            : (uint32_t)((((long long)gid * P + p) * g.nty + ty) * g.ntx + tx);
                        }
                        if (cnt && cv >= (g.ny >> 1)) atomicAdd(cnt + ((size_t)gid * g.ny + cv) * g.nx + cu, nok);   // NEXT-2: one hit per visibility
                    }
                }
            }
        }
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            Staged& o = s ? s1 : s0;
            uint32_t hold = 0xFFFFFFFFu;
            bool global_now = false;
            if (o.bin != kNoBin) {
                uint32_t slot = (o.bin * 2654435761u) >> 22;
                global_now = true;
#pragma unroll
                for (int probe = 0; probe < 2; ++probe) {
                    const uint32_t old = atomicCAS(&s_tag[slot], kNoBin, o.bin);
                    if (old == kNoBin || old == o.bin) {
                        hold = slot << 16 | atomicAdd(&s_num[slot], 1u);
                        global_now = false;
                        break;
                    }
                    slot = (slot + 1u) & (kHashSlots - 1);
                }
            }
            if (it < 4) held[2 * it + s] = hold;
            if (__any_sync(0xffffffffu, global_now)) {                // both probes taken: warp-aggregated global atomic
                const unsigned full_ = 0xffffffffu;
                const int lane_ = threadIdx.x & 31;
                const uint32_t key = global_now ? o.bin : kNoBin;
                const unsigned m = __match_any_sync(full_, key);
                const int leader = __ffs(m) - 1;
                uint32_t b0 = 0;
                if (global_now && lane_ == leader) b0 = atomicAdd(&bin_count[o.bin], (uint32_t)__popc(m));
                b0 = __shfl_sync(full_, b0, leader);
                if (global_now) o.rank = b0 + (uint32_t)__popc(m & ((1u << lane_) - 1u));
            }
        }
        if (k < nvis) {
            uint4* dst = reinterpret_cast<uint4*>(staged + 2 * k);
            const uint4* a = reinterpret_cast<const uint4*>(&s0);
            const uint4* b = reinterpret_cast<const uint4*>(&s1);
            if (s0.bin != kNoBin) dst[0] = a[0];
            dst[1] = a[1];
            if (s1.bin != kNoBin) dst[2] = b[0];
            dst[3] = b[1];
        }
    }
    // every occupied slot reserves its run in its bin; the ranks held by the threads become global
    __syncthreads();
    for (int i = threadIdx.x; i < kHashSlots; i += 256) {
        const uint32_t tag = s_tag[i];
        if (tag != kNoBin) s_num[i] = atomicAdd(&bin_count[tag], s_num[i]);
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const long long k = base + (long long)it * 256 + threadIdx.x;
        if (it >= iters || k >= nvis) continue;
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const uint32_t hold = held[2 * it + s];
            if (hold != 0xFFFFFFFFu) staged[2 * k + s].rank = s_num[hold >> 16] + (hold & 0xFFFFu);
        }
    }
    // block reduction of the counters, one atomic set per block
    __shared__ int s_cnt[3][8];
    __shared__ double s_w[3][8];
    const unsigned full = 0xffffffffu;
    int c0 = __reduce_add_sync(full, kept), c1 = __reduce_add_sync(full, dropped), c2 = __reduce_add_sync(full, flagged);
    for (int o = 16; o > 0; o >>= 1) {
        wsum += __shfl_xor_sync(full, wsum, o);
        v2sum += __shfl_xor_sync(full, v2sum, o);
        w2sum += __shfl_xor_sync(full, w2sum, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { s_cnt[0][warp] = c0; s_cnt[1][warp] = c1; s_cnt[2][warp] = c2; s_w[0][warp] = wsum; s_w[1][warp] = v2sum; s_w[2][warp] = w2sum; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int t0 = 0, t1 = 0, t2 = 0;
        double tw = 0.0, tv2 = 0.0, tw2 = 0.0;
        for (int w = 0; w < 8; ++w) {
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

// ------------------------------------------------------------------------------------------------- K2
// Exclusive scan of the tile histogram -> sample offsets and work items of <= chunk samples; re-zeroes the histogram
// for the next call.  Multi-CTA: per-block totals (4096 bins per CTA), one CTA scans the totals, every CTA writes its
// block (one launch when the histogram fits one block).
struct Scan2 { uint32_t c, n; };
__device__ __forceinline__ Scan2 block_scan2(Scan2 v, Scan2& total, uint32_t (*s_w)[32]) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    Scan2 inc = v;
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t xc = __shfl_up_sync(0xffffffffu, inc.c, o), xn = __shfl_up_sync(0xffffffffu, inc.n, o);
        if (lane >= o) { inc.c += xc; inc.n += xn; }
    }
    if (lane == 31) { s_w[0][warp] = inc.c; s_w[1][warp] = inc.n; }
    __syncthreads();
    if (warp == 0) {
        uint32_t wc = s_w[0][lane], wn = s_w[1][lane];
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t xc = __shfl_up_sync(0xffffffffu, wc, o), xn = __shfl_up_sync(0xffffffffu, wn, o);
            if (lane >= o) { wc += xc; wn += xn; }
        }
        s_w[0][lane] = wc; s_w[1][lane] = wn;
    }
    __syncthreads();
    Scan2 ex;
    ex.c = (warp ? s_w[0][warp - 1] : 0u) + inc.c - v.c;
    ex.n = (warp ? s_w[1][warp - 1] : 0u) + inc.n - v.n;
    total.c = s_w[0][31]; total.n = s_w[1][31];
    __syncthreads();
    return ex;
}
__device__ __forceinline__ Scan2 scan_load4(const Geom& g, const uint32_t* __restrict__ bin_count, uint32_t b0, uint32_t c[4]) {
    Scan2 t = {0u, 0u};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        c[j] = (b0 + j < g.nbins) ? bin_count[b0 + j] : 0u;
        t.c += c[j];
        t.n += (c[j] + (uint32_t)g.chunk - 1u) / (uint32_t)g.chunk;
    }
    return t;
}

__global__ void __launch_bounds__(1024) k_scan_items_reduce(const Geom g, const uint32_t* __restrict__ bin_count,
                                                            uint32_t* __restrict__ tops) {
    __shared__ uint32_t s_w[2][32];
    uint32_t c[4];
    const Scan2 t = scan_load4(g, bin_count, blockIdx.x * 4096u + 4u * threadIdx.x, c);
    Scan2 total;
    block_scan2(t, total, s_w);
    if (threadIdx.x == 0) { tops[2 * blockIdx.x] = total.c; tops[2 * blockIdx.x + 1] = total.n; }
}

__global__ void __launch_bounds__(1024) k_scan_items_tops(const Geom g, const uint32_t nblocks, uint32_t* __restrict__ tops,
                                                          uint32_t* __restrict__ bin_offset, uint32_t* __restrict__ nitems) {
    __shared__ uint32_t s_w[2][32];
    Scan2 carry = {0u, 0u};
    for (uint32_t base = 0; base < nblocks; base += 1024) {
        const uint32_t b = base + threadIdx.x;
        Scan2 v = {0u, 0u};
        if (b < nblocks) { v.c = tops[2 * b]; v.n = tops[2 * b + 1]; }
        Scan2 total;
        const Scan2 ex = block_scan2(v, total, s_w);
        if (b < nblocks) { tops[2 * b] = carry.c + ex.c; tops[2 * b + 1] = carry.n + ex.n; }
        carry.c += total.c; carry.n += total.n;
    }
    if (threadIdx.x == 0) { bin_offset[g.nbins] = carry.c; if (nitems) *nitems = carry.n; }
}

template <int SINGLE>
__global__ void __launch_bounds__(1024) k_scan_items_write(const Geom g, uint32_t* __restrict__ bin_count,
                                                           const uint32_t* __restrict__ tops, uint32_t* __restrict__ bin_offset,
                                                           Item* __restrict__ items, uint32_t* __restrict__ nitems) {
    __shared__ uint32_t s_w[2][32];
    const uint32_t b0 = blockIdx.x * 4096u + 4u * threadIdx.x;
    uint32_t c[4];
    const Scan2 t = scan_load4(g, bin_count, b0, c);
    Scan2 total;
    const Scan2 ex = block_scan2(t, total, s_w);
    uint32_t off = ex.c, ioff = ex.n;
    if (SINGLE) {
        if (threadIdx.x == 0) { bin_offset[g.nbins] = total.c; if (nitems) *nitems = total.n; }
    } else {
        off += tops[2 * blockIdx.x]; ioff += tops[2 * blockIdx.x + 1];
    }
    const uint32_t CH = (uint32_t)g.chunk;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t b = b0 + j;
        if (b < g.nbins) {
            bin_offset[b] = off;
            if (c[j]) bin_count[b] = 0;
            const uint32_t n = (c[j] + CH - 1u) / CH;
            for (uint32_t q = 0; items && q < n; ++q) {
                Item it;
                it.bin = b; it.start = off + q * CH; it.count = min(CH, c[j] - q * CH);
                items[ioff + q] = it;
            }
            off += c[j]; ioff += n;
        }
    }
}

// ------------------------------------------------------------------------------------------------- K3
__global__ void __launch_bounds__(256) k_scatter(const Geom g, const Staged* __restrict__ staged,
                                                 const long long nsamples, const uint32_t* __restrict__ bin_offset,
                                                 Sample* __restrict__ sorted) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nsamples) return;
    const uint4* src = reinterpret_cast<const uint4*>(staged + i);
    const uint4 b = src[1];                                            // b: phase bin rank gp
    if (b.y == kNoBin) return;                                         // (a was not written)
    const uint4 a = src[0];                                            // a: re im wt cell
    const uint32_t tb = g.wtile ? b.y / (uint32_t)g.nplanes : b.y;          // tile-major order: plane is the minor index
    const uint32_t tx = tb % (uint32_t)g.ntx, ty = (tb / (uint32_t)g.ntx) % (uint32_t)g.nty;
    const int cu = (int)(a.w & 0xFFFFu), cv = (int)(a.w >> 16);
    const int lx = cu - ((int)tx * kTile - kTile / 2), ly = cv - ((int)ty * kTile - kTile / 2);
    const uint32_t rx = b.x & 511u, ry = (b.x >> 9) & 511u, kc = (b.x >> 18) & 1u;
    uint4 o;
    o.x = a.x; o.y = a.y; o.z = a.z;
    o.w = (uint32_t)lx | ((uint32_t)ly << 5) | (rx << 10) | (ry << 19) | (kc << 28);
    reinterpret_cast<uint4*>(sorted)[bin_offset[b.y] + b.z] = o;
}

// ------------------------------------------------------------------------------------------------- K4 tiled
__device__ __forceinline__ void decode_bin(const Geom& g, uint32_t bin, int& gi, int& p, int& ty, int& tx) {
    tx = (int)(bin % (uint32_t)g.ntx); bin /= (uint32_t)g.ntx;
    ty = (int)(bin % (uint32_t)g.nty); bin /= (uint32_t)g.nty;
    const uint32_t P = g.wmode ? (uint32_t)g.nplanes : 1u;
    p = (int)(bin % P);
    gi = (int)(bin / P);
}

// Generic tiled gridder (any support, 2-D or w mode): one work item = <= chunk samples of one (grid, plane,
// tile).  The CTA accumulates the tile plus its halo ((32+2h)^2 cells) in shared memory, then adds the touched cells
// to the grids with vector reductions.
//   - the plane's kernel table is staged in shared memory per item (<= 16.6 KB at S = 31, Q = 64);
//   - a sample is handled by S lanes, lane = footprint COLUMN jx, looping over the S rows: the row's ky * (wt V) and
//     ky * wt are formed once per row (separable kernel), each lane then needs one complex multiply per grid;
//     floor(32 / S) samples share a warp (4 at S = 7, 2 at S = 11..15, 1 above);
//   - the region is accumulated in 32-bit FIXED POINT: integer shared-memory adds are native single instructions,
//     fp32 adds are compare-and-swap loops.  Per item the scales map the largest possible cell sum (sum of
//     |wt Re V| + |wt Im V| resp. wt over the item's samples, times the plane's bound on |kx ky|) to 0.98 * 2^31.
template <int WMODE>
__global__ void __launch_bounds__(256) k_grid_tiled_generic(const Geom g, const Sample* __restrict__ sorted,
                                                            const Item* __restrict__ items,
                                                            const uint32_t* __restrict__ nitems,
                                                            const PlaneMeta* __restrict__ planes,
                                                            const float* __restrict__ tables, GridPtrs grids,
                                                            const int region_ints) {
    extern __shared__ __align__(16) int smem_i[];
    float* s_tab = reinterpret_cast<float*>(smem_i + region_ints);  // TT[r][j] of the item's plane (floats, or float2 in w mode)
    __shared__ float s_sum[8][2];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t n_items = *nitems;
    for (uint32_t it = blockIdx.x; it < n_items; it += gridDim.x) {
        const Item item = items[it];
        int gi, p, ty, tx;
        decode_bin(g, item.bin, gi, p, ty, tx);
        const PlaneMeta pm = planes[p];
        const int S = pm.support, h = (S - 1) >> 1, R = kTile + 2 * h, RR = R * R;
        constexpr int NPL = WMODE ? 4 : 3;                          // planes: G.re G.im W(.re) [W.im]
        for (int i = threadIdx.x; i < NPL * RR; i += blockDim.x) smem_i[i] = 0;
        {   // stage the plane's table
            const int nfl = (g.Q + 1) * pm.pitch * (WMODE ? 2 : 1);
            const float* src = tables + (size_t)pm.offset * (WMODE ? 2 : 1);
            for (int i = threadIdx.x; i < nfl; i += blockDim.x) s_tab[i] = __ldg(src + i);
        }
        float mv = 0.f, mw = 0.f;
        for (uint32_t i = threadIdx.x; i < item.count; i += blockDim.x) {
            const uint4 a = __ldg(reinterpret_cast<const uint4*>(sorted + item.start + i));
            mv += fabsf(__uint_as_float(a.x)) + fabsf(__uint_as_float(a.y));
            mw += __uint_as_float(a.z);
        }
        for (int o = 16; o > 0; o >>= 1) { mv += __shfl_xor_sync(0xffffffffu, mv, o); mw += __shfl_xor_sync(0xffffffffu, mw, o); }
        if (lane == 0) { s_sum[warp][0] = mv; s_sum[warp][1] = mw; }
        __syncthreads();
        mv = 0.f; mw = 0.f;
        for (int w = 0; w < 8; ++w) { mv += s_sum[w][0]; mw += s_sum[w][1]; }
        const float kb = __int_as_float(pm.pad);                    // bound on |kx ky| of this plane (>= 1)
        const float sv = 2104533975.0f / fmaxf(mv * kb, 1e-30f), sw = 2104533975.0f / fmaxf(mw * kb, 1e-30f);
        const int per = 32 / S > 0 ? 32 / S : 1;                    // samples per warp pass (S <= 63: S > 32 takes two column passes)
        const int sub = lane / S, j0 = lane - sub * S;
        const bool on = sub < per;
        for (uint32_t i0 = (uint32_t)(warp * per); i0 < item.count; i0 += 8u * per) {
            const uint32_t i = i0 + (uint32_t)sub;
            if (!on || i >= item.count) continue;
            const uint4 a = __ldg(reinterpret_cast<const uint4*>(sorted + item.start + i));
            const float re = __uint_as_float(a.x) * sv, im = __uint_as_float(a.y) * sv, wt = __uint_as_float(a.z) * sw;
            const int lx = (int)(a.w & 31u), ly = (int)((a.w >> 5) & 31u);
            const int rx = (int)((a.w >> 10) & 511u), ry = (int)((a.w >> 19) & 511u), kc = (int)((a.w >> 28) & 1u);
            for (int jx = j0; jx < S; jx += 32) {                   // one pass unless S > 32
                int* cell = smem_i + ly * R + lx + jx;               // region origin is (tile origin - h)
                if (WMODE == 0) {
                    const float kx = s_tab[rx * pm.pitch + jx];
                    const float* kyp = s_tab + ry * pm.pitch;
                    for (int jy = 0; jy < S; ++jy, cell += R) {
                        const float kk = kx * kyp[jy];
                        atomicAdd(cell, __float2int_rn(kk * re));
                        atomicAdd(cell + RR, __float2int_rn(kk * im));
                        atomicAdd(cell + 2 * RR, __float2int_rn(kk * wt));
                    }
                } else {
                    const float2* tc = reinterpret_cast<const float2*>(s_tab);
                    float2 kx = tc[rx * pm.pitch + jx];
                    const float cs = kc ? -1.0f : 1.0f;               // conjugate kernel for w < 0
                    kx.y *= cs;
                    const float2* kyp = tc + ry * pm.pitch;
                    for (int jy = 0; jy < S; ++jy, cell += R) {
                        float2 ky = kyp[jy];
                        ky.y *= cs;
                        // row factors (same for every lane of the sample), then one complex multiply per grid
                        const float tr = ky.x * re - ky.y * im, ti = ky.x * im + ky.y * re;
                        const float ur = ky.x * wt, ui = ky.y * wt;
                        atomicAdd(cell, __float2int_rn(kx.x * tr - kx.y * ti));
                        atomicAdd(cell + RR, __float2int_rn(kx.x * ti + kx.y * tr));
                        atomicAdd(cell + 2 * RR, __float2int_rn(kx.x * ur - kx.y * ui));
                        atomicAdd(cell + 3 * RR, __float2int_rn(kx.x * ui + kx.y * ur));
                    }
                }
            }
        }
        __syncthreads();
        const float iv = 1.0f / sv, iw = 1.0f / sw;
        const int x0 = tx * kTile - kTile / 2 - h, y0 = ty * kTile - kTile / 2 - h;
        const size_t gbase = (size_t)gi * g.ny * g.nx;
        for (int y = warp; y < R; y += 8)
          for (int x = lane; x < R; x += 32) {
            const int i = y * R + x;
            const int gx = x0 + x, gy = y0 + y;
            if (gx < 0 || gx >= g.nx || gy < (g.ny >> 1) || gy >= g.ny) continue;   // the stored half-plane only
            const size_t idx = gbase + (size_t)gy * g.nx + gx;
            const int vr = smem_i[i], vi = smem_i[RR + i], wr = smem_i[2 * RR + i];
            if (vr | vi) atomicAdd(&grids.G[idx], make_float2((float)vr * iv, (float)vi * iv));
            if (WMODE == 0) {
                if (wr) atomicAdd(&grids.Gw[idx], (float)wr * iw);
            } else {
                const int wi = smem_i[3 * RR + i];
                if (wr | wi) atomicAdd(reinterpret_cast<float2*>(grids.Gw) + idx, make_float2((float)wr * iw, (float)wi * iw));
            }
        }
        __syncthreads();
    }
}

// Fast path: 2-D mode, support 7.  Per work item the CTA (1) counting-sorts its <= 512 samples by nearest
// cell inside the tile, (2) lets each warp walk an equal slice of the sorted list with the 7x7 footprint held
// in registers (lane = (row jy, column jx), two rows per lane), flushing to the shared tile only when the
// nearest cell changes -- MUSER's uv coverage puts many samples on the same cell -- and (3) adds the touched
// cells of the 38x38 region to the grids.
constexpr int kFastChunk = 512;
constexpr int kFastR = 38, kFastPitch = 40;                 // pitch 40 = 8 mod 32: the 4 rows of a warp hit disjoint banks

__global__ void __launch_bounds__(256) k_grid_tiled_s7(const Geom g, const Sample* __restrict__ sorted,
                                                       const Item* __restrict__ items,
                                                       const uint32_t* __restrict__ nitems,
                                                       const PlaneMeta* __restrict__ planes,
                                                       const float* __restrict__ tables, GridPtrs grids) {
    extern __shared__ __align__(16) float smem[];
    constexpr int PL = kFastR * kFastPitch;                 // floats per accumulator plane
    int* s_re = reinterpret_cast<int*>(smem);               // 32-bit fixed point (native shared adds; an fp32 add is a CAS loop)
    int* s_im = s_re + PL;
    int* s_w = s_re + 2 * PL;
    uint32_t* s_hist = reinterpret_cast<uint32_t*>(smem + 3 * PL);           // 1024 cells of the tile
    float4* s_rec = reinterpret_cast<float4*>(smem + 3 * PL + 1024);         // kFastChunk samples, cell-sorted
    float* s_tt = smem + 3 * PL + 1024 + 4 * kFastChunk;                    // (Q+1) x 8 transposed table
    __shared__ uint32_t s_wsum[8];
    __shared__ float s_bound[8][2];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int jx = lane & 7, jy = lane >> 3;
    const PlaneMeta pm = planes[0];
    for (int i = threadIdx.x; i < (g.Q + 1) * 8; i += blockDim.x) s_tt[i] = __ldg(tables + pm.offset + i);
    const uint32_t n_items = *nitems;
    for (uint32_t it = blockIdx.x; it < n_items; it += gridDim.x) {
        const Item item = items[it];
        int gi, p, ty, tx;
        decode_bin(g, item.bin, gi, p, ty, tx);
        {   // zero accumulators and histogram
            float4* z = reinterpret_cast<float4*>(smem);
            for (int i = threadIdx.x; i < (3 * PL + 1024) / 4; i += blockDim.x) z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        __syncthreads();
        // (1) local counting sort by cell
        float4 rec[kFastChunk / 256];
        float bv = 0.f, bw = 0.f;
        uint32_t rnk[kFastChunk / 256];
#pragma unroll
        for (int j = 0; j < kFastChunk / 256; ++j) {
            const uint32_t i = threadIdx.x + j * 256;
            if (i < item.count) {
                rec[j] = __ldg(reinterpret_cast<const float4*>(sorted + item.start + i));
                rnk[j] = atomicAdd(&s_hist[__float_as_uint(rec[j].w) & 1023u], 1u);
                bv += fabsf(rec[j].x) + fabsf(rec[j].y);
                bw += rec[j].z;
            }
        }
        for (int o = 16; o > 0; o >>= 1) { bv += __shfl_xor_sync(0xffffffffu, bv, o); bw += __shfl_xor_sync(0xffffffffu, bw, o); }
        if (lane == 0) { s_bound[warp][0] = bv; s_bound[warp][1] = bw; }
        __syncthreads();
        bv = 0.f; bw = 0.f;
        for (int w = 0; w < 8; ++w) { bv += s_bound[w][0]; bw += s_bound[w][1]; }
        // the item's largest possible cell sum (the kernel never exceeds 1) maps to 0.98 * 2^31
        const float sv = 2104533975.0f / fmaxf(bv, 1e-30f), sw = 2104533975.0f / fmaxf(bw, 1e-30f);
        {
            uint4 hv = reinterpret_cast<uint4*>(s_hist)[threadIdx.x];
            const uint32_t tot = hv.x + hv.y + hv.z + hv.w;
            uint32_t inc = tot;
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            if (lane == 31) s_wsum[warp] = inc;
            __syncthreads();
            uint32_t base = inc - tot;
            for (int w = 0; w < warp; ++w) base += s_wsum[w];
            uint4 ov;
            ov.x = base; ov.y = base + hv.x; ov.z = ov.y + hv.y; ov.w = ov.z + hv.z;
            reinterpret_cast<uint4*>(s_hist)[threadIdx.x] = ov;
        }
        __syncthreads();
#pragma unroll
        for (int j = 0; j < kFastChunk / 256; ++j) {
            const uint32_t i = threadIdx.x + j * 256;
            if (i < item.count) s_rec[s_hist[__float_as_uint(rec[j].w) & 1023u] + rnk[j]] = rec[j];
        }
        __syncthreads();
        // (2) register accumulation over runs of equal cell
        {
            const int n = (int)item.count, per = (n + 7) >> 3;
            const int b = warp * per, e = min(n, b + per);
            float a0r = 0.f, a0i = 0.f, a0w = 0.f, a1r = 0.f, a1i = 0.f, a1w = 0.f;
            int cur = -1;
            auto flush = [&]() {
                if (cur >= 0 && jx < 7) {
                    const int lx = cur & 31, ly = cur >> 5;
                    const int s0 = (ly + jy) * kFastPitch + lx + jx;
                    atomicAdd(&s_re[s0], __float2int_rn(a0r * sv)); atomicAdd(&s_im[s0], __float2int_rn(a0i * sv)); atomicAdd(&s_w[s0], __float2int_rn(a0w * sw));
                    if (jy < 3) {
                        const int s1 = s0 + 4 * kFastPitch;
                        atomicAdd(&s_re[s1], __float2int_rn(a1r * sv)); atomicAdd(&s_im[s1], __float2int_rn(a1i * sv)); atomicAdd(&s_w[s1], __float2int_rn(a1w * sw));
                    }
                }
            };
            for (int i = b; i < e; ++i) {
                const float4 r = s_rec[i];
                const uint32_t pk = __float_as_uint(r.w);
                const int cell = (int)(pk & 1023u);
                if (cell != cur) {
                    flush();
                    cur = cell;
                    a0r = a0i = a0w = a1r = a1i = a1w = 0.f;
                }
                const int rx = (int)((pk >> 10) & 511u), ry = (int)((pk >> 19) & 511u);
                const float kx = s_tt[rx * 8 + jx];
                const float ky0 = s_tt[ry * 8 + jy], ky1 = s_tt[ry * 8 + jy + 4];
                const float k0 = kx * ky0, k1 = kx * ky1;
                a0r = fmaf(k0, r.x, a0r); a0i = fmaf(k0, r.y, a0i); a0w = fmaf(k0, r.z, a0w);
                a1r = fmaf(k1, r.x, a1r); a1i = fmaf(k1, r.y, a1i); a1w = fmaf(k1, r.z, a1w);
            }
            flush();
        }
        __syncthreads();
        // (3) add the touched cells of the region to the grids
        const float isv = 1.0f / sv, isw = 1.0f / sw;
        const int x0 = tx * kTile - kTile / 2 - 3, y0 = ty * kTile - kTile / 2 - 3;
        const size_t gbase = (size_t)gi * g.ny * g.nx;
        for (int i = threadIdx.x; i < PL; i += blockDim.x) {
            const int y = i / kFastPitch, x = i - y * kFastPitch;
            const int gx = x0 + x, gy = y0 + y;
            if (x >= kFastR || gx < 0 || gx >= g.nx || gy < (g.ny >> 1) || gy >= g.ny) continue;   // the stored half-plane only
            const size_t idx = gbase + (size_t)gy * g.nx + gx;
            const int vr = s_re[i], vi = s_im[i], vw = s_w[i];
            if (vr | vi) atomicAdd(&grids.G[idx], make_float2((float)vr * isv, (float)vi * isv));
            if (vw) atomicAdd(&grids.Gw[idx], (float)vw * isw);
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------- mirror
// The owner-tile gridder stores only the half-plane of rows ny/2 .. ny-1 (the grids are Hermitian: "half
// the grid (as the data is Hermitian)").  This kernel rebuilds rows 0 .. ny/2-1 for consumers of the full grids:
// G[y][x] = conj G[ny-y][nx-x], Gw[y][x] = Gw[ny-y][nx-x] (conjugated in w mode); row 0 and column 0 have no mirror
// and are empty by the drop rule R5.
template <int WMODE>
__global__ void __launch_bounds__(256) k_mirror_lower(const int nx, const int ny, const size_t total, float2* __restrict__ G,
                                                      float* __restrict__ Gw, int* __restrict__ cnt) {
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;      // over [ngrids][ny/2][nx]
    if (t >= total) return;
    const int x = (int)(t % nx);
    const size_t row = t / nx;
    const int y = (int)(row % (ny >> 1));
    const size_t gbase = (row / (ny >> 1)) * (size_t)ny * nx;
    const size_t dst = gbase + (size_t)y * nx + x;
    float2 v = make_float2(0.f, 0.f), w = make_float2(0.f, 0.f);
    int c = 0;
    if (x > 0 && y > 0) {
        const size_t src = gbase + (size_t)(ny - y) * nx + (nx - x);
        v = G[src];
        v.y = -v.y;
        if (WMODE) { w = reinterpret_cast<const float2*>(Gw)[src]; w.y = -w.y; }
        else w.x = Gw[src];
        if (cnt) c = cnt[src];
    }
    if (cnt) cnt[dst] = c;
    G[dst] = v;
    if (WMODE) reinterpret_cast<float2*>(Gw)[dst] = w;
    else Gw[dst] = w.x;
}

// ------------------------------------------------------------------------------------------------- pack, K5
// H = G + i*alpha*Gw: G and Gw are both Hermitian, so their inverse transforms are real and one complex FFT of
// H returns the dirty image in the real part and alpha * beam in the imaginary part.  alpha is the power of two
// nearest to rms|wt*V| / rms(wt): it balances the two parts so that fp32 rounding of the (much larger) beam does
// not leak into the dirty image; a power of two keeps the scaling exact.
template <int WMODE>
__global__ void __launch_bounds__(256) k_pack(const size_t ncell2, const float4* __restrict__ G,
                                              const float* __restrict__ Gw, const int* __restrict__ cnt,
                                              float4* __restrict__ H, Stats* __restrict__ stats) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;      // two cells per thread
    const double v2 = stats->sum_val2, w2 = stats->sum_wt2;
    float al = 1.0f;
    if (v2 > 0.0 && w2 > 0.0) al = exp2f(rintf(0.5f * log2f((float)(v2 / w2))));
    al = fminf(fmaxf(al, 9.5367431640625e-07f), 1048576.0f);
    if (i == 0) { stats->alpha = al; stats->inv_alpha = 1.0f / al; }
    if (i >= ncell2) return;
    float4 gv = G[i];
    // wgtGrid_kernel (Alg. 1 l.1-16): uniform mode multiplies a cell by 1 / count where count != 0
    float u0 = 1.0f, u1 = 1.0f;
    if (cnt) {
        const int2 c = reinterpret_cast<const int2*>(cnt)[i];
        if (c.x) u0 = 1.0f / (float)c.x;
        if (c.y) u1 = 1.0f / (float)c.y;
        gv.x *= u0; gv.y *= u0; gv.z *= u1; gv.w *= u1;
    }
    float4 o;
    if (WMODE == 0) {
        const float2 w = reinterpret_cast<const float2*>(Gw)[i];
        o = make_float4(gv.x, gv.y + al * (w.x * u0), gv.z, gv.w + al * (w.y * u1));
    } else {
        const float4 w = reinterpret_cast<const float4*>(Gw)[i];
        o = make_float4(gv.x - al * (w.y * u0), gv.y + al * (w.x * u0), gv.z - al * (w.w * u1), gv.w + al * (w.z * u1));
    }
    H[i] = o;
}

// A6: img[y][x] = (-1)^(x+y) * F_raw[(y+ny/2)%ny][(x+nx/2)%nx] * icx[x] * icy[y]  (nx/2, ny/2 even);
// dirty from the real part, beam from the imaginary part.  Four pixels per thread.
__global__ void __launch_bounds__(256) k_correct(const int nx, const int ny, const int ngrids,
                                                 const float2* __restrict__ F, const float* __restrict__ icx,
                                                 const float* __restrict__ icy, const Stats* __restrict__ stats,
                                                 float* __restrict__ dirty, float* __restrict__ psf,
                                                 PeakSlot* __restrict__ peaks) {
    const int nx4 = nx >> 2;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t total = (size_t)ngrids * ny * nx4;
    if (t >= total) return;
    const int x = (int)(t % nx4) << 2;
    const size_t row = t / nx4;
    const int y = (int)(row % ny);
    const size_t gi = row / ny;
    const int sy = (y + (ny >> 1)) % ny;
    const int sx0 = (x + (nx >> 1)) % nx, sx2 = (x + 2 + (nx >> 1)) % nx;  // pairs never wrap (nx/2 is even)
    const float2* srow = F + (gi * ny + sy) * (size_t)nx;
    const float4 f01 = *reinterpret_cast<const float4*>(srow + sx0);
    const float4 f23 = *reinterpret_cast<const float4*>(srow + sx2);
    const float4 cx = *reinterpret_cast<const float4*>(icx + x);
    const float cy = (y & 1) ? -icy[y] : icy[y];                         // x is a multiple of 4: sign = (-1)^y * (+,-,+,-)
    const float m0 = cx.x * cy, m1 = -cx.y * cy, m2 = cx.z * cy, m3 = -cx.w * cy;
    const size_t o = (gi * ny + y) * (size_t)nx + x;
    if (dirty) {
        const float4 d = make_float4(f01.x * m0, f01.z * m1, f23.x * m2, f23.z * m3);
        *reinterpret_cast<float4*>(dirty + o) = d;
        if (peaks) {                                                     // NEXT-4: strength and position of the peak, minimum
            const unsigned int base = (unsigned int)((size_t)y * nx + x);
            const float v[4] = {d.x, d.y, d.z, d.w};
            unsigned long long best = 0ull;
            unsigned int lo = 0u;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const unsigned int ord = peak_ordered(v[i]);
                const unsigned long long key = ((unsigned long long)ord << 32) | (unsigned long long)(~(base + i));
                best = key > best ? key : best;
                lo = max(lo, ~ord);
            }
            atomicMax(&peaks[gi].maxkey, best);
            atomicMax(&peaks[gi].minkey, lo);
        }
    }
    if (psf) {
        const float ia = stats->inv_alpha;                               // exact power of two
        *reinterpret_cast<float4*>(psf + o) = make_float4(f01.y * m0 * ia, f01.w * m1 * ia, f23.y * m2 * ia, f23.w * m3 * ia);
    }
}

// The grids as wgtGrid_kernel leaves them (for inspection; the imaging path applies the same factor at the FFT input).
template <int WMODE>
__global__ void __launch_bounds__(256) k_weighted_copy(const size_t ncell, const float2* __restrict__ G,
                                                       const float* __restrict__ Gw, const int* __restrict__ cnt,
                                                       float2* __restrict__ G_out, float* __restrict__ Gw_out) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ncell) return;
    float u = 1.0f;
    if (cnt) { const int c = cnt[i]; if (c) u = 1.0f / (float)c; }
    if (G_out) { const float2 v = G[i]; G_out[i] = make_float2(v.x * u, v.y * u); }
    if (Gw_out) {
        if (WMODE) { const float2 w = reinterpret_cast<const float2*>(Gw)[i]; reinterpret_cast<float2*>(Gw_out)[i] = make_float2(w.x * u, w.y * u); }
        else Gw_out[i] = Gw[i] * u;
    }
}

// NEXT-4: "the data from a dirty image is divided into 2000 ranges".  bin = floor((v - lo) * (nbins /
// (hi - lo))) in fp32 without contraction, hi itself in the last bin, values outside [lo, hi] not counted; lo >= hi: the
// grid's own minimum and maximum from the peak search.  Shared-memory histogram per CTA, one global add per non-empty bin.
__global__ void __launch_bounds__(256) k_histogram(const float* __restrict__ image, const size_t npix, const int nbins,
                                                   float lo, float hi, const PeakSlot* __restrict__ peaks,
                                                   unsigned int* __restrict__ hist) {
    extern __shared__ unsigned int s_h[];
    const int gi = blockIdx.y;
    for (int i = threadIdx.x; i < nbins; i += 256) s_h[i] = 0u;
    if (!(lo < hi) && peaks) {
        hi = peak_unordered((unsigned int)(peaks[gi].maxkey >> 32));
        lo = peak_unordered(~peaks[gi].minkey);
    }
    const float scale = (lo < hi) ? __fdiv_rn((float)nbins, __fsub_rn(hi, lo)) : 0.0f;     // constant image (own range, hi == lo): everything in bin 0
    __syncthreads();
    const float* img = image + (size_t)gi * npix;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < npix; i += (size_t)gridDim.x * 256) {
        const float v = img[i];
        if (v >= lo && v <= hi) {
            const int b = min((int)floorf(__fmul_rn(__fsub_rn(v, lo), scale)), nbins - 1);
            atomicAdd(&s_h[b], 1u);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nbins; i += 256)
        if (s_h[i]) atomicAdd(&hist[(size_t)gi * nbins + i], s_h[i]);
}

// ------------------------------------------------------------------------------------------------- launchers
static inline unsigned blocks_for(long long n, int per) { return (unsigned)((n + per - 1) / per); }

cudaError_t launch_coords(const Geom& g, const float* uvw, const double* freq, const float2* vis, const float* wt,
                          const int* grid_id, long long nvis, const RowsShapeG* rows, double wstep, const PlaneMeta* planes,
                          Staged* staged, uint32_t* bin_count, Stats* stats, int* cnt, cudaStream_t s) {
    int iters = 4;                                                     // (the kernel holds the ranks of at most 4 blocks) enough CTAs to fill the machine a few times over
    while (iters > 1 && nvis / (256 * iters) < 148 * 8) iters >>= 1;
    if (rows) k_coords<1><<<blocks_for(nvis, 256 * iters), 256, 0, s>>>(g, *rows, uvw, freq, vis, wt, grid_id, nvis, iters, wstep, planes, staged,
                                                                       bin_count, stats, cnt);
    else k_coords<0><<<blocks_for(nvis, 256 * iters), 256, 0, s>>>(g, RowsShapeG{}, uvw, freq, vis, wt, grid_id, nvis, iters, wstep, planes, staged,
                                                                   bin_count, stats, cnt);
    return cudaGetLastError();
}

cudaError_t launch_scan_items(const Geom& g, uint32_t* bin_count, uint32_t* bin_offset, Item* items,
                              uint32_t* nitems, uint32_t* tops, cudaStream_t s) {
    const uint32_t nblocks = (g.nbins + 4095u) / 4096u;
    if (nblocks == 1) {
        k_scan_items_write<1><<<1, 1024, 0, s>>>(g, bin_count, tops, bin_offset, items, nitems);
        return cudaGetLastError();
    }
    k_scan_items_reduce<<<nblocks, 1024, 0, s>>>(g, bin_count, tops);
    k_scan_items_tops<<<1, 1024, 0, s>>>(g, nblocks, tops, bin_offset, nitems);
    k_scan_items_write<0><<<nblocks, 1024, 0, s>>>(g, bin_count, tops, bin_offset, items, nitems);
    return cudaGetLastError();
}

cudaError_t launch_scatter(const Geom& g, const Staged* staged, long long nsamples, const uint32_t* bin_offset,
                           Sample* sorted, cudaStream_t s) {
    k_scatter<<<blocks_for(nsamples, 256), 256, 0, s>>>(g, staged, nsamples, bin_offset, sorted);
    return cudaGetLastError();
}

static int generic_region_ints(int wmode, int smax) {
    const int R = kTile + (smax - 1);
    return ((wmode ? 4 : 3) * R * R + 3) & ~3;
}
static size_t generic_smem_bytes(int wmode, int smax, int Q, int pitch_max) {
    return (size_t)generic_region_ints(wmode, smax) * sizeof(int) + (size_t)(Q + 1) * pitch_max * (wmode ? 2 : 1) * sizeof(float);
}
static size_t fast_smem_bytes(int Q) {
    return (size_t)(3 * kFastR * kFastPitch + 1024 + 4 * kFastChunk + (Q + 1) * 8) * sizeof(float);
}

cudaError_t tiled_kernel_setup(int max_smem_bytes) {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(k_grid_tiled_generic<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes - 1024))) return e;
    if ((e = cudaFuncSetAttribute(k_grid_tiled_generic<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes - 1024))) return e;
    if ((e = cudaFuncSetAttribute(k_grid_tiled_s7, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes - 1024))) return e;
    return cudaSuccess;
}

cudaError_t launch_grid_tiled(const Geom& g, const Sample* sorted, const Item* items, const uint32_t* nitems,
                              const PlaneMeta* planes, const PlaneMeta* planes_host, const float* tables,
                              GridPtrs grids, int num_sms, cudaStream_t s) {
    const int P = g.wmode ? g.nplanes : 1;
    int smax = 1;
    for (int p = 0; p < P; ++p) smax = planes_host[p].support > smax ? planes_host[p].support : smax;
    if (!g.wmode && smax == 7 && g.chunk == kFastChunk) {
        k_grid_tiled_s7<<<num_sms * 4, 256, fast_smem_bytes(g.Q), s>>>(g, sorted, items, nitems, planes, tables, grids);
    } else {
        int pitch_max = 4;
        for (int p = 0; p < P; ++p) pitch_max = planes_host[p].pitch > pitch_max ? planes_host[p].pitch : pitch_max;
        const size_t smem = generic_smem_bytes(g.wmode, smax, g.Q, pitch_max);
        const int region = generic_region_ints(g.wmode, smax);
        int per_sm = (int)(220 * 1024 / (smem + 1024));
        per_sm = per_sm < 1 ? 1 : (per_sm > 4 ? 4 : per_sm);
        if (g.wmode) k_grid_tiled_generic<1><<<num_sms * per_sm, 256, smem, s>>>(g, sorted, items, nitems, planes, tables, grids, region);
        else k_grid_tiled_generic<0><<<num_sms * per_sm, 256, smem, s>>>(g, sorted, items, nitems, planes, tables, grids, region);
    }
    return cudaGetLastError();
}

cudaError_t launch_pack(const Geom& g, GridPtrs grids, float2* H, Stats* stats, cudaStream_t s) {
    const size_t ncell2 = (size_t)g.ngrids * g.ny * g.nx / 2;
    const unsigned blocks = (unsigned)((ncell2 + 255) / 256);
    const int* cnt = g.uniform ? grids.cnt : nullptr;
    if (g.wmode) k_pack<1><<<blocks, 256, 0, s>>>(ncell2, reinterpret_cast<const float4*>(grids.G), grids.Gw, cnt, reinterpret_cast<float4*>(H), stats);
    else k_pack<0><<<blocks, 256, 0, s>>>(ncell2, reinterpret_cast<const float4*>(grids.G), grids.Gw, cnt, reinterpret_cast<float4*>(H), stats);
    return cudaGetLastError();
}

cudaError_t launch_mirror_lower(const Geom& g, GridPtrs grids, cudaStream_t s) {
    const size_t total = (size_t)g.ngrids * (g.ny / 2) * g.nx;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    if (g.wmode) k_mirror_lower<1><<<blocks, 256, 0, s>>>(g.nx, g.ny, total, grids.G, grids.Gw, grids.cnt);
    else k_mirror_lower<0><<<blocks, 256, 0, s>>>(g.nx, g.ny, total, grids.G, grids.Gw, grids.cnt);
    return cudaGetLastError();
}

cudaError_t launch_weighted_copy(const Geom& g, GridPtrs grids, float2* G_out, float* Gw_out, cudaStream_t s) {
    const size_t ncell = (size_t)g.ngrids * g.ny * g.nx;
    const unsigned blocks = (unsigned)((ncell + 255) / 256);
    const int* cnt = g.uniform ? grids.cnt : nullptr;
    if (g.wmode) k_weighted_copy<1><<<blocks, 256, 0, s>>>(ncell, grids.G, grids.Gw, cnt, G_out, Gw_out);
    else k_weighted_copy<0><<<blocks, 256, 0, s>>>(ncell, grids.G, grids.Gw, cnt, G_out, Gw_out);
    return cudaGetLastError();
}

cudaError_t launch_histogram(const float* image, size_t npix, int ngrids, int nbins, float lo, float hi, const PeakSlot* peaks,
                             unsigned int* hist, cudaStream_t s) {
    const unsigned bx = (unsigned)std::min<size_t>((npix + 256 * 16 - 1) / (256 * 16), 592);
    k_histogram<<<dim3(bx ? bx : 1, (unsigned)ngrids), 256, (size_t)nbins * sizeof(unsigned int), s>>>(image, npix, nbins, lo, hi,
                                                                                                         peaks, hist);
    return cudaGetLastError();
}

cudaError_t launch_correct(const Geom& g, const float2* F, const float* icx, const float* icy, const Stats* stats,
                           float* dirty, float* psf, PeakSlot* peaks, cudaStream_t s) {
    const size_t total = (size_t)g.ngrids * g.ny * (g.nx / 4);
    k_correct<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(g.nx, g.ny, g.ngrids, F, icx, icy, stats, dirty, psf, peaks);
    return cudaGetLastError();
}

}  // namespace muser
