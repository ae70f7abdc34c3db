// Internal declarations shared by the kernels (muser_kernels.cu) and the C ABI (muser_api.cu).
// Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace muser {

constexpr int kTile = 32;          // uv tile edge in cells (A1 sort key, A2 shared-memory accumulator)
constexpr int kTileShift = 5;
constexpr int kMaxPlanes = 64;
constexpr uint32_t kNoBin = 0xFFFFFFFFu;

// Geometry and mode, passed by value to every kernel.
struct Geom {
    int nx, ny, Q, ngrids, nplanes, wmode;
    double su, sv;                 // nx*cell, ny*cell (rad): u_pix = u_lambda*su + nx/2 (O1)
    int ntx, nty;                  // tiles per axis; tile tx covers cells [tx*32-16, tx*32+16) so DC sits mid-tile
    uint32_t nbins;                // ngrids*max(nplanes,1)*nty*ntx
    int chunk;                     // samples per work item of the tiled gridder
    int S;                         // support of plane 0 (the 2-D kernel)
    int ntiles;                    // nty*ntx
    int otx, oty, ontiles;         // owner-tile path: tiles per row (kOwTileW cells wide), tile rows of the stored
                                   // half-plane (rows ny/2 .. ny-1, 32 cells tall), tiles per grid = oty*otx
    uint32_t onbins;               // ngrids*ontiles
    int phase_on;                  // NEXT-3: V *= exp(+2 pi i (u dl + v dm)) before gridding
    double dl, dm;
    int uniform;                   // NEXT-2: hit counts are accumulated and wgtGrid (cell / count) is applied at the FFT input
    int wtile;                     // generic binning: bins ordered (grid, tile, plane) instead of (grid, plane, tile) -- the
                                   // w-projection window gridder (muser_wgrid.cu) works through a tile's planes in one item
};

// Per-plane kernel metadata in constant-ish device memory.
struct PlaneMeta {
    int support;                   // S_p (odd)
    int pitch;                     // row pitch of the transposed table TT[r][j], j < pitch, entries >= S_p are 0
    int offset;                    // offset of the plane's TT in the table buffer (floats in 2-D mode, float2 in w mode)
    int pad;                       // float bits: bound (>= 1) on |kx ky| of the plane's table (fixed-point scale of the tiled gridder)
    double wc;                     // plane centre in |w| wavelengths
};

// K1 output, one per SAMPLE (2 per visibility; slot 2k = primary, 2k+1 = conjugate).
struct __align__(16) Staged {
    float re, im, wt;              // wt*Re V, +-wt*Im V, wt
    uint32_t cell;                 // iu0 | iv0 << 16 (nearest grid cell)
    uint32_t phase;                // rx | ry << 9 | kconj << 18, rx = Q/2 - ru in [0, Q]
    uint32_t bin;                  // ((g*P + p)*nty + ty)*ntx + tx, or kNoBin if the sample is not gridded
    uint32_t rank;                 // arrival order inside the bin (tiled strategy)
    uint32_t gp;                   // grid | plane << 24
};

// K3 output, tile-sorted, 16 B: what the tiled gridder streams.
struct __align__(16) Sample {
    float re, im, wt;
    uint32_t packed;               // lx | ly << 5 | rx << 10 | ry << 19 | kconj << 28 (lx, ly: cell inside the tile)
};

struct Item {                      // work item of the tiled gridder: <= chunk samples of one bin
    uint32_t bin, start, count;
};

struct Stats {
    double sum_weights;
    unsigned long long n_gridded, n_dropped, n_flagged;
    double sum_val2, sum_wt2;      // sum |wt*V|^2 and sum wt^2 over kept visibilities: scale of G against Gw
    float alpha, inv_alpha;        // written by k_pack: H = G + i*alpha*Gw, alpha a power of two
};

struct GridPtrs {
    float2* G;                     // [ngrids][ny][nx] complex
    float* Gw;                     // [ngrids][ny][nx] real (2-D) or complex interleaved (w mode)
    int* cnt;                      // [ngrids][ny][nx] hit counts (uniform weighting only, else null); rows >= ny/2 are
                                   // accumulated, the rest is mirrored on demand like G
};

// NEXT-3 (PAPER.md:174 step 3, :286): V * exp(+2 pi i (u dl + v dm)), u, v in wavelengths; the phase is reduced in fp64,
// the rotation is fp32
__device__ __forceinline__ float2 phase_rotate(const Geom& g, float um, float vm, double f, float2 V) {
    const double il = __ddiv_rn(f, 299792458.0);
    double x = __dmul_rn((double)um, il) * g.dl + __dmul_rn((double)vm, il) * g.dm;
    x -= rint(x);
    float sn, cs;
    sincospif(2.0f * (float)x, &sn, &cs);
    return make_float2(V.x * cs - V.y * sn, V.x * sn + V.y * cs);
}

// NEXT-4: per-grid peak search of the dirty image.  key = ordered(value) << 32 | ~flat index: atomicMax keeps the largest
// value and, among equal values, the lowest index; the minimum is kept as the maximum of the inverted ordered value.
struct PeakSlot { unsigned long long maxkey; unsigned int minkey; unsigned int pad; };
__device__ __forceinline__ unsigned int peak_ordered(float v) {
    const unsigned int b = __float_as_uint(v);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float peak_unordered(unsigned int o) {
    return __uint_as_float((o & 0x80000000u) ? (o & 0x7FFFFFFFu) : ~o);
}

// ---- launch wrappers (muser_kernels.cu); all asynchronous on `s` -------------------------------------------
// channelised input of the generic binning kernel: elements (t, po, c, r), npi polarisations summed per element
struct RowsShapeG { int ntime, npo, npi, nchan, nrow; };
// nvis: visibilities (flat call, rows == nullptr) or elements (rows call).  wstep > 0: the plane centres are exactly the
// ladder p * wstep (the nearest plane is then found in O(1))
cudaError_t launch_coords(const Geom& g, const float* uvw, const double* freq, const float2* vis, const float* wt,
                          const int* grid_id, long long nvis, const RowsShapeG* rows, double wstep, const PlaneMeta* planes, Staged* staged,
                          uint32_t* bin_count, Stats* stats, int* cnt, cudaStream_t s);
// items == nullptr: offsets only (the caller builds its own work items from them)
cudaError_t launch_scan_items(const Geom& g, uint32_t* bin_count, uint32_t* bin_offset, Item* items,
                              uint32_t* nitems, uint32_t* tops, cudaStream_t s);
cudaError_t launch_scatter(const Geom& g, const Staged* staged, long long nsamples, const uint32_t* bin_offset,
                           Sample* sorted, cudaStream_t s);
cudaError_t launch_grid_tiled(const Geom& g, const Sample* sorted, const Item* items, const uint32_t* nitems,
                              const PlaneMeta* planes, const PlaneMeta* planes_host, const float* tables,
                              GridPtrs grids, int num_sms, cudaStream_t s);
cudaError_t launch_pack(const Geom& g, GridPtrs grids, float2* H, Stats* stats, cudaStream_t s);
cudaError_t launch_weighted_copy(const Geom& g, GridPtrs grids, float2* G_out, float* Gw_out, cudaStream_t s);
cudaError_t launch_histogram(const float* image, size_t npix, int ngrids, int nbins, float lo, float hi, const PeakSlot* peaks,
                             unsigned int* hist, cudaStream_t s);
cudaError_t launch_mirror_lower(const Geom& g, GridPtrs grids, cudaStream_t s);
cudaError_t launch_correct(const Geom& g, const float2* F, const float* icx, const float* icy, const Stats* stats,
                           float* dirty, float* psf, PeakSlot* peaks, cudaStream_t s);
cudaError_t tiled_kernel_setup(int max_smem_bytes);

// ---- w-projection window gridder (muser_wgrid.cu): w mode, every plane support <= 31
bool wgrid_supported(const PlaneMeta* planes_host, int P, int Q, int max_smem_bytes);
cudaError_t wgrid_kernel_setup(int max_smem_bytes);
size_t wgrid_list_cap(const Geom& g, size_t nsamples);
cudaError_t launch_wtile_items(const Geom& g, const uint32_t* bin_offset, const PlaneMeta* planes, Item* items, uint32_t* lists,
                               uint32_t list_cap, uint32_t* nitems, uint32_t* ctl, cudaStream_t s);
int launch_wgrid(const Geom& g, const Sample* sorted, const Item* items, const uint32_t* lists, uint32_t list_cap, uint32_t* ctl,
                 const uint32_t* bin_offset, const PlaneMeta* planes, const PlaneMeta* planes_host, const float* tables,
                 GridPtrs grids, int num_sms, cudaStream_t s, const cudaStream_t* side, const cudaEvent_t* ev, cudaError_t* err);

// ---- owner-tile path (muser_owner.cu): 2-D mode, support 7.  The grids are Hermitian (every visibility is gridded
// with its conjugate), so only the half-plane of rows ny/2 .. ny-1 is computed and stored; k_mirror_lower rebuilds
// the other half for consumers that want the full grid.  Every 64x32 tile of the stored half-plane has exactly one
// writer, so it is written with plain stores (no memset, no global atomics); samples whose footprint crosses a tile
// edge are listed in every tile they touch.
constexpr int kOwTileW = 64;                 // owner tiles are 64 cells wide, 32 tall
constexpr int kOwTileFloats = kOwTileW * 32 * 3;   // one partial tile in the scratch buffer: A[32][W] float2 + B[32][W] float
// two-parity transposed table TT2[(par*(Q+1) + r)*8 + i]: par 0: i = j (j = 0..6: T[j*Q + r]), [7] = 0;
// par 1: [0] = 0, i = j + 1
struct OwItem {                              // one chunk of a heavy tile (more than item_size samples)
    uint32_t bin, start, count, first_slot, nchunks, chunk;
};
int owner_bin_iters(long long nvis, int forced);
size_t owner_bin_ctas(long long nvis, int iters);
cudaError_t launch_owner_count(const Geom& g, const float* uvw, const double* freq, const float2* vis, const float* wt,
                               const int* grid_id, long long nvis, uint32_t* bin_count, uint32_t* cta_hist, Stats* stats,
                               uint4* loc, int iters, cudaStream_t s);
cudaError_t launch_owner_scan(const Geom& g, uint32_t* bin_count, uint32_t* cursor, uint32_t* bin_offset, OwItem* items,
                              uint32_t* nitems, uint32_t item_size, uint4* work, uint32_t* ctl, uint32_t* tops,
                              uint32_t* valid_reset, cudaStream_t s);   // valid_reset != nullptr: clear the tile flags (first call after a reset)
cudaError_t launch_owner_scatter(const Geom& g, const uint4* loc, const float* uvw, const double* freq, const float2* vis,
                                 const float* wt, const int* grid_id, long long nvis, const uint32_t* bin_offset,
                                 const uint32_t* cta_hist, uint32_t* cursor, uint4* sorted, int* cnt, int iters,
                                 cudaStream_t s);
// channelised entry point (NEXT-1): elements (t, po, c, r); pols_split = 0: the polarisations of an element are summed
int rows_cpc(int ntime, int npo, int nchan, int nrow);
size_t rows_ctas(int ntime, int npol, int nchan, int nrow, int pols_split, int cpc);
cudaError_t launch_rows_count(const Geom& g, int ntime, int npol, int nchan, int nrow, int pols_split, int cpc, const float* uvw,
                              const double* freq, const float2* vis, const float* wt, const int* grid_id, uint32_t* bin_count,
                              uint32_t* cta_hist, Stats* stats, uint4* loc, cudaStream_t s);
cudaError_t launch_rows_scatter(const Geom& g, int ntime, int npol, int nchan, int nrow, int pols_split, int cpc,
                                const uint4* loc, const float* uvw, const double* freq, const float2* vis, const float* wt,
                                const int* grid_id, const uint32_t* bin_offset, const uint32_t* cta_hist, uint32_t* cursor,
                                uint4* sorted, int* cnt, cudaStream_t s);
int rows_max_channels();
cudaError_t owner_kernel_setup(int max_smem_bytes);
cudaError_t launch_owner_grid(const Geom& g, const uint4* sorted, const uint32_t* bin_offset,
                              const OwItem* items, const uint32_t* nitems, const uint4* work, uint32_t* ctl,
                              const float* tt2, GridPtrs grids, float* scratch, uint32_t* tickets, uint32_t* valid,
                              int first, int num_sms, cudaStream_t s);   // first: first call after a reset (every tile is stored)
// valid [ngrids * ontiles (+ pad to a multiple of 4)]: 0 = the tile has not been written since the last reset (its cells
// stand for zeros whatever they hold).  Zero those tiles and flag them:
cudaError_t launch_owner_fill_invalid(const Geom& g, GridPtrs grids, uint32_t* valid, cudaStream_t s);

// ---- fused column transform + correction (muser_fft.cu): ny = 256, 512, 1024, 2048 or 4096, nx a multiple of 16
bool fft_cols_supported(int nx, int ny);
int fft_cols_first_radix(int ny);
cudaError_t fft_cols_setup();
// row pass on the stored half-plane (nx a power of two in [64, 4096]): Z = row transform of G + i alpha Gw, all ny rows
bool fft_rows_supported(int nx, int ny, int wmode);
int fft_rows_first_radix(int nx);
cudaError_t fft_rows_setup();
// valid != nullptr: tile flags of the owner gridder (tiles at 0 stand for zeros and are not loaded); at most 96 tiles per row
cudaError_t launch_fft_rows_half(const Geom& g, const float2* G, const float* Gw, const int* cnt, const float2* tw,
                                 Stats* stats, float2* Z, const uint32_t* valid, int grid_begin, int grid_count, int num_sms,
                                 cudaStream_t s);                       // grids [grid_begin, grid_begin + grid_count)
// tmap128 != nullptr: the strip is staged by TMA (tensor map from fft_cols_make_tmap), else by per-lane loads
bool fft_cols_make_tmap(void* map128, const float2* F1, int nx, int ny, int ngrids);
// tw8 != nullptr (ny = 512, 1024, with the TMA staging): two radix-8 stages after the first one instead of three radix-4 ones
bool fft_cols_radix8(int ny);
cudaError_t launch_fft_cols_correct(const Geom& g, const float2* F1, const float2* tw, const float2* tw8, const float* icx,
                                    const float* icy, const Stats* stats, float* dirty, float* psf, PeakSlot* peaks,
                                    const void* tmap128, int grid_begin, int grid_count, cudaStream_t s);

}  // namespace muser
