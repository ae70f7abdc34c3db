/* muser.h -- C ABI of the B200-native MUSER dirty-imaging hot path (arXiv 1712.06913).
 *
 * The path: calibrated visibilities -> [A1] coordinates + binning (counting sort by uv tile)
 *        -> [A2/A3/A4] convolutional gridding (2-D, w-projection planes, batched grids)
 *        -> [A5] 2-D inverse FFT (the library's own half-plane row pass + column pass for power-of-two sizes, cuFFT otherwise)
 *        -> [A6] grid correction + fftshift + real part (the column pass's epilogue)
 *        -> dirty image and dirty beam (PSF).
 * Paper passages (PAPER.md = the paper's text; DESIGN.md restates every reading R1..R21):
 *   "Gridding is the convolution of the visibilities with a particular function, which resamples the
 *    visibilities to lie on a regular rectangular grid"                        PAPER.md:78  (sec. 2)
 *   truncated spheroidal gridding convolution function                          PAPER.md:136-138 (sec. 3.2.3)
 *   "Inverse FFT is performed after gridding for generating dirty image"
 *   inputs "Visibilities and UVW (Phase corrected, Flagged)"                     PAPER.md:213 (Alg. 1)
 *   grid is float2, row-major iv*nu+iu, Hermitian                               PAPER.md:216-228 (Alg. 1 l.1-6)
 *   natural weighting multiplies by 1                                           PAPER.md:240-243 (Alg. 1 l.12-13)
 *   DIRTY_IMAGE: w-projection, gridding, inverse FFT "with the sun disk at the center",
 *   returns dirty image and dirty beam                                          PAPER.md:249-256 (Alg. 1 l.17-20)
 *   w-projection is used for the w-term                                         PAPER.md:126 (sec. 3.2.2)
 *
 * General rules
 *   - Plain C, no C++/torch types.  Every pointer argument says HOST or DEVICE.  DEVICE pointers must be on
 *     the CUDA device that was current when the handle was created.
 *   - The caller owns every data buffer; the library never frees or keeps them beyond the work it enqueues.
 *     The library owns the handle: grids, sort scratch, tables, correctors, cuFFT plan.  Scratch only grows.
 *   - Calls taking a muser_stream only ENQUEUE work on it (no host synchronisation) unless stated.
 *   - Every int-returning call returns MUSER_OK (0) or an error code; no exception or abort crosses the ABI.
 *     muser_last_error(h) gives the text of the last error on that handle (h = NULL: last create error).
 *   - Arrays are row-major [y][x] = [v][u].  Grid cell (iu, iv) <-> u = (iu - nx/2)/(nx*cell) wavelengths.
 *     Image pixel (x, y) <-> direction cosines l = (x - nx/2)*cell, m = (y - ny/2)*cell (no sky flip).
 *   - Outputs are un-normalised: a unit point source at the phase centre gives a peak of sum_weights
 *     (sum over gridded samples, conjugates included).
 *   - There is no CPU fallback anywhere: without a CUDA device create fails with MUSER_ECUDA.
 */
#ifndef MUSER_H_
#define MUSER_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct muser_imager muser_imager;     /* opaque; owned by the library */
typedef void* muser_stream;                   /* a cudaStream_t; NULL = the legacy default stream */

enum { MUSER_OK = 0, MUSER_EINVAL = 1, MUSER_ECUDA = 2, MUSER_ENOMEM = 3, MUSER_ESTATE = 4, MUSER_EUNSUPPORTED = 5 };
enum { MUSER_KERNEL_PSWF = 0, MUSER_KERNEL_GAUSS = 1 };
/* gridding strategies (muser_set_strategy).  OWNER: the grids are Hermitian, so only the half-plane of rows
 * ny/2 .. ny-1 is computed; every 64x32-cell tile of it has one writer that accumulates it in registers / fixed-point
 * shared memory and stores it once (no memset, no global atomics; 2-D mode with support 7 only, else
 * MUSER_EUNSUPPORTED at muser_grid); the other half-plane is rebuilt on demand (muser_get_grid).  TILED: work items of
 * <= 512 samples per 32x32 tile, shared memory accumulation, global reductions at the flush (any support, w planes).
 * WPLANE (w mode, PAPER.md:126, and 2-D mode with a support other than 7; every support <= 31): work items of <= 4096 records of one 32x32 tile, sorted by
 * plane; a run of records whose footprints share a 2x2-aligned (S+1) x (S+1) window is accumulated in registers and
 * merged into a fixed-point shared-memory region, which is added to the grids once per item.
 * AUTO picks OWNER where it applies, else WPLANE where it applies, else TILED.  (Value 1 was a per-sample
 * global-reduction strategy; it missed the image tolerance on dense grids and was removed.) */
enum { MUSER_STRATEGY_AUTO = 0, MUSER_STRATEGY_TILED = 2, MUSER_STRATEGY_OWNER = 3, MUSER_STRATEGY_WPLANE = 4 };
/* stage ids of muser_get_profile.  On the fused imaging path (ny = 256 ... 4096 a power of two, nx a multiple of 16) FFT is
 * the row pass (the library's own on the stored half-plane when nx is a power of two in [64, 4096], else cuFFT's on the
 * packed grid) and CORRECT the library's own column transform with the shift/correction epilogue; otherwise FFT is
 * cuFFT's 2-D transform and CORRECT the stand-alone correction kernel.  PACK only runs on the cuFFT paths. */
enum { MUSER_STAGE_BIN = 0, MUSER_STAGE_GRID = 1, MUSER_STAGE_PACK = 2, MUSER_STAGE_FFT = 3, MUSER_STAGE_CORRECT = 4,
       MUSER_STAGE_COUNT = 5 };

/* ---- A0 setup -------------------------------------------------------------------------------------------
 * Create an imager for nx x ny grids/images with pixel size cell_arcsec, a separable gridding kernel of FULL
 * width `support` cells (odd, R1) tabulated at `oversample` sub-cell phases (even), PSWF by default
 * (R2).  Requirements: nx, ny multiples of 4 and >= 2*(support+1); support odd in [1,63];
 * oversample even in [2,256]; cell_arcsec > 0.  Builds the table and the per-axis correctors (fp64 on the
 * host), allocates grids (zeroed), makes the cuFFT plan.  May synchronise.  Returns NULL on error. */
muser_imager* muser_imager_create(int nx, int ny, double cell_arcsec, int support, int oversample);
/* Frees everything the handle owns.  NULL is a no-op.  Synchronises the device. */
int muser_imager_destroy(muser_imager* h);
/* Choose the 2-D kernel: MUSER_KERNEL_PSWF (param ignored) or MUSER_KERNEL_GAUSS (param = a in cells of
 * exp(-(x/a)^2), 0 -> 1.55; R3).  Rebuilds table + correctors, leaves w-plane mode, zeroes the grids. */
int muser_set_kernel(muser_imager* h, int kind, double param);
/* Number of independent grids (A4, batched imaging: one grid per frame/channel/polarisation).
 * Reallocates and zeroes the grids.  ngrids >= 1. */
int muser_set_batch(muser_imager* h, int ngrids);
/* A3: w-projection with nplanes planes (R15).  HOST arrays, copied: w_centres[p] >= 0 (plane
 * centres in wavelengths of |w|), supports[p] odd in [1,63]; tables_c64[p] = supports[p]*oversample+1
 * interleaved (re,im) FLOAT pairs of the per-axis kernel, or tables_c64 == NULL: the library generates the
 * Fresnel-separable kernels of R15.  Caller tables must be EVEN, T[t] = T[S*Q - t] to 1e-5 of their maximum (else MUSER_EINVAL):
 * the gridders compute the Hermitian half-plane only, which equals the full gridding for even kernels (every gridding
 * kernel is).  Plane 0's (real part) table defines the grid correction.
 * nplanes == 0 returns to 2-D mode.  Zeroes the grids (the beam grid becomes complex). */
int muser_set_wplanes(muser_imager* h, int nplanes, const double* w_centres, const int* supports,
                      const float* const* tables_c64);
int muser_set_strategy(muser_imager* h, int strategy);
/* Tuning knobs of the OWNER strategy (results do not depend on them beyond fp32 summation order).  ITEM_SIZE: records
 * per chunk of a heavy tile (a tile with more records is split into chunks gridded by different CTAs and summed);
 * 0 (default) = chosen from the size of the call.  BIN_ITERS: blocks of 256 visibilities a binning CTA loops over
 * (1..64; 0 = automatic).  COLS_TMA: how the fused column transform fetches its strip of 8 columns: 1 = per-lane loads,
 * 2 = cp.async.bulk.tensor (TMA) into shared memory, 0 = the library's default.  FFT_SUBBATCH: grids per rows -> columns
 * sub-batch of the fused transform (the row transform of a sub-batch stays in L2 until its column pass has read it);
 * 0 (default) or >= ngrids = all rows, then all columns, which measured fastest. */
enum { MUSER_TUNE_ITEM_SIZE = 0, MUSER_TUNE_BIN_ITERS = 1, MUSER_TUNE_COLS_TMA = 2, MUSER_TUNE_FFT_SUBBATCH = 3, MUSER_TUNE_COUNT = 4 };
int muser_set_tuning(muser_imager* h, int key, int value);
/* 1 (default): A6 divides by the kernel's transform; 0: A6 only shifts/takes the real part (parity gate R9(i)). */
int muser_set_grid_correction(muser_imager* h, int enabled);
/* Weighting mode of Alg. 1 ("weighting mode: weight_mode, natural or uniform").  NATURAL (default): the
 * per-visibility weight only.  UNIFORM: the gridder also keeps the integer hit-count grid `cnt` (one hit per gridded
 * sample -- visibility or conjugate -- at its nearest cell) and the paper's wgtGrid_kernel is applied where the grids
 * enter the FFT: a cell of the visibility grid AND of the beam grid is multiplied by 1/cnt where cnt != 0, and left
 * alone where cnt == 0 (reading R22).  The accumulated grids are not modified; muser_get_weighted_grid shows the
 * weighted ones.  Changing the mode reallocates and zeroes the grids.  May synchronise. */
enum { MUSER_WEIGHT_NATURAL = 0, MUSER_WEIGHT_UNIFORM = 1 };
int muser_set_weighting(muser_imager* h, int mode);
/* Phase correction of the visibilities (PAPER.md:174 step 3, :286 Alg. 1 IMPROVED_CLEAN; Table 3 row 4), fused into A1:
 * from the next muser_grid on, every visibility is multiplied by exp(+2 pi i (u dl + v dm)) (u, v in wavelengths) before
 * it is gridded, which moves the point at direction cosines (dl, dm) -- the measured offset of the solar disk -- to the
 * phase centre (reading R24).  (0, 0) switches it off.  The beam does not depend on it. */
int muser_set_phase_offset(muser_imager* h, double dl, double dm);
/* NEXT-2b: CLEAN wants a beam twice the size of the image.  When enabled, every muser_grid /
 * muser_grid_batched call also grids the weights onto a second set of grids of 2nx x 2ny cells (same cell size, same
 * kernel), and muser_psf2x returns that beam: DEVICE float [ngrids][2ny][2nx].  muser_frame_host(_async) grids it too.  Later
 * muser_set_kernel / muser_set_strategy / muser_set_batch / muser_set_weighting calls apply to it as well.  2-D mode only:
 * while it is enabled muser_set_wplanes(n > 0) returns MUSER_EUNSUPPORTED.  May synchronise. */
int muser_set_psf2x(muser_imager* h, int enabled);
int muser_psf2x(muser_imager* h, float* beam2x_out, muser_stream s);

/* ---- A1..A4 gridding --------------------------------------------------------------------------------------
 * Zero the grids, the sum of weights and the counters (asynchronous on s).  On the OWNER strategy the zeroing is lazy: the
 * tiles of the stored half-plane that the following muser_grid calls do not touch are flagged as zeros and never written
 * (the row transform skips them); muser_get_grid and every other consumer of the dense grids see exact zeros there. */
int muser_reset(muser_imager* h, muser_stream s);
/* Grid nvis visibilities AND their Hermitian conjugates (-u,-v,-w, conj V) (R6), accumulating
 * onto what is already there (time integration; R16).  DEVICE pointers:
 *   uvw_m   float  [nvis][3]  baseline coordinates in metres
 *   freq_hz double [nvis]     observing frequency of each visibility (u_lambda = u_m * freq/c)
 *   vis_c64 float  [nvis][2]  complex visibility (re, im)
 *   weight  float  [nvis]     weight; <= 0 or non-finite inputs flag the visibility (skipped and counted)
 * Visibilities whose kernel footprint (either sample's) leaves cells [1, n-1] are dropped and counted (R5).
 * nvis == 0 is a no-op.  grid_id (batched): int [nvis], 0 <= grid_id < ngrids, else flagged. */
int muser_grid(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64,
               const float* weight, long long nvis, muser_stream s);
int muser_grid_batched(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64,
                       const float* weight, const int* grid_id, long long nvis, muser_stream s);

/* NEXT-1, the channelised call (a 3 ms frame is 16 channels x 2 polarisations of the SAME baselines): the
 * same gridding as muser_grid on the visibilities (t, p, c, r) with coordinates uvw_m[t][r] * freq_hz[c] / c, in the
 * instrument's own layout, 12.4 instead of 32 bytes per visibility.  DEVICE pointers:
 *   uvw_m   float  [ntime][nrow][3]           baseline coordinates in metres, one set per time step
 *   freq_hz double [nchan]                    channel frequencies
 *   vis_c64 float  [ntime][npol][nchan][nrow][2]
 *   weight  float  [ntime][npol][nchan][nrow]
 *   grid_id int    MUSER_POLS_SUM:   [ntime][nchan]        the polarisations of a (time, channel) go onto one grid; their
 *                                                          weighted visibilities are added up before gridding (one
 *                                                          kernel evaluation per baseline and channel instead of npol)
 *                  MUSER_POLS_SPLIT: [ntime][npol][nchan]  one grid per polarisation (the paper's per-channel,
 *                                                          per-polarisation images)
 *                  NULL: everything onto grid 0
 * The result is that of muser_grid(_batched) on the flattened arrays (the order of the fp32 sums differs); flags, drops
 * and counters are per visibility as there.  npol <= 8.  Every strategy has the channelised binning kernels (owner tiles:
 * k_rows_count / k_rows_scatter; w planes and other supports: k_coords<ROWS>). */
enum { MUSER_POLS_SUM = 0, MUSER_POLS_SPLIT = 1 };
int muser_grid_rows(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64, const float* weight,
                    const int* grid_id, long long nrow, int nchan, int npol, int ntime, int pol_mode, muser_stream s);

/* ---- A5 + A6 imaging --------------------------------------------------------------------------------------
 * DEVICE outputs float [ngrids][ny][nx].  One complex inverse FFT of H = G + i*Gw yields both images (the
 * dirty image is its real part, the beam its imaginary part, because G and Gw are Hermitian); muser_dirty and
 * muser_psf share that transform when called back to back.  The accumulated grids are NOT destroyed: both may
 * be called, in either order, and gridding may continue afterwards.  Either output of muser_dirty_psf may be NULL. */
int muser_dirty(muser_imager* h, float* image_out, muser_stream s);
int muser_psf(muser_imager* h, float* beam_out, muser_stream s);
int muser_dirty_psf(muser_imager* h, float* image_out, float* beam_out, muser_stream s);

/* ---- consumers of the dirty image (NEXT-4) -----------------------------------------------------------------------
 * "Find the strength and position of the peak in the dirty map" (Alg. 1 l.33/36): when enabled, every
 * muser_dirty / muser_dirty_psf also keeps, per grid, the maximum of the dirty image with its position (lowest index
 * among equal values) and the minimum, found in the epilogue that writes the image (no extra pass).  muser_get_peak
 * synchronises the last stream; HOST outputs of ngrids entries, any may be NULL. */
int muser_set_peak_search(muser_imager* h, int enabled);
int muser_get_peak(muser_imager* h, float* peak_value, int* peak_x, int* peak_y, float* min_value);
/* "the data from a dirty image is divided into 2000 ranges" (the input of the GMM): histogram of `image`
 * (DEVICE float [ngrids][ny][nx]) into nbins equal ranges of [lo, hi]: bin = floor((v - lo) * (nbins / (hi - lo))) in
 * fp32, hi itself in the last bin, values outside not counted.  lo >= hi: each grid's own minimum and maximum from the
 * peak search of the last muser_dirty (reading R23); MUSER_ESTATE if the peak search is off or no dirty image has been made
 * since it was switched on; a constant image (minimum == maximum) goes to bin 0.  hist_out: DEVICE unsigned [ngrids][nbins], overwritten. */
int muser_histogram(muser_imager* h, const float* image, int nbins, float lo, float hi, unsigned int* hist_out, muser_stream s);

/* The same own-range histogram for callers that cannot allocate device memory: no handle, no cudaMalloc / cudaFree and no
 * allocating library call, on any call.  Meant for a steady-state monitoring loop, where cudaMalloc would
 * synchronise the device and stall the imaging streams, and for processes in which another allocator (a framework's caching
 * pool) already holds the HBM so that cudaMalloc fails.  The only scratch the histogram needs -- one minimum / maximum slot per
 * image -- is a fixed __device__ array inside the library (16 KB, held by every GPU that loads libmuser.so until exit).
 *   image    DEVICE float [ngrids][npix]      any images (non-finite pixels are ignored), on the CURRENT device
 *   hist_out DEVICE unsigned [ngrids][nbins]  overwritten; image g is binned over its own [min, max] exactly as
 *                                             muser_histogram(lo >= hi) bins the dirty image (reading R23); an image without a
 *                                             finite pixel gives zeros, a constant image puts everything into bin 0
 *   err_out  HOST char [err_cap] or NULL      text of the error when the return code is not MUSER_OK
 * Limits and sharing: 1 <= ngrids <= MUSER_STATIC_MAX_GRIDS, else MUSER_EINVAL and nothing is enqueued; 1 <= nbins <= 8192;
 * npix >= 1.  All calls on a device share the one array.  Each call first clears the slots it uses (they still hold the
 * previous call's values), so calls queued on ONE stream are independent of each other; calls that may overlap on the GPU
 * (different streams without an event between them) race on the slots.  The first call on each device also looks up the
 * array's device address (cudaGetSymbolAddress; the runtime loads the module then): make it at start-up, before any stream
 * capture.  Only enqueues on s (two memsets, two kernels); the caller synchronises s before reading hist_out. */
#define MUSER_STATIC_MAX_GRIDS 1024
int muser_histogram_static(const float* image, long long npix, int ngrids, int nbins, unsigned int* hist_out, muser_stream s,
                           char* err_out, int err_cap);

/* ---- whole path with HOST buffers (end-to-end entry point) ------------------------------------------------
 * reset -> copy the inputs to the device -> grid -> dirty + psf -> copy the images back, all on s, then
 * synchronises s.  HOST pointers (pinned memory makes the copies asynchronous); grid_id may be NULL;
 * image_out / beam_out (float [ngrids][ny][nx]) may each be NULL. */
int muser_frame_host(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64,
                     const float* weight, const int* grid_id, long long nvis, float* image_out, float* beam_out,
                     muser_stream s);
/* The same without the final synchronisation (after the first call has sized the staging buffers it only enqueues):
 * with pinned HOST buffers, two handles on two streams overlap one batch's copy back with the next batch's upload and
 * imaging.  The caller synchronises the stream before reading the images or re-using the input buffers. */
int muser_frame_host_async(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64,
                           const float* weight, const int* grid_id, long long nvis, float* image_out, float* beam_out,
                           muser_stream s);

/* ---- inspection ---------------------------------------------------------------------------------------------
 * Copy the centred grids (DC at [ny/2][nx/2]) to DEVICE buffers: grid_c64_out float [ngrids][ny][nx][2];
 * wgrid_out float [ngrids][ny][nx] (2-D mode) or [ngrids][ny][nx][2] (w mode).  Either may be NULL. */
int muser_get_grid(muser_imager* h, void* grid_c64_out, float* wgrid_out, muser_stream s);
/* Uniform mode only: the hit counts, DEVICE int [ngrids][ny][nx]; and the grids as wgtGrid_kernel leaves them (same
 * layouts as muser_get_grid; in natural mode the same as muser_get_grid). */
int muser_get_counts(muser_imager* h, int* counts_out, muser_stream s);
int muser_get_weighted_grid(muser_imager* h, void* grid_c64_out, float* wgrid_out, muser_stream s);
/* Kernel table of `plane` as used on the device, in the oracle's order T[t], t = 0..S*Q (2-D mode: floats;
 * w mode: (re,im) pairs).  HOST output; *len in: capacity in floats, out: floats written. */
int muser_get_table(muser_imager* h, int plane, float* table_out_host, int* len);
/* HOST outputs (any may be NULL).  Synchronises the last stream used.  sum_weights counts both samples of a
 * kept visibility; n_gridded counts kept visibilities. */
int muser_get_stats(muser_imager* h, double* sum_weights, long long* n_gridded, long long* n_dropped,
                    long long* n_flagged);
const char* muser_last_error(const muser_imager* h);

/* ---- measurement -----------------------------------------------------------------------------------------
 * enabled = 1: bracket every stage with CUDA events on the caller's stream (adds host work; do not enable it
 * inside a throughput measurement).  muser_get_profile synchronises and returns, per stage, the summed device
 * time in milliseconds and the number of launches since profiling was enabled (HOST arrays of MUSER_STAGE_COUNT). */
int muser_set_profiling(muser_imager* h, int enabled);
int muser_get_profile(muser_imager* h, double* stage_ms, long long* stage_launches);
/* Number of the library's own kernels launched on this handle since creation (cuFFT's and memsets not counted). */
long long muser_get_launch_count(const muser_imager* h);

/* ---- host-only helpers (no GPU needed; used by the table-parity tests) ---------------------------------------
 * The library's own fp64 generators: kernel table T[t], t = 0..S*Q (kind as above; param: Gaussian a), and
 * the per-axis corrector c[x], x = 0..n-1, of a real table.  HOST outputs of S*Q+1 and n doubles. */
int muser_host_table(int kind, int support, int oversample, double param, double* table_out);
int muser_host_wtable(int support, int oversample, double w_lambda, double fov_rad, double* table_out_re_im);
int muser_host_corrector(const double* table, int support, int oversample, int n, double* corr_out);
const char* muser_version(void);
/* Device microbenchmarks behind the roofline discussion; needs a GPU, synchronises the device.
 * kind 0: FP32 FMA (flop/s), 1: packed FFMA2 (flop/s), 2: native 32-bit shared-memory integer adds (adds/s),
 * 3: fp32 shared-memory adds = compare-and-swap loops (adds/s), 4: fp32 global reductions over 256 MB (adds/s).
 * HOST output. */
int muser_microbench(int kind, double* rate_out);

#ifdef __cplusplus
}
#endif
#endif /* MUSER_H_ */
