// C ABI of the MUSER dirty-imaging library (include/muser.h): handle, validation, setup (A0), stage sequencing.
// Every step of the data path runs in the kernels of muser_kernels.cu (+ cuFFT for A5); this file only
// validates, allocates and enqueues.
#include "../../include/muser.h"
#include "muser_internal.h"
#include "tables.h"

#include <cufft.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

using namespace muser;

static thread_local std::string g_create_error;
static const double kArcsec = 3.14159265358979323846 / 648000.0;
static const bool kColsTmaDefault = true;      // column pass staged by TMA unless MUSER_TUNE_COLS_TMA says otherwise (measured: DESIGN.md 5)

struct StageEvent {
    cudaEvent_t a, b;
    int stage;
};

struct muser_imager {
    int nx = 0, ny = 0, S = 0, Q = 0;
    double cell_arcsec = 0;
    int kind = MUSER_KERNEL_PSWF;
    double gauss_a = 1.55;
    int ngrids = 1, nplanes = 0, strategy = MUSER_STRATEGY_AUTO, correction = 1;
    int device = 0, num_sms = 148, max_smem = 0;
    int tune[MUSER_TUNE_COUNT] = {0};
    Geom geom{};
    std::vector<PlaneMeta> planes_h;
    std::vector<std::vector<float>> tables_f32;     // per plane, oracle order T[t] (floats or (re,im) pairs)
    PlaneMeta* planes_d = nullptr;
    float* tables_d = nullptr;
    float *icx_d = nullptr, *icy_d = nullptr, *ones_d = nullptr;
    float2* G = nullptr;
    float* Gw = nullptr;
    float2* H = nullptr;
    int* cnt = nullptr;                     // hit counts (uniform weighting only)
    int weighting = MUSER_WEIGHT_NATURAL;
    double off_l = 0.0, off_m = 0.0;        // phase-centre offset (NEXT-3)
    bool peak_search = false;               // NEXT-4: peak / minimum of the dirty image kept per grid
    PeakSlot* peaks_d = nullptr;
    bool peaks_valid = false;               // a dirty image has filled peaks_d since the search was enabled / the grids were (re)allocated
    muser_imager* child2x = nullptr;        // NEXT-2b: imager of 2nx x 2ny pixels gridding the weights only
    Staged* staged = nullptr;
    Sample* sorted = nullptr;
    size_t sample_cap = 0;
    uint32_t *bin_count = nullptr, *bin_offset = nullptr, *nitems_d = nullptr, *bin_tops = nullptr;
    Item* items = nullptr;
    size_t bins_cap = 0, items_cap = 0;
    Stats* stats_d = nullptr;
    // owner-tile path
    float* ttp_d = nullptr;                 // padded transposed table (2-D mode, support 7), else null
    OwItem* ow_items = nullptr;
    uint32_t* ow_tickets = nullptr;
    float* ow_scratch = nullptr;
    size_t ow_items_cap = 0, ow_sorted_cap = 0, ow_bins_cap = 0;
    uint4 *ow_sorted = nullptr, *ow_loc = nullptr;          // tile-sorted records; per-visibility integer result of O1
    uint32_t *ow_count = nullptr, *ow_cursor = nullptr, *ow_offset = nullptr, *ow_ctl = nullptr, *ow_tops = nullptr;
    uint4* ow_work = nullptr;
    uint32_t* wg_ctl = nullptr;             // work counters and list lengths of the w-plane window gridder (per window shape)
    uint32_t* wg_lists = nullptr;           // per shape: the items that hold records of it
    size_t wg_list_cap = 0;
    cudaStream_t wg_side[7] = {};           // side streams / fork-join events of its per-shape kernels
    cudaEvent_t wg_ev[8] = {};
    bool wg_streams_ok = false;
    alignas(64) unsigned char tmap[128] = {};   // CUtensorMap of H (column pass staged by TMA)
    bool tmap_tried = false, tmap_ok = false;
    double wstep = 0.0;                     // > 0: the plane centres are the ladder p * wstep (O(1) plane search in K1)
    uint32_t* ow_cta_hist = nullptr;        // per binning CTA: its shared tile histogram (k_owner_count -> k_owner_scatter)
    size_t ow_cta_hist_cap = 0;
    bool weights_only = false;              // the 2x-beam child: muser_grid is called without visibilities
    bool zero_pending = false;              // muser_reset was called and the grids have not been zeroed yet
    uint32_t* ow_valid = nullptr;           // owner path: per (grid, tile) flag, 0 = not written since the last reset (stands for zeros)
    bool sparse = false;                    // some flags may be 0: G, Gw are not dense (flush_zero makes them so)
    bool lower_valid = true;                // rows 0 .. ny/2-1 of G, Gw are up to date (the owner gridder stores rows >= ny/2 only)
    cufftHandle plan = 0, plan_rows = 0;
    bool plan_ok = false, plan_rows_ok = false, fft_valid = false;
    bool fused_fft = false;                 // row pass by cuFFT, column pass + correction by k_fft_cols_correct
    bool fused_rows = false;                // row pass by k_fft_rows_half on the stored half-plane (nx a power of two)
    float2* tw_d = nullptr;                 // per-stage twiddles of the fused column transform
    float2* tw8_d = nullptr;                // ... of its radix-8 variant (ny = 512, 1024)
    float2* tw_rows_d = nullptr;            // ... and of the row transform
    cudaStream_t last_stream = nullptr;
    // host-frame staging (muser_frame_host)
    float* in_uvw = nullptr; double* in_freq = nullptr; float2* in_vis = nullptr; float* in_wt = nullptr; int* in_gid = nullptr;
    size_t in_cap = 0;
    float *out_dirty = nullptr, *out_psf = nullptr;
    // profiling
    bool profiling = false;
    std::vector<StageEvent> ev_used, ev_free;
    double stage_ms[MUSER_STAGE_COUNT] = {0};
    long long stage_n[MUSER_STAGE_COUNT] = {0};
    long long n_launches = 0;
    std::string err;
};

static int fail(muser_imager* h, int code, const std::string& msg) {
    if (h) h->err = msg; else g_create_error = msg;
    return code;
}
#define CU(h, expr)                                                                                   \
    do {                                                                                              \
        cudaError_t e_ = (expr);                                                                      \
        if (e_ != cudaSuccess)                                                                        \
            return fail(h, e_ == cudaErrorMemoryAllocation ? MUSER_ENOMEM : MUSER_ECUDA,              \
                        std::string(#expr) + ": " + cudaGetErrorString(e_));                          \
    } while (0)

namespace {

struct StageScope {       // brackets a stage with events when profiling is on
    muser_imager* h; cudaStream_t s; StageEvent ev; bool on;
    StageScope(muser_imager* h_, int stage, cudaStream_t s_) : h(h_), s(s_), on(h_->profiling) {
        if (!on) return;
        if (!h->ev_free.empty()) { ev = h->ev_free.back(); h->ev_free.pop_back(); }
        else { cudaEventCreate(&ev.a); cudaEventCreate(&ev.b); }
        ev.stage = stage;
        cudaEventRecord(ev.a, s);
    }
    ~StageScope() {
        if (!on) return;
        cudaEventRecord(ev.b, s);
        h->ev_used.push_back(ev);
    }
};

size_t grid_cells(const muser_imager* h) { return (size_t)h->ngrids * h->ny * h->nx; }
bool wmode(const muser_imager* h) { return h->nplanes > 0; }

void free_grids(muser_imager* h) {
    cudaFree(h->G); cudaFree(h->Gw); cudaFree(h->H); cudaFree(h->out_dirty); cudaFree(h->out_psf); cudaFree(h->cnt);
    cudaFree(h->peaks_d); cudaFree(h->ow_valid); h->ow_valid = nullptr;
    h->tmap_tried = h->tmap_ok = false;
    h->G = nullptr; h->Gw = nullptr; h->H = nullptr; h->out_dirty = h->out_psf = nullptr; h->cnt = nullptr; h->peaks_d = nullptr;
    if (h->plan_ok) { cufftDestroy(h->plan); h->plan_ok = false; }
    if (h->plan_rows_ok) { cufftDestroy(h->plan_rows); h->plan_rows_ok = false; }
}

void free_bins(muser_imager* h) {
    cudaFree(h->bin_count); cudaFree(h->bin_offset); cudaFree(h->items); cudaFree(h->bin_tops);
    h->bin_count = h->bin_offset = h->bin_tops = nullptr; h->items = nullptr; h->bins_cap = h->items_cap = 0;
    cudaFree(h->ow_count); cudaFree(h->ow_cursor); cudaFree(h->ow_offset); cudaFree(h->ow_work); cudaFree(h->ow_tops);
    cudaFree(h->ow_cta_hist);
    h->ow_count = h->ow_cursor = h->ow_offset = h->ow_tops = nullptr; h->ow_work = nullptr; h->ow_bins_cap = 0;
    h->ow_cta_hist = nullptr; h->ow_cta_hist_cap = 0;
}

int rebuild_geom(muser_imager* h) {
    Geom& g = h->geom;
    g.nx = h->nx; g.ny = h->ny; g.Q = h->Q; g.ngrids = h->ngrids;
    g.nplanes = wmode(h) ? h->nplanes : 1;
    g.wmode = wmode(h) ? 1 : 0;
    const double cell = h->cell_arcsec * kArcsec;       // same operation order as DESIGN.md O1
    g.su = (double)h->nx * cell;
    g.sv = (double)h->ny * cell;
    g.ntx = (h->nx - 1 + kTile / 2) / kTile + 1;
    g.nty = (h->ny - 1 + kTile / 2) / kTile + 1;
    const unsigned long long nb = (unsigned long long)h->ngrids * g.nplanes * g.nty * g.ntx;
    if (nb >= 0x7FFFFFFFull) return fail(h, MUSER_EUNSUPPORTED, "too many (grid, plane, tile) bins");
    g.nbins = (uint32_t)nb;
    g.chunk = 512;
    g.S = h->planes_h.empty() ? h->S : h->planes_h[0].support;
    g.ntiles = g.nty * g.ntx;
    g.otx = (h->nx - 1 + kOwTileW / 2) / kOwTileW + 1;
    g.oty = (h->ny / 2 + kTile - 1) / kTile;
    g.ontiles = g.oty * g.otx;
    g.onbins = (uint32_t)h->ngrids * (uint32_t)g.ontiles;
    g.phase_on = (h->off_l != 0.0 || h->off_m != 0.0) ? 1 : 0;
    g.dl = h->off_l; g.dm = h->off_m;
    g.uniform = h->weighting == MUSER_WEIGHT_UNIFORM ? 1 : 0;
    g.wtile = 0;
    return MUSER_OK;
}

// (re)allocate and zero the grids for the current nx, ny, ngrids, mode.  Called from the set_* calls only, which may
// synchronise: the memsets run on the legacy stream and the device is synchronised before returning, so that work the
// caller later enqueues on ANY stream (non-blocking ones included) sees the zeros.
int alloc_grids(muser_imager* h) {
    free_grids(h);
    free_bins(h);
    const size_t nc = grid_cells(h);
    CU(h, cudaMalloc(&h->G, nc * sizeof(float2)));
    CU(h, cudaMalloc(&h->Gw, nc * (wmode(h) ? sizeof(float2) : sizeof(float))));
    CU(h, cudaMalloc(&h->H, nc * sizeof(float2)));
    CU(h, cudaMemset(h->G, 0, nc * sizeof(float2)));
    CU(h, cudaMemset(h->Gw, 0, nc * (wmode(h) ? sizeof(float2) : sizeof(float))));
    CU(h, cudaMemset(h->stats_d, 0, sizeof(Stats)));
    if (h->weighting == MUSER_WEIGHT_UNIFORM) {
        CU(h, cudaMalloc(&h->cnt, nc * sizeof(int)));
        CU(h, cudaMemset(h->cnt, 0, nc * sizeof(int)));
    }
    {
        const size_t nb = ((size_t)h->geom.onbins + 8) & ~(size_t)3;
        CU(h, cudaMalloc(&h->ow_valid, nb * sizeof(uint32_t)));
        CU(h, cudaMemset(h->ow_valid, 0xFF, nb * sizeof(uint32_t)));  // the grids are zeroed and dense
    }
    h->sparse = false;
    CU(h, cudaMalloc(&h->peaks_d, (size_t)h->ngrids * sizeof(PeakSlot)));
    CU(h, cudaMemset(h->peaks_d, 0, (size_t)h->ngrids * sizeof(PeakSlot)));
    h->peaks_valid = false;
    CU(h, cudaDeviceSynchronize());
    h->fft_valid = false;
    h->zero_pending = false;
    h->lower_valid = true;
    return MUSER_OK;
}

GridPtrs grid_ptrs(const muser_imager* h) { return GridPtrs{h->G, h->Gw, h->cnt}; }

// the lazily deferred part of muser_reset: zero the grids now (every consumer but the owner-tile gridder needs it)
int flush_zero(muser_imager* h, cudaStream_t s) {
    if (h->zero_pending) {
        const size_t nc = grid_cells(h);
        CU(h, cudaMemsetAsync(h->G, 0, nc * sizeof(float2), s));
        CU(h, cudaMemsetAsync(h->Gw, 0, nc * (wmode(h) ? sizeof(float2) : sizeof(float)), s));
        CU(h, cudaMemsetAsync(h->ow_valid, 0xFF, (((size_t)h->geom.onbins + 8) & ~(size_t)3) * sizeof(uint32_t), s));
        h->zero_pending = false;
        h->sparse = false;
        h->lower_valid = true;
        return MUSER_OK;
    }
    if (h->sparse) {
        // the owner gridder left the tiles it did not write untouched (flag 0 = zeros): make the stored half-plane dense
        CU(h, launch_owner_fill_invalid(h->geom, grid_ptrs(h), h->ow_valid, s));
        h->n_launches += 1;
        h->sparse = false;
    }
    return MUSER_OK;
}


// rebuild rows 0 .. ny/2-1 of the grids from the stored half-plane (consumers of the full grids call this first)
int ensure_lower(muser_imager* h, cudaStream_t s) {
    if (h->lower_valid) return MUSER_OK;
    CU(h, launch_mirror_lower(h->geom, grid_ptrs(h), s));
    h->n_launches += 1;
    h->lower_valid = true;
    return MUSER_OK;
}

bool owner_capable(const muser_imager* h) { return !wmode(h) && h->ttp_d != nullptr; }

// upload tables (transposed TT[r][j] = T[j*Q + r]) + plane metadata + correctors from fp64 host tables
int upload_tables(muser_imager* h, const std::vector<std::vector<double>>& t64, const std::vector<int>& supports,
                  const std::vector<double>& wc) {
    const int P = (int)t64.size(), Q = h->Q;
    const bool wm = wmode(h);
    h->planes_h.assign(P, PlaneMeta{});
    h->tables_f32.assign(P, {});
    std::vector<float> dev;
    for (int p = 0; p < P; ++p) {
        const int S = supports[p], pitch = (S + 4) & ~3, comp = wm ? 2 : 1;
        PlaneMeta& pm = h->planes_h[p];
        pm.support = S; pm.pitch = pitch; pm.offset = (int)(dev.size() / comp); pm.wc = wc[p];
        {   // bound on |kx ky| = (max |T|)^2, at least 1 (library tables peak at 1; caller-supplied ones may not)
            double m2 = 1.0;
            for (size_t i = 0; i < (size_t)S * Q + 1; ++i) {
                const double v2 = wm ? t64[p][2 * i] * t64[p][2 * i] + t64[p][2 * i + 1] * t64[p][2 * i + 1] : t64[p][i] * t64[p][i];
                m2 = std::max(m2, v2);
            }
            const float kb = (float)(m2 * 1.0001);
            std::memcpy(&pm.pad, &kb, sizeof(float));
        }
        const size_t L = (size_t)S * Q + 1;
        h->tables_f32[p].resize(L * comp);
        for (size_t i = 0; i < L * comp; ++i) h->tables_f32[p][i] = (float)t64[p][i];
        const size_t base = dev.size();
        dev.resize(base + (size_t)(Q + 1) * pitch * comp, 0.f);
        for (int r = 0; r <= Q; ++r)
            for (int j = 0; j < S; ++j)
                for (int c = 0; c < comp; ++c)
                    dev[base + ((size_t)r * pitch + j) * comp + c] = h->tables_f32[p][((size_t)j * Q + r) * comp + c];
    }
    // a ladder of centres wc[p] = p * wc[1] (to rounding), strictly increasing: K1 searches three planes instead of all
    h->wstep = 0.0;
    if (wm && P >= 2 && wc[0] == 0.0 && wc[1] > 0.0) {
        bool ladder = true;
        for (int p = 1; p < P; ++p)
            ladder = ladder && wc[p] > wc[p - 1] && std::fabs(wc[p] - (double)p * wc[1]) <= 1e-9 * wc[1];
        if (ladder) h->wstep = wc[1];
    }
    cudaFree(h->tables_d); cudaFree(h->planes_d);
    h->tables_d = nullptr; h->planes_d = nullptr;
    CU(h, cudaMalloc(&h->tables_d, dev.size() * sizeof(float)));
    CU(h, cudaMemcpy(h->tables_d, dev.data(), dev.size() * sizeof(float), cudaMemcpyHostToDevice));
    CU(h, cudaMalloc(&h->planes_d, P * sizeof(PlaneMeta)));
    CU(h, cudaMemcpy(h->planes_d, h->planes_h.data(), P * sizeof(PlaneMeta), cudaMemcpyHostToDevice));
    // owner-tile path: two-parity transposed table TT2[(par*(Q+1) + r)*8 + par + j] = T[j*Q + r], other entries 0
    cudaFree(h->ttp_d); h->ttp_d = nullptr;
    if (!wm && P == 1 && supports[0] == 7) {
        std::vector<float> ttp((size_t)2 * (Q + 1) * 8, 0.f);
        for (int par = 0; par < 2; ++par)
            for (int r = 0; r <= Q; ++r)
                for (int j = 0; j < 7; ++j)
                    ttp[((size_t)par * (Q + 1) + r) * 8 + par + j] = h->tables_f32[0][(size_t)j * Q + r];
        CU(h, cudaMalloc(&h->ttp_d, ttp.size() * sizeof(float)));
        CU(h, cudaMemcpy(h->ttp_d, ttp.data(), ttp.size() * sizeof(float), cudaMemcpyHostToDevice));
    }
    // correctors from plane 0 (real part), fp64 -> reciprocal -> fp32
    std::vector<double> t0((size_t)supports[0] * Q + 1);
    for (size_t i = 0; i < t0.size(); ++i) t0[i] = wm ? t64[0][2 * i] : t64[0][i];
    const std::vector<double> cx = muser_host::corrector(t0.data(), supports[0], Q, h->nx);
    const std::vector<double> cy = muser_host::corrector(t0.data(), supports[0], Q, h->ny);
    std::vector<float> icx(h->nx), icy(h->ny), ones(std::max(h->nx, h->ny), 1.0f);
    for (int x = 0; x < h->nx; ++x) icx[x] = (float)(1.0 / cx[x]);
    for (int y = 0; y < h->ny; ++y) icy[y] = (float)(1.0 / cy[y]);
    if (!h->icx_d) {
        CU(h, cudaMalloc(&h->icx_d, h->nx * sizeof(float)));
        CU(h, cudaMalloc(&h->icy_d, h->ny * sizeof(float)));
        CU(h, cudaMalloc(&h->ones_d, ones.size() * sizeof(float)));
        CU(h, cudaMemcpy(h->ones_d, ones.data(), ones.size() * sizeof(float), cudaMemcpyHostToDevice));
    }
    CU(h, cudaMemcpy(h->icx_d, icx.data(), h->nx * sizeof(float), cudaMemcpyHostToDevice));
    CU(h, cudaMemcpy(h->icy_d, icy.data(), h->ny * sizeof(float), cudaMemcpyHostToDevice));
    return MUSER_OK;
}

int build_2d_tables(muser_imager* h) {
    std::vector<std::vector<double>> t64(1);
    t64[0] = h->kind == MUSER_KERNEL_GAUSS ? muser_host::table_gauss(h->S, h->Q, h->gauss_a)
                                           : muser_host::table_pswf(h->S, h->Q);
    return upload_tables(h, t64, {h->S}, {0.0});
}

int ensure_scratch(muser_imager* h, long long nvis, cudaStream_t s) {
    const size_t ns = (size_t)2 * (size_t)nvis;
    if (ns > h->sample_cap) {
        cudaFree(h->staged); cudaFree(h->sorted);
        h->staged = nullptr; h->sorted = nullptr; h->sample_cap = 0;
        const size_t cap = ns + ns / 8 + 1024;
        CU(h, cudaMalloc(&h->staged, cap * sizeof(Staged)));
        CU(h, cudaMalloc(&h->sorted, cap * sizeof(Sample)));
        h->sample_cap = cap;
    }
    const size_t nb = h->geom.nbins;
    if (nb + 1 > h->bins_cap) {
        cudaFree(h->bin_count); cudaFree(h->bin_offset); cudaFree(h->bin_tops);
        h->bin_count = h->bin_offset = h->bin_tops = nullptr; h->bins_cap = 0;
        CU(h, cudaMalloc(&h->bin_tops, (nb / 4096 + 2) * 2 * sizeof(uint32_t)));
        CU(h, cudaMalloc(&h->bin_count, (nb + 1) * sizeof(uint32_t)));
        CU(h, cudaMalloc(&h->bin_offset, (nb + 1) * sizeof(uint32_t)));
        // K2 re-zeroes the histogram after every use; this first zeroing is ordered on the caller's stream
        CU(h, cudaMemsetAsync(h->bin_count, 0, (nb + 1) * sizeof(uint32_t), s));
        h->bins_cap = nb + 1;
    }
    const size_t ni = std::min(nb, h->sample_cap) + h->sample_cap / (size_t)h->geom.chunk + 2;
    if (ni > h->items_cap) {
        cudaFree(h->items); h->items = nullptr; h->items_cap = 0;
        CU(h, cudaMalloc(&h->items, ni * sizeof(Item)));
        h->items_cap = ni;
    }
    return MUSER_OK;
}

bool wplane_capable(const muser_imager* h) {     // w mode, or 2-D mode (one plane, real table); every support <= 31
    return !h->planes_h.empty() && wgrid_supported(h->planes_h.data(), (int)h->planes_h.size(), h->Q, h->max_smem);
}

int pick_strategy(const muser_imager* h) {
    if (h->strategy != MUSER_STRATEGY_AUTO) return h->strategy;
    if (owner_capable(h)) return MUSER_STRATEGY_OWNER;
    return wplane_capable(h) ? MUSER_STRATEGY_WPLANE : MUSER_STRATEGY_TILED;
}

uint32_t owner_item_size(long long nvis, int num_sms, int item_override) {
    // Heavy tiles are split into chunks of item_size samples.  4096 (the gridder sorts a chunk in units of kOwUnit = 4096
    // records; a larger chunk -- MUSER_TUNE_ITEM_SIZE up to 2^20, or the growth rule below -- is several units) when the call has
    // enough work to fill the machine; down to 256 for a single small frame, whose latency is the critical path of
    // one chunk (a third of a MUSER frame sits in the tile around the uv origin; the partial tiles are summed in two
    // levels, so 147 chunks cost less than 37 did: measured 76 us per frame at 256 against 88 at 1024).  For huge inputs
    // the chunk grows so that the partial-tile scratch (at most 16*nvis/item_size + 2 tiles) stays under 256 MB.
    if (item_override > 0) return (uint32_t)item_override;
    uint32_t item = 4096;
    const double units = 2.4 * (double)nvis / 4096.0;                // ~2.4 records per visibility on MUSER frames
    while (item > 256 && units * (4096.0 / item) < 4.0 * num_sms) item /= 2;
    while ((16.0 * (double)nvis / item + 2.0) * kOwTileFloats * sizeof(float) > 256.0 * 1048576.0) item *= 2;
    return item;
}

int ensure_owner_scratch(muser_imager* h, long long nvis, uint32_t item_size, uint32_t* max_items_out, cudaStream_t s) {
    const size_t nrec = (size_t)8 * (size_t)nvis;                    // <= 2 samples x 4 tiles per visibility
    if (nrec > h->ow_sorted_cap) {
        cudaFree(h->ow_sorted); cudaFree(h->ow_loc); h->ow_sorted = h->ow_loc = nullptr; h->ow_sorted_cap = 0;
        const size_t cap = nrec + nrec / 8 + 1024;
        CU(h, cudaMalloc(&h->ow_sorted, cap * sizeof(uint4)));
        CU(h, cudaMalloc(&h->ow_loc, (cap / 8 + 1) * sizeof(uint4)));
        h->ow_sorted_cap = cap;
    }
    const size_t nb = ((size_t)h->geom.onbins + 8) & ~(size_t)3;
    if (nb > h->ow_bins_cap) {
        cudaFree(h->ow_count); cudaFree(h->ow_cursor); cudaFree(h->ow_offset); cudaFree(h->ow_work); cudaFree(h->ow_tops);
        h->ow_count = h->ow_cursor = h->ow_offset = h->ow_tops = nullptr; h->ow_work = nullptr; h->ow_bins_cap = 0;
        CU(h, cudaMalloc(&h->ow_count, nb * sizeof(uint32_t)));
        CU(h, cudaMalloc(&h->ow_cursor, nb * sizeof(uint32_t)));
        CU(h, cudaMalloc(&h->ow_offset, nb * sizeof(uint32_t)));
        CU(h, cudaMalloc(&h->ow_work, nb * sizeof(uint4)));
        CU(h, cudaMalloc(&h->ow_tops, (nb / 4096 + 3) * 4 * sizeof(uint32_t)));
        CU(h, cudaMemsetAsync(h->ow_tops, 0, (nb / 4096 + 3) * 4 * sizeof(uint32_t), s));   // flags of the chained scan: zero when idle
        if (!h->ow_ctl) CU(h, cudaMalloc(&h->ow_ctl, 4 * sizeof(uint32_t)));
        CU(h, cudaMemsetAsync(h->ow_count, 0, nb * sizeof(uint32_t), s));   // ordered on the caller's stream; every later use leaves it zeroed
        h->ow_bins_cap = nb;
    }
    const size_t ni = (size_t)(16.0 * (double)nvis / item_size) + 2;
    if (ni > h->ow_items_cap) {
        cudaFree(h->ow_items); cudaFree(h->ow_tickets); cudaFree(h->ow_scratch);
        h->ow_items = nullptr; h->ow_tickets = nullptr; h->ow_scratch = nullptr; h->ow_items_cap = 0;
        const size_t cap = ni + ni / 4 + 16;
        CU(h, cudaMalloc(&h->ow_items, cap * sizeof(OwItem)));
        CU(h, cudaMalloc(&h->ow_tickets, cap * sizeof(uint32_t)));
        CU(h, cudaMemsetAsync(h->ow_tickets, 0, cap * sizeof(uint32_t), s));   // the last chunk of a tile re-zeroes its ticket
        CU(h, cudaMalloc(&h->ow_scratch, cap * kOwTileFloats * sizeof(float)));
        h->ow_items_cap = cap;
    }
    *max_items_out = (uint32_t)ni;
    return MUSER_OK;
}

// TILED and WPLANE strategies: generic binning (K1-K3) + their gridders.  n = visibilities (flat call) or elements
// (channelised call, rows != nullptr: the polarisations of an element are summed by K1).
int grid_generic(muser_imager* h, int strat, const float* uvw, const double* freq, const void* vis, const float* wt,
                 const int* gid, long long nvis, const RowsShapeG* rows, cudaStream_t s) {
    const Geom& g = h->geom;
    GridPtrs gp = grid_ptrs(h);
    if (strat != MUSER_STRATEGY_TILED && strat != MUSER_STRATEGY_WPLANE) return fail(h, MUSER_EUNSUPPORTED, "unknown gridding strategy");
    if (strat == MUSER_STRATEGY_WPLANE && !wplane_capable(h))
        return fail(h, MUSER_EUNSUPPORTED, "the window strategy needs every support <= 31 (and a table that fits shared memory)");
    int rc = ensure_scratch(h, nvis, s);
    if (rc) return rc;
    if ((rc = flush_zero(h, s))) return rc;
    h->last_stream = s;
    h->fft_valid = false;
    h->lower_valid = false;                                           // like the owner path, it grids rows >= ny/2 only
    if (strat == MUSER_STRATEGY_WPLANE) {
        // bins ordered (grid, tile, plane); work items = <= 4096 consecutive records of one tile
        Geom gw = g;
        gw.wtile = 1;
        if (!h->wg_ctl) CU(h, cudaMalloc(&h->wg_ctl, 16 * sizeof(uint32_t)));
        const size_t list_cap = wgrid_list_cap(gw, h->sample_cap);
        if (list_cap > h->wg_list_cap) {
            cudaFree(h->wg_lists); h->wg_lists = nullptr; h->wg_list_cap = 0;
            CU(h, cudaMalloc(&h->wg_lists, 8 * list_cap * sizeof(uint32_t)));
            h->wg_list_cap = list_cap;
        }
        {
            StageScope sc(h, MUSER_STAGE_BIN, s);
            CU(h, launch_coords(gw, uvw, freq, (const float2*)vis, wt, gid, nvis, rows, h->wstep, h->planes_d, h->staged, h->bin_count,
                                h->stats_d, h->cnt, s));
            CU(h, launch_scan_items(gw, h->bin_count, h->bin_offset, nullptr, nullptr, h->bin_tops, s));
            CU(h, launch_wtile_items(gw, h->bin_offset, h->planes_d, h->items, h->wg_lists, (uint32_t)h->wg_list_cap, h->nitems_d, h->wg_ctl, s));
            CU(h, launch_scatter(gw, h->staged, 2 * nvis, h->bin_offset, h->sorted, s));
            h->n_launches += g.nbins <= 4096u ? 4 : 6;
        }
        StageScope sc(h, MUSER_STAGE_GRID, s);
        cudaError_t ce = cudaSuccess;
        if (!h->wg_streams_ok) {
            for (int i = 0; i < 7; ++i) CU(h, cudaStreamCreateWithFlags(&h->wg_side[i], cudaStreamNonBlocking));
            for (int i = 0; i < 8; ++i) CU(h, cudaEventCreateWithFlags(&h->wg_ev[i], cudaEventDisableTiming));
            h->wg_streams_ok = true;
        }
        h->n_launches += launch_wgrid(gw, h->sorted, h->items, h->wg_lists, (uint32_t)h->wg_list_cap, h->wg_ctl, h->bin_offset, h->planes_d,
                                      h->planes_h.data(), h->tables_d, gp, h->num_sms, s, h->wg_side, h->wg_ev, &ce);
        CU(h, ce);
        return MUSER_OK;
    }
    {
        StageScope sc(h, MUSER_STAGE_BIN, s);
        CU(h, launch_coords(g, uvw, freq, (const float2*)vis, wt, gid, nvis, rows, h->wstep, h->planes_d, h->staged, h->bin_count,
                            h->stats_d, h->cnt, s));
        CU(h, launch_scan_items(g, h->bin_count, h->bin_offset, h->items, h->nitems_d, h->bin_tops, s));
        CU(h, launch_scatter(g, h->staged, 2 * nvis, h->bin_offset, h->sorted, s));
        h->n_launches += g.nbins <= 4096u ? 3 : 5;
    }
    {
        StageScope sc(h, MUSER_STAGE_GRID, s);
        CU(h, launch_grid_tiled(g, h->sorted, h->items, h->nitems_d, h->planes_d, h->planes_h.data(), h->tables_d,
                                gp, h->num_sms, s));
        h->n_launches += 1;
    }
    return MUSER_OK;
}

int grid_impl(muser_imager* h, const float* uvw, const double* freq, const void* vis, const float* wt,
              const int* gid, long long nvis, cudaStream_t s) {
    if (nvis < 0 || nvis > (1LL << 30)) return fail(h, MUSER_EINVAL, "nvis out of range [0, 2^30]");
    if (nvis == 0) return MUSER_OK;
    if (!uvw || !freq || !wt || (!vis && !h->weights_only)) return fail(h, MUSER_EINVAL, "null input pointer");
    int strat = pick_strategy(h);
    const Geom& g = h->geom;
    GridPtrs gp = grid_ptrs(h);
    if (strat == MUSER_STRATEGY_WPLANE && (unsigned long long)h->ngrids * g.ntiles + (unsigned long long)nvis / 2048 + 2 >= (1ull << 24)) {
        // its work lists hold 24-bit item indices
        if (h->strategy != MUSER_STRATEGY_AUTO) return fail(h, MUSER_EUNSUPPORTED, "too many tiles for the w-plane window strategy");
        strat = MUSER_STRATEGY_TILED;
    }
    if (strat == MUSER_STRATEGY_OWNER) {
        if (!owner_capable(h)) return fail(h, MUSER_EUNSUPPORTED, "the owner-tile strategy needs 2-D mode and support 7");
        const uint32_t item_size = owner_item_size(nvis, h->num_sms, h->tune[MUSER_TUNE_ITEM_SIZE]);
        uint32_t max_items = 0;
        int rc = ensure_owner_scratch(h, nvis, item_size, &max_items, s);
        if (rc) return rc;
        const int iters = owner_bin_iters(nvis, h->tune[MUSER_TUNE_BIN_ITERS]);
        {
            const size_t need = owner_bin_ctas(nvis, iters) * (size_t)g.ontiles;
            if (need > h->ow_cta_hist_cap) {
                cudaFree(h->ow_cta_hist); h->ow_cta_hist = nullptr; h->ow_cta_hist_cap = 0;
                CU(h, cudaMalloc(&h->ow_cta_hist, (need + need / 4) * sizeof(uint32_t)));
                h->ow_cta_hist_cap = need + need / 4;
            }
        }
        if (g.oty > 65535 || g.otx > 1024 + 8) return fail(h, MUSER_EUNSUPPORTED, "too many tiles per axis");
        h->last_stream = s;
        h->fft_valid = false;
        {
            StageScope sc(h, MUSER_STAGE_BIN, s);
            CU(h, launch_owner_count(g, uvw, freq, (const float2*)vis, wt, gid, nvis, h->ow_count, h->ow_cta_hist, h->stats_d,
                                     h->ow_loc, iters, s));
            CU(h, launch_owner_scan(g, h->ow_count, h->ow_cursor, h->ow_offset, h->ow_items, h->nitems_d, item_size,
                                    h->ow_work, h->ow_ctl, h->ow_tops, h->zero_pending ? h->ow_valid : nullptr, s));
            CU(h, launch_owner_scatter(g, h->ow_loc, uvw, freq, (const float2*)vis, wt, gid, nvis, h->ow_offset, h->ow_cta_hist,
                                       h->ow_cursor, h->ow_sorted, h->cnt, iters, s));
        }
        {
            StageScope sc(h, MUSER_STAGE_GRID, s);
            CU(h, launch_owner_grid(g, h->ow_sorted, h->ow_offset, h->ow_items, h->nitems_d, h->ow_work,
                                    h->ow_ctl, h->ttp_d, gp, h->ow_scratch, h->ow_tickets, h->ow_valid, h->zero_pending ? 1 : 0, h->num_sms, s));
        }
        h->n_launches += g.onbins <= 4096u * 1024u ? 4 : 6;           // count, scan (1 launch up to 4 M bins, else 3), scatter, grid
        if (h->zero_pending) h->sparse = true;                        // first call after a reset: the tiles it did not write keep flag 0
        h->zero_pending = false;
        h->lower_valid = false;                                       // rows < ny/2 are rebuilt on demand (ensure_lower)
        return MUSER_OK;
    }
    return grid_generic(h, strat, uvw, freq, vis, wt, gid, nvis, nullptr, s);
}

// NEXT-1: the channelised call.  Every strategy: the owner-tile path has its own rows binning kernels (k_rows_count /
// k_rows_scatter); TILED and WPLANE go through grid_generic with k_coords<ROWS>.
int grid_rows_impl(muser_imager* h, const float* uvw, const double* freq, const void* vis, const float* wt, const int* gid,
                   long long nrow, int nchan, int npol, int ntime, int pol_mode, cudaStream_t s) {
    if (nrow < 0 || nchan < 1 || npol < 1 || ntime < 1 || nchan > rows_max_channels() || npol > 8)
        return fail(h, MUSER_EINVAL, "rows call: need nrow >= 0, 1 <= nchan <= 65535, 1 <= npol <= 8, ntime >= 1");
    if ((long long)ntime * npol * nchan > 32768LL * 65535LL) return fail(h, MUSER_EINVAL, "rows call: too many (time, pol, channel) blocks");
    if (pol_mode != MUSER_POLS_SUM && pol_mode != MUSER_POLS_SPLIT) return fail(h, MUSER_EINVAL, "unknown pol_mode");
    const long long nvis = nrow * nchan * npol * ntime;
    if (nrow > (1LL << 30) || nvis > (1LL << 30)) return fail(h, MUSER_EINVAL, "too many visibilities in one call (2^30)");
    if (nvis == 0) return MUSER_OK;
    if (!uvw || !freq || !wt || (!vis && !h->weights_only)) return fail(h, MUSER_EINVAL, "null input pointer");
    const Geom& g = h->geom;
    const int split = pol_mode == MUSER_POLS_SPLIT ? 1 : 0;
    const long long nelem = split ? nvis : nvis / npol;
    int strat = pick_strategy(h);
    if (strat == MUSER_STRATEGY_OWNER && !owner_capable(h))
        return fail(h, MUSER_EUNSUPPORTED, "the owner-tile strategy needs 2-D mode and support 7");
    if (strat != MUSER_STRATEGY_OWNER) {
        // w planes / other supports: the generic binning kernel has the channelised variant, the rest of the path is the flat one
        if (strat == MUSER_STRATEGY_WPLANE && (unsigned long long)h->ngrids * g.ntiles + (unsigned long long)nelem / 2048 + 2 >= (1ull << 24)) {
            if (h->strategy != MUSER_STRATEGY_AUTO) return fail(h, MUSER_EUNSUPPORTED, "too many tiles for the w-plane window strategy");
            strat = MUSER_STRATEGY_TILED;
        }
        const RowsShapeG sh = {ntime, split ? npol : 1, split ? 1 : npol, nchan, (int)nrow};
        return grid_generic(h, strat, uvw, freq, vis, wt, gid, nelem, &sh, s);
    }
    const uint32_t item_size = owner_item_size(nelem, h->num_sms, h->tune[MUSER_TUNE_ITEM_SIZE]);
    uint32_t max_items = 0;
    int rc = ensure_owner_scratch(h, nelem, item_size, &max_items, s);
    if (rc) return rc;
    if (g.oty > 65535 || g.otx > 1024 + 8) return fail(h, MUSER_EUNSUPPORTED, "too many tiles per axis");
    const int cpc = rows_cpc(ntime, split ? npol : 1, nchan, (int)nrow);
    {
        const size_t need = rows_ctas(ntime, npol, nchan, (int)nrow, split, cpc) * (size_t)g.ontiles;
        if (need > h->ow_cta_hist_cap) {
            cudaFree(h->ow_cta_hist); h->ow_cta_hist = nullptr; h->ow_cta_hist_cap = 0;
            CU(h, cudaMalloc(&h->ow_cta_hist, (need + need / 4) * sizeof(uint32_t)));
            h->ow_cta_hist_cap = need + need / 4;
        }
    }
    h->last_stream = s;
    h->fft_valid = false;
    {
        StageScope sc(h, MUSER_STAGE_BIN, s);
        CU(h, launch_rows_count(g, ntime, npol, nchan, (int)nrow, split, cpc, uvw, freq, (const float2*)vis, wt, gid, h->ow_count,
                                h->ow_cta_hist, h->stats_d, h->ow_loc, s));
        CU(h, launch_owner_scan(g, h->ow_count, h->ow_cursor, h->ow_offset, h->ow_items, h->nitems_d, item_size, h->ow_work,
                                h->ow_ctl, h->ow_tops, h->zero_pending ? h->ow_valid : nullptr, s));
        CU(h, launch_rows_scatter(g, ntime, npol, nchan, (int)nrow, split, cpc, h->ow_loc, uvw, freq, (const float2*)vis, wt, gid,
                                  h->ow_offset, h->ow_cta_hist, h->ow_cursor, h->ow_sorted, h->cnt, s));
    }
    {
        StageScope sc(h, MUSER_STAGE_GRID, s);
        CU(h, launch_owner_grid(g, h->ow_sorted, h->ow_offset, h->ow_items, h->nitems_d, h->ow_work, h->ow_ctl, h->ttp_d,
                                grid_ptrs(h), h->ow_scratch, h->ow_tickets, h->ow_valid, h->zero_pending ? 1 : 0, h->num_sms, s));
    }
    h->n_launches += g.onbins <= 4096u * 1024u ? 4 : 6;
    if (h->zero_pending) h->sparse = true;
    h->zero_pending = false;
    h->lower_valid = false;
    return MUSER_OK;
}

// tensor map of H for the TMA-staged column pass (MUSER_TUNE_COLS_TMA: 0 = default, 1 = per-lane loads, 2 = TMA)
const void* cols_tmap(muser_imager* h) {
    const int mode = h->tune[MUSER_TUNE_COLS_TMA];
    if (mode == 1 || (mode == 0 && !kColsTmaDefault)) return nullptr;
    if (!h->tmap_tried) {
        h->tmap_tried = true;
        h->tmap_ok = fft_cols_make_tmap(h->tmap, h->H, h->nx, h->ny, h->ngrids);
    }
    return h->tmap_ok ? h->tmap : nullptr;
}

// Grids per rows -> columns sub-batch of the fused transform: MUSER_TUNE_FFT_SUBBATCH, or (0, the default) every grid in
// one batch.  Measured on cfg 3 (80 x 1024^2) and on 1024 x 512^2 (round 3): the partial waves of the smaller
// launches cost more than the L2 hits of the column pass save at every sub-batch size, so the knob stays off.
int fft_subbatch(const muser_imager* h) {
    const int t = h->tune[MUSER_TUNE_FFT_SUBBATCH];
    return t > 0 ? std::min(t, h->ngrids) : h->ngrids;
}

int image_impl(muser_imager* h, float* dirty, float* psf, cudaStream_t s) {
    if (!dirty && !psf) return MUSER_OK;
    h->last_stream = s;
    // the half-plane row pass takes the owner gridder's tile flags (unwritten tiles are not loaded); every other path wants
    // dense grids
    const bool rows_take_flags = h->fused_fft && h->fused_rows && !h->zero_pending && h->geom.otx <= 96;
    if (!rows_take_flags) {
        int rcz = flush_zero(h, s);
        if (rcz) return rcz;
    }
    if (h->fused_fft && h->fused_rows) {
        // A5 rows by k_fft_rows_half straight from the stored half-planes of G and Gw (H = G + i alpha Gw is never
        // materialised and rows < ny/2 are never read), A5 columns + A6 by the fused column kernel; H keeps the row
        // transform, so muser_dirty followed by muser_psf repeats only the column pass
        const float* cx = h->correction ? h->icx_d : h->ones_d;
        const float* cy = h->correction ? h->icy_d : h->ones_d;
        PeakSlot* peaks = (h->peak_search && dirty) ? h->peaks_d : nullptr;
        if (peaks) { CU(h, cudaMemsetAsync(peaks, 0, (size_t)h->ngrids * sizeof(PeakSlot), s)); h->peaks_valid = true; }
        // The row transform H of one grid (8 B per cell) is written by the row pass and read once by the column pass.  Running
        // rows -> columns over sub-batches of a few grids would keep that round trip inside the 126 MB L2 instead of DRAM
        // (MUSER_TUNE_FFT_SUBBATCH); measured slower than one batch at every size, so the default is one batch.
        const int sub = fft_subbatch(h);
        const void* tmap = cols_tmap(h);
        const bool need_rows = !h->fft_valid;
        for (int g0 = 0; g0 < h->ngrids; g0 += sub) {
            const int gc = std::min(sub, h->ngrids - g0);
            if (need_rows) {
                StageScope sc(h, MUSER_STAGE_FFT, s);
                CU(h, launch_fft_rows_half(h->geom, h->G, h->Gw, h->cnt, h->tw_rows_d, h->stats_d, h->H, h->sparse ? h->ow_valid : nullptr,
                                           g0, gc, h->num_sms, s));
                h->n_launches += 1;
            }
            StageScope sc(h, MUSER_STAGE_CORRECT, s);
            CU(h, launch_fft_cols_correct(h->geom, h->H, h->tw_d, h->tw8_d, cx, cy, h->stats_d, dirty, psf, peaks, tmap, g0, gc, s));
            h->n_launches += 1;
        }
        h->fft_valid = true;
        return MUSER_OK;
    }
    if (h->fused_fft) {
        // nx not a power of two: rows by cuFFT (contiguous 1-D transforms of the packed full grid), then as above
        if (!h->plan_rows_ok) {
            int dims[1] = {h->nx};
            cufftResult r = cufftPlanMany(&h->plan_rows, 1, dims, nullptr, 1, h->nx, nullptr, 1, h->nx, CUFFT_C2C, h->ngrids * h->ny);
            if (r != CUFFT_SUCCESS) return fail(h, MUSER_ECUDA, "cufftPlanMany (rows) failed: " + std::to_string((int)r));
            h->plan_rows_ok = true;
        }
        if (!h->fft_valid) {
            {
                int rc = ensure_lower(h, s);
                if (rc) return rc;
                StageScope sc(h, MUSER_STAGE_PACK, s);
                CU(h, launch_pack(h->geom, grid_ptrs(h), h->H, h->stats_d, s));
                h->n_launches += 1;
            }
            StageScope sc(h, MUSER_STAGE_FFT, s);
            cufftResult r = cufftSetStream(h->plan_rows, s);
            if (r == CUFFT_SUCCESS) r = cufftExecC2C(h->plan_rows, (cufftComplex*)h->H, (cufftComplex*)h->H, CUFFT_INVERSE);
            if (r != CUFFT_SUCCESS) return fail(h, MUSER_ECUDA, "cufftExecC2C (rows) failed: " + std::to_string((int)r));
            h->fft_valid = true;
        }
        StageScope sc(h, MUSER_STAGE_CORRECT, s);
        const float* cx = h->correction ? h->icx_d : h->ones_d;
        const float* cy = h->correction ? h->icy_d : h->ones_d;
        PeakSlot* peaks = (h->peak_search && dirty) ? h->peaks_d : nullptr;
        if (peaks) { CU(h, cudaMemsetAsync(peaks, 0, (size_t)h->ngrids * sizeof(PeakSlot), s)); h->peaks_valid = true; }
        CU(h, launch_fft_cols_correct(h->geom, h->H, h->tw_d, h->tw8_d, cx, cy, h->stats_d, dirty, psf, peaks, cols_tmap(h), 0, h->ngrids, s));
        h->n_launches += 1;
        return MUSER_OK;
    }
    if (!h->plan_ok) {
        int dims[2] = {h->ny, h->nx};
        cufftResult r = cufftPlanMany(&h->plan, 2, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2C, h->ngrids);
        if (r != CUFFT_SUCCESS) return fail(h, MUSER_ECUDA, "cufftPlanMany failed: " + std::to_string((int)r));
        h->plan_ok = true;
    }
    if (!h->fft_valid) {
        {
            int rc = ensure_lower(h, s);
            if (rc) return rc;
            StageScope sc(h, MUSER_STAGE_PACK, s);
            CU(h, launch_pack(h->geom, grid_ptrs(h), h->H, h->stats_d, s));
            h->n_launches += 1;
        }
        {
            StageScope sc(h, MUSER_STAGE_FFT, s);
            cufftResult r = cufftSetStream(h->plan, s);
            if (r == CUFFT_SUCCESS) r = cufftExecC2C(h->plan, (cufftComplex*)h->H, (cufftComplex*)h->H, CUFFT_INVERSE);
            if (r != CUFFT_SUCCESS) return fail(h, MUSER_ECUDA, "cufftExecC2C failed: " + std::to_string((int)r));
        }
        h->fft_valid = true;
    }
    {
        StageScope sc(h, MUSER_STAGE_CORRECT, s);
        const float* cx = h->correction ? h->icx_d : h->ones_d;
        const float* cy = h->correction ? h->icy_d : h->ones_d;
        PeakSlot* peaks = (h->peak_search && dirty) ? h->peaks_d : nullptr;
        if (peaks) { CU(h, cudaMemsetAsync(peaks, 0, (size_t)h->ngrids * sizeof(PeakSlot), s)); h->peaks_valid = true; }
        CU(h, launch_correct(h->geom, h->H, cx, cy, h->stats_d, dirty, psf, peaks, s));
        h->n_launches += 1;
    }
    return MUSER_OK;
}

int reset_impl(muser_imager* h, cudaStream_t s) {
    h->last_stream = s;
    h->fft_valid = false;
    // The grids are zeroed lazily: the next owner-tile muser_grid clears the tile flags, stores the tiles it grids and leaves
    // the others alone (flag 0 = zeros; the row transform skips them), so a reset followed by muser_grid needs no memset and
    // no zero fill at all; any consumer of the dense grids calls flush_zero first.
    h->zero_pending = true;
    if (!(owner_capable(h) && pick_strategy(h) == MUSER_STRATEGY_OWNER)) {
        int rc = flush_zero(h, s);
        if (rc) return rc;
    }
    CU(h, cudaMemsetAsync(h->stats_d, 0, sizeof(Stats), s));
    if (h->cnt) CU(h, cudaMemsetAsync(h->cnt, 0, grid_cells(h) * sizeof(int), s));
    if (h->child2x) return reset_impl(h->child2x, s);
    return MUSER_OK;
}

// The set_* calls reset on the legacy stream; a caller's cudaStreamNonBlocking stream is not ordered after that stream, so
// they wait for the memsets here (they are set-up calls: every one of them synchronises the device at entry already).
int reset_sync(muser_imager* h) {
    int rc = reset_impl(h, nullptr);
    if (rc) return rc;
    CU(h, cudaDeviceSynchronize());
    return MUSER_OK;
}

}  // namespace

// =================================================================================================== ABI
extern "C" {

const char* muser_version(void) { return "muser-b200 0.1 (sm_100a)"; }

const char* muser_last_error(const muser_imager* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

muser_imager* muser_imager_create(int nx, int ny, double cell_arcsec, int support, int oversample) {
    g_create_error.clear();
    if (support < 1 || support > 63 || (support & 1) == 0) { fail(nullptr, MUSER_EINVAL, "support must be odd in [1,63]"); return nullptr; }
    if (oversample < 2 || oversample > 256 || (oversample & 1)) { fail(nullptr, MUSER_EINVAL, "oversample must be even in [2,256]"); return nullptr; }
    if (nx < 2 * (support + 1) || ny < 2 * (support + 1) || (nx & 3) || (ny & 3) || nx > 32768 || ny > 32768) {
        fail(nullptr, MUSER_EINVAL, "nx, ny must be multiples of 4 in [2*(support+1), 32768]"); return nullptr;
    }
    if (!(cell_arcsec > 0) || !std::isfinite(cell_arcsec)) { fail(nullptr, MUSER_EINVAL, "cell_arcsec must be > 0"); return nullptr; }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        fail(nullptr, MUSER_ECUDA, std::string("no CUDA device (there is no CPU fallback): ") + cudaGetErrorString(e));
        return nullptr;
    }
    muser_imager* h = new muser_imager();
    h->nx = nx; h->ny = ny; h->cell_arcsec = cell_arcsec; h->S = support; h->Q = oversample;
    cudaGetDevice(&h->device);
    cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, h->device);
    cudaDeviceGetAttribute(&h->max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
    int rc = rebuild_geom(h);
    auto bail = [&](const char* what) -> muser_imager* {
        g_create_error = std::string(what) + ": " + h->err;
        muser_imager_destroy(h);
        return nullptr;
    };
    if (rc) return bail("geometry");
    if (tiled_kernel_setup(h->max_smem) != cudaSuccess || owner_kernel_setup(h->max_smem) != cudaSuccess ||
        wgrid_kernel_setup(h->max_smem) != cudaSuccess) { h->err = cudaGetErrorString(cudaGetLastError()); return bail("kernel setup"); }
    if (cudaMalloc(&h->stats_d, sizeof(Stats)) != cudaSuccess || cudaMalloc(&h->nitems_d, sizeof(uint32_t)) != cudaSuccess) {
        h->err = "cudaMalloc failed"; return bail("alloc");
    }
    if (build_2d_tables(h)) return bail("tables");
    if (rebuild_geom(h)) return bail("geometry");
    if (alloc_grids(h)) return bail("grids");
    // per-stage twiddles of the radix-4 stages of a length-n transform in thread order: tw[(3 stage + i - 1) T + j],
    // T = n/4, = exp(+2 pi i * i * (j mod Ns) / (4 Ns)), Ns = R1 * 4^stage, R1 = 16 or 8 (fp64 on the host)
    auto twiddles = [&](int n, int r1, float2** out) -> bool {
        const int T = n / 4;
        std::vector<float2> tw;
        for (int Ns = r1; Ns < n; Ns *= 4)
            for (int i = 1; i <= 3; ++i)
                for (int j = 0; j < T; ++j) {
                    const double a = 2.0 * 3.14159265358979323846 * (double)i * (double)(j % Ns) / (4.0 * (double)Ns);
                    tw.push_back(make_float2((float)std::cos(a), (float)std::sin(a)));
                }
        return cudaMalloc(out, tw.size() * sizeof(float2)) == cudaSuccess &&
               cudaMemcpy(*out, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice) == cudaSuccess;
    };
    // radix-8 stages: tw8[(7 stage + i - 1) (n/8) + j] = exp(+2 pi i * i * (j mod Ns) / (8 Ns)), Ns = R1 * 8^stage
    auto twiddles8 = [&](int n, int r1, float2** out) -> bool {
        const int T8 = n / 8;
        std::vector<float2> tw;
        for (int Ns = r1; Ns < n; Ns *= 8)
            for (int i = 1; i <= 7; ++i)
                for (int j = 0; j < T8; ++j) {
                    const double a = 2.0 * 3.14159265358979323846 * (double)i * (double)(j % Ns) / (8.0 * (double)Ns);
                    tw.push_back(make_float2((float)std::cos(a), (float)std::sin(a)));
                }
        return cudaMalloc(out, tw.size() * sizeof(float2)) == cudaSuccess &&
               cudaMemcpy(*out, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice) == cudaSuccess;
    };
    if (fft_cols_supported(nx, ny) && fft_cols_setup() == cudaSuccess) {
        if (!twiddles(ny, fft_cols_first_radix(ny), &h->tw_d)) { h->err = "twiddle table"; return bail("fft"); }
        if (fft_cols_radix8(ny) && !twiddles8(ny, fft_cols_first_radix(ny), &h->tw8_d)) { h->err = "twiddle table"; return bail("fft"); }
        h->fused_fft = true;
        if (fft_rows_supported(nx, ny, 0) && fft_rows_supported(nx, ny, 1) && fft_rows_setup() == cudaSuccess) {
            if (!twiddles(nx, fft_rows_first_radix(nx), &h->tw_rows_d)) { h->err = "twiddle table"; return bail("fft"); }
            h->fused_rows = true;
        }
    }
    return h;
}

int muser_imager_destroy(muser_imager* h) {
    if (!h) return MUSER_OK;
    if (h->child2x) { muser_imager_destroy(h->child2x); h->child2x = nullptr; }
    cudaDeviceSynchronize();
    free_grids(h);
    free_bins(h);
    cudaFree(h->staged); cudaFree(h->sorted); cudaFree(h->stats_d); cudaFree(h->nitems_d);
    cudaFree(h->tables_d); cudaFree(h->planes_d); cudaFree(h->icx_d); cudaFree(h->icy_d); cudaFree(h->ones_d);
    cudaFree(h->in_uvw); cudaFree(h->in_freq); cudaFree(h->in_vis); cudaFree(h->in_wt); cudaFree(h->in_gid);
    cudaFree(h->ttp_d); cudaFree(h->ow_items); cudaFree(h->ow_tickets); cudaFree(h->ow_scratch);
    cudaFree(h->ow_sorted); cudaFree(h->ow_loc); cudaFree(h->ow_ctl); cudaFree(h->wg_ctl); cudaFree(h->wg_lists); cudaFree(h->tw_d); cudaFree(h->tw8_d); cudaFree(h->tw_rows_d);
    if (h->wg_streams_ok) {
        for (int i = 0; i < 7; ++i) cudaStreamDestroy(h->wg_side[i]);
        for (int i = 0; i < 8; ++i) cudaEventDestroy(h->wg_ev[i]);
    }
    for (auto& ev : h->ev_used) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
    for (auto& ev : h->ev_free) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
    delete h;
    return MUSER_OK;
}

int muser_set_kernel(muser_imager* h, int kind, double param) {
    if (!h) return MUSER_EINVAL;
    if (kind != MUSER_KERNEL_PSWF && kind != MUSER_KERNEL_GAUSS) return fail(h, MUSER_EINVAL, "unknown kernel kind");
    if (kind == MUSER_KERNEL_GAUSS && (param < 0 || !std::isfinite(param))) return fail(h, MUSER_EINVAL, "gaussian width must be >= 0");
    cudaDeviceSynchronize();
    h->kind = kind;
    h->gauss_a = (kind == MUSER_KERNEL_GAUSS && param > 0) ? param : 1.55;
    const bool was_w = wmode(h);
    h->nplanes = 0;
    int rc = rebuild_geom(h);
    if (rc) return rc;
    if ((rc = build_2d_tables(h))) return rc;
    rc = was_w ? alloc_grids(h) : reset_sync(h);
    if (rc == MUSER_OK && h->child2x) {                               // the 2x beam is gridded with the same kernel
        rc = muser_set_kernel(h->child2x, kind, param);
        if (rc) h->err = "2x beam: " + h->child2x->err;
    }
    return rc;
}

int muser_set_batch(muser_imager* h, int ngrids) {
    if (!h) return MUSER_EINVAL;
    if (ngrids < 1 || ngrids > (1 << 24) - 1) return fail(h, MUSER_EINVAL, "ngrids must be in [1, 2^24)");
    cudaDeviceSynchronize();
    const int old = h->ngrids;
    h->ngrids = ngrids;
    int rc = rebuild_geom(h);
    if (rc) { h->ngrids = old; rebuild_geom(h); return rc; }
    if ((rc = alloc_grids(h))) return rc;
    if (h->child2x) return muser_set_batch(h->child2x, ngrids);
    return MUSER_OK;
}

int muser_set_wplanes(muser_imager* h, int nplanes, const double* w_centres, const int* supports,
                      const float* const* tables_c64) {
    if (!h) return MUSER_EINVAL;
    if (nplanes < 0 || nplanes > kMaxPlanes) return fail(h, MUSER_EINVAL, "nplanes must be in [0, 64]");
    cudaDeviceSynchronize();
    if (nplanes == 0) {
        const bool was_w = wmode(h);
        h->nplanes = 0;
        int rc = rebuild_geom(h);
        if (rc) return rc;
        if ((rc = build_2d_tables(h))) return rc;
        return was_w ? alloc_grids(h) : reset_sync(h);
    }
    if (h->child2x) return fail(h, MUSER_EUNSUPPORTED, "the 2x beam is built in 2-D mode only: switch it off (muser_set_psf2x(h, 0)) before entering w mode");
    if (!w_centres || !supports) return fail(h, MUSER_EINVAL, "w_centres and supports are required");
    std::vector<int> sup(nplanes);
    std::vector<double> wc(nplanes);
    for (int p = 0; p < nplanes; ++p) {
        sup[p] = supports[p]; wc[p] = w_centres[p];
        if (sup[p] < 1 || sup[p] > 63 || !(sup[p] & 1)) return fail(h, MUSER_EINVAL, "plane supports must be odd in [1,63]");
        if (!(wc[p] >= 0) || !std::isfinite(wc[p])) return fail(h, MUSER_EINVAL, "plane centres must be finite and >= 0");
        if (h->nx < 2 * (sup[p] + 1) || h->ny < 2 * (sup[p] + 1)) return fail(h, MUSER_EINVAL, "grid too small for a plane support");
    }
    std::vector<std::vector<double>> t64(nplanes);
    if (tables_c64) {
        for (int p = 0; p < nplanes; ++p) {
            if (!tables_c64[p]) return fail(h, MUSER_EINVAL, "null plane table");
            const size_t L = ((size_t)sup[p] * h->Q + 1) * 2;
            t64[p].resize(L);
            for (size_t i = 0; i < L; ++i) t64[p][i] = (double)tables_c64[p][i];
            // the gridders compute the Hermitian half-plane only and take the other half as its conjugate mirror: that holds
            // for EVEN kernels, k(-x) = k(x) (every gridding kernel is: PSWF, Gaussian, the Fresnel w-kernels)
            double tmax = 0.0, asym = 0.0;
            const size_t n1 = (size_t)sup[p] * h->Q;
            for (size_t t = 0; t <= n1; ++t) {
                tmax = std::max(tmax, std::hypot(t64[p][2 * t], t64[p][2 * t + 1]));
                asym = std::max(asym, std::hypot(t64[p][2 * t] - t64[p][2 * (n1 - t)], t64[p][2 * t + 1] - t64[p][2 * (n1 - t) + 1]));
            }
            if (!(asym <= 1e-5 * tmax)) return fail(h, MUSER_EINVAL, "plane tables must be even: T[t] = T[S*Q - t]");
        }
    } else {
        const muser_host::WKernelGen gen(4096);
        const double fov = (double)h->nx * (h->cell_arcsec * kArcsec);
        for (int p = 0; p < nplanes; ++p) {
            const auto t = gen.table(sup[p], h->Q, wc[p], fov);
            t64[p].resize(t.size() * 2);
            for (size_t i = 0; i < t.size(); ++i) { t64[p][2 * i] = t[i].real(); t64[p][2 * i + 1] = t[i].imag(); }
        }
    }
    h->nplanes = nplanes;
    int rc = rebuild_geom(h);
    if (!rc) rc = upload_tables(h, t64, sup, wc);
    if (!rc) rc = alloc_grids(h);
    if (rc) {
        // do not leave the handle half-way (w mode with the 2-D beam grid or the old tables): fall back to 2-D mode
        const std::string why = h->err;
        h->nplanes = 0;
        if (rebuild_geom(h) == MUSER_OK && build_2d_tables(h) == MUSER_OK) alloc_grids(h);
        h->err = why + " (the handle is back in 2-D mode)";
    }
    return rc;
}

int muser_set_strategy(muser_imager* h, int strategy) {
    if (!h) return MUSER_EINVAL;
    if (strategy != MUSER_STRATEGY_AUTO && strategy != MUSER_STRATEGY_TILED && strategy != MUSER_STRATEGY_OWNER &&
        strategy != MUSER_STRATEGY_WPLANE)
        return fail(h, MUSER_EINVAL, "unknown strategy");
    if (h->zero_pending || h->sparse) {                               // do not carry a deferred reset / unwritten tiles across strategies
        int rc = flush_zero(h, h->last_stream);
        if (rc) return rc;
    }
    h->strategy = strategy;
    if (h->child2x) {
        int rc = muser_set_strategy(h->child2x, strategy);
        if (rc) { h->err = "2x beam: " + h->child2x->err; return rc; }
    }
    return MUSER_OK;
}

int muser_set_tuning(muser_imager* h, int key, int value) {
    if (!h) return MUSER_EINVAL;
    if (key < 0 || key >= MUSER_TUNE_COUNT) return fail(h, MUSER_EINVAL, "unknown tuning key");
    if (key == MUSER_TUNE_ITEM_SIZE && value != 0 && (value < 64 || value > (1 << 20))) return fail(h, MUSER_EINVAL, "item_size must be 0 (automatic) or in [64, 2^20]");
    if (key == MUSER_TUNE_BIN_ITERS && (value < 0 || value > 64)) return fail(h, MUSER_EINVAL, "bin_iters must be in [0, 64]");
    if (key == MUSER_TUNE_COLS_TMA && (value < 0 || value > 2)) return fail(h, MUSER_EINVAL, "cols_tma must be 0, 1 or 2");
    if (key == MUSER_TUNE_FFT_SUBBATCH && value < 0) return fail(h, MUSER_EINVAL, "fft_subbatch must be 0 (automatic) or a number of grids >= 1");
    h->tune[key] = value;
    return rebuild_geom(h);
}

int muser_set_grid_correction(muser_imager* h, int enabled) {
    if (!h) return MUSER_EINVAL;
    h->correction = enabled ? 1 : 0;
    if (h->child2x) h->child2x->correction = h->correction;
    return MUSER_OK;
}

int muser_set_weighting(muser_imager* h, int mode) {
    if (!h) return MUSER_EINVAL;
    if (mode != MUSER_WEIGHT_NATURAL && mode != MUSER_WEIGHT_UNIFORM) return fail(h, MUSER_EINVAL, "unknown weighting mode");
    cudaDeviceSynchronize();
    const int old = h->weighting;
    h->weighting = mode;
    int rc = rebuild_geom(h);
    if (rc == MUSER_OK) rc = alloc_grids(h);
    if (rc) { h->weighting = old; rebuild_geom(h); return rc; }
    if (h->child2x) return muser_set_weighting(h->child2x, mode);
    return MUSER_OK;
}

int muser_set_phase_offset(muser_imager* h, double dl, double dm) {
    if (!h) return MUSER_EINVAL;
    if (!std::isfinite(dl) || !std::isfinite(dm) || std::fabs(dl) > 1.0 || std::fabs(dm) > 1.0)
        return fail(h, MUSER_EINVAL, "phase offset must be finite direction cosines");
    h->off_l = dl; h->off_m = dm;
    return rebuild_geom(h);                                           // the beam does not depend on it: the 2x child is left alone
}

int muser_set_peak_search(muser_imager* h, int enabled) {
    if (!h) return MUSER_EINVAL;
    if ((enabled != 0) != h->peak_search) h->peaks_valid = false;
    h->peak_search = enabled != 0;
    return MUSER_OK;
}

int muser_get_peak(muser_imager* h, float* peak_value, int* peak_x, int* peak_y, float* min_value) {
    if (!h) return MUSER_EINVAL;
    if (!h->peak_search) return fail(h, MUSER_ESTATE, "peak search is off (muser_set_peak_search)");
    CU(h, cudaStreamSynchronize(h->last_stream));
    std::vector<PeakSlot> p((size_t)h->ngrids);
    CU(h, cudaMemcpy(p.data(), h->peaks_d, p.size() * sizeof(PeakSlot), cudaMemcpyDeviceToHost));
    for (int g = 0; g < h->ngrids; ++g) {
        if (p[g].maxkey == 0ull) return fail(h, MUSER_ESTATE, "no dirty image has been made since the peak search was enabled");
        const unsigned int ord = (unsigned int)(p[g].maxkey >> 32), idx = ~(unsigned int)(p[g].maxkey & 0xFFFFFFFFull);
        const unsigned int lo = ~p[g].minkey;
        float v, m;
        const unsigned int vb = (ord & 0x80000000u) ? (ord & 0x7FFFFFFFu) : ~ord, mb = (lo & 0x80000000u) ? (lo & 0x7FFFFFFFu) : ~lo;
        std::memcpy(&v, &vb, 4); std::memcpy(&m, &mb, 4);
        if (peak_value) peak_value[g] = v;
        if (peak_x) peak_x[g] = (int)(idx % (unsigned int)h->nx);
        if (peak_y) peak_y[g] = (int)(idx / (unsigned int)h->nx);
        if (min_value) min_value[g] = m;
    }
    return MUSER_OK;
}

int muser_histogram(muser_imager* h, const float* image, int nbins, float lo, float hi, unsigned int* hist_out, muser_stream sv) {
    if (!h) return MUSER_EINVAL;
    if (!image || !hist_out) return fail(h, MUSER_EINVAL, "null pointer");
    if (nbins < 1 || nbins > 8192) return fail(h, MUSER_EINVAL, "nbins must be in [1, 8192]");
    const bool own_range = !(lo < hi);
    if (own_range && !h->peak_search) return fail(h, MUSER_ESTATE, "lo >= hi asks for the image's own range: enable the peak search first");
    if (own_range && !h->peaks_valid) return fail(h, MUSER_ESTATE, "lo >= hi asks for the image's own range: no dirty image has been made since the peak search was enabled");
    if (h->ngrids > 65535) return fail(h, MUSER_EUNSUPPORTED, "histogram of more than 65535 grids per call");
    cudaStream_t s = (cudaStream_t)sv;
    h->last_stream = s;
    CU(h, cudaMemsetAsync(hist_out, 0, (size_t)h->ngrids * nbins * sizeof(unsigned int), s));
    CU(h, launch_histogram(image, (size_t)h->ny * h->nx, h->ngrids, nbins, lo, hi, own_range ? h->peaks_d : nullptr, hist_out, s));
    h->n_launches += 1;
    return MUSER_OK;
}

int muser_get_counts(muser_imager* h, int* counts_out, muser_stream sv) {
    if (!h) return MUSER_EINVAL;
    if (!counts_out) return fail(h, MUSER_EINVAL, "counts_out is null");
    if (!h->cnt) return fail(h, MUSER_ESTATE, "hit counts exist in uniform weighting mode only");
    cudaStream_t s = (cudaStream_t)sv;
    h->last_stream = s;
    int rc = flush_zero(h, s);
    if (rc == MUSER_OK) rc = ensure_lower(h, s);
    if (rc) return rc;
    CU(h, cudaMemcpyAsync(counts_out, h->cnt, grid_cells(h) * sizeof(int), cudaMemcpyDeviceToDevice, s));
    return MUSER_OK;
}

int muser_get_weighted_grid(muser_imager* h, void* grid_c64_out, float* wgrid_out, muser_stream sv) {
    if (!h) return MUSER_EINVAL;
    cudaStream_t s = (cudaStream_t)sv;
    h->last_stream = s;
    int rc = flush_zero(h, s);
    if (rc == MUSER_OK) rc = ensure_lower(h, s);
    if (rc) return rc;
    CU(h, launch_weighted_copy(h->geom, grid_ptrs(h), (float2*)grid_c64_out, wgrid_out, s));
    h->n_launches += 1;
    return MUSER_OK;
}

int muser_set_psf2x(muser_imager* h, int enabled) {
    if (!h) return MUSER_EINVAL;
    cudaDeviceSynchronize();
    if (!enabled) {
        if (h->child2x) { muser_imager_destroy(h->child2x); h->child2x = nullptr; }
        return MUSER_OK;
    }
    if (h->child2x) return MUSER_OK;
    if (wmode(h)) return fail(h, MUSER_EUNSUPPORTED, "the 2x beam is built in 2-D mode only");
    if (2 * h->nx > 32768 || 2 * h->ny > 32768) return fail(h, MUSER_EINVAL, "2x beam too large");
    muser_imager* c = muser_imager_create(2 * h->nx, 2 * h->ny, h->cell_arcsec, h->S, h->Q);
    if (!c) return fail(h, MUSER_ENOMEM, std::string("2x beam: ") + g_create_error);
    c->weights_only = true;
    int rc = MUSER_OK;
    if (h->kind != MUSER_KERNEL_PSWF) rc = muser_set_kernel(c, h->kind, h->gauss_a);
    if (rc == MUSER_OK && h->ngrids != 1) rc = muser_set_batch(c, h->ngrids);
    if (rc == MUSER_OK && h->weighting != MUSER_WEIGHT_NATURAL) rc = muser_set_weighting(c, h->weighting);
    if (rc == MUSER_OK) rc = muser_set_strategy(c, h->strategy);
    if (rc) { h->err = "2x beam: " + c->err; muser_imager_destroy(c); return rc; }
    c->correction = h->correction;
    h->child2x = c;
    return MUSER_OK;
}

int muser_psf2x(muser_imager* h, float* beam2x_out, muser_stream s) {
    if (!h) return MUSER_EINVAL;
    if (!beam2x_out) return fail(h, MUSER_EINVAL, "beam2x_out is null");
    if (!h->child2x) return fail(h, MUSER_ESTATE, "the 2x beam is off (muser_set_psf2x)");
    int rc = image_impl(h->child2x, nullptr, beam2x_out, (cudaStream_t)s);
    if (rc) h->err = "2x beam: " + h->child2x->err;
    return rc;
}

int muser_reset(muser_imager* h, muser_stream s) {
    if (!h) return MUSER_EINVAL;
    return reset_impl(h, (cudaStream_t)s);
}

int muser_grid(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64, const float* weight,
               long long nvis, muser_stream s) {
    if (!h) return MUSER_EINVAL;
    int rc = grid_impl(h, uvw_m, freq_hz, vis_c64, weight, nullptr, nvis, (cudaStream_t)s);
    if (rc == MUSER_OK && h->child2x) {
        rc = grid_impl(h->child2x, uvw_m, freq_hz, nullptr, weight, nullptr, nvis, (cudaStream_t)s);
        if (rc) h->err = "2x beam: " + h->child2x->err;
    }
    return rc;
}

int muser_grid_batched(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64,
                       const float* weight, const int* grid_id, long long nvis, muser_stream s) {
    if (!h) return MUSER_EINVAL;
    if (!grid_id && nvis > 0) return fail(h, MUSER_EINVAL, "grid_id is required");
    int rc = grid_impl(h, uvw_m, freq_hz, vis_c64, weight, grid_id, nvis, (cudaStream_t)s);
    if (rc == MUSER_OK && h->child2x) {
        rc = grid_impl(h->child2x, uvw_m, freq_hz, nullptr, weight, grid_id, nvis, (cudaStream_t)s);
        if (rc) h->err = "2x beam: " + h->child2x->err;
    }
    return rc;
}

int muser_grid_rows(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64, const float* weight,
                    const int* grid_id, long long nrow, int nchan, int npol, int ntime, int pol_mode, muser_stream s) {
    if (!h) return MUSER_EINVAL;
    int rc = grid_rows_impl(h, uvw_m, freq_hz, vis_c64, weight, grid_id, nrow, nchan, npol, ntime, pol_mode, (cudaStream_t)s);
    if (rc == MUSER_OK && h->child2x) {
        rc = grid_rows_impl(h->child2x, uvw_m, freq_hz, nullptr, weight, grid_id, nrow, nchan, npol, ntime, pol_mode, (cudaStream_t)s);
        if (rc) h->err = "2x beam: " + h->child2x->err;
    }
    return rc;
}

int muser_dirty(muser_imager* h, float* image_out, muser_stream s) {
    if (!h) return MUSER_EINVAL;
    if (!image_out) return fail(h, MUSER_EINVAL, "image_out is null");
    return image_impl(h, image_out, nullptr, (cudaStream_t)s);
}

int muser_psf(muser_imager* h, float* beam_out, muser_stream s) {
    if (!h) return MUSER_EINVAL;
    if (!beam_out) return fail(h, MUSER_EINVAL, "beam_out is null");
    return image_impl(h, nullptr, beam_out, (cudaStream_t)s);
}

int muser_dirty_psf(muser_imager* h, float* image_out, float* beam_out, muser_stream s) {
    if (!h) return MUSER_EINVAL;
    return image_impl(h, image_out, beam_out, (cudaStream_t)s);
}

static int frame_host_impl(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64,
                           const float* weight, const int* grid_id, long long nvis, float* image_out, float* beam_out,
                           muser_stream sv, bool synchronise) {
    if (!h) return MUSER_EINVAL;
    if (nvis < 0 || nvis > (1LL << 30)) return fail(h, MUSER_EINVAL, "nvis out of range");
    if (nvis > 0 && (!uvw_m || !freq_hz || !vis_c64 || !weight)) return fail(h, MUSER_EINVAL, "null input pointer");
    cudaStream_t s = (cudaStream_t)sv;
    if ((size_t)nvis > h->in_cap) {
        cudaFree(h->in_uvw); cudaFree(h->in_freq); cudaFree(h->in_vis); cudaFree(h->in_wt); cudaFree(h->in_gid);
        h->in_uvw = nullptr; h->in_freq = nullptr; h->in_vis = nullptr; h->in_wt = nullptr; h->in_gid = nullptr; h->in_cap = 0;
        const size_t cap = (size_t)nvis + 1024;
        CU(h, cudaMalloc(&h->in_uvw, cap * 3 * sizeof(float)));
        CU(h, cudaMalloc(&h->in_freq, cap * sizeof(double)));
        CU(h, cudaMalloc(&h->in_vis, cap * sizeof(float2)));
        CU(h, cudaMalloc(&h->in_wt, cap * sizeof(float)));
        CU(h, cudaMalloc(&h->in_gid, cap * sizeof(int)));
        h->in_cap = cap;
    }
    const size_t img_bytes = grid_cells(h) * sizeof(float);
    if (image_out && !h->out_dirty) CU(h, cudaMalloc(&h->out_dirty, img_bytes));
    if (beam_out && !h->out_psf) CU(h, cudaMalloc(&h->out_psf, img_bytes));
    int rc = reset_impl(h, s);
    if (rc) return rc;
    if (nvis > 0) {
        CU(h, cudaMemcpyAsync(h->in_uvw, uvw_m, (size_t)nvis * 3 * sizeof(float), cudaMemcpyHostToDevice, s));
        CU(h, cudaMemcpyAsync(h->in_freq, freq_hz, (size_t)nvis * sizeof(double), cudaMemcpyHostToDevice, s));
        CU(h, cudaMemcpyAsync(h->in_vis, vis_c64, (size_t)nvis * sizeof(float2), cudaMemcpyHostToDevice, s));
        CU(h, cudaMemcpyAsync(h->in_wt, weight, (size_t)nvis * sizeof(float), cudaMemcpyHostToDevice, s));
        if (grid_id) CU(h, cudaMemcpyAsync(h->in_gid, grid_id, (size_t)nvis * sizeof(int), cudaMemcpyHostToDevice, s));
        rc = grid_impl(h, h->in_uvw, h->in_freq, h->in_vis, h->in_wt, grid_id ? h->in_gid : nullptr, nvis, s);
        if (rc) return rc;
        if (h->child2x) {                                             // reset_impl above has reset the child as well
            rc = grid_impl(h->child2x, h->in_uvw, h->in_freq, nullptr, h->in_wt, grid_id ? h->in_gid : nullptr, nvis, s);
            if (rc) { h->err = "2x beam: " + h->child2x->err; return rc; }
        }
    }
    rc = image_impl(h, image_out ? h->out_dirty : nullptr, beam_out ? h->out_psf : nullptr, s);
    if (rc) return rc;
    if (image_out) CU(h, cudaMemcpyAsync(image_out, h->out_dirty, img_bytes, cudaMemcpyDeviceToHost, s));
    if (beam_out) CU(h, cudaMemcpyAsync(beam_out, h->out_psf, img_bytes, cudaMemcpyDeviceToHost, s));
    if (synchronise) CU(h, cudaStreamSynchronize(s));
    return MUSER_OK;
}

int muser_frame_host(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64,
                     const float* weight, const int* grid_id, long long nvis, float* image_out, float* beam_out,
                     muser_stream s) {
    return frame_host_impl(h, uvw_m, freq_hz, vis_c64, weight, grid_id, nvis, image_out, beam_out, s, true);
}

int muser_frame_host_async(muser_imager* h, const float* uvw_m, const double* freq_hz, const void* vis_c64,
                           const float* weight, const int* grid_id, long long nvis, float* image_out, float* beam_out,
                           muser_stream s) {
    return frame_host_impl(h, uvw_m, freq_hz, vis_c64, weight, grid_id, nvis, image_out, beam_out, s, false);
}

int muser_get_grid(muser_imager* h, void* grid_c64_out, float* wgrid_out, muser_stream sv) {
    if (!h) return MUSER_EINVAL;
    cudaStream_t s = (cudaStream_t)sv;
    const size_t nc = grid_cells(h);
    h->last_stream = s;
    int rcz = flush_zero(h, s);
    if (rcz) return rcz;
    if ((rcz = ensure_lower(h, s))) return rcz;
    if (grid_c64_out) CU(h, cudaMemcpyAsync(grid_c64_out, h->G, nc * sizeof(float2), cudaMemcpyDeviceToDevice, s));
    if (wgrid_out) CU(h, cudaMemcpyAsync(wgrid_out, h->Gw, nc * (wmode(h) ? sizeof(float2) : sizeof(float)), cudaMemcpyDeviceToDevice, s));
    return MUSER_OK;
}

int muser_get_table(muser_imager* h, int plane, float* table_out_host, int* len) {
    if (!h || !len) return MUSER_EINVAL;
    if (plane < 0 || plane >= (int)h->tables_f32.size()) return fail(h, MUSER_EINVAL, "plane out of range");
    const std::vector<float>& t = h->tables_f32[plane];
    if (!table_out_host || *len < (int)t.size()) { *len = (int)t.size(); return table_out_host ? fail(h, MUSER_EINVAL, "table buffer too small") : MUSER_OK; }
    std::memcpy(table_out_host, t.data(), t.size() * sizeof(float));
    *len = (int)t.size();
    return MUSER_OK;
}

int muser_get_stats(muser_imager* h, double* sum_weights, long long* n_gridded, long long* n_dropped, long long* n_flagged) {
    if (!h) return MUSER_EINVAL;
    CU(h, cudaStreamSynchronize(h->last_stream));
    Stats st;
    CU(h, cudaMemcpy(&st, h->stats_d, sizeof(Stats), cudaMemcpyDeviceToHost));
    if (sum_weights) *sum_weights = st.sum_weights;
    if (n_gridded) *n_gridded = (long long)st.n_gridded;
    if (n_dropped) *n_dropped = (long long)st.n_dropped;
    if (n_flagged) *n_flagged = (long long)st.n_flagged;
    return MUSER_OK;
}

int muser_set_profiling(muser_imager* h, int enabled) {
    if (!h) return MUSER_EINVAL;
    cudaDeviceSynchronize();
    for (auto& ev : h->ev_used) h->ev_free.push_back(ev);
    h->ev_used.clear();
    for (int i = 0; i < MUSER_STAGE_COUNT; ++i) { h->stage_ms[i] = 0; h->stage_n[i] = 0; }
    h->profiling = enabled != 0;
    return MUSER_OK;
}

int muser_get_profile(muser_imager* h, double* stage_ms, long long* stage_launches) {
    if (!h) return MUSER_EINVAL;
    CU(h, cudaDeviceSynchronize());
    for (auto& ev : h->ev_used) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, ev.a, ev.b) == cudaSuccess) { h->stage_ms[ev.stage] += ms; h->stage_n[ev.stage] += 1; }
        h->ev_free.push_back(ev);
    }
    h->ev_used.clear();
    for (int i = 0; i < MUSER_STAGE_COUNT; ++i) {
        if (stage_ms) stage_ms[i] = h->stage_ms[i];
        if (stage_launches) stage_launches[i] = h->stage_n[i];
    }
    return MUSER_OK;
}

long long muser_get_launch_count(const muser_imager* h) { return h ? h->n_launches : 0; }

int muser_host_table(int kind, int support, int oversample, double param, double* table_out) {
    if (!table_out || support < 1 || support > 63 || !(support & 1) || oversample < 2 || oversample > 256 || (oversample & 1)) return MUSER_EINVAL;
    std::vector<double> t;
    if (kind == MUSER_KERNEL_PSWF) t = muser_host::table_pswf(support, oversample);
    else if (kind == MUSER_KERNEL_GAUSS) t = muser_host::table_gauss(support, oversample, param > 0 ? param : 1.55);
    else return MUSER_EINVAL;
    std::memcpy(table_out, t.data(), t.size() * sizeof(double));
    return MUSER_OK;
}

int muser_host_wtable(int support, int oversample, double w_lambda, double fov_rad, double* table_out_re_im) {
    if (!table_out_re_im || support < 1 || support > 63 || !(support & 1) || oversample < 2 || oversample > 256 || (oversample & 1)) return MUSER_EINVAL;
    const muser_host::WKernelGen gen(4096);
    const auto t = gen.table(support, oversample, w_lambda, fov_rad);
    for (size_t i = 0; i < t.size(); ++i) { table_out_re_im[2 * i] = t[i].real(); table_out_re_im[2 * i + 1] = t[i].imag(); }
    return MUSER_OK;
}

int muser_host_corrector(const double* table, int support, int oversample, int n, double* corr_out) {
    if (!table || !corr_out || support < 1 || oversample < 2 || n < 1) return MUSER_EINVAL;
    const std::vector<double> c = muser_host::corrector(table, support, oversample, n);
    std::memcpy(corr_out, c.data(), c.size() * sizeof(double));
    return MUSER_OK;
}

}  // extern "C"
