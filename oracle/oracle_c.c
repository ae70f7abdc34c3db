/* CPU fp64 ORACLE (plain C) for the MUSER gridding hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A second, loop-by-loop transcription of steps O1 (coordinates), O3 (gridding) and O6 (w-planes) of
 * SURVEY.md §8(c) / DESIGN.md, and of the direct-DFT definition (I), fast enough for the full-size
 * configs and for bench.py's cpu_baseline.  It shares nothing with paper_1712_06913_b200/csrc and is
 * cross-checked against the numpy transcription in muser_oracle.py (tests/test_oracle_c.py).
 * Single thread, sequential sums, no blocking, no reordering.
 *
 * Paper passages followed: gridding = convolution of visibilities with a GCF onto a regular grid
 * (PAPER.md:78, 136-138); grid is complex, row-major iv*nu+iu (Alg. 1); both Hermitian
 * halves are gridded explicitly (reading R6 of "half the grid (as the data is Hermitian)");
 * natural weighting multiplies by the per-visibility weight (reading R10);
 * w-projection selects a kernel by |w| (reading R15).
 */
#include <math.h>
#include <stddef.h>

#define C_M_S 299792458.0
#define ARCSEC (3.14159265358979323846 / 648000.0)

/* O1 for one axis: nearest cell and oversample phase, floor(x+0.5) rounding for both (R4). */
static void cell_phase(double c_lambda, double scale, int n, int Q, double* i0, double* r) {
    double p = c_lambda * scale + (double)(n / 2);
    *i0 = floor(p + 0.5);
    double fr = p - *i0;
    *r = floor(fr * (double)Q + 0.5);
}

/* tables[p]: S_p*Q+1 doubles (2-D mode, wmode=0) or S_p*Q+1 (re,im) pairs (wmode=1).
 * G: [ngrids][ny][nx] (re,im) doubles.  Gw: [ngrids][ny][nx] doubles (wmode=0) or (re,im) pairs (wmode=1).
 * stats[4]: sum_weights, n_gridded (kept visibilities), n_dropped (off grid), n_flagged (weight<=0 / non-finite).
 * cnt (may be NULL): [ngrids][ny][nx] hit counts, +1 per gridded sample at its nearest cell (Alg. 1 l.1 `cnt`).
 * (dl, dm): phase-centre offset; V is multiplied by exp(+2 pi i (u dl + v dm)) first (PAPER.md:174 step 3; 0, 0 = none).
 * Accumulates into G, Gw, cnt, stats (callers zero them). */
int oracle_grid(const float* uvw_m, const double* freq_hz, const float* vis_ri, const float* weight,
                const int* grid_id, long long nvis, int nx, int ny, double cell_arcsec, int Q,
                int nplanes, const double* wc, const int* supports, const double* const* tables, int wmode,
                double dl, double dm, double* G, double* Gw, long long* cnt, double* stats) {
    const double cell = cell_arcsec * ARCSEC;
    const double su = (double)nx * cell, sv = (double)ny * cell;
    for (long long k = 0; k < nvis; ++k) {
        const double il = freq_hz[k] / C_M_S;
        const double ul = (double)uvw_m[3 * k + 0] * il;
        const double vl = (double)uvw_m[3 * k + 1] * il;
        const double wl = (double)uvw_m[3 * k + 2] * il;
        const double wt = (double)weight[k];
        double vr = (double)vis_ri[2 * k], vi = (double)vis_ri[2 * k + 1];
        if (!(isfinite(ul) && isfinite(vl) && isfinite(wl) && isfinite(wt) && isfinite(vr) && isfinite(vi) &&
              isfinite(freq_hz[k]) && wt > 0.0)) {
            stats[3] += 1.0;
            continue;
        }
        if (dl != 0.0 || dm != 0.0) {          /* NEXT-3: V * exp(+2 pi i (u dl + v dm)) */
            const double ph = 2.0 * 3.14159265358979323846 * (ul * dl + vl * dm);
            const double c = cos(ph), s = sin(ph), r0 = vr, i0 = vi;
            vr = r0 * c - i0 * s;
            vi = r0 * s + i0 * c;
        }
        int p = 0;
        if (wmode) {                          /* O6: nearest plane centre in |w|, tie -> lower p */
            double best = fabs(fabs(wl) - wc[0]);
            for (int q = 1; q < nplanes; ++q) {
                double d = fabs(fabs(wl) - wc[q]);
                if (d < best) { best = d; p = q; }
            }
        }
        const int S = supports[p], h = (S - 1) / 2;
        double iu0[2], iv0[2], ru[2], rv[2];
        int inside = 1;
        for (int s = 0; s < 2; ++s) {
            const double sgn = s ? -1.0 : 1.0;
            cell_phase(sgn * ul, su, nx, Q, &iu0[s], &ru[s]);
            cell_phase(sgn * vl, sv, ny, Q, &iv0[s], &rv[s]);
            if (!(iu0[s] >= h + 1 && iu0[s] <= nx - 1 - h && iv0[s] >= h + 1 && iv0[s] <= ny - 1 - h)) inside = 0;
        }
        if (!inside) { stats[2] += 1.0; continue; }
        stats[0] += 2.0 * wt;
        stats[1] += 1.0;
        const double* T = tables[p];
        const size_t g = grid_id ? (size_t)grid_id[k] : 0;
        for (int s = 0; s < 2; ++s) {
            const double sgn = s ? -1.0 : 1.0;
            const double valr = wt * vr, vali = wt * (s ? -vi : vi);     /* conjugate sample carries conj V */
            const int kconj = wmode && (sgn * wl < 0.0);                 /* conjugate kernel iff sample's w < 0 */
            const int cu = (int)iu0[s], cv = (int)iv0[s], pu = (int)ru[s], pv = (int)rv[s];
            if (cnt) cnt[(g * (size_t)ny + (size_t)cv) * (size_t)nx + (size_t)cu] += 1;
            for (int jy = -h; jy <= h; ++jy) {
                const int ty = jy * Q - pv + S * Q / 2;
                for (int jx = -h; jx <= h; ++jx) {
                    const int tx = jx * Q - pu + S * Q / 2;
                    const size_t cellidx = (g * (size_t)ny + (size_t)(cv + jy)) * (size_t)nx + (size_t)(cu + jx);
                    if (!wmode) {
                        const double kk = T[tx] * T[ty];
                        G[2 * cellidx] += kk * valr;
                        G[2 * cellidx + 1] += kk * vali;
                        Gw[cellidx] += kk * wt;
                    } else {
                        double kxr = T[2 * tx], kxi = T[2 * tx + 1], kyr = T[2 * ty], kyi = T[2 * ty + 1];
                        if (kconj) { kxi = -kxi; kyi = -kyi; }
                        const double kr = kxr * kyr - kxi * kyi, ki = kxr * kyi + kxi * kyr;
                        G[2 * cellidx] += kr * valr - ki * vali;
                        G[2 * cellidx + 1] += kr * vali + ki * valr;
                        Gw[2 * cellidx] += kr * wt;
                        Gw[2 * cellidx + 1] += ki * wt;
                    }
                }
            }
        }
    }
    return 0;
}

/* (I): out[k] = sum_s (valr+i vali)_s exp(+2 pi i (u l + v m [+ w (sqrt(1-l^2-m^2)-1)])) at direction cosines (l,m). */
int oracle_dft(long long ns, const double* u, const double* v, const double* w, const double* valr,
               const double* vali, long long npix, const double* l, const double* m, int use_w,
               double* out_re, double* out_im) {
    const double twopi = 2.0 * 3.14159265358979323846;
    for (long long k = 0; k < npix; ++k) {
        const double nn = use_w ? sqrt(1.0 - l[k] * l[k] - m[k] * m[k]) - 1.0 : 0.0;
        double sr = 0.0, si = 0.0;
        for (long long s = 0; s < ns; ++s) {
            const double ph = twopi * (u[s] * l[k] + v[s] * m[k] + (use_w ? w[s] * nn : 0.0));
            const double c = cos(ph), sn = sin(ph);
            sr += valr[s] * c - vali[s] * sn;
            si += valr[s] * sn + vali[s] * c;
        }
        out_re[k] = sr;
        out_im[k] = si;
    }
    return 0;
}
