// Host-side fp64 generators of the library (A0 setup): gridding-kernel tables and grid correctors.
//
// PAPER.md:136-138 (sec. 3.2.3): the gridding convolution function is a truncated spheroidal function.
// DESIGN.md R2: the exact order-0 prolate spheroidal wave function psi_0(eta; c), c = pi*S/2, from its
// definition -- here through its Legendre-series eigenproblem (the differential operator
// (1-x^2) d2/dx2 - 2x d/dx - c^2 x^2 is tridiagonal in the normalised Legendre basis).  This generator is
// the library's own: it shares nothing with oracle/ (which calls scipy's special function).
#include "tables.h"

#include <algorithm>
#include <cmath>
#include <cstddef>

namespace muser_host {

static const double kPi = 3.14159265358979323846;

// Smallest eigenpair of a symmetric tridiagonal matrix (diag d[0..n), off-diag e[0..n-1)) by bisection on the
// Sturm count followed by inverse iteration.
static void smallest_eigvec_tridiag(const std::vector<double>& d, const std::vector<double>& e,
                                    std::vector<double>& vec) {
    const int n = (int)d.size();
    double lo = d[0], hi = d[0];
    for (int i = 0; i < n; ++i) {
        const double r = (i > 0 ? std::fabs(e[i - 1]) : 0.0) + (i + 1 < n ? std::fabs(e[i]) : 0.0);
        lo = std::min(lo, d[i] - r);
        hi = std::max(hi, d[i] + r);
    }
    auto count_below = [&](double x) {      // number of eigenvalues < x
        int cnt = 0;
        double q = d[0] - x;
        if (q < 0) ++cnt;
        for (int i = 1; i < n; ++i) {
            if (q == 0.0) q = 1e-300;
            q = d[i] - x - e[i - 1] * e[i - 1] / q;
            if (q < 0) ++cnt;
        }
        return cnt;
    };
    for (int it = 0; it < 200 && hi - lo > 1e-15 * std::max(1.0, std::fabs(lo) + std::fabs(hi)); ++it) {
        const double mid = 0.5 * (lo + hi);
        if (count_below(mid) >= 1) hi = mid; else lo = mid;
    }
    const double lam = 0.5 * (lo + hi) - 1e-9 * std::max(1.0, std::fabs(hi));   // shift just below it
    // inverse iteration: solve (A - lam I) y = x by the Thomas algorithm (A - lam I is positive definite)
    vec.assign(n, 1.0);
    std::vector<double> cp(n), y(n);
    for (int it = 0; it < 60; ++it) {
        double b = d[0] - lam;
        cp[0] = e.empty() ? 0.0 : e[0] / b;
        y[0] = vec[0] / b;
        for (int i = 1; i < n; ++i) {
            b = d[i] - lam - e[i - 1] * cp[i - 1];
            cp[i] = (i + 1 < n) ? e[i] / b : 0.0;
            y[i] = (vec[i] - e[i - 1] * y[i - 1]) / b;
        }
        for (int i = n - 2; i >= 0; --i) y[i] -= cp[i] * y[i + 1];
        double nrm = 0.0;
        for (int i = 0; i < n; ++i) nrm += y[i] * y[i];
        nrm = std::sqrt(nrm);
        for (int i = 0; i < n; ++i) vec[i] = y[i] / nrm;
    }
}

Pswf::Pswf(double c) {
    // even normalised Legendre indices k = 0, 2, ..., 2(N-1)
    const int N = std::max(40, (int)(c * 1.5) + 30);
    std::vector<double> d(N), e(N - 1);
    const double c2 = c * c;
    for (int j = 0; j < N; ++j) {
        const double k = 2.0 * j;
        d[j] = k * (k + 1.0) + c2 * (2.0 * k * (k + 1.0) - 1.0) / ((2.0 * k + 3.0) * (2.0 * k - 1.0));
        if (j + 1 < N)
            e[j] = c2 * (k + 2.0) * (k + 1.0) / ((2.0 * k + 3.0) * std::sqrt((2.0 * k + 1.0) * (2.0 * k + 5.0)));
    }
    smallest_eigvec_tridiag(d, e, beta_);
    norm0_ = 1.0;
    norm0_ = raw(0.0);
}

double Pswf::raw(double x) const {
    // sum_j beta_j * sqrt(2j + 1/2) * P_{2j}(x), Legendre three-term recurrence
    const int N = (int)beta_.size();
    double pkm1 = 1.0, pk = x, sum = beta_[0] * std::sqrt(0.5);
    for (int k = 1; k < 2 * N - 1; ++k) {          // pk = P_k
        const double pkp1 = ((2.0 * k + 1.0) * x * pk - k * pkm1) / (k + 1.0);
        pkm1 = pk;
        pk = pkp1;                                   // now P_{k+1}
        if (((k + 1) & 1) == 0) sum += beta_[(k + 1) / 2] * std::sqrt((k + 1) + 0.5) * pk;
    }
    return sum / norm0_;
}

double Pswf::operator()(double eta) const {
    eta = std::fabs(eta);
    if (eta > 1.0) eta = 1.0;
    return raw(eta);
}

std::vector<double> table_pswf(int S, int Q) {
    const Pswf psi(kPi * S / 2.0);
    const int L = S * Q + 1;
    std::vector<double> T(L);
    for (int t = 0; t <= (L - 1) / 2; ++t) {        // the table is built exactly symmetric about its centre
        const double x = ((double)t - S * Q / 2.0) / Q;
        const double val = psi(2.0 * x / S);
        T[t] = val;
        T[L - 1 - t] = val;
    }
    return T;
}

std::vector<double> table_gauss(int S, int Q, double a) {
    const int L = S * Q + 1;
    std::vector<double> T(L);
    for (int t = 0; t <= (L - 1) / 2; ++t) {
        const double x = ((double)t - S * Q / 2.0) / Q;
        const double val = std::exp(-(x / a) * (x / a));
        T[t] = val;
        T[L - 1 - t] = val;
    }
    return T;
}

// Gauss-Legendre nodes/weights on [-1, 1] (Newton iteration on P_n).
static void gauss_legendre(int n, std::vector<double>& x, std::vector<double>& w) {
    x.resize(n);
    w.resize(n);
    for (int i = 0; i < (n + 1) / 2; ++i) {
        double z = std::cos(kPi * (i + 0.75) / (n + 0.5));
        double pp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) {
                const double p3 = p2;
                p2 = p1;
                p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
            }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            const double dz = p1 / pp;
            z -= dz;
            if (std::fabs(dz) < 1e-16) break;
        }
        x[i] = -z;
        x[n - 1 - i] = z;
        w[i] = w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

WKernelGen::WKernelGen(int nquad) {
    // taper A(l) = psi(2 l), c = 3.5 pi, on l in [-1/2, 1/2]; integrand is even in l -> keep l > 0 only
    std::vector<double> xg, wg;
    gauss_legendre(nquad, xg, wg);
    const Pswf psi(3.5 * kPi);
    norm_ = 0.0;
    for (int i = 0; i < nquad; ++i) {
        if (xg[i] <= 0.0) continue;
        ell_.push_back(0.5 * xg[i]);
        const double aw = psi(xg[i]) * 0.5 * wg[i];
        aw_.push_back(aw);
        norm_ += 2.0 * aw;
    }
}

std::vector<std::complex<double>> WKernelGen::table(int S, int Q, double w, double fov) const {
    // k_w(D) = Int A(l) exp(-i pi w (l fov)^2) exp(-2 pi i D l) dl / Int A  = 2 Int_{l>0} A chirp cos(2 pi D l) dl / Int A
    const int L = S * Q + 1, nq = (int)ell_.size();
    std::vector<double> cr(nq), ci(nq);
    for (int i = 0; i < nq; ++i) {
        const double ph = -kPi * w * (ell_[i] * fov) * (ell_[i] * fov);
        cr[i] = aw_[i] * std::cos(ph);
        ci[i] = aw_[i] * std::sin(ph);
    }
    std::vector<std::complex<double>> T(L);
    for (int t = 0; t <= (L - 1) / 2; ++t) {
        const double D = ((double)t - S * Q / 2.0) / Q;
        double sr = 0.0, si = 0.0;
        for (int i = 0; i < nq; ++i) {
            const double cs = std::cos(2.0 * kPi * D * ell_[i]);
            sr += cr[i] * cs;
            si += ci[i] * cs;
        }
        const std::complex<double> val(2.0 * sr / norm_, 2.0 * si / norm_);
        T[t] = val;
        T[L - 1 - t] = val;
    }
    return T;
}

std::vector<double> corrector(const double* T, int S, int Q, int n) {
    // c[x] = (1/Q) sum_t om_t T[t] cos(2 pi l_x x_t), l_x = (x - n/2)/n, trapezoid weights (O5)
    const int L = S * Q + 1;
    std::vector<double> c(n);
    for (int x = 0; x < n; ++x) {
        const double ell = ((double)x - n / 2) / n;
        double sum = 0.0;
        for (int t = 0; t < L; ++t) {
            const double xt = ((double)t - S * Q / 2.0) / Q;
            const double om = (t == 0 || t == L - 1) ? 0.5 : 1.0;
            sum += om * T[t] * std::cos(2.0 * kPi * ell * xt);
        }
        c[x] = sum / Q;
    }
    return c;
}

}  // namespace muser_host
