// Host-side fp64 table generators of the library (see tables.cpp).  Not shared with oracle/.
#pragma once
#include <complex>
#include <vector>

namespace muser_host {

// Order-0 prolate spheroidal wave function psi_0(eta; c) on |eta| <= 1, normalised psi(0) = 1 (R2).
class Pswf {
public:
    explicit Pswf(double c);
    double operator()(double eta) const;

private:
    double raw(double x) const;
    std::vector<double> beta_;   // coefficients on the even normalised Legendre polynomials
    double norm0_;
};

// O2 tables T[t] = C((t - S*Q/2)/Q), t = 0..S*Q.
std::vector<double> table_pswf(int S, int Q);
std::vector<double> table_gauss(int S, int Q, double a);

// R15 Fresnel-separable w-kernels (one axis), taper psi(2 l) at c = 3.5 pi, Gauss-Legendre quadrature.
class WKernelGen {
public:
    explicit WKernelGen(int nquad = 4096);
    std::vector<std::complex<double>> table(int S, int Q, double w_lambda, double fov_rad) const;

private:
    std::vector<double> ell_, aw_;
    double norm_;
};

// O5 per-axis corrector of a real table.
std::vector<double> corrector(const double* T, int S, int Q, int n);

}  // namespace muser_host
