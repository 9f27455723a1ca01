// field_kernels.cuh -- SURVEY.md 8(f) N2: the field step of the Vlasov-Poisson system on the periodic x grid.
//
//   rho_c = rho_fac * (moment - mean),   -Laplace(phi) = rho_c   (eq (2))   or
//   phi = phi_fac * (moment - mean)                              (eq (11), adiabatic electrons),
//   E = -grad(phi), pseudo-spectral.
//
// The x grid is tiny next to f (n_x^3 <= ~1e5 points against n_x^3 * n_v^3), so the transform is a plain
// separable DFT: one thread per output coefficient, n complex multiply-adds along the transformed axis with a
// twiddle table exp(-2 pi i m / n) indexed by (j*k) mod n.  That is O(n) more arithmetic than an FFT and still
// microseconds (3 * 48^3 * 48 complex MACs at C5), works for any extent (48 is not a power of two), and keeps the
// library free of a cuFFT dependency.  The k = 0 mode is dropped (reading F1), Nyquist modes have no first
// derivative (reading F2).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace bsl6d {

// DFT along one axis of a C-order array viewed as [outer][n][inner].
//   REAL_IN : input is real (double) instead of complex (double2)
//   REAL_OUT: write scale * Re(result) as double (last axis of an inverse transform)
//   inverse : use conj(w)
template <bool REAL_IN, bool REAL_OUT>
__global__ void dft_axis_kernel(const void* __restrict__ in_, void* __restrict__ out_, const double2* __restrict__ w,
                                uint32_t n, uint32_t inner, uint32_t total, int inverse, double scale) {
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= total) return;
    const uint32_t i = e % inner;
    const uint32_t k = (e / inner) % n;
    const uint32_t o = e / (inner * n);
    const size_t base = (size_t)o * n * inner + i;
    double re = 0.0, im = 0.0;
    uint32_t m = 0;                                           // (j*k) mod n, updated incrementally
    for (uint32_t j = 0; j < n; ++j) {
        double2 t = w[m];
        if (inverse) t.y = -t.y;
        double xr, xi;
        if (REAL_IN) {
            xr = static_cast<const double*>(in_)[base + (size_t)j * inner];
            xi = 0.0;
        } else {
            const double2 x = static_cast<const double2*>(in_)[base + (size_t)j * inner];
            xr = x.x;
            xi = x.y;
        }
        re += xr * t.x - xi * t.y;
        im += xr * t.y + xi * t.x;
        m += k;
        if (m >= n) m -= n;
    }
    if (REAL_OUT) static_cast<double*>(out_)[e] = scale * re;
    else static_cast<double2*>(out_)[e] = make_double2(re, im);
}

struct FieldArgs {
    uint32_t n[3];
    double L[3];            // period of each x dim
    int adiabatic;          // 0: phi_hat = rho_hat / |kappa|^2 ; 1: phi_hat = rho_hat  (c1 already holds phi_fac)
    double c1;              // rho_fac (Poisson) or phi_fac (adiabatic)
};

// rho_hat (moment's DFT) -> the three E_hat_d = -i kappa'_d phi_hat, written to e0, e1, e2.
__global__ void spectral_field_kernel(const double2* __restrict__ rho_hat, double2* __restrict__ e0,
                                      double2* __restrict__ e1, double2* __restrict__ e2, const FieldArgs a) {
    const uint32_t total = a.n[0] * a.n[1] * a.n[2];
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= total) return;
    uint32_t idx[3];
    idx[2] = e % a.n[2];
    idx[1] = (e / a.n[2]) % a.n[1];
    idx[0] = e / (a.n[2] * a.n[1]);
    double klap[3], kder[3];
    const double two_pi = 6.283185307179586476925286766559;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const uint32_t n = a.n[d], m = idx[d];
        double mm = (m < (n + 1) / 2) ? (double)m : (double)m - (double)n;
        const bool nyq = (n % 2 == 0) && (m == n / 2);
        if (nyq) mm = 0.5 * (double)n;
        klap[d] = two_pi * mm / a.L[d];
        kder[d] = nyq ? 0.0 : klap[d];
    }
    const double2 r = rho_hat[e];
    double pr, pi;
    if (e == 0) {                                             // k = 0: the mean is dropped
        pr = 0.0;
        pi = 0.0;
    } else if (a.adiabatic) {
        pr = a.c1 * r.x;
        pi = a.c1 * r.y;
    } else {
        const double k2 = klap[0] * klap[0] + klap[1] * klap[1] + klap[2] * klap[2];
        pr = a.c1 * r.x / k2;
        pi = a.c1 * r.y / k2;
    }
    // -i * k * (pr + i pi) = k*pi - i*k*pr
    e0[e] = make_double2(kder[0] * pi, -kder[0] * pr);
    e1[e] = make_double2(kder[1] * pi, -kder[1] * pr);
    e2[e] = make_double2(kder[2] * pi, -kder[2] * pr);
}

}  // namespace bsl6d
