// pointwise_kernels.cuh -- SURVEY.md 8(f) N3: odd stencil width with one displacement per POINT.
//
// PAPER.md:86-89 eq (6): for odd q the stencil stays centred on the grid point,
//     f(x_j + alpha) = sum_{m=-h..h} l_m(alpha) f(x_{j+m}),   h = (q-1)/2,   |alpha| < dx,
// and PAPER.md:100, 194, 244: the displacement may depend on all six coordinates -- the paper's own section-5
// benchmark runs exactly this ("random shifts alpha/dx in [-1,1]", widths 3, 5, 7, 9, 37^6 points).
// alpha is a full-size array in cells, so a sweep moves 24 B/point (f in, alpha in, f out) and the weights are
// evaluated per point (5q flops + q FMAs).  As in sweep_kernels.cuh one thread owns one pencil and keeps it in
// registers; because there is no integer part k here, every stencil index -- wrap or zero fill included -- is a
// compile-time constant.  All loads of a pencil precede its stores => f_in == f_out is legal (alpha must not alias).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace bsl6d {

template <int Q>
struct OddDen {
    double r[Q];
    constexpr OddDen() : r() {
        for (int i = 0; i < Q; ++i) {
            double d = 1.0;
            for (int j = 0; j < Q; ++j)
                if (j != i) d *= (double)(i - j);
            r[i] = 1.0 / d;
        }
    }
};

// l_m(alpha) on nodes m = i - H, i = 0..Q-1.  Prefix/suffix products (3Q multiplies) times compile-time reciprocal
// denominators; a whole-cell alpha in [-H, H] is mapped to the exact unit vector (reading S11 carried over), so that
// whole-cell displacements stay exact permutations.
template <int Q>
__device__ __forceinline__ void lagrange_weights_odd(double alpha, double (&w)[Q]) {
    constexpr OddDen<Q> den{};
    constexpr int H = (Q - 1) / 2;
    double d[Q], pre[Q], suf[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) d[i] = alpha - (double)(i - H);
    pre[0] = 1.0;
#pragma unroll
    for (int i = 1; i < Q; ++i) pre[i] = pre[i - 1] * d[i - 1];
    suf[Q - 1] = 1.0;
#pragma unroll
    for (int i = Q - 2; i >= 0; --i) suf[i] = suf[i + 1] * d[i + 1];
#pragma unroll
    for (int i = 0; i < Q; ++i) w[i] = (pre[i] * suf[i]) * den.r[i];
    if (alpha == rint(alpha) && fabs(alpha) <= (double)H) {       // whole-cell displacement: rare, exact
#pragma unroll
        for (int i = 0; i < Q; ++i) w[i] = (d[i] == 0.0) ? 1.0 : 0.0;
    }
}

struct PointwiseArgs {
    const double* in;
    double* out;
    const double* alpha;   // same shape and layout as f, displacement in cells
    uint32_t inner, outer; // as in SweepArgs
    uint32_t npencil;      // inner * outer
};

template <int N, int Q, bool PERIODIC>
__device__ __forceinline__ double stencil_at(const double (&u)[N], const double (&w)[Q], int j) {
    constexpr int H = (Q - 1) / 2;
    double acc = 0.0;
    bool first = true;
#pragma unroll
    for (int m = 0; m < Q; ++m) {
        const int jj = j + m - H;
        double v;
        if (PERIODIC) v = u[((jj % N) + N) % N];
        else {
            if (jj < 0 || jj >= N) continue;              // zero extension: the term vanishes
            v = u[jj];
        }
        acc = first ? w[m] * v : fma(w[m], v, acc);
        first = false;
    }
    return acc;
}

// strided dims (inner > 1)
template <int N, int Q, bool PERIODIC, int T, int MINB>
__global__ void __launch_bounds__(T, MINB) pointwise_strided_kernel(const PointwiseArgs a) {
    // lanes run along the flattened pencil index (o, i): full lane use for any `inner` (37 is not a power of two)
    const uint32_t p = blockIdx.x * T + threadIdx.x;
    if (p >= a.npencil) return;
    const uint32_t o = p / a.inner, i = p - o * a.inner;
    const size_t stride = a.inner;
    const size_t base = (size_t)o * N * stride + i;
    const double* pin = a.in + base;
    const double* pal = a.alpha + base;
    double* pout = a.out + base;
    // every load of the pencil -- values and displacements -- is issued before the first store: 2N loads in flight
    // per thread, and stores to f_out can never be ordered between them (f_out may alias f_in)
    double u[N], al[N];
#pragma unroll
    for (int t = 0; t < N; ++t) u[t] = __ldcs(pin + (size_t)t * stride);
#pragma unroll
    for (int t = 0; t < N; ++t) al[t] = __ldcs(pal + (size_t)t * stride);
#pragma unroll
    for (int j = 0; j < N; ++j) {
        double w[Q];
        lagrange_weights_odd<Q>(al[j], w);
        __stcs(pout + (size_t)j * stride, stencil_at<N, Q, PERIODIC>(u, w, j));
    }
}

// unit-stride dim (inner == 1, always a v dim): PB pencils per block, f and alpha transposed through two padded
// shared-memory tiles (odd row pitch: "lane = pencil" accesses are conflict-free); results overwrite the alpha tile
// (alpha_j is consumed by the one thread that produces out_j).  A pencil is cut into S segments of R = ceil(N/S)
// outputs, one thread each (the lanes of a warp share the segment): a thread then holds R+Q-1 values instead of N and
// evaluates R weight sets instead of N, so that a block has S times the warps for the same tile -- the one-thread-
// per-pencil version of round 1 ran 8 warps per SM (3.5-4.5 TB/s at 37^6).
template <int N, int Q, int S, int PB, int MINB>
__global__ void __launch_bounds__(PB * S, MINB) pointwise_unit_kernel(const PointwiseArgs a) {
    extern __shared__ double tiles[];                      // 2 x PB x LD
    constexpr int T = PB * S;
    constexpr int LD = N | 1;
    constexpr int H = (Q - 1) / 2;
    constexpr int R = (N + S - 1) / S;
    double* tf = tiles;
    double* ta = tiles + PB * LD;
    const size_t p0 = (size_t)blockIdx.x * PB;
    const uint32_t np = (uint32_t)(((size_t)a.outer - p0) < (size_t)PB ? ((size_t)a.outer - p0) : (size_t)PB);
    const uint32_t nelem = np * N;
    const double* pin = a.in + p0 * N;
    const double* pal = a.alpha + p0 * N;
    double* pout = a.out + p0 * N;
#pragma unroll 4
    for (uint32_t e = threadIdx.x; e < nelem; e += T) {
        const uint32_t s = (e / N) * LD + (e % N);
        tf[s] = __ldcs(pin + e);
        ta[s] = __ldcs(pal + e);
    }
    __syncthreads();
    const uint32_t pl = threadIdx.x % PB;
    const int j0 = (int)(threadIdx.x / PB) * R;
    if (pl < np) {
        const double* rowf = tf + pl * LD;
        double* rowa = ta + pl * LD;
        double u[R + Q - 1];                               // u[t] = f[j0 - H + t], zero outside the pencil
#pragma unroll
        for (int t = 0; t < R + Q - 1; ++t) {
            const int c = j0 - H + t;
            u[t] = (c >= 0 && c < N) ? rowf[c] : 0.0;
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int j = j0 + r;
            if (j < N) {
                double w[Q];
                lagrange_weights_odd<Q>(rowa[j], w);
                // the terms of stencil_at<N, Q, false> in the same order; a node outside the pencil contributes nothing
                double acc = 0.0;
                bool first = true;
#pragma unroll
                for (int m = 0; m < Q; ++m) {
                    const int jj = j + m - H;
                    if (jj < 0 || jj >= N) continue;
                    acc = first ? w[m] * u[r + m] : fma(w[m], u[r + m], acc);
                    first = false;
                }
                rowa[j] = acc;
            }
        }
    }
    __syncthreads();
#pragma unroll 4
    for (uint32_t e = threadIdx.x; e < nelem; e += T) __stcs(pout + e, ta[(e / N) * LD + (e % N)]);
}

}  // namespace bsl6d
