// pointwise_kernels.cuh -- SURVEY.md 8(f) N3: odd stencil width with one displacement per POINT.
//
// PAPER.md:86-89 eq (6): for odd q the stencil stays centred on the grid point,
//     f(x_j + alpha) = sum_{m=-h..h} l_m(alpha) f(x_{j+m}),   h = (q-1)/2,   |alpha| < dx,
// and PAPER.md:100, 194, 244: the displacement may depend on all six coordinates -- the paper's own section-5
// benchmark runs exactly this ("random shifts alpha/dx in [-1,1]", widths 3, 5, 7, 9, 37^6 points).
// alpha is a full-size array in cells, so a sweep moves 24 B/point (f in, alpha in, f out) and the interpolant is
// evaluated per point.  Because there is no integer part k here, every stencil index -- wrap or zero fill included --
// is a compile-time constant in the kernels compiled per extent.
//
// Round 2 (second half): (i) the per-point evaluation uses the symmetry of the centred equidistant nodes
// (interp_odd below: about 4.5q fp64 instructions instead of 6q for q separate weights -- 41 against 52 at q = 9),
// because widths 7 and 9 were co-limited by the fp64 pipe; (ii) the strided kernel no longer holds the displacements of a whole
// pencil in registers: f and alpha stream through a look-ahead of D rows (loads issued D outputs ahead of their
// use, stores in between), which halves the registers and doubles the resident warps; (iii) run-time-extent kernels
// (pointwise_generic_kernel, pointwise_generic_unit_kernel) serve every extent without a compiled instance.
// In every kernel a value of f_in is loaded before the output with the same index is stored, and the values a
// periodic wrap needs again at the end of the pencil are kept in registers => f_in == f_out is legal (alpha must not
// alias f_out).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace bsl6d {

// c[m] = 1 / prod_{j != m, |j| <= H} (m - j) for m = 0..H (c[-m] == c[m]: q - 1 is even)
template <int Q>
struct OddSym {
    double c[(Q + 1) / 2];
    constexpr OddSym() : c() {
        constexpr int H = (Q - 1) / 2;
        for (int m = 0; m <= H; ++m) {
            double d = 1.0;
            for (int j = -H; j <= H; ++j)
                if (j != m) d *= (double)(m - j);
            c[m] = 1.0 / d;
        }
    }
};

// sum_{m=-H..H} l_m(alpha) v[H+m] for the Lagrange basis on the nodes -H..H (eq (6)), written with the node symmetry:
//     e_i = alpha^2 - i^2,  E_m = prod_{i>=1, i != m} e_i,  E_0 = prod_{i>=1} e_i,
//     l_{+-m}(alpha) = c_m alpha E_m (alpha +- m)   (m >= 1),      l_0(alpha) = c_0 E_0,
//     sum = c_0 E_0 v_0 + alpha * sum_{m>=1} c_m E_m [ alpha (v_m + v_-m) + m (v_m - v_-m) ].
// Same polynomial as q separate weights (differences: a few ulp of max|v|).  A whole-cell alpha in [-H, H] returns
// v[H + alpha] itself, so that whole-cell displacements stay exact permutations (reading S11 carried over).
template <int Q>
__device__ __forceinline__ double interp_odd(double alpha, const double (&v)[Q]) {
    constexpr int H = (Q - 1) / 2;
    constexpr OddSym<Q> k{};
    double r, e0_all = 0.0;
    if constexpr (H == 0) {
        r = v[0];
    } else {
        double e[H + 1], pre[H + 2], suf[H + 2];               // pre[m] = prod_{1<=i<m} e_i, suf[m] = prod_{m<i<=H} e_i
#pragma unroll
        for (int i = 1; i <= H; ++i) e[i] = fma(alpha, alpha, -(double)(i * i));
        pre[1] = 1.0;
#pragma unroll
        for (int m = 2; m <= H + 1; ++m) pre[m] = (m == 2) ? e[1] : pre[m - 1] * e[m - 1];
        suf[H] = 1.0;
#pragma unroll
        for (int m = H - 1; m >= 1; --m) suf[m] = (m == H - 1) ? e[H] : suf[m + 1] * e[m + 1];
        double acc = 0.0;
#pragma unroll
        for (int m = 1; m <= H; ++m) {
            const double s = v[H + m] + v[H - m], d = v[H + m] - v[H - m];
            const double t = fma(alpha, s, (m == 1) ? d : (double)m * d);
            // c_m E_m: E_m = pre[m] * suf[m], with the unit factors at the ends left out
            const double g = (H == 1) ? k.c[1] : (m == 1 ? k.c[m] * suf[m] : (m == H ? k.c[m] * pre[m] : k.c[m] * (pre[m] * suf[m])));
            acc = (m == 1) ? g * t : fma(g, t, acc);
        }
        r = fma(alpha, acc, (k.c[0] * pre[H + 1]) * v[H]);
        e0_all = pre[H + 1];
    }
    // whole-cell displacement (rare): alpha * E_0 = prod_{|i| <= H} (alpha - i) is zero exactly when alpha is one of the
    // nodes (alpha^2 - i^2 is formed with one rounding), or so small that v[H] is the answer to the last bit anyway
    bool whole;
    if constexpr (H == 0) whole = true;
    else whole = alpha * e0_all == 0.0;
    if (whole) {
        const int ia = (int)alpha;
#pragma unroll
        for (int m = -H; m <= H; ++m)
            if (ia == m) r = v[H + m];
    }
    return r;
}

struct PointwiseArgs {
    const double* in;
    double* out;
    const double* alpha;   // same shape and layout as f, displacement in cells
    uint32_t inner, outer; // as in SweepArgs
    uint32_t npencil;      // inner * outer
    uint32_t n;            // extent of the swept dim (run-time-extent kernels only)
    uint32_t periodic;     //   "   boundary kind
    uint32_t pb, ld;       // pointwise_generic_unit_kernel: pencils per block, row pitch of the tiles
};

// strided dims (inner > 1), extent N compiled in.  Thread = pencil, lanes along the flattened pencil index (o, i)
// (full lane use for any `inner`: 37 is not a power of two).  Loads run D outputs ahead of their use.
template <int N, int Q, bool PERIODIC, int T, int MINB, int D>
__global__ void __launch_bounds__(T, MINB) pointwise_strided_kernel(const PointwiseArgs a) {
    constexpr int H = (Q - 1) / 2;
    const uint32_t p = blockIdx.x * T + threadIdx.x;
    if (p >= a.npencil) return;
    const uint32_t o = p / a.inner, i = p - o * a.inner;
    const size_t stride = a.inner;
    const size_t base = (size_t)o * N * stride + i;
    const double* pin = a.in + base;
    const double* pal = a.alpha + base;
    double* pout = a.out + base;
    // u[] and al[] are fully unrolled: each element is a register that lives from its load to its last use.  The
    // stores in between pin the loads where they are written (f_out may alias f_in, and alpha carries no
    // __restrict__ on purpose: hoisting all N alpha loads to the top is what this kernel avoids).
    double u[N], al[N];
    constexpr int TAIL0 = (PERIODIC && N - H > 0) ? N - H : N;    // periodic: rows N-H..N-1 are needed by output 0
#pragma unroll
    for (int t = TAIL0; t < N; ++t) u[t] = __ldcs(pin + (size_t)t * stride);
#pragma unroll
    for (int t = 0; t < N && t <= H + D && t < TAIL0; ++t) u[t] = __ldcs(pin + (size_t)t * stride);
#pragma unroll
    for (int t = 0; t < N && t <= D; ++t) al[t] = __ldcs(pal + (size_t)t * stride);
#pragma unroll
    for (int j = 0; j < N; ++j) {
        const int tf = j + H + D + 1, ta = j + D + 1;
        if (tf < TAIL0) u[tf] = __ldcs(pin + (size_t)tf * stride);
        if (ta < N) al[ta] = __ldcs(pal + (size_t)ta * stride);
        double v[Q];
#pragma unroll
        for (int m = 0; m < Q; ++m) {
            const int jj = j + m - H;
            if (PERIODIC) v[m] = u[((jj % N) + N) % N];
            else v[m] = (jj < 0 || jj >= N) ? 0.0 : u[jj];       // zero extension
        }
        __stcs(pout + (size_t)j * stride, interp_odd<Q>(al[j], v));
    }
}

// strided dims, run-time extent n (any n >= 1; periodic: the stencil may wrap more than once when n < q).
// The same streaming scheme with register rings whose indices are static because the pencil is walked in blocks of
// Q outputs: win[(j + t) % Q] = f[j - H + t], qf[j % Q] = f[j + H + Q] on its way, qa[j % Q] = alpha[j + Q] on its way.
template <int Q, int T>
__global__ void __launch_bounds__(T) pointwise_generic_kernel(const PointwiseArgs a) {
    constexpr int H = (Q - 1) / 2;
    const uint32_t p = blockIdx.x * T + threadIdx.x;
    if (p >= a.npencil) return;
    const uint32_t o = p / a.inner, i = p - o * a.inner;
    const int n = (int)a.n;
    const bool periodic = a.periodic != 0;
    const size_t stride = a.inner;
    const size_t base = (size_t)o * n * stride + i;
    const double* pin = a.in + base;
    const double* pal = a.alpha + base;
    double* pout = a.out + base;
    // rows 0..H-1 are needed again at the end of a periodic pencil, when an in-place sweep has overwritten them
    double first[H > 0 ? H : 1];
#pragma unroll
    for (int t = 0; t < H; ++t) first[t] = (periodic && n > 0) ? __ldcs(pin + (size_t)(t % n) * stride) : 0.0;
    // f at (virtual) row r: r in [0, n) from memory, beyond the ends by wrap or zero.  `early` rows (r < H after the
    // wrap) come from `first` once outputs have been stored.
    auto row_value = [&](int r, bool stored_some) -> double {
        if (periodic) {
            if (stored_some) {
                if (r >= n) r -= n;                            // in the loop r < n + H: at most one wrap
            } else {
                r %= n;
                if (r < 0) r += n;
            }
            if (stored_some && r < H) {
                double x = 0.0;
#pragma unroll
                for (int t = 0; t < H; ++t)
                    if (r == t) x = first[t];
                return x;
            }
            return __ldcs(pin + (size_t)r * stride);
        }
        return (r >= 0 && r < n) ? __ldcs(pin + (size_t)r * stride) : 0.0;
    };
    double win[Q], qf[Q], qa[Q];
#pragma unroll
    for (int t = 0; t < Q; ++t) win[t] = row_value(t - H, false);                 // window of output 0
#pragma unroll
    for (int t = 0; t < Q; ++t) qf[t] = row_value(t + H + 1, false);              // rows H+1 .. H+Q (outputs 1..Q)
#pragma unroll
    for (int t = 0; t < Q; ++t) qa[t] = (t < n) ? __ldcs(pal + (size_t)t * stride) : 0.0;
    // rows up to H+Q have been read before the first store: an in-place wrap is only a hazard for rows < H read later
    for (int jb = 0; jb < n; jb += Q) {
#pragma unroll
        for (int d = 0; d < Q; ++d) {
            const int j = jb + d;
            if (j < n) {
                double v[Q];
#pragma unroll
                for (int t = 0; t < Q; ++t) v[t] = win[(d + t) % Q];
                const double alpha = qa[d];
                const double nextf = qf[d];                                        // f[j + H + 1]
                if (j + Q < n) qa[d] = __ldcs(pal + (size_t)(j + Q) * stride);
                // f[j + 1 + H + Q] for output j + 1 + Q (only if that output exists)
                if (j + 1 + Q < n) qf[d] = row_value(j + 1 + H + Q, true);
                __stcs(pout + (size_t)j * stride, interp_odd<Q>(alpha, v));
                win[d % Q] = nextf;                                                // slot of f[j - H] becomes f[j + H + 1]
            }
        }
    }
}

// unit-stride dim (inner == 1, always a v dim), extent N compiled in: PB pencils per block, f and alpha transposed
// through two padded shared-memory tiles (odd row pitch: "lane = pencil" accesses are conflict-free; filled by
// asynchronous copies, see below); results overwrite the alpha tile (alpha_j is consumed by the one thread that
// produces out_j).  A pencil is cut into S segments of R = ceil(N/S) outputs, one thread each (the lanes of a warp
// share the segment): a thread holds R+Q-1 values instead of N, so that a block has S times the warps for the same tile.
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
    // fill both tiles with 8-byte asynchronous copies (cp.async): nothing is staged in registers and every copy of
    // every resident block is in flight at once -- with a register-staged fill (4 loads ahead) v3 took 12.0-14.5 ms at
    // 37^6, with this one 8.6-9.9 ms
    for (uint32_t e = threadIdx.x; e < nelem; e += T) {
        const uint32_t s = (e / N) * LD + (e % N);
        const uint32_t df = (uint32_t)__cvta_generic_to_shared(tf + s), da = (uint32_t)__cvta_generic_to_shared(ta + s);
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(df), "l"(pin + e) : "memory");
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(da), "l"(pal + e) : "memory");
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
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
                double v[Q];
#pragma unroll
                for (int m = 0; m < Q; ++m) v[m] = u[r + m];
                rowa[j] = interp_odd<Q>(rowa[j], v);
            }
        }
    }
    __syncthreads();
#pragma unroll 4
    for (uint32_t e = threadIdx.x; e < nelem; e += T) __stcs(pout + e, ta[(e / N) * LD + (e % N)]);
}

// The same with a run-time extent: a.pb pencils per block (a multiple of 32 chosen by the host so that the two tiles
// fit), S = blockDim.x / a.pb segments per pencil, a register window of Q values sliding along the segment.
template <int Q>
__global__ void pointwise_generic_unit_kernel(const PointwiseArgs a) {
    extern __shared__ double tiles[];                      // 2 x pb x ld
    constexpr int H = (Q - 1) / 2;
    const int n = (int)a.n;
    const uint32_t PB = a.pb, LD = a.ld, T = blockDim.x;
    const int S = (int)(T / PB);
    double* tf = tiles;
    double* ta = tiles + (size_t)PB * LD;
    const size_t p0 = (size_t)blockIdx.x * PB;
    const uint32_t np = (uint32_t)(((size_t)a.outer - p0) < (size_t)PB ? ((size_t)a.outer - p0) : (size_t)PB);
    const uint32_t nelem = np * (uint32_t)n;
    const double* pin = a.in + p0 * n;
    const double* pal = a.alpha + p0 * n;
    double* pout = a.out + p0 * n;
    // (row, col) = (e / n, e % n) advanced by (T / n, T % n) per step instead of two run-time divisions per element
    const uint32_t un = (uint32_t)n, dq = T / un, dr = T % un;
    const uint32_t row0 = threadIdx.x / un, col0 = threadIdx.x % un;
    {
        uint32_t row = row0, col = col0;
        for (uint32_t e = threadIdx.x; e < nelem; e += T) {              // asynchronous fill, as above
            const uint32_t s = row * LD + col;
            const uint32_t df = (uint32_t)__cvta_generic_to_shared(tf + s), da = (uint32_t)__cvta_generic_to_shared(ta + s);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(df), "l"(pin + e) : "memory");
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(da), "l"(pal + e) : "memory");
            row += dq;
            col += dr;
            if (col >= un) { col -= un; ++row; }
        }
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
    const uint32_t pl = threadIdx.x % PB;
    const int seg = (int)(threadIdx.x / PB);
    if (pl < np) {
        const int R = (n + S - 1) / S;
        const int j0 = seg * R, j1 = (j0 + R < n) ? j0 + R : n;
        const double* rowf = tf + pl * LD;
        double* rowa = ta + pl * LD;
        auto fetch = [&](int c) -> double { return (c >= 0 && c < n) ? rowf[c] : 0.0; };
        double win[Q];
#pragma unroll
        for (int m = 0; m < Q - 1; ++m) win[m + 1] = fetch(j0 - H + m);
        for (int j = j0; j < j1; ++j) {
#pragma unroll
            for (int m = 0; m < Q - 1; ++m) win[m] = win[m + 1];
            win[Q - 1] = fetch(j + H);
            rowa[j] = interp_odd<Q>(rowa[j], win);
        }
    }
    __syncthreads();
    {
        uint32_t row = row0, col = col0;
        for (uint32_t e = threadIdx.x; e < nelem; e += T) {
            __stcs(pout + e, ta[row * LD + col]);
            row += dq;
            col += dr;
            if (col >= un) { col -= un; ++row; }
        }
    }
}

}  // namespace bsl6d
