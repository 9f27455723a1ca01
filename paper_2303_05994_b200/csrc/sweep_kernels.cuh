// sweep_kernels.cuh -- device code of the 1-D advection sweep (sm_100a).
//
// One sweep = for every pencil p along the swept dim:  out[p,j] = sum_m l_m(theta_p) * in[p, j+k_p+m]
// (eq (7), 69-72 eq (5); include/bsl6d.h).  The 6-D array is viewed as [outer][N][inner].
//
// Design: a pencil is owned by exactly ONE thread, which
//   1. evaluates the shift of its pencil (a1) and the q Lagrange weights (a2) in registers,
//   2. loads the whole pencil into registers *in shifted order*: register t holds in[(r0+t) mod N]
//      (periodic) or in[r0+t]-or-zero (zero extension) with r0 = k - q/2 + 1, so the data-dependent
//      displacement k only ever appears in a load ADDRESS,
//   3. forms out[j] = sum_{m'} w[m'] * u[j+m'] with compile-time register indices (fully unrolled) and
//      streams the results out.
// Every element of f is therefore read once and written once (16 B/point), no halo is re-read, and because
// all loads of a pencil precede its stores, f_in == f_out is safe.
//   * strided dims (inner > 1): lanes run along `inner`, so every load/store instruction of a warp is one
//     contiguous 256 B segment per pencil row -- no shared memory at all.
//   * unit-stride dim (inner == 1): a block first transposes T pencils through padded shared memory.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

// Cache hints of the streaming accesses to f (every element is touched once per sweep): evict-first loads and stores.
// f_in == f_out is legal for every sweep, so the f pointers carry no __restrict__ and BSL6D_LD must stay a coherent
// load (never ld.global.nc / __ldg): a thread's loads of its pencil must not be moved past its stores.
#ifndef BSL6D_LD
#define BSL6D_LD __ldcs
#endif
#ifndef BSL6D_ST
#define BSL6D_ST __stcs
#endif

namespace bsl6d {

constexpr int kMaxSrcTerms = 5;
constexpr uint32_t kFlatPencils = 31;                      // SweepArgs::ti_log2 value selecting flattened pencil indexing

// Where a pencil finds its shift source: the array seen along the swept dim is [outer][N][inner]; the source is a
// dense C-order array over a subset of the other dims, so its index is a sum of up to five
// (divide, modulo, stride) terms of the pencil's outer or inner index.
struct SrcTerms {
    uint32_t nterms;       // src index = sum_t ((g_t / below_t) % extent_t) * sstride_t,  g_t = outer or inner index
    uint32_t t_inner[kMaxSrcTerms];   // 1: term decodes the inner index, 0: the outer index
    uint32_t t_below[kMaxSrcTerms];
    uint32_t t_extent[kMaxSrcTerms];  // 0 = slowest term of its group: no wrap needed
    uint32_t t_sstride[kMaxSrcTerms];
};

struct SweepArgs {
    const double* in;
    double* out;
    const double* src;     // shift source (device), indexed by `terms`
    double scale;          // alpha_cells = -(src * scale)
    uint32_t inner;        // product of extents of dims faster than the swept one
    uint32_t outer;        // product of extents of dims slower than the swept one
    uint32_t n;            // extent of the swept dim (== template N in the specialised kernels)
    uint32_t ti_log2;      // strided: threads of a block along `inner` = 1 << ti_log2
    uint32_t nib;          // strided: number of inner chunks (= ceil(inner / TI)); flattened mode: number of pencils
    SrcTerms terms;
    const double* left;    // sweep_stream_kernel<.., PEER = true> only: the ring neighbours' arrays (same shape as `in`)
    const double* right;
};

// ---- a2: Lagrange basis on the nodes m_i = i - Q/2 + 1, i = 0..Q-1 ------------------------------------------
// w_i = prod_{j != i} (theta - m_j) / prod_{j != i} (m_i - m_j).  Numerators by prefix/suffix products
// (3Q multiplies), denominators (-1)^(Q-1-i) i! (Q-1-i)! folded into compile-time reciprocals.  theta == 0 and
// theta == 1 are mapped to exact unit vectors so that integer-cell shifts are exact permutations (reading S11).
template <int Q>
struct LagrangeDen {
    double r[Q];
    constexpr LagrangeDen() : r() {
        for (int i = 0; i < Q; ++i) {
            double d = 1.0;
            for (int j = 0; j < Q; ++j)
                if (j != i) d *= (double)(i - j);
            r[i] = 1.0 / d;
        }
    }
};

template <int Q>
__device__ __forceinline__ void lagrange_weights(double theta, double (&w)[Q]) {
    constexpr LagrangeDen<Q> den{};
    double d[Q], pre[Q], suf[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) d[i] = theta - (double)(i - Q / 2 + 1);
    pre[0] = 1.0;
#pragma unroll
    for (int i = 1; i < Q; ++i) pre[i] = pre[i - 1] * d[i - 1];
    suf[Q - 1] = 1.0;
#pragma unroll
    for (int i = Q - 2; i >= 0; --i) suf[i] = suf[i + 1] * d[i + 1];
    const bool at0 = (theta == 0.0), at1 = (theta == 1.0);
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        double v = (pre[i] * suf[i]) * den.r[i];
        if (at0) v = (i == Q / 2 - 1) ? 1.0 : 0.0;
        if (at1) v = (i == Q / 2) ? 1.0 : 0.0;
        w[i] = v;
    }
}

// ---- a1: displacement of one pencil -> integer part k and fraction theta -----------------------------------
__device__ __forceinline__ void split_shift(double a, double scale, long long& k, double& theta) {
    const double alpha = -(a * scale);
    double kf = floor(alpha);
    theta = alpha - kf;                                   // exact; in [0,1]
    kf = fmin(fmax(kf, -4.0e18), 4.0e18);
    k = (long long)kf;
}

__device__ __forceinline__ uint32_t src_offset(const SrcTerms& a, uint32_t o, uint32_t i) {
    uint32_t off = 0;
    for (uint32_t t = 0; t < a.nterms; ++t) {
        uint32_t g = a.t_inner[t] ? i : o;
        if (a.t_below[t] != 1u) g /= a.t_below[t];
        if (a.t_extent[t] != 0u) g %= a.t_extent[t];
        off += g * a.t_sstride[t];
    }
    return off;
}

// ---- a4: strided sweep, one column per thread, no shared memory --------------------------------------------
// S > 1 cuts a pencil into S segments of R = N/S outputs, one thread each (the threads of a pencil sit in different
// warps of the same block): a thread then holds R+Q-1 instead of N values, which keeps long pencils with wide
// stencils (N = 48, Q = 10) under the register budget of 4 resident blocks per SM.  The Q-1 rows two neighbouring
// segments share are loaded by both threads (L1/L2 hits, never HBM); a block barrier between the load and the store
// phase keeps f_in == f_out legal.
template <int N, int Q, bool PERIODIC, int T, int MINB, int S = 1>
__global__ void __launch_bounds__(T, MINB) sweep_strided_kernel(const SweepArgs a) {
    static_assert(N % S == 0 && T % S == 0, "segments must tile the pencil and the block");
    constexpr int TP = T / S;                              // pencils per block
    constexpr int R = N / S;                               // outputs per thread
    const uint32_t tp = S == 1 ? threadIdx.x : threadIdx.x % TP;
    const int seg = S == 1 ? 0 : (int)(threadIdx.x / TP);
    uint32_t i, o;
    bool live;
    if (a.ti_log2 == kFlatPencils) {
        // `inner` is not a multiple of the warp width (37^k): lanes run along the flattened pencil index so that
        // every lane has work; a warp then covers the tail of one row segment and the head of the next
        const uint32_t p = blockIdx.x * TP + tp;
        live = p < a.nib;                                   // nib = number of pencils in this mode
        o = p / a.inner;
        i = p - o * a.inner;
    } else {
        const uint32_t ti_mask = (1u << a.ti_log2) - 1u;
        const uint32_t bo = blockIdx.x / a.nib;
        const uint32_t bi = blockIdx.x - bo * a.nib;
        i = (bi << a.ti_log2) + (tp & ti_mask);
        o = bo * (TP >> a.ti_log2) + (tp >> a.ti_log2);
        live = i < a.inner && o < a.outer;
    }
    if (S == 1 && !live) return;

    long long k = 0;
    double theta = 0.0;
    if (live) split_shift(__ldg(a.src + src_offset(a.terms, o, i)), a.scale, k, theta);

    const size_t stride = a.inner;
    const size_t base = (size_t)o * N * stride + i;
    const double* pin = a.in + base;
    double* pout = a.out + base;

    constexpr int NU = (PERIODIC && S == 1) ? N : R + Q - 1;
    static_assert(NU <= N || !PERIODIC, "a segment's window must not wrap onto itself");
    double u[NU];
    if (live) {
        if (PERIODIC) {
            int r0 = (int)((k + (long long)(1 - Q / 2 + seg * R)) % (long long)N);
            if (r0 < 0) r0 += N;
#pragma unroll
            for (int t = 0; t < NU; ++t) {
                int row = r0 + t;
                if (row >= N) row -= N;
                u[t] = BSL6D_LD(pin + (size_t)row * stride);
            }
        } else {
            // rows r0 .. r0+R+Q-2; anything outside [0,N) is the zero extension
            long long kc = k < -(long long)(2 * N + 2 * Q) ? -(long long)(2 * N + 2 * Q) : k;
            kc = kc > (long long)(2 * N + 2 * Q) ? (long long)(2 * N + 2 * Q) : kc;
            const int r0 = (int)kc + (1 - Q / 2) + seg * R;
#pragma unroll
            for (int t = 0; t < NU; ++t) {
                const int row = r0 + t;
                u[t] = (row >= 0 && row < N) ? BSL6D_LD(pin + (size_t)row * stride) : 0.0;
            }
        }
    }
    if (S > 1) __syncthreads();                            // every segment of a pencil has loaded before any stores
    if (!live) return;

    double w[Q];
    lagrange_weights<Q>(theta, w);

#pragma unroll
    for (int j = 0; j < R; ++j) {
        double acc = w[0] * u[(PERIODIC && S == 1) ? (j % N) : j];
#pragma unroll
        for (int m = 1; m < Q; ++m) acc = fma(w[m], u[(PERIODIC && S == 1) ? ((j + m) % N) : (j + m)], acc);
        BSL6D_ST(pout + (size_t)(seg * R + j) * stride, acc);
    }
}

// ---- a4, out of place: the same sweep with the pencil STREAMED through a register window --------------------
// Only for f_in != f_out (an output row may be stored before the input rows behind it have been read).  A thread still
// owns a pencil, but holds Q-1+D+1 of its values at a time instead of all N: row t (in shifted order) is loaded D
// outputs before the first output that needs it, the stores in between keep the loads where they are written.  For
// long pencils with wide stencils (N = 48, Q = 10: 162-168 registers, 12 warps per SM in sweep_strided_kernel) this
// roughly halves the registers.  Periodic pencils keep their first Q-1 rows for the wrap at the end.  Arithmetic and
// its order are those of sweep_strided_kernel: bit-identical results.
// PEER = true (x1 sweep of a slab, outer == 1, see sweep_peer_kernel below): the N planes of the slab continue into the
// neighbours' arrays -- virtual plane r < 0 is plane r+N of a.left, r >= N is plane r-N of a.right -- so the only
// change is WHERE a row is loaded from; there is no wrap (PERIODIC must be false) and no zero fill within one slab width.
template <int N, int Q, bool PERIODIC, int T, int MINB, int D, bool PEER = false>
__global__ void __launch_bounds__(T, MINB) sweep_stream_kernel(const SweepArgs a) {
    static_assert(!(PEER && PERIODIC), "a slab's pencil does not wrap: it continues into its neighbours");
    const uint32_t tp = threadIdx.x;
    uint32_t i, o;
    bool live;
    if (a.ti_log2 == kFlatPencils) {
        const uint32_t p = blockIdx.x * T + tp;
        live = p < a.nib;
        o = p / a.inner;
        i = p - o * a.inner;
    } else {
        const uint32_t ti_mask = (1u << a.ti_log2) - 1u;
        const uint32_t bo = blockIdx.x / a.nib;
        const uint32_t bi = blockIdx.x - bo * a.nib;
        i = (bi << a.ti_log2) + (tp & ti_mask);
        o = bo * (T >> a.ti_log2) + (tp >> a.ti_log2);
        live = i < a.inner && o < a.outer;
    }
    if (!live) return;
    long long k;
    double theta;
    split_shift(__ldg(a.src + src_offset(a.terms, o, i)), a.scale, k, theta);
    const size_t stride = a.inner;
    const size_t base = (size_t)o * N * stride + i;
    const double* pin = a.in + base;
    double* pout = a.out + base;
    int r0;
    if (PERIODIC) {
        r0 = (int)((k + (long long)(1 - Q / 2)) % (long long)N);
        if (r0 < 0) r0 += N;
    } else {
        long long kc = k < -(long long)(2 * N + 2 * Q) ? -(long long)(2 * N + 2 * Q) : k;
        kc = kc > (long long)(2 * N + 2 * Q) ? (long long)(2 * N + 2 * Q) : kc;
        r0 = (int)kc + (1 - Q / 2);
    }
    auto load_row = [&](int t) -> double {                 // shifted row t = 0 .. N+Q-2
        int row = r0 + t;
        if (PERIODIC) {
            if (row >= N) row -= N;
            return BSL6D_LD(pin + (size_t)row * stride);
        }
        if (PEER) {                                        // outer == 1: the pencil's offset in every array is i
            if (row < -N || row >= 2 * N) return 0.0;
            const double* b = row < 0 ? a.left + (size_t)(row + N) * stride
                                      : (row >= N ? a.right + (size_t)(row - N) * stride : a.in + (size_t)row * stride);
            return BSL6D_LD(b + i);
        }
        return (row >= 0 && row < N) ? BSL6D_LD(pin + (size_t)row * stride) : 0.0;
    };
    // u[t], t = 0 .. N+Q-2: fully unrolled, each element lives from its load to its last use; periodic: u[N+t] is u[t]
    constexpr int NU = N + Q - 1;
    constexpr int NL = PERIODIC ? N : NU;                  // rows that are loaded
    double u[NU];
#pragma unroll
    for (int t = 0; t < NL && t < Q - 1 + D; ++t) u[t] = load_row(t);
    double w[Q];
    lagrange_weights<Q>(theta, w);
#pragma unroll
    for (int j = 0; j < N; ++j) {
        const int tl = j + Q - 1 + D;
        if (tl < NL) u[tl] = load_row(tl);
        double acc = w[0] * u[(PERIODIC && j >= N) ? j - N : j];
#pragma unroll
        for (int m = 1; m < Q; ++m) acc = fma(w[m], u[(PERIODIC && j + m >= N) ? j + m - N : j + m], acc);
        BSL6D_ST(pout + (size_t)j * stride, acc);
    }
}

// ---- a3: unit-stride sweep (swept dim is the contiguous one; always a v dim => zero extension) -------------
// A block owns PB = T/S consecutive pencils = one contiguous chunk of PB*N doubles.  Coalesced load -> padded
// smem (row stride N+1 doubles: conflict-free for "lane = pencil" access).  A pencil is cut into S segments of
// R = N/S outputs; thread (pencil p, segment s) reads the R+Q-1 inputs of its segment in shifted order into
// registers (all lanes of a warp share s, so every smem access of a warp is conflict-free), forms its R outputs,
// and after a barrier writes them back into the same smem row -> coalesced store.  S > 1 keeps the register
// window small for long pencils (N = 48, 64) so that >= 3-4 blocks stay resident per SM and overlap their
// load / compute / store phases.
template <int N, int Q, int S, int T, int MINB, bool ASYNC = false>
__global__ void __launch_bounds__(T, MINB) sweep_unit_kernel(const SweepArgs a) {
    static_assert(N % S == 0 && T % (32 * S) == 0, "segments must tile the pencil and the block");
    extern __shared__ double tile[];                       // PB * LD
    constexpr int LD = N | 1;                              // odd row pitch: "lane = pencil" accesses are conflict-free
    constexpr int PB = T / S;                              // pencils per block
    constexpr int R = N / S;                               // outputs per thread
    constexpr int NE = PB * N;                             // elements per full block
    const size_t p0 = (size_t)blockIdx.x * PB;             // first pencil of this block
    const uint32_t np = (uint32_t)(((size_t)a.outer - p0) < (size_t)PB ? ((size_t)a.outer - p0) : (size_t)PB);
    const double* pin = a.in + p0 * N;
    double* pout = a.out + p0 * N;
    const uint32_t nelem = np * N;

    // thread -> (pencil, segment): warp w serves segment w % S of pencils 32*(w/S) .. 32*(w/S)+31
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    const uint32_t seg = warp % S;
    const uint32_t pl = (warp / S) * 32u + lane;           // pencil within the block

    // shift source first: its latency overlaps the tile load
    double sval = 0.0;
    if (pl < np) sval = __ldg(a.src + src_offset(a.terms, (uint32_t)(p0 + pl), 0u));

    if (ASYNC) {
        // 8-byte asynchronous copies instead of loads staged in registers: measured +4 to +7 % for N = 64 (where the
        // freed registers also allow 6 instead of 4 blocks per SM) and N = 32 with q = 8, -1.6 % for N = 32 with q = 10
#pragma unroll
        for (int it = 0; it < (NE + T - 1) / T; ++it) {
            const uint32_t e = it * T + threadIdx.x;
            if (e < nelem) {
                const uint32_t dst = (uint32_t)__cvta_generic_to_shared(tile + (e / N) * LD + (e % N));
                asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(pin + e) : "memory");
            }
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
    } else {
#pragma unroll
        for (int it = 0; it < (NE + T - 1) / T; ++it) {
            const uint32_t e = it * T + threadIdx.x;
            if (e < nelem) tile[(e / N) * LD + (e % N)] = __ldcs(pin + e);
        }
    }
    __syncthreads();

    double res[R];
    if (pl < np) {
        long long k;
        double theta;
        split_shift(sval, a.scale, k, theta);
        long long kc = k < -(long long)(2 * N + 2 * Q) ? -(long long)(2 * N + 2 * Q) : k;
        kc = kc > (long long)(2 * N + 2 * Q) ? (long long)(2 * N + 2 * Q) : kc;
        const int r0 = (int)kc + (1 - Q / 2) + (int)seg * R;
        const double* row = tile + pl * LD;
        constexpr int NU = R + Q - 1;
        double u[NU];
#pragma unroll
        for (int t = 0; t < NU; ++t) {
            const int c = r0 + t;
            u[t] = (c >= 0 && c < N) ? row[c] : 0.0;
        }
        double w[Q];
        lagrange_weights<Q>(theta, w);
#pragma unroll
        for (int j = 0; j < R; ++j) {
            double acc = w[0] * u[j];
#pragma unroll
            for (int m = 1; m < Q; ++m) acc = fma(w[m], u[j + m], acc);
            res[j] = acc;
        }
    }
    if (S > 1) __syncthreads();                            // other segments of my row may still be reading it
    if (pl < np) {
        double* row = tile + pl * LD + seg * R;
#pragma unroll
        for (int j = 0; j < R; ++j) row[j] = res[j];
    }
    __syncthreads();

#pragma unroll
    for (int it = 0; it < (NE + T - 1) / T; ++it) {
        const uint32_t e = it * T + threadIdx.x;
        if (e < nelem) __stcs(pout + e, tile[(e / N) * LD + (e % N)]);
    }
}

// ---- fallback for extents without a specialised instance (any n, even q <= 12) -------------------------------
// One pencil per thread, lanes along the flattened pencil index (full lane use for any `inner`).  The column is
// staged in shared memory as tile[row * T + tid] (all n loads in flight, and f_in == f_out stays legal), then a
// register window of Q values slides along it: one shared-memory read and Q FMAs per output, the same
// split_shift / lagrange_weights / fma order as the specialised kernels (so the numbers are bit-identical).
template <int Q, int T>
__global__ void __launch_bounds__(T) sweep_generic_kernel(const SweepArgs a, int periodic) {
    extern __shared__ double tile[];                       // n * T
    const uint32_t p = blockIdx.x * T + threadIdx.x;
    if (p >= a.inner * a.outer) return;
    const uint32_t o = p / a.inner, i = p - o * a.inner;
    const int n = (int)a.n;
    long long k;
    double theta;
    split_shift(__ldg(a.src + src_offset(a.terms, o, i)), a.scale, k, theta);
    const size_t stride = a.inner;
    const size_t base = (size_t)o * n * stride + i;
    double* col = tile + threadIdx.x;
    {   // 8-byte asynchronous copies: all n rows of the column in flight, nothing staged in registers
        const uint32_t dcol = (uint32_t)__cvta_generic_to_shared(col);
        const double* src = a.in + base;
        for (int r = 0; r < n; ++r)
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dcol + (uint32_t)(r * T * 8)), "l"(src + (size_t)r * stride) : "memory");
        asm volatile("cp.async.wait_all;" ::: "memory");       // a thread reads only what it copied itself
    }

    double w[Q];
    lagrange_weights<Q>(theta, w);

    // row of the first stencil node of output 0, then advanced by one per output
    long long kk = k + (long long)(1 - Q / 2);
    int row;
    if (periodic) {
        kk %= n;
        if (kk < 0) kk += n;
        row = (int)kk;
    } else {
        const long long lim = 2LL * n + 32;
        kk = kk < -lim ? -lim : (kk > lim ? lim : kk);
        row = (int)kk;
    }
    auto fetch = [&](int r) -> double {
        if (periodic) return col[r * T];
        return (r >= 0 && r < n) ? col[r * T] : 0.0;
    };
    auto next = [&](int r) -> int {
        ++r;
        if (periodic && r >= n) r -= n;
        return r;
    };
    double win[Q];
#pragma unroll
    for (int m = 0; m < Q - 1; ++m) {
        win[m + 1] = fetch(row);                             // win[1..Q-1] primed; shifted down in the loop
        row = next(row);
    }
    for (int j = 0; j < n; ++j) {
#pragma unroll
        for (int m = 0; m < Q - 1; ++m) win[m] = win[m + 1];
        win[Q - 1] = fetch(row);
        row = next(row);
        double acc = w[0] * win[0];
#pragma unroll
        for (int m = 1; m < Q; ++m) acc = fma(w[m], win[m], acc);
        __stcs(a.out + base + (size_t)j * stride, acc);
    }
}

// ---- x1 sweep of a SLAB whose neighbours' planes are read where they are ---------------
// The slab holds planes 0..n-1 of its part of dim 0; the w planes below come from the END of `left`'s array and the
// w planes above from the START of `right`'s (both arrays have the slab's own shape: n planes).  left / right may be
// peer memory of another GPU (loads travel over NVLink: the halo "exchange" IS the sweep's own loads -- no halo
// planes, no copy, no separate communication step), arrays of other slabs on the same device, or `in` itself (one
// slab: the periodic ring closes on itself).  Out of place only: the neighbours read this slab's input meanwhile.
// Structure and arithmetic of sweep_generic_kernel (pencil staged in shared memory by cp.async, sliding register
// window): results are bit-identical to the periodic sweep on the undivided grid as long as no foot lies more than
// w - q/2 cells away (the caller's promise, as for halo planes; rows beyond the staged range read as zero).
struct PeerArgs {
    const double* in;
    const double* left;
    const double* right;
    double* out;
    const double* src;
    double scale;
    uint32_t inner;        // product of the extents of dims 1..5
    uint32_t n;            // planes of this slab
    uint32_t w;            // neighbour planes staged on either side (<= n)
    uint32_t pad_;
    SrcTerms terms;
};

template <int Q, int T>
__global__ void __launch_bounds__(T) sweep_peer_kernel(const PeerArgs a) {
    extern __shared__ double tile[];                       // (n + 2w) * T
    const uint32_t i = blockIdx.x * T + threadIdx.x;
    if (i >= a.inner) return;
    const int n = (int)a.n, w = (int)a.w;
    long long k;
    double theta;
    split_shift(__ldg(a.src + src_offset(a.terms, 0u, i)), a.scale, k, theta);
    const size_t stride = a.inner;
    double* col = tile + threadIdx.x;
    {
        const uint32_t dcol = (uint32_t)__cvta_generic_to_shared(col);
        for (int r = -w; r < n + w; ++r) {                 // virtual plane r -> whose array, which plane
            const double* src = r < 0 ? a.left + (size_t)(r + n) * stride
                                      : (r >= n ? a.right + (size_t)(r - n) * stride : a.in + (size_t)r * stride);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dcol + (uint32_t)((r + w) * T * 8)), "l"(src + i) : "memory");
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
    }
    double wgt[Q];
    lagrange_weights<Q>(theta, wgt);
    const long long lim = 2LL * n + 32;
    long long kk = k + (long long)(1 - Q / 2);
    kk = kk < -lim ? -lim : (kk > lim ? lim : kk);
    int row = (int)kk;                                      // virtual plane of the first stencil node of output 0
    auto fetch = [&](int r) -> double { return (r >= -w && r < n + w) ? col[(r + w) * T] : 0.0; };
    double win[Q];
#pragma unroll
    for (int m = 0; m < Q - 1; ++m) win[m + 1] = fetch(row++);
    for (int j = 0; j < n; ++j) {
#pragma unroll
        for (int m = 0; m < Q - 1; ++m) win[m] = win[m + 1];
        win[Q - 1] = fetch(row++);
        double acc = wgt[0] * win[0];
#pragma unroll
        for (int m = 1; m < Q; ++m) acc = fma(wgt[m], win[m], acc);
        __stcs(a.out + (size_t)j * stride + i, acc);
    }
}

// The same for the unit-stride dim (inner == 1; always a v dim => zero extension): a block owns PB consecutive
// pencils = one contiguous chunk, moved coalesced through two shared-memory tiles (input rows, output rows) with an
// odd row pitch, so that "lane = pencil" accesses are conflict-free.  A pencil is cut into S segments of
// ceil(n/S) outputs, one thread each (the lanes of a warp share the segment), which gives a block S times the warps
// for the same tile (with one thread per pencil the kernel ran 10 warps per SM: 3.4 TB/s at 36^6).
// Round 2 (second half): ONE tile instead of two.  The number of segments per pencil is chosen at launch so that a
// thread forms at most RMAX = 16 (n <= 256; else 32) outputs (S = ceil(n / RMAX) = blockDim.x / PB); it keeps them in registers (fully
// unrolled, predicated), and after a barrier -- every segment of a row has read its inputs -- writes them over the
// row.  Half the shared memory per block (twice the resident blocks) and no second tile to fill.
template <int Q, int PB, int RMAX>
__global__ void __launch_bounds__(512) sweep_generic_unit_kernel(const SweepArgs a) {
    extern __shared__ double tile[];                       // PB * LD
    const uint32_t T = blockDim.x;                         // PB * S
    const int S = (int)(T / PB);
    const int n = (int)a.n;
    const int LD = n | 1;
    const size_t p0 = (size_t)blockIdx.x * PB;
    const uint32_t np = (uint32_t)(((size_t)a.outer - p0) < (size_t)PB ? ((size_t)a.outer - p0) : (size_t)PB);
    const uint32_t nelem = np * (uint32_t)n;
    const double* pin = a.in + p0 * n;
    double* pout = a.out + p0 * n;
    // element e of the chunk sits at (row, col) = (e / n, e % n): with a run-time n these two divisions per element and
    // loop (fill, store) were the kernel's largest cost (~80 of its instructions per point), so (row, col) is advanced
    // by (T / n, T % n) instead -- two divisions per thread
    const uint32_t un = (uint32_t)n, dq = T / un, dr = T % un;
    const uint32_t row0 = threadIdx.x / un, col0 = threadIdx.x % un;
    {
        uint32_t row = row0, col = col0;
        for (uint32_t e = threadIdx.x; e < nelem; e += T) {
            const uint32_t dst = (uint32_t)__cvta_generic_to_shared(tile + row * LD + col);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(pin + e) : "memory");
            row += dq;
            col += dr;
            if (col >= un) { col -= un; ++row; }
        }
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
    const uint32_t pl = threadIdx.x % PB;
    const int seg = (int)(threadIdx.x / PB);
    const int R = (n + S - 1) / S;                         // <= RMAX by the choice of S
    const int j0 = seg * R, j1 = (j0 + R < n) ? j0 + R : n;
    double res[RMAX];
    if (pl < np && j0 < n) {
        long long k;
        double theta;
        split_shift(__ldg(a.src + src_offset(a.terms, (uint32_t)(p0 + pl), 0u)), a.scale, k, theta);
        double w[Q];
        lagrange_weights<Q>(theta, w);
        const long long lim = 2LL * n + 32;
        long long kk = k + (long long)(1 - Q / 2);
        kk = kk < -lim ? -lim : (kk > lim ? lim : kk);
        int row = (int)kk + j0;                            // first stencil node of output j0
        const double* rin = tile + pl * LD;
        double win[Q];                                     // ring with static indices: win[(r + m) % Q] = node m of output j0 + r
#pragma unroll
        for (int m = 0; m < Q - 1; ++m) {
            win[m] = (row >= 0 && row < n) ? rin[row] : 0.0;
            ++row;
        }
#pragma unroll
        for (int r = 0; r < RMAX; ++r) {
            if (j0 + r < j1) {
                win[(r + Q - 1) % Q] = (row >= 0 && row < n) ? rin[row] : 0.0;
                ++row;
                double acc = w[0] * win[r % Q];
#pragma unroll
                for (int m = 1; m < Q; ++m) acc = fma(w[m], win[(r + m) % Q], acc);
                res[r] = acc;
            }
        }
    }
    __syncthreads();                                       // every segment of every row has read its inputs
    if (pl < np && j0 < n) {
        double* rout = tile + pl * LD + j0;
#pragma unroll
        for (int r = 0; r < RMAX; ++r)
            if (j0 + r < j1) rout[r] = res[r];
    }
    __syncthreads();
    {
        uint32_t row = row0, col = col0;
        for (uint32_t e = threadIdx.x; e < nelem; e += T) {
            __stcs(pout + e, tile[row * LD + col]);
            row += dq;
            col += dr;
            if (col >= un) { col -= un; ++row; }
        }
    }
}

}  // namespace bsl6d
