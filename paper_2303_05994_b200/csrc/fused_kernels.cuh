// fused_kernels.cuh -- SURVEY.md 8(f) N1: several consecutive 1-D sweeps over TWO dims a < b in ONE pass.
//
// The Lie-split step applies 1-D sweeps one after another.  Consecutive sweeps that act along
// only two dims a, b (x1 then x2; x3 then v1; the three shears v_a, v_b, v_a of a rotation) touch, for fixed
// values of every other index, one N_a x N_b plane.  A block stages a tile of C such planes that are adjacent in
// memory -- [N_a][N_b][C] doubles, C contiguous -- so that f is read from HBM once and written once for the
// whole group: 16 B/point per PASS instead of per sweep.
//
//   phase "a, global -> smem":  thread (ib, c) loads its column along a from global memory in shifted order into
//                               registers (exactly the strided sweep kernel), sweeps, writes the column into the tile
//   phase "b, smem -> smem":    thread (ia, c) reads its row along b from the tile, sweeps, writes it back in place
//   phase "b, smem -> global":  the same, results streamed to global memory (segments of C contiguous doubles)
//   phase "a, smem -> global":  thread (ib, c) reads its column from the tile, sweeps, streams it out
//
// Patterns: AB = a,b   ABA = a,b,a.  Per sweep the arithmetic (split_shift, lagrange_weights, the fma chain) is the
// one of sweep_kernels.cuh, so a fused pass is bit-identical to the same sweeps launched one by one.
// Shared-memory traffic is 16 B/point for AB and 32 B/point for ABA (the first sweep reads global memory straight
// into registers, the last one writes registers straight to global memory).
// The tile row pitch is N_b*C + PAD doubles with PAD chosen so that both the "lanes along (ib,c)" and the
// "lanes along (ia,c)" access patterns are bank-conflict free for 8-byte words.
// All global loads of a block precede its global stores and blocks own disjoint tiles => f_in == f_out is legal.
#pragma once
#include "sweep_kernels.cuh"

namespace bsl6d {

constexpr int kMaxFused = 3;
enum FusedPattern { kPatAB = 0, kPatABA = 1 };

struct FusedSweep {
    const double* src;
    double scale;
    SrcTerms terms;        // in terms of the (outer, inner) index of that sweep's own [outer][N][inner] view
};

struct FusedArgs {
    const double* in;
    double* out;
    uint32_t mid;          // product of the extents of the dims between a and b
    uint32_t inner_b;      // product of the extents of the dims faster than b  (> 1)
    uint32_t nchunks;      // inner_b / C
    uint32_t pad_;
    FusedSweep sw[kMaxFused];
};

// One pencil: shift -> (k, theta) -> load in shifted order -> weights -> N outputs in res[].
// GLOBAL: streaming loads from global memory; otherwise plain loads (shared memory).
template <int N, int Q, bool PERIODIC, bool GLOBAL>
__device__ __forceinline__ void sweep_pencil(const double* pin, size_t stride, double sval, double scale,
                                             double (&res)[N]) {
    long long k;
    double theta;
    split_shift(sval, scale, k, theta);
    constexpr int NU = PERIODIC ? N : N + Q - 1;
    double u[NU];
    if (PERIODIC) {
        int r0 = (int)((k + (long long)(1 - Q / 2)) % (long long)N);
        if (r0 < 0) r0 += N;
#pragma unroll
        for (int t = 0; t < N; ++t) {
            int row = r0 + t;
            if (row >= N) row -= N;
            u[t] = GLOBAL ? __ldcs(pin + (size_t)row * stride) : pin[(size_t)row * stride];
        }
    } else {
        long long kc = k < -(long long)(2 * N + 2 * Q) ? -(long long)(2 * N + 2 * Q) : k;
        kc = kc > (long long)(2 * N + 2 * Q) ? (long long)(2 * N + 2 * Q) : kc;
        const int r0 = (int)kc + (1 - Q / 2);
#pragma unroll
        for (int t = 0; t < NU; ++t) {
            const int row = r0 + t;
            double v = 0.0;
            if (row >= 0 && row < N) v = GLOBAL ? __ldcs(pin + (size_t)row * stride) : pin[(size_t)row * stride];
            u[t] = v;
        }
    }
    double w[Q];
    lagrange_weights<Q>(theta, w);
#pragma unroll
    for (int j = 0; j < N; ++j) {
        double acc = w[0] * u[PERIODIC ? (j % N) : j];
#pragma unroll
        for (int m = 1; m < Q; ++m) acc = fma(w[m], u[PERIODIC ? ((j + m) % N) : (j + m)], acc);
        res[j] = acc;
    }
}

template <int NA, int NB, int C>
struct FusedGeom {
    static constexpr int gcd_(int x, int y) { return y == 0 ? x : gcd_(y, x % y); }
    static constexpr int T = gcd_(NA, NB) * C;             // threads per block: tiles both pencil sets
    static constexpr int RA = NB * C / T;                  // columns (along a) per thread
    static constexpr int RB = NA * C / T;                  // rows (along b) per thread
    static constexpr int PAD = C >= 16 ? 0 : C;
    static constexpr int LDS = NB * C + PAD;               // tile row pitch (doubles)
    static constexpr size_t kSmemBytes = sizeof(double) * (size_t)NA * LDS;
    static_assert((NB * C) % T == 0 && (NA * C) % T == 0, "threads must tile both pencil sets");
    static_assert(T % 32 == 0 && T <= 1024, "block shape");
};

template <int NA, int NB, int Q, bool PA, bool PB, int C, int PATTERN, int MINB>
__global__ void __launch_bounds__(FusedGeom<NA, NB, C>::T, MINB) sweep_fused_kernel(const FusedArgs a) {
    using G = FusedGeom<NA, NB, C>;
    extern __shared__ double tile[];                       // [NA][LDS]
    constexpr int T = G::T, LDS = G::LDS;

    // block -> (o, m, chunk)
    const uint32_t ch = blockIdx.x % a.nchunks;
    const uint32_t om = blockIdx.x / a.nchunks;            // o * mid + m
    const uint32_t m = om % a.mid;
    const uint32_t o = om / a.mid;
    const size_t strideB = a.inner_b;
    const size_t strideA = (size_t)a.mid * NB * strideB;
    const size_t base = ((size_t)o * NA * a.mid + m) * NB * strideB + (size_t)ch * C;
    const uint32_t i0 = ch * C;

    // ---- sweep 0: along a, global -> tile ------------------------------------------------------------------
#pragma unroll
    for (int r = 0; r < G::RA; ++r) {
        const uint32_t p = r * T + threadIdx.x;            // column index = ib * C + c
        const uint32_t ib = p / C, c = p % C;
        // a-view of the array: outer index o, inner index (m*NB + ib)*inner_b + i
        const uint32_t inner_idx = (m * NB + ib) * a.inner_b + i0 + c;
        const double sval = __ldg(a.sw[0].src + src_offset(a.sw[0].terms, o, inner_idx));
        double res[NA];
        sweep_pencil<NA, Q, PA, true>(a.in + base + (size_t)ib * strideB + c, strideA, sval, a.sw[0].scale, res);
#pragma unroll
        for (int j = 0; j < NA; ++j) tile[j * LDS + p] = res[j];
    }
    __syncthreads();

    // ---- sweep 1: along b ----------------------------------------------------------------------------------------
    if (PATTERN == kPatAB) {
#pragma unroll
        for (int r = 0; r < G::RB; ++r) {
            const uint32_t p = r * T + threadIdx.x;        // row index = ia * C + c
            const uint32_t ia = p / C, c = p % C;
            // b-view: outer index (o*NA + ia)*mid + m, inner index i
            const uint32_t outer_idx = (o * NA + ia) * a.mid + m;
            const double sval = __ldg(a.sw[1].src + src_offset(a.sw[1].terms, outer_idx, i0 + c));
            double res[NB];
            sweep_pencil<NB, Q, PB, false>(tile + ia * LDS + c, (size_t)C, sval, a.sw[1].scale, res);
            double* pout = a.out + base + (size_t)ia * strideA + c;
#pragma unroll
            for (int j = 0; j < NB; ++j) __stcs(pout + (size_t)j * strideB, res[j]);
        }
        return;
    }

    // PATTERN == kPatABA: b in place in the tile (a thread owns its whole row: it has read all of it into registers
    // before it writes any of it back), then a from the tile to global memory
#pragma unroll
    for (int r = 0; r < G::RB; ++r) {
        const uint32_t p = r * T + threadIdx.x;
        const uint32_t ia = p / C, c = p % C;
        const uint32_t outer_idx = (o * NA + ia) * a.mid + m;
        const double sval = __ldg(a.sw[1].src + src_offset(a.sw[1].terms, outer_idx, i0 + c));
        double res[NB];
        sweep_pencil<NB, Q, PB, false>(tile + ia * LDS + c, (size_t)C, sval, a.sw[1].scale, res);
#pragma unroll
        for (int j = 0; j < NB; ++j) tile[ia * LDS + j * C + c] = res[j];
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < G::RA; ++r) {
        const uint32_t p = r * T + threadIdx.x;
        const uint32_t ib = p / C, c = p % C;
        const uint32_t inner_idx = (m * NB + ib) * a.inner_b + i0 + c;
        const double sval = __ldg(a.sw[2].src + src_offset(a.sw[2].terms, o, inner_idx));
        double res[NA];
        sweep_pencil<NA, Q, PA, false>(tile + p, (size_t)LDS, sval, a.sw[2].scale, res);
        double* pout = a.out + base + (size_t)ib * strideB + c;
#pragma unroll
        for (int j = 0; j < NA; ++j) __stcs(pout + (size_t)j * strideA, res[j]);
    }
}

}  // namespace bsl6d
