// ptile_kernels.cuh -- SURVEY.md 8(f) N1, second generation: a chain of sweeps along TWO dims a < b in ONE pass,
// as a persistent, warp-specialised, TMA-fed pipeline (sm_100a).
//
// Tile = [N_a][N_b][C = 8 contiguous doubles] (64 KB at 32 x 32), the same tile as fused_kernels.cuh, but:
//   * one CTA per SM lives for the whole launch and walks over tiles  blockIdx.x, blockIdx.x + gridDim.x, ...
//   * tiles arrive in a ring of NBUF shared-memory buffers, one cp.async.bulk.tensor.5d per tile (TMA, completion on
//     an mbarrier) -- no register staging, no address math, and a tile is in flight while others are worked on;
//   * two CONSUMER groups of GT threads each take alternate tiles: wait on the tile's `full` barrier, run the whole
//     chain of sweeps in place in shared memory (thread owns a pencil: shifted-order loads into registers, Q-term
//     FMA chains, results back), then one elected thread issues the TMA store and, as soon as the store has read
//     the buffer, the TMA load that refills it (so no producer warp and no `empty` barriers are needed: 16 warps,
//     128 registers each).
// While one group computes, the other computes too and the ring's third buffer is storing / loading: HBM, the fp64
// pipe and the shared-memory pipe overlap instead of taking turns (the round-1 kernels ran 2 lock-stepped blocks per
// SM: load, then compute, then store).
// The shared-memory tile is dense (a TMA box cannot be padded): sweeps along a are bank-conflict free, sweeps along b
// would see 2-way conflicts (two rows 2 KB apart per half-warp); pencil_in_place's `rot` removes them without a second
// pass through shared memory by letting the odd rows run one element ahead.
// Per sweep the arithmetic (split_shift, lagrange_weights, the fma chain) is that of sweep_kernels.cuh, so a pass is
// bit-identical to the same sweeps launched one by one.
#pragma once
#include <cuda.h>

#include "sweep_kernels.cuh"

constexpr auto kPtileRot = 1;
constexpr auto kPtileStream = 1;          // zero-extended pencils: stream through a register window where that is safe
constexpr auto kPtileStreamD = 4;

namespace bsl6d {

constexpr int kMaxPSweeps = 8;
constexpr int kPTileC = 8;                                 // contiguous doubles per tile row

struct PSweep {
    const double* src;
    double scale;
    int32_t along_b;       // 0: sweep along a, 1: along b
    SrcTerms terms;        // in terms of the (outer, inner) index of that sweep's own [outer][N][inner] view
};

struct PTileArgs {
    uint32_t nsweeps;
    uint32_t ntiles;       // outer * mid * nchunks
    uint32_t mid;          // product of the extents of the dims between a and b
    uint32_t inner_b;      // product of the extents of the dims faster than b (a multiple of 8)
    uint32_t nchunks;      // inner_b / 8
    uint32_t pad_;
    PSweep sw[kMaxPSweeps];
};

namespace pt {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t phase) {
    asm volatile(
        "{\n\t"
        ".reg .pred P1;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
        "@P1 bra DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "DONE:\n\t"
        "}" ::"r"(bar), "r"(phase) : "memory");
}
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2,
                                            int c3, int c4) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], "
        "[%2];" ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}
__device__ __forceinline__ void tma_store_5d(const CUtensorMap* map, uint32_t src, int c0, int c1, int c2, int c3,
                                             int c4) {
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5, %6}], [%1];" ::"l"(map),
                 "r"(src), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}
__device__ __forceinline__ double lds_f64(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_f64(uint32_t addr, double v) {
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}
__device__ __forceinline__ void group_sync(int id, int count) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}

// One pencil of N points at shared-memory address `base`, element j at base + j*STRIDE bytes: in place.
// Loads in shifted order (all before the first store), weights, FMA chains: the arithmetic of sweep_strided_kernel.
//
// rot (0 or 1) turns the order in which the thread touches its pencil by one element: with rot = 1 the t-th load
// instruction reads the element AFTER the one a rot = 0 thread reads, and the j-th store writes output j+1.  The
// values are the same; only which instruction moves which element changes.  Sweeps along b pass par = i_a & 1 and get
// rot = (r0 + par) & 1, so that the row a thread touches at instruction t has the parity of i_a + t whatever its
// displacement: the two pencils of a half-warp there lie a whole plane (a multiple of 128 bytes) apart, i.e. in the
// same banks when they touch the same row, and the turn keeps them one 64-byte tile row -- half the banks -- apart.
// The dense tile a TMA box writes is then swept without bank conflicts in both directions (ncu, C2 v1+v2: 1.7e8
// conflict wavefronts of 4.6e8 before).  Periodic pencils: a cyclic turn of the N registers.  Zero-extended pencils
// hold N+Q-1 values u[t] = in[r0 + (t + rot) mod NU]; outputs j+rot come out of registers j..j+Q-1 for j < N-1, and the
// one output left (N-1 for rot = 0, 0 for rot = 1) out of a register set picked by rot.  par < 0: no turn.
// Measured (alternating runs on one box, ms per pass): v1+v2 2.90 -> 2.75 at C2, 11.34 -> 11.08 at C5 -- the passes are
// bound by dependent latency at 16 warps per SM more than by the shared-memory pipe.  For x3+v1 (a periodic) no gain
// could be shown (C2: 3.03 without, 3.56 with the turn in one pair of runs, but the same kernel without the turn also
// measured 3.95 on another box: that pass varies more from run to run than the turn could win), so the turn is applied
// only where a is zero-extended.
template <int N, int Q, bool PERIODIC, uint32_t STRIDE>
__device__ __forceinline__ void pencil_in_place(uint32_t base, double sval, double scale, int par = -1) {
    long long k;
    double theta;
    split_shift(sval, scale, k, theta);
    constexpr int NU = PERIODIC ? N : N + Q - 1;
    double u[NU];
    int rot;
    if (PERIODIC) {
        int r0 = (int)((k + (long long)(1 - Q / 2)) % (long long)N);
        if (r0 < 0) r0 += N;
        rot = par < 0 ? 0 : ((r0 + par) & 1);
        r0 += rot;
        if (r0 >= N) r0 -= N;
#pragma unroll
        for (int t = 0; t < N; ++t) {
            int row = r0 + t;
            if (row >= N) row -= N;
            u[t] = lds_f64(base + (uint32_t)row * STRIDE);
        }
    } else {
        long long kc = k < -(long long)(2 * N + 2 * Q) ? -(long long)(2 * N + 2 * Q) : k;
        kc = kc > (long long)(2 * N + 2 * Q) ? (long long)(2 * N + 2 * Q) : kc;
        const int r0 = (int)kc + (1 - Q / 2);
        rot = par < 0 ? 0 : ((r0 + par) & 1);
        if (kPtileStream && r0 > -Q) {
            // Streaming form (ncu: in the all-loads-first form below the fp64 pipe is the top stall of a pass and yet
            // only half busy -- every warp alternates a burst of shared-memory loads with a burst of DFMAs).  Rows are
            // read in increasing order, D outputs ahead of their first use, and output j (row j + rot) is stored as
            // soon as it is formed: the next row to be read, r0 + j + Q + D + rot, lies above it whenever r0 > -Q, so
            // nothing is overwritten before it is read.  The turn's wrapped element (row r0 for rot = 1) is read
            // first.  Same values, same order of operations per output: bit-identical to the form below.
            // Measured (alternating runs, ms): v1+v2 at C5 10.57 -> 10.27, three shears at C2 3.84 -> 3.75, Strang step
            // at C2 23.1 -> 22.6; look-ahead 2 or 8 instead of 4: no better.
            constexpr int D = kPtileStreamD;
            auto ld = [&](int t) -> double {
                int tt = t + rot;
                if (tt >= NU) tt -= NU;
                const int row = r0 + tt;
                double v = 0.0;
                if (row >= 0 && row < N) v = lds_f64(base + (uint32_t)row * STRIDE);
                return v;
            };
            u[NU - 1] = ld(NU - 1);
#pragma unroll
            for (int t = 0; t < NU - 1 && t < Q - 1 + D; ++t) u[t] = ld(t);
            double w[Q];
            lagrange_weights<Q>(theta, w);
#pragma unroll
            for (int j = 0; j < N - 1; ++j) {
                const int tl = j + Q - 1 + D;
                if (tl < NU - 1) u[tl] = ld(tl);
                double acc = w[0] * u[j];
#pragma unroll
                for (int m = 1; m < Q; ++m) acc = fma(w[m], u[j + m], acc);
                sts_f64(base + (uint32_t)(j + rot) * STRIDE, acc);
            }
            double acc = w[0] * (rot ? u[NU - 1] : u[N - 1]);
#pragma unroll
            for (int m = 1; m < Q; ++m) acc = fma(w[m], rot ? u[m - 1] : u[N - 1 + m], acc);
            sts_f64(base + (uint32_t)(rot ? 0 : N - 1) * STRIDE, acc);
            return;
        }
#pragma unroll
        for (int t = 0; t < NU; ++t) {
            int tt = t + rot;
            if (tt >= NU) tt -= NU;
            const int row = r0 + tt;
            double v = 0.0;
            if (row >= 0 && row < N) v = lds_f64(base + (uint32_t)row * STRIDE);
            u[t] = v;
        }
    }
    double w[Q];
    lagrange_weights<Q>(theta, w);
    if (PERIODIC) {
#pragma unroll
        for (int j = 0; j < N; ++j) {
            double acc = w[0] * u[j % N];
#pragma unroll
            for (int m = 1; m < Q; ++m) acc = fma(w[m], u[(j + m) % N], acc);
            int jo = j + rot;
            if (jo >= N) jo -= N;
            sts_f64(base + (uint32_t)jo * STRIDE, acc);
        }
    } else {
#pragma unroll
        for (int j = 0; j < N - 1; ++j) {
            double acc = w[0] * u[j];
#pragma unroll
            for (int m = 1; m < Q; ++m) acc = fma(w[m], u[j + m], acc);
            sts_f64(base + (uint32_t)(j + rot) * STRIDE, acc);
        }
        // the output left: N-1 from in[r0+N-1+m] = u[N-1+m] (rot = 0), or 0 from in[r0+m] = u[m-1], u[NU-1] for m = 0 (rot = 1)
        double acc = w[0] * (rot ? u[NU - 1] : u[N - 1]);
#pragma unroll
        for (int m = 1; m < Q; ++m) acc = fma(w[m], rot ? u[m - 1] : u[N - 1 + m], acc);
        sts_f64(base + (uint32_t)(rot ? 0 : N - 1) * STRIDE, acc);
    }
}

}  // namespace pt

template <int NA, int NB>
struct PTileGeom {
    static constexpr int C = kPTileC;
    static constexpr int ROW = C * 8;                      // bytes per tile row
    static constexpr int PLANE = NB * ROW;                 // bytes per i_a plane
    static constexpr int TILE = NA * PLANE;                // bytes per tile
    static constexpr int NBUF_ = (220 * 1024) / TILE;
    static constexpr int NBUF = NBUF_ > 4 ? 4 : NBUF_;     // ring depth (3 at 32 x 32)
    static constexpr int GT = (NA > 32 || NB > 32) ? 128 : 256;   // threads per consumer group (register budget)
    static constexpr int THREADS = 2 * GT;                 // two consumer groups (16 warps: 128 registers each)
    static constexpr size_t kSmemBytes = (size_t)NBUF * TILE + 1024;
    static_assert(NBUF >= 2, "tile too large for a ring of two");
};

template <int NA, int NB, int Q, bool PA, bool PB>
__global__ void __launch_bounds__((PTileGeom<NA, NB>::THREADS), 1)
    ptile_kernel(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_out,
                 const __grid_constant__ PTileArgs a) {
    using G = PTileGeom<NA, NB>;
    constexpr int C = G::C, ROW = G::ROW, PLANE = G::PLANE, TILE = G::TILE, NBUF = G::NBUF, GT = G::GT;
    extern __shared__ unsigned char pt_smem_raw[];
    // Completion barriers.  Ring slot b is used for this CTA's tiles b, b+NBUF, b+2*NBUF, ...; with an odd ring the
    // slot alternates between the two consumer groups, and an mbarrier wait only knows the PARITY of the phase it
    // waits for: a group that runs ahead of the other group's load of the previous use would sail through.  Two
    // barriers per slot (even uses, odd uses) make every barrier single-consumer and strictly in order.
    __shared__ __align__(8) unsigned long long pt_bars[2 * NBUF];
    const uint32_t buf0 = (pt::smem_u32(pt_smem_raw) + 1023u) & ~1023u;
    const uint32_t full0 = pt::smem_u32(&pt_bars[0]);
    const uint32_t stride_tiles = gridDim.x;

    // tile id -> TMA coordinates (chunk*C, 0, m, 0, o) and one load of the CTA's i-th tile into ring slot i % NBUF
    auto issue_load = [&](uint32_t i) {
        const uint32_t t = blockIdx.x + i * stride_tiles;
        if (t >= a.ntiles) return;
        const uint32_t b = i % NBUF, use = i / NBUF;
        const uint32_t bar = full0 + 8 * (2 * b + (use & 1));
        const uint32_t ch = t % a.nchunks, om = t / a.nchunks;
        const uint32_t m = om % a.mid, o = om / a.mid;
        pt::mbar_expect_tx(bar, (uint32_t)TILE);
        pt::tma_load_5d(buf0 + b * TILE, &tm_in, bar, (int)(ch * C), 0, (int)m, 0, (int)o);
    };

    if (threadIdx.x == 0) {
#pragma unroll
        for (int b = 0; b < 2 * NBUF; ++b) pt::mbar_init(full0 + 8 * b, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
        for (int b = 0; b < NBUF; ++b) issue_load((uint32_t)b);       // fill the ring
    }
    __syncthreads();

    // ---- consumer groups: group g takes this CTA's tiles g, g+2, g+4, ... ------------------------------------------
    const int g = threadIdx.x >= GT ? 1 : 0;
    const int gt = (int)threadIdx.x - g * GT;
    uint32_t i = (uint32_t)g;
    for (uint32_t t = blockIdx.x + (uint32_t)g * stride_tiles; t < a.ntiles; t += 2 * stride_tiles, i += 2) {
        const uint32_t b = i % NBUF, use = i / NBUF;
        const uint32_t buf = buf0 + b * TILE;
        const uint32_t ch = t % a.nchunks, om = t / a.nchunks;
        const uint32_t m = om % a.mid, o = om / a.mid;
        const uint32_t i0 = ch * C;

        // The shift source of a pencil is a (small, cached) global load at the head of every sweep: a dependent
        // latency of several hundred cycles per sweep with only four warps per scheduler to cover it.  The value for
        // the thread's first pencil of sweep s+1 is therefore fetched while sweep s runs (and the one for sweep 0
        // while the tile is still in flight).
        auto shift_source = [&](uint32_t s, int p) -> double {
            const PSweep& sw = a.sw[s];
            if (!sw.along_b) {
                // pencil (i_b, c) along a: a-view of the array has outer index o, inner index (m*NB + i_b)*inner_b + i
                const uint32_t ib = (uint32_t)p / C, c = (uint32_t)p % C;
                return __ldg(sw.src + src_offset(sw.terms, o, (m * NB + ib) * a.inner_b + i0 + c));
            }
            // pencil (i_a, c) along b: b-view has outer index (o*NA + i_a)*mid + m, inner index i
            const uint32_t ia = (uint32_t)p / C, c = (uint32_t)p % C;
            return __ldg(sw.src + src_offset(sw.terms, (o * NA + ia) * a.mid + m, i0 + c));
        };
        double sval_next = 0.0;
        if (a.nsweeps > 0 && gt < (a.sw[0].along_b ? NA * C : NB * C)) sval_next = shift_source(0, gt);
        pt::mbar_wait(full0 + 8 * (2 * b + (use & 1)), (use >> 1) & 1);

        for (uint32_t s = 0; s < a.nsweeps; ++s) {
            const PSweep& sw = a.sw[s];
            const double sval_first = sval_next;
            if (s + 1 < a.nsweeps && gt < (a.sw[s + 1].along_b ? NA * C : NB * C)) sval_next = shift_source(s + 1, gt);
            if (!sw.along_b) {
                for (int p = gt; p < NB * C; p += GT) {
                    const double sval = p == gt ? sval_first : shift_source(s, p);
                    pt::pencil_in_place<NA, Q, PA, (uint32_t)PLANE>(buf + (uint32_t)p * 8u, sval, sw.scale);
                }
            } else {
                for (int p = gt; p < NA * C; p += GT) {
                    const uint32_t ia = (uint32_t)p / C, c = (uint32_t)p % C;
                    const double sval = p == gt ? sval_first : shift_source(s, p);
                    pt::pencil_in_place<NB, Q, PB, (uint32_t)ROW>(buf + ia * (uint32_t)PLANE + c * 8u, sval, sw.scale, (kPtileRot && !PA) ? (int)(ia & 1u) : -1);
                }
            }
            pt::group_sync(1 + g, GT);
        }
        // generic-proxy writes -> visible to the async proxy, then one bulk store; as soon as the store has read the
        // buffer the same thread refills it with the tile NBUF places further down this CTA's list
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        pt::group_sync(1 + g, GT);
        if (gt == 0) {
            pt::tma_store_5d(&tm_out, buf, (int)i0, 0, (int)m, 0, (int)o);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            issue_load(i + NBUF);
        }
    }
}

}  // namespace bsl6d
