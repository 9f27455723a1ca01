// vblock_kernels.cuh -- SURVEY.md 8(f) N1: EVERY velocity-space sweep of a step in ONE pass over f (sm_100a).
//
// In C order each x-point owns one contiguous block of nv1*nv2*nv3 doubles (256 KB at 32^3), and the whole v-part of
// the Lie chain -- the three E-sweeps v1,v2,v3 and the shears of the rotation -- acts inside it.
// A thread-block CLUSTER of CL CTAs stages one x-point's v-block on chip, cut along v3: CTA r holds
//     tile[j1][j2][c],  c = 0..CW-1  <->  j3 = r*CW + c,   CW = NV/CL      (64 KB per CTA at 32^3 with CL = 4)
// fetched by ONE TMA bulk-tensor copy (cp.async.bulk.tensor.4d + mbarrier; no register staging), and written back
// by one TMA store.  All sweeps run in place in shared memory: HBM traffic is 16 B/point for the whole group.
//
//   v1 / v2 sweeps  thread owns the pencil (j2,c) / (j1,c): whole pencil -> registers in shifted order ->
//                   Q-term FMA chains -> back into the tile.  Entirely CTA-local.
//   v3 sweeps       the pencil crosses the cluster.  Default: the block is RE-TILED THROUGH L2 into the other cut
//                   (each CTA: a quarter of the j1-planes, all of v3) by TMA stores / cluster barrier / TMA loads, the
//                   sweep runs locally, and the block is re-tiled back.  Alternative (V3PATH = kV3ViaDsmem): the
//                   CW+Q-1 inputs are read through distributed shared memory (mapa + ld.shared::cluster) from
//                   whichever CTA owns the column.  Both are measured slower than a v3 pass of its own (section 10).
//
// The tile rows are CW*8 = 64 or 128 bytes, written by the TMA with the matching 64B / 128B swizzle (16-byte chunk
// index XOR row bits), which is what makes the v3 sweeps (lanes along rows) and the v1/v2 sweeps (lanes along c)
// both bank-conflict-light without padding -- TMA boxes cannot be padded.
// Per sweep the arithmetic (split_shift, lagrange_weights, the fma chain) is that of sweep_kernels.cuh, so a pass is
// bit-identical to the same sweeps launched one by one.
#pragma once
#include <cuda.h>
#include <cooperative_groups.h>

#include "sweep_kernels.cuh"

namespace bsl6d {

constexpr int kMaxVSweeps = 12;

struct VSweep {
    const double* src;
    double scale;
    int32_t dim;           // 3, 4 or 5
    SrcTerms terms;        // in terms of the (outer, inner) index of that sweep's own [outer][N][inner] view
};

struct VBlockArgs {
    uint32_t nsweeps;
    uint32_t nx;           // number of x-points = number of v-blocks
    VSweep sw[kMaxVSweeps];
};

namespace vb {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
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
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2,
                                            int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_store_4d(const CUtensorMap* map, uint32_t src, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];" ::"l"(map),
                 "r"(src), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ double lds_f64(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_f64(uint32_t addr, double v) {
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}
// read a double of CTA `rank`'s shared memory at this CTA's address `addr` (distributed shared memory)
__device__ __forceinline__ double ld_cluster_f64(uint32_t addr, uint32_t rank) {
    uint32_t ra;
    double v;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(addr), "r"(rank));
    asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(v) : "r"(ra));
    return v;
}

// Outputs j0 .. j0+NOUT-1 of a zero-extended pencil of N points: load the NOUT+Q-1 inputs in shifted order through
// `ld(row)` (row in [0,N) guaranteed), weights, FMA chains -- the arithmetic of sweep_pencil<N,Q,false,...>.
template <int N, int NOUT, int Q, class Load>
__device__ __forceinline__ void window_sweep(double sval, double scale, int j0, Load&& ld, double (&res)[NOUT]) {
    long long k;
    double theta;
    split_shift(sval, scale, k, theta);
    long long kc = k < -(long long)(2 * N + 2 * Q) ? -(long long)(2 * N + 2 * Q) : k;
    kc = kc > (long long)(2 * N + 2 * Q) ? (long long)(2 * N + 2 * Q) : kc;
    const int r0 = (int)kc + (1 - Q / 2) + j0;
    constexpr int NU = NOUT + Q - 1;
    double u[NU];
#pragma unroll
    for (int t = 0; t < NU; ++t) {
        const int row = r0 + t;
        double v = 0.0;
        if (row >= 0 && row < N) v = ld(row);
        u[t] = v;
    }
    double w[Q];
    lagrange_weights<Q>(theta, w);
#pragma unroll
    for (int j = 0; j < NOUT; ++j) {
        double acc = w[0] * u[j];
#pragma unroll
        for (int m = 1; m < Q; ++m) acc = fma(w[m], u[j + m], acc);
        res[j] = acc;
    }
}

}  // namespace vb

template <int NV, int CL>
struct VBlockGeom {
    static constexpr int CW = NV / CL;                     // columns (v3 values) per CTA
    static constexpr int RB = CW * 8;                      // tile row bytes: 64 or 128 (= the TMA swizzle span)
    static constexpr uint32_t SWZ = RB == 128 ? 7u : 3u;   // 16-byte chunk index ^= row bits & SWZ
    static constexpr int PLANE = NV * RB;                  // bytes per j1 plane
    static constexpr int TILE = NV * PLANE;                // bytes per CTA tile
    static constexpr int T = NV * CW < 512 ? (NV * CW < 32 ? 32 : NV * CW) : 512;   // threads per CTA: one per v1/v2 pencil
    static constexpr size_t kSmemBytes = (size_t)TILE + 1024;   // + alignment slack (swizzle pattern repeats at 1 KB)
    static_assert(NV % CL == 0 && (RB == 64 || RB == 128), "tile rows must be 64 or 128 bytes");
    static_assert(PLANE % 1024 == 0 || (RB == 64 && PLANE % 512 == 0), "j1 planes must not disturb the swizzle bits");
};

// How a v3 sweep is served when the v-block is cut along v3 over CL > 1 CTAs:
//   kV3ViaL2   (default) RE-TILE THROUGH L2.  The cluster stores its four [j1][j2][c] tiles (TMA store to f_out, which
//              lands in the 126 MB L2), synchronises, and every CTA loads the block again in the OTHER cut --
//              [its NV/CL j1-planes][j2][all of v3], two TMA boxes of 128-byte half rows with the 128B swizzle -- runs the
//              v3 sweep entirely locally (thread owns a row), stores, synchronises, and loads its [j1][j2][c] tile
//              back.  Two extra round trips through L2 per v3 sweep (32 B/point of L2 traffic, none to HBM: the lines
//              are still dirty in L2 and are overwritten there), all by bulk tensor copies.
//   kV3ViaDsmem          the pencil's CW+Q-1 inputs are read from whichever CTA owns them through distributed shared
//              memory (mapa + ld.shared::cluster) between cluster barriers.  Measured ~3 clk per scattered 8-byte
//              request on B200: ~9 ms per v3 sweep at C2.  Kept for comparison.
enum V3Path { kV3ViaL2 = 0, kV3ViaDsmem = 1 };

template <int NV, int Q, int CL, int MINB, int V3PATH>
__global__ void __cluster_dims__(CL, 1, 1) __launch_bounds__((VBlockGeom<NV, CL>::T), MINB)
    vblock_kernel(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_out,
                  const __grid_constant__ CUtensorMap tm_inB, const __grid_constant__ CUtensorMap tm_outB,
                  const __grid_constant__ VBlockArgs a) {
    using G = VBlockGeom<NV, CL>;
    constexpr int CW = G::CW, RB = G::RB, PLANE = G::PLANE, T = G::T;
    constexpr uint32_t SWZ = G::SWZ;
    constexpr bool RETILE = CL > 1 && V3PATH == kV3ViaL2;
    // the other cut (RETILE only): BJ1 = NV/CL j1-planes x NV rows of NV doubles, as NV/16 boxes of 128-byte half rows
    constexpr int BJ1 = NV / CL, BROWS = BJ1 * NV, BHALVES = (NV * 8) / 128, BBOX = BROWS * 128;
    static_assert(!RETILE || (NV * 8) % 128 == 0, "re-tiling wants rows of whole 128-byte halves");
    static_assert(!RETILE || BHALVES * BBOX == G::TILE, "both cuts fill the same buffer");
    extern __shared__ unsigned char vb_smem_raw[];
    __shared__ __align__(8) unsigned long long vb_mbar;
    const uint32_t tile = (vb::smem_u32(vb_smem_raw) + 1023u) & ~1023u;
    const uint32_t bar = vb::smem_u32(&vb_mbar);
    const uint32_t rank = CL > 1 ? (blockIdx.x % CL) : 0u;
    const uint32_t x = blockIdx.x / CL;
    const int c_lo = (int)rank * CW;                       // first v3 index of this CTA (cut A)

    if (threadIdx.x == 0) {
        vb::mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    uint32_t phase = 0;                                    // parity of the next TMA-load completion
    bool stored = false;                                   // has the block been written to f_out yet?
    int cut = -1;                                          // what the buffer holds: -1 nothing, 0 cut A, 1 cut B
    auto load_cut = [&](int want) {
        if (threadIdx.x == 0) {
            vb::mbar_expect_tx(bar, (uint32_t)G::TILE);
            if (want == 0) {
                vb::tma_load_4d(tile, stored ? &tm_out : &tm_in, bar, c_lo, 0, 0, (int)x);
            } else {
#pragma unroll
                for (int h = 0; h < BHALVES; ++h)
                    vb::tma_load_4d(tile + h * BBOX, stored ? &tm_outB : &tm_inB, bar, 16 * h, 0, (int)rank * BJ1, (int)x);
            }
        }
        vb::mbar_wait(bar, phase);
        phase ^= 1u;
        cut = want;
    };
    auto store_cut = [&](bool complete) {
        // generic-proxy writes -> visible to the async proxy, then bulk store(s) of the buffer to f_out
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (threadIdx.x == 0) {
            if (cut == 0) {
                vb::tma_store_4d(&tm_out, tile, c_lo, 0, 0, (int)x);
            } else {
#pragma unroll
                for (int h = 0; h < BHALVES; ++h) vb::tma_store_4d(&tm_outB, tile + h * BBOX, 16 * h, 0, (int)rank * BJ1, (int)x);
            }
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            if (complete) {
                asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");     // the WRITES are done, not just the reads
                asm volatile("fence.proxy.async;" ::: "memory");
                __threadfence();
            } else {
                asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            }
        }
        stored = true;
    };
    // switch the buffer to the cut the next sweep needs (RETILE): store, let the whole cluster finish storing, reload
    auto want_cut = [&](int want) {
        if (cut == want) return;
        if (cut >= 0) {
            store_cut(true);
            cooperative_groups::this_cluster().sync();     // (also a CTA barrier: thread 0's store is complete for all)
            asm volatile("fence.proxy.async;" ::: "memory");
        }
        load_cut(want);
    };

    for (uint32_t s = 0; s < a.nsweeps; ++s) {
        const VSweep& sw = a.sw[s];
        if (RETILE) want_cut(sw.dim == 5 ? 1 : 0);
        else if (cut < 0) load_cut(0);
        if (sw.dim == 3) {
            // ---- along v1: pencil (j2, c), element j1 at  p_off + j1*PLANE  (swizzle term does not depend on j1)
            for (int p = threadIdx.x; p < NV * CW; p += T) {
                const uint32_t j2 = p / CW, c = p % CW;
                const uint32_t off = j2 * RB + c * 8;
                const uint32_t base = tile + (off ^ (((off >> 7) & SWZ) << 4));
                const double sval = __ldg(sw.src + src_offset(sw.terms, x, j2 * NV + (uint32_t)c_lo + c));
                double res[NV];
                vb::window_sweep<NV, NV, Q>(sval, sw.scale, 0,
                                            [&](int row) { return vb::lds_f64(base + (uint32_t)row * PLANE); }, res);
#pragma unroll
                for (int j = 0; j < NV; ++j) vb::sts_f64(base + (uint32_t)j * PLANE, res[j]);
            }
        } else if (sw.dim == 4) {
            // ---- along v2: pencil (j1, c), element j2 at  j1*PLANE + swz(j2*RB + c*8)
            for (int p = threadIdx.x; p < NV * CW; p += T) {
                const uint32_t j1 = p / CW, c = p % CW;
                const uint32_t base = tile + j1 * PLANE;
                const uint32_t c8 = c * 8;
                const double sval = __ldg(sw.src + src_offset(sw.terms, x * NV + j1, (uint32_t)c_lo + c));
                double res[NV];
                vb::window_sweep<NV, NV, Q>(sval, sw.scale, 0,
                                            [&](int row) {
                                                const uint32_t o = (uint32_t)row * RB;
                                                return vb::lds_f64(base + o + (c8 ^ (((o >> 7) & SWZ) << 4)));
                                            },
                                            res);
#pragma unroll
                for (int j = 0; j < NV; ++j) {
                    const uint32_t o = (uint32_t)j * RB;   // compile-time
                    vb::sts_f64(base + o + (c8 ^ (((o >> 7) & SWZ) << 4)), res[j]);
                }
            }
        } else if (RETILE) {
            // ---- along v3, cut B: thread owns the whole row (j1 = rank*BJ1 + p/NV, j2 = p%NV); column col lives in half
            // col/16 at  row*128 + ((col%16)*8 ^ (row&7)<<4)
            for (int p = threadIdx.x; p < BROWS; p += T) {
                const uint32_t rbase = tile + (uint32_t)p * 128u;
                const uint32_t sx = ((uint32_t)p & 7u) << 4;
                const uint32_t grow = (rank * BJ1 + (uint32_t)p / NV) * NV + (uint32_t)p % NV;      // j1*NV + j2
                const double sval = __ldg(sw.src + src_offset(sw.terms, x * (NV * NV) + grow, 0u));
                double res[NV];
                vb::window_sweep<NV, NV, Q>(sval, sw.scale, 0,
                                            [&](int col) {
                                                const uint32_t h = (uint32_t)col >> 4, cl = (uint32_t)col & 15u;
                                                return vb::lds_f64(rbase + h * BBOX + ((cl * 8) ^ sx));
                                            },
                                            res);
#pragma unroll
                for (int j = 0; j < NV; ++j)
                    vb::sts_f64(rbase + (uint32_t)(j >> 4) * BBOX + (((uint32_t)(j & 15) * 8) ^ sx), res[j]);
            }
        } else {
            // ---- along v3, cut A: row piece (j1, j2) x this CTA's CW outputs; inputs from any CTA of the cluster
            // Hazard: a neighbour reads my boundary columns of row p while I want to overwrite row p.  Rows are
            // handled in RP rounds (round r = rows r*T .. r*T+T-1 in EVERY CTA of the cluster, each thread one row
            // piece); within a round everyone reads, the cluster synchronises, everyone writes.  Later rounds touch
            // other rows, so one barrier per round (plus one up front for the previous sweep's writes) is enough.
            constexpr int RP = (NV * NV + T - 1) / T;      // rounds
            if (CL > 1) cooperative_groups::this_cluster().sync();
#pragma unroll 1
            for (int r = 0; r < RP; ++r) {
                const uint32_t p = r * T + threadIdx.x;    // row = j1*NV + j2
                const uint32_t roff = p * RB;
                const uint32_t sx = ((roff >> 7) & SWZ) << 4;
                double res[CW];
                if (p < NV * NV) {
                    const uint32_t rbase = tile + roff;
                    const double sval = __ldg(sw.src + src_offset(sw.terms, x * (NV * NV) + p, 0u));
                    vb::window_sweep<NV, CW, Q>(sval, sw.scale, c_lo,
                                                [&](int col) {
                                                    const uint32_t owner = (uint32_t)col / CW, cl = (uint32_t)col % CW;
                                                    const uint32_t ad = rbase + ((cl * 8) ^ sx);
                                                    if (CL > 1 && owner != rank) return vb::ld_cluster_f64(ad, owner);
                                                    return vb::lds_f64(ad);
                                                },
                                                res);
                }
                if (CL > 1) cooperative_groups::this_cluster().sync();     // every CTA has read this round's rows
                if (p < NV * NV) {
#pragma unroll
                    for (int j = 0; j < CW; ++j) vb::sts_f64(tile + roff + (((uint32_t)j * 8) ^ sx), res[j]);
                }
            }
        }
        __syncthreads();
    }
    if (cut < 0) load_cut(0);                              // an empty chain is a copy
    store_cut(false);
}

}  // namespace bsl6d
