// fused_api.h -- internal interface between bsl6d_api.cu and the fused-pass translation units (one per stencil
// width q, so that they compile in parallel).  Not part of the C ABI.
#pragma once
#include <cstddef>

namespace bsl6d {

struct FusedChoice {
    const void* fn;        // __global__ void (*)(FusedArgs)
    int threads;
    size_t smem;           // dynamic shared memory, bytes
    int C;                 // contiguous doubles per tile row segment
};

// Is there a fused kernel for sweeps along dims a < b of extents na, nb, stencil width q, boundary kinds
// (periodic_a, periodic_b) and `pattern` (FusedPattern)?  One function per compiled q.
bool fused_lookup_q6(int na, int nb, bool pa, bool pb, int pattern, FusedChoice& out);
bool fused_lookup_q8(int na, int nb, bool pa, bool pb, int pattern, FusedChoice& out);
bool fused_lookup_q10(int na, int nb, bool pa, bool pb, int pattern, FusedChoice& out);

}  // namespace bsl6d

// ---- whole-v-block passes (vblock_kernels.cuh, bsl6d_vblock.cu) ----------------------------------------------------
#include <cstdint>
#include <cuda_runtime.h>
namespace bsl6d {
struct VBlockArgs;
struct VBlockChoice {
    const void* fn;        // __global__ void (*)(CUtensorMap in, out, in (other cut), out (other cut), VBlockArgs)
    int threads;
    size_t smem;
    int cl;                // CTAs per cluster = CTAs per v-block
    int cw;                // v3 columns per CTA
};
// Is there a whole-v-block kernel for a cubic velocity grid nv^3 and stencil width q (and a TMA-capable driver)?
bool vblock_lookup(int nv1, int nv2, int nv3, int q, VBlockChoice& out);
// Encode the tensor maps of f_in / f_out ([nx][nv][nv][nv] doubles) and enqueue one pass.
cudaError_t vblock_launch(const VBlockChoice& vc, const double* f_in, double* f_out, uint32_t nx, int nv,
                          const VBlockArgs& args, cudaStream_t stream);
}  // namespace bsl6d

// ---- persistent TMA-fed two-dim tile passes (ptile_kernels.cuh, bsl6d_ptile.cu) -----------------------------------
namespace bsl6d {
struct PTileArgs;
struct PTileChoice {
    const void* fn;        // __global__ void (*)(CUtensorMap, CUtensorMap, PTileArgs)
    int threads;
    size_t smem;
    int na, nb;
};
bool ptile_lookup_q6(int na, int nb, bool pa, bool pb, PTileChoice& out);
bool ptile_lookup_q8(int na, int nb, bool pa, bool pb, PTileChoice& out);
bool ptile_lookup_q10(int na, int nb, bool pa, bool pb, PTileChoice& out);
bool ptile_available();    // is cuTensorMapEncodeTiled reachable through the runtime?
cudaError_t ptile_launch(const PTileChoice& pc, const double* f_in, double* f_out, uint64_t outer, uint64_t mid,
                         uint64_t inner_b, const PTileArgs& args, int num_sms, cudaStream_t stream);
}  // namespace bsl6d

// ---- pointwise (odd q, per-point displacement) kernels, bsl6d_pointwise.cu -------------------------------------
namespace bsl6d {
struct PointwiseChoice {
    const void* fn;        // __global__ void (*)(PointwiseArgs)
    int threads;
    size_t smem;
    int unit;              // > 0: unit-stride kernel, a block takes this many pencils
    int generic;           // run-time-extent kernel: PointwiseArgs::n / periodic / pb / ld are read
};
bool pointwise_lookup(int n, int q, bool periodic, bool unit_stride, PointwiseChoice& out);
}  // namespace bsl6d
