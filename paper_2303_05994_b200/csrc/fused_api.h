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

// ---- pointwise (odd q, per-point displacement) kernels, bsl6d_pointwise.cu -------------------------------------
namespace bsl6d {
struct PointwiseChoice {
    const void* fn;        // __global__ void (*)(PointwiseArgs)
    int threads;
    size_t smem;
    int unit;              // 1: unit-stride kernel (block = `threads` pencils)
};
bool pointwise_lookup(int n, int q, bool periodic, bool unit_stride, PointwiseChoice& out);
}  // namespace bsl6d
