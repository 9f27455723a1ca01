// bsl6d_pointwise.cu -- instantiations of the odd-q / per-point-displacement sweep kernels.
#include "fused_api.h"
#include "pointwise_kernels.cuh"

namespace bsl6d {
namespace {

template <int N, int Q>
constexpr int pw_minblocks() {
    constexpr int est = 4 * N + 6 * Q + 40;                 // registers a thread wants (pencil + shifts + weight scratch)
    return est <= 128 ? 4 : (est <= 170 ? 3 : 2);
}

template <int N, int Q>
bool by_kind(bool periodic, bool unit, PointwiseChoice& c) {
    constexpr int T = 128;
    if (unit) {
        if (periodic) return false;
        constexpr int S = N >= 16 ? 4 : 1, PB = 64;        // 64 pencils x 4 segments per block
        constexpr size_t smem = 2 * sizeof(double) * PB * (N | 1);
#ifndef BSL6D_TUNE_PWMINB
#define BSL6D_TUNE_PWMINB 3
#endif
        constexpr int MINB = S == 1 ? 8 : BSL6D_TUNE_PWMINB;   // the weight evaluation wants ~85 registers
        c = PointwiseChoice{(const void*)pointwise_unit_kernel<N, Q, S, PB, MINB>, PB * S, smem, PB};
    } else if (periodic) {
        c = PointwiseChoice{(const void*)pointwise_strided_kernel<N, Q, true, T, pw_minblocks<N, Q>()>, T, 0, 0};
    } else {
        c = PointwiseChoice{(const void*)pointwise_strided_kernel<N, Q, false, T, pw_minblocks<N, Q>()>, T, 0, 0};
    }
    return true;
}

template <int N>
bool by_q(int q, bool periodic, bool unit, PointwiseChoice& c) {
    switch (q) {
        case 3: return by_kind<N, 3>(periodic, unit, c);
        case 5: return by_kind<N, 5>(periodic, unit, c);
        case 7: return by_kind<N, 7>(periodic, unit, c);
        case 9: return by_kind<N, 9>(periodic, unit, c);
        default: return false;
    }
}

}  // namespace

bool pointwise_lookup(int n, int q, bool periodic, bool unit_stride, PointwiseChoice& out) {
    switch (n) {
        case 8: return by_q<8>(q, periodic, unit_stride, out);
        case 16: return by_q<16>(q, periodic, unit_stride, out);
        case 32: return by_q<32>(q, periodic, unit_stride, out);
        case 37: return by_q<37>(q, periodic, unit_stride, out);     // the paper's benchmark extent
        default: return false;
    }
}

}  // namespace bsl6d
