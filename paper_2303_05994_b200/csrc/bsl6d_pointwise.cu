// bsl6d_pointwise.cu -- instantiations of the odd-q / per-point-displacement sweep kernels.
#include "fused_api.h"
#include "pointwise_kernels.cuh"

namespace bsl6d {
namespace {

// Strided kernel, per stencil width: look-ahead D (outputs) and the resident blocks per SM it is compiled for (the
// register cap).  Measured on 37^6 (B200, ms per sweep, x dims / v1,v2): q = 7: D=8,MINB=4 11.4 / 12.6, D=12,MINB=3
// 11.3 / 11.25; q = 9: D=8,MINB=4 13.0 / 15.6 (spills), D=4,MINB=5 12.7 / 12.4.  Unit-stride kernel: 32 pencils x 4
// segments per block (128 threads), 6 blocks per SM (q = 3/5/7/9: 8.6 / 10.2 / 9.3 / 9.9-11.0 ms; 64 pencils x 4
// segments, 4 blocks per SM: 9.0 / 10.5 / 10.2 / 10.1).  A shared-memory tile variant of the strided kernel (same
// structure as the unit-stride one, rows of 32 or 64 pencils) was measured too: no better than the register kernel
// (q = 9: 12.5-13.6 against 11.9-12.4 ms) and dropped.
constexpr auto kTunePwt = 128;
constexpr auto kTunePwd7 = 12;
constexpr auto kTunePwm7 = 3;
constexpr auto kTunePwd9 = 4;
constexpr auto kTunePwm9 = 5;
constexpr auto kTunePwminb = 6;
constexpr auto kTunePwpb = 32;

template <int Q> constexpr int pw_lookahead() { return Q >= 9 ? kTunePwd9 : (Q >= 7 ? kTunePwd7 : 8); }
template <int Q> constexpr int pw_minblocks() { return Q >= 9 ? kTunePwm9 : (Q >= 7 ? kTunePwm7 : 4); }

template <int N, int Q>
bool by_kind(bool periodic, bool unit, PointwiseChoice& c) {
    constexpr int T = kTunePwt, D = pw_lookahead<Q>(), MB = pw_minblocks<Q>();
    c = PointwiseChoice{};
    if (unit) {
        if (periodic) return false;
        constexpr int S = N >= 48 ? 8 : (N >= 16 ? 4 : 1), PB = kTunePwpb;      // PB pencils x S segments per block
        constexpr size_t smem = 2 * sizeof(double) * PB * (N | 1);
        constexpr int MINB = S == 1 ? 8 : (S == 8 ? 3 : kTunePwminb);
        c.fn = (const void*)pointwise_unit_kernel<N, Q, S, PB, MINB>;
        c.threads = PB * S;
        c.smem = smem;
        c.unit = PB;
    } else {
        c.fn = periodic ? (const void*)pointwise_strided_kernel<N, Q, true, T, MB, D>
                        : (const void*)pointwise_strided_kernel<N, Q, false, T, MB, D>;
        c.threads = T;
    }
    return true;
}

template <int Q>
bool generic(int n, bool periodic, bool unit, PointwiseChoice& c) {
    c = PointwiseChoice{};
    c.generic = 1;
    if (unit && !periodic) {
        // two tiles of pb x (n|1) doubles; 4 segments per pencil; as many pencils as fit ~96 KB (two blocks per SM)
        const size_t row = 2 * sizeof(double) * (size_t)(n | 1);
        int pb = 64;
        while (pb > 32 && row * pb > 96 * 1024) pb -= 32;
        if (row * pb > 200 * 1024) return false;                         // extent above ~400: no staging possible
        c.fn = (const void*)pointwise_generic_unit_kernel<Q>;
        c.threads = pb * 4;
        c.smem = row * pb;
        c.unit = pb;
    } else {                                                              // (a periodic dim with inner == 1 included)
        c.fn = (const void*)pointwise_generic_kernel<Q, 128>;
        c.threads = 128;
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

bool generic_by_q(int n, int q, bool periodic, bool unit, PointwiseChoice& c) {
    switch (q) {
        case 1: return generic<1>(n, periodic, unit, c);
        case 3: return generic<3>(n, periodic, unit, c);
        case 5: return generic<5>(n, periodic, unit, c);
        case 7: return generic<7>(n, periodic, unit, c);
        case 9: return generic<9>(n, periodic, unit, c);
        case 11: return generic<11>(n, periodic, unit, c);
        default: return false;
    }
}

}  // namespace

bool pointwise_lookup(int n, int q, bool periodic, bool unit_stride, PointwiseChoice& out) {
    {
        bool ok = false;
        switch (n) {
            case 8: ok = by_q<8>(q, periodic, unit_stride, out); break;
            case 16: ok = by_q<16>(q, periodic, unit_stride, out); break;
            case 32: ok = by_q<32>(q, periodic, unit_stride, out); break;
            case 37: ok = by_q<37>(q, periodic, unit_stride, out); break;    // the paper's benchmark extent
            case 48: ok = by_q<48>(q, periodic, unit_stride, out); break;
            case 64: ok = by_q<64>(q, periodic, unit_stride, out); break;
            default: break;
        }
        if (ok) return true;
    }
    return generic_by_q(n, q, periodic, unit_stride, out);
}

}  // namespace bsl6d
