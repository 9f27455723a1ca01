// bsl6d_fused.cu -- instantiations of sweep_fused_kernel for one stencil width (compile with -DBSL6D_FUSED_Q=6|8|10).
#include "fused_api.h"
#include "fused_kernels.cuh"

#ifndef BSL6D_FUSED_Q
#error "compile with -DBSL6D_FUSED_Q=<6|8|10>"
#endif

namespace bsl6d {
namespace {

constexpr int Q = BSL6D_FUSED_Q;

constexpr int cgcd(int a, int b) { return b == 0 ? a : cgcd(b, a % b); }

// Tile shape policy: C = 8 contiguous doubles (64 B segments) while the tile stays <= ~100 KB, else 4.
template <int NA, int NB> constexpr int fused_C() { return NA * NB <= 1536 ? 8 : 4; }

template <int NA, int NB, bool PA, bool PB, int PAT>
constexpr int fused_minblocks() {
    constexpr int C = fused_C<NA, NB>();
    using G = FusedGeom<NA, NB, C>;
    constexpr int nmax = NA > NB ? NA : NB;
    constexpr int est = 2 * (nmax + Q - 1) + 2 * Q + 32;           // registers a thread wants
    constexpr int by_regs = 65536 / (est * G::T);
    constexpr int by_smem = (int)((220 * 1024) / G::kSmemBytes);
    constexpr int mb = by_regs < by_smem ? by_regs : by_smem;
    return mb < 1 ? 1 : (mb > 4 ? 4 : mb);
}

template <int NA, int NB, bool PA, bool PB, int PAT>
FusedChoice choice() {
    constexpr int C = fused_C<NA, NB>();
    using G = FusedGeom<NA, NB, C>;
    constexpr int MINB = fused_minblocks<NA, NB, PA, PB, PAT>();
    return FusedChoice{(const void*)sweep_fused_kernel<NA, NB, Q, PA, PB, C, PAT, MINB>, G::T, G::kSmemBytes, C};
}

// same-extent pairs: x-x (periodic, periodic), x-v (periodic, zero), v-v (zero, zero) for AB; v-v for ABA
template <int N>
bool same_extent(bool pa, bool pb, int pattern, FusedChoice& out) {
    if (pattern == kPatAB) {
        if (pa && pb) { out = choice<N, N, true, true, kPatAB>(); return true; }
        if (pa && !pb) { out = choice<N, N, true, false, kPatAB>(); return true; }
        if (!pa && !pb) { out = choice<N, N, false, false, kPatAB>(); return true; }
        return false;
    }
    if (pattern == kPatABA && !pa && !pb) { out = choice<N, N, false, false, kPatABA>(); return true; }
    return false;
}

// mixed extents only occur as (x3, v1): periodic then zero-extended, AB
template <int NA, int NB>
bool mixed_extent(bool pa, bool pb, int pattern, FusedChoice& out) {
    if (pattern == kPatAB && pa && !pb) { out = choice<NA, NB, true, false, kPatAB>(); return true; }
    return false;
}

}  // namespace

#define BSL6D_CAT_(a, b) a##b
#define BSL6D_CAT(a, b) BSL6D_CAT_(a, b)

bool BSL6D_CAT(fused_lookup_q, BSL6D_FUSED_Q)(int na, int nb, bool pa, bool pb, int pattern, FusedChoice& out) {
    if (na == nb) {
        switch (na) {
            case 8: return same_extent<8>(pa, pb, pattern, out);
            case 16: return same_extent<16>(pa, pb, pattern, out);
            case 32: return same_extent<32>(pa, pb, pattern, out);
            case 48: return same_extent<48>(pa, pb, pattern, out);
            case 64: return same_extent<64>(pa, pb, pattern, out);
            default: return false;
        }
    }
    if (na == 8 && nb == 16) return mixed_extent<8, 16>(pa, pb, pattern, out);
    if (na == 16 && nb == 64) return mixed_extent<16, 64>(pa, pb, pattern, out);
    if (na == 48 && nb == 32) return mixed_extent<48, 32>(pa, pb, pattern, out);
    return false;
}

}  // namespace bsl6d
