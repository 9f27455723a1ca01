// bsl6d_ptile.cu -- instantiations of ptile_kernel for one stencil width (compile with -DBSL6D_PTILE_Q=6|8|10), and,
// in the Q = 8 unit, the tensor maps and the launch.  Not part of the C ABI; called by the pass planner.
#include "fused_api.h"
#include "ptile_kernels.cuh"

#ifndef BSL6D_PTILE_Q
#error "compile with -DBSL6D_PTILE_Q=<6|8|10>"
#endif

namespace bsl6d {
namespace {

constexpr int Q = BSL6D_PTILE_Q;

template <int NA, int NB, bool PA, bool PB>
PTileChoice choice() {
    using G = PTileGeom<NA, NB>;
    return PTileChoice{(const void*)ptile_kernel<NA, NB, Q, PA, PB>, G::THREADS, G::kSmemBytes, NA, NB};
}

// same-extent pairs: x-x (periodic, periodic), x-v (periodic, zero), v-v (zero, zero)
template <int N>
bool same_extent(bool pa, bool pb, PTileChoice& out) {
    if (pa && pb) { out = choice<N, N, true, true>(); return true; }
    if (pa && !pb) { out = choice<N, N, true, false>(); return true; }
    if (!pa && !pb) { out = choice<N, N, false, false>(); return true; }
    return false;
}

template <int NA, int NB>
bool mixed_extent(bool pa, bool pb, PTileChoice& out) {        // only occurs as (x3, v1): periodic, zero-extended
    if (pa && !pb) { out = choice<NA, NB, true, false>(); return true; }
    return false;
}

}  // namespace

#define BSL6D_CAT_(a, b) a##b
#define BSL6D_CAT(a, b) BSL6D_CAT_(a, b)

bool BSL6D_CAT(ptile_lookup_q, BSL6D_PTILE_Q)(int na, int nb, bool pa, bool pb, PTileChoice& out) {
    if (na == nb) {
        switch (na) {
            case 8: return same_extent<8>(pa, pb, out);
            case 16: return same_extent<16>(pa, pb, out);
            case 32: return same_extent<32>(pa, pb, out);
            default: return false;
        }
    }
    if (na == 8 && nb == 16) return mixed_extent<8, 16>(pa, pb, out);
    if (na == 48 && nb == 32) return mixed_extent<48, 32>(pa, pb, out);
    return false;
}

#if BSL6D_PTILE_Q == 8
namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        else
            (void)cudaGetLastError();
    }
    return fn;
}

// f seen as [outer][na][mid][nb][inner_b] doubles; box = one tile [1][na][1][nb][8], dense in shared memory.
bool make_map(CUtensorMap* m, const double* f, uint64_t outer, int na, uint64_t mid, int nb, uint64_t inner_b) {
    EncodeTiledFn enc = encode_fn();
    if (!enc) return false;
    const cuuint64_t dims[5] = {inner_b, (cuuint64_t)nb, mid, (cuuint64_t)na, outer};
    const cuuint64_t sb = inner_b * 8, sm = sb * (cuuint64_t)nb, sa = sm * mid, so = sa * (cuuint64_t)na;
    const cuuint64_t strides[4] = {sb, sm, sa, so};
    const cuuint32_t box[5] = {(cuuint32_t)kPTileC, (cuuint32_t)nb, 1u, (cuuint32_t)na, 1u};
    const cuuint32_t estr[5] = {1u, 1u, 1u, 1u, 1u};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, const_cast<double*>(f), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

bool ptile_available() { return encode_fn() != nullptr; }

cudaError_t ptile_launch(const PTileChoice& pc, const double* f_in, double* f_out, uint64_t outer, uint64_t mid,
                         uint64_t inner_b, const PTileArgs& args, int num_sms, cudaStream_t stream) {
    CUtensorMap tin, tout;
    if (!make_map(&tin, f_in, outer, pc.na, mid, pc.nb, inner_b) ||
        !make_map(&tout, f_out, outer, pc.na, mid, pc.nb, inner_b))
        return cudaErrorInvalidValue;
    const unsigned grid = args.ntiles < (uint32_t)num_sms ? args.ntiles : (unsigned)num_sms;
    void* kargs[] = {(void*)&tin, (void*)&tout, (void*)&args};
    return cudaLaunchKernel(pc.fn, dim3(grid), dim3((unsigned)pc.threads), kargs, pc.smem, stream);
}
#endif

}  // namespace bsl6d
