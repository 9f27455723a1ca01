// bsl6d_vblock.cu -- instantiations, tensor maps and launch of vblock_kernel (all velocity-space
// sweeps of a step in one pass).  Not part of the C ABI; called by the pass planner in bsl6d_api.cu.
#include "fused_api.h"
#include "vblock_kernels.cuh"

#include <cstring>

namespace bsl6d {
namespace {

// cuTensorMapEncodeTiled is a driver-API entry point; it is fetched through the runtime so that the library links
// against the static CUDA runtime only (no -lcuda).
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

// f seen as [nx][nv][nv][nv] doubles; box = one CTA's share of one v-block: [1][nv][nv][cw], rows swizzled.
bool make_map(CUtensorMap* m, const double* f, uint32_t nx, int nv, int cw) {
    EncodeTiledFn enc = encode_fn();
    if (!enc) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)nv, (cuuint64_t)nv, (cuuint64_t)nv, (cuuint64_t)nx};
    const cuuint64_t strides[3] = {(cuuint64_t)nv * 8, (cuuint64_t)nv * nv * 8, (cuuint64_t)nv * nv * nv * 8};
    const cuuint32_t box[4] = {(cuuint32_t)cw, (cuuint32_t)nv, (cuuint32_t)nv, 1u};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUtensorMapSwizzle swz = cw * 8 == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B;
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(f), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

constexpr auto kTuneV3path = kV3ViaL2;

template <int NV, int Q, int CL, int MINB>
VBlockChoice choice() {
    using G = VBlockGeom<NV, CL>;
    return VBlockChoice{(const void*)vblock_kernel<NV, Q, CL, MINB, kTuneV3path>, G::T, G::kSmemBytes, CL, G::CW};
}

// The other cut of the same block: box = [1][nv/cl j1-planes][nv][16 doubles], 128-byte half rows, 128B swizzle.
bool make_map_b(CUtensorMap* m, const double* f, uint32_t nx, int nv, int cl) {
    EncodeTiledFn enc = encode_fn();
    if (!enc) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)nv, (cuuint64_t)nv, (cuuint64_t)nv, (cuuint64_t)nx};
    const cuuint64_t strides[3] = {(cuuint64_t)nv * 8, (cuuint64_t)nv * nv * 8, (cuuint64_t)nv * nv * nv * 8};
    const cuuint32_t box[4] = {16u, (cuuint32_t)nv, (cuuint32_t)(nv / cl), 1u};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(f), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

constexpr auto kTuneVcl = 4;
constexpr auto kTuneVminb = 2;

template <int Q>
bool by_nv(int nv, VBlockChoice& out) {
    switch (nv) {
        case 8: out = choice<8, Q, 1, 4>(); return true;
        case 16: out = choice<16, Q, 1, 3>(); return true;
        case 32: out = choice<32, Q, kTuneVcl, kTuneVminb>(); return true;
        default: return false;
    }
}

}  // namespace

bool vblock_lookup(int nv1, int nv2, int nv3, int q, VBlockChoice& out) {
    if (nv1 != nv2 || nv2 != nv3) return false;
    if (!encode_fn()) return false;
    switch (q) {
        case 6: return by_nv<6>(nv1, out);
        case 8: return by_nv<8>(nv1, out);
        case 10: return by_nv<10>(nv1, out);
        default: return false;
    }
}

cudaError_t vblock_launch(const VBlockChoice& vc, const double* f_in, double* f_out, uint32_t nx, int nv,
                          const VBlockArgs& args, cudaStream_t stream) {
    CUtensorMap tin, tout, tinb, toutb;
    if (!make_map(&tin, f_in, nx, nv, vc.cw) || !make_map(&tout, f_out, nx, nv, vc.cw)) return cudaErrorInvalidValue;
    if (vc.cl > 1 && nv >= 16) {
        if (!make_map_b(&tinb, f_in, nx, nv, vc.cl) || !make_map_b(&toutb, f_out, nx, nv, vc.cl)) return cudaErrorInvalidValue;
    } else {
        tinb = tin;                                        // unused by a single-CTA block
        toutb = tout;
    }
    void* kargs[] = {(void*)&tin, (void*)&tout, (void*)&tinb, (void*)&toutb, (void*)&args};
    return cudaLaunchKernel(vc.fn, dim3(nx * (unsigned)vc.cl), dim3((unsigned)vc.threads), kargs, vc.smem, stream);
}

}  // namespace bsl6d
