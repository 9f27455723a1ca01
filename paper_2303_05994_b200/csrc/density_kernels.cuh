// density_kernels.cuh -- a6: rho[x] = dv^3 * sum_v f[x, v]   (eq (2)).
//
// In C order every x-point owns one contiguous segment of S = nv1*nv2*nv3 doubles, so the moment is a
// segmented streaming reduction: 8 B/point read once.  A segment is cut into G equal chunks, one block per
// (x, chunk); per thread four independent accumulators over 16-byte loads, then a warp-shuffle tree, then one
// value per warp through shared memory.  The order of additions is fixed => bitwise reproducible.
// G > 1 writes partials that density_finish_kernel adds in chunk order.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace bsl6d {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    return v;
}

template <int T, bool VEC>
__global__ void __launch_bounds__(T) density_kernel(const double* __restrict__ f, double* __restrict__ out,
                                                    size_t seg, uint32_t G, size_t chunk, double scale) {
    const size_t x = blockIdx.x / G;
    const uint32_t g = blockIdx.x - (uint32_t)x * G;
    const size_t lo = (size_t)g * chunk;
    size_t hi = lo + chunk;
    if (hi > seg) hi = seg;
    const double* __restrict__ p = f + x * seg + lo;
    const size_t len = hi - lo;

    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    if (VEC) {
        const double2* __restrict__ p2 = reinterpret_cast<const double2*>(p);
        const size_t len2 = len >> 1;
        size_t e = threadIdx.x;
        for (; e + 3 * (size_t)T < len2; e += 4 * (size_t)T) {
            const double2 v0 = __ldcs(p2 + e), v1 = __ldcs(p2 + e + T), v2 = __ldcs(p2 + e + 2 * T),
                          v3 = __ldcs(p2 + e + 3 * T);
            a0 += v0.x + v0.y;
            a1 += v1.x + v1.y;
            a2 += v2.x + v2.y;
            a3 += v3.x + v3.y;
        }
        for (; e < len2; e += T) {
            const double2 v0 = __ldcs(p2 + e);
            a0 += v0.x + v0.y;
        }
        if ((len & 1) && threadIdx.x == 0) a1 += p[len - 1];
    } else {
        for (size_t e = threadIdx.x; e < len; e += T) a0 += __ldcs(p + e);
    }
    double s = warp_sum((a0 + a1) + (a2 + a3));

    __shared__ double part[T / 32];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < T / 32 ? part[threadIdx.x] : 0.0;
        v = warp_sum(v);
        if (threadIdx.x == 0) out[blockIdx.x] = (G == 1) ? scale * v : v;
    }
}

__global__ void density_finish_kernel(const double* __restrict__ part, double* __restrict__ rho, size_t nx,
                                      uint32_t G, double scale) {
    const size_t x = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= nx) return;
    double s = 0.0;
    for (uint32_t g = 0; g < G; ++g) s += part[x * G + g];
    rho[x] = scale * s;
}

}  // namespace bsl6d
