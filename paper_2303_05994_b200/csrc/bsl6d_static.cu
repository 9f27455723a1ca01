// bsl6d_static.cu -- bsl6d_density_static: the density moment (a6, eq (2)) for callers that cannot allocate
// device memory.
//
// Who that is: code that runs where cudaMalloc / cudaFree are off limits -- a plug-in inside a host application that
// hands out every byte of device memory itself (a solver framework with its own pool, a Kokkos or PyTorch caching
// allocator that must see all allocations to keep its accounting right), a real-time or in-situ diagnostic that runs
// between time steps and must not take the implicit device-wide synchronisation cudaFree / cudaMalloc can cause, or a
// process already so close to its memory limit that an allocation in the middle of a run may fail.  The rest of this
// library keeps its scratch in the context (bsl6d_create calls cudaMalloc); this entry point needs no context at all.
//
// What it does differently from bsl6d_density: when the velocity block of one x-point is longer than 32768 doubles
// the moment is formed in two launches -- partial sums of G chunks per x-point, then their sum -- and the partial sums
// need nx*G doubles of scratch.  bsl6d_density keeps them in memory the context got from cudaMalloc.  Here they live
// in a file-scope __device__ array of BSL6D_STATIC_SCRATCH_DOUBLES doubles (2 MiB) that is part of the library image:
// every GPU that loads this translation unit's module holds those 2 MiB until the process exits, whether the entry
// point is ever called or not, and nothing is allocated or freed at run time.  The arithmetic (chunking, order of
// additions) is the same as in density_kernels.cuh, so the two entry points give the same bits.
//
// The array is shared by every call on a device and keeps whatever the last call left in it.  Nothing in it has to
// start at zero: a call writes each of its nx*G slots in the first launch before the second launch reads them, and
// reads no other slot.  Two calls whose kernels can overlap on the GPU (different streams, no dependency between them)
// race on the array and produce garbage; calls on one stream, or ordered by events, are fine.
#include <cmath>
#include <cstdint>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/bsl6d.h"

namespace {

// Partial sums of split v-blocks.  In HOST code this name is only a stand-in the runtime uses to look the symbol up:
// it is not a device address and must never be passed to a kernel as one.  Host code gets the address from
// cudaGetSymbolAddress (scratch_of_current_device below); device code could also name the array directly.
static __device__ __align__(256) double g_static_partials[BSL6D_STATIC_SCRATCH_DOUBLES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
double* g_partials_addr[kMaxDevices];      // device address of g_static_partials on device i, once looked up

// The address of g_static_partials on the CURRENT device, looked up once per device (the array exists once per GPU
// that loaded the module, at a different address on each).  The first look-up on a device may make the runtime load
// this module there, which is why the first call on a device should not sit inside a stream capture.
int scratch_of_current_device(double** out, cudaError_t* err) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { *err = e; return BSL6D_ECUDA; }
    if (dev < 0 || dev >= kMaxDevices) return BSL6D_EUNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_partials_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_partials);
        if (e != cudaSuccess || !p) { *err = e; (void)cudaGetLastError(); return BSL6D_ECUDA; }
        g_partials_addr[dev] = static_cast<double*>(p);
    }
    *out = g_partials_addr[dev];
    return BSL6D_OK;
}

__device__ __forceinline__ double warp_sum_static(double v) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    return v;
}

// One block per (x, chunk): the sum over chunk g of the v-block of x-point x, four accumulators over 16-byte loads,
// a shuffle tree per warp, one value per warp through shared memory -- the order of additions of density_kernel.
// G == 1: out = rho and the value is scaled; G > 1: out = the scratch array, unscaled partial sums.
template <int T, bool VEC>
__global__ void __launch_bounds__(T) density_static_kernel(const double* __restrict__ f, double* __restrict__ out,
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
    const double s = warp_sum_static((a0 + a1) + (a2 + a3));

    __shared__ double part[T / 32];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < T / 32 ? part[threadIdx.x] : 0.0;
        v = warp_sum_static(v);
        if (threadIdx.x == 0) out[blockIdx.x] = (G == 1) ? scale * v : v;
    }
}

// rho[x] = scale * (partials of x added in chunk order)
__global__ void density_static_finish_kernel(const double* __restrict__ part, double* __restrict__ rho, size_t nx,
                                             uint32_t G, double scale) {
    const size_t x = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= nx) return;
    double s = 0.0;
    for (uint32_t g = 0; g < G; ++g) s += part[x * G + g];
    rho[x] = scale * s;
}

}  // namespace

extern "C" int bsl6d_density_static(const int32_t n[6], const double dv[3], const double* f, double* rho, void* stream,
                                    int* cuda_error) {
    if (cuda_error) *cuda_error = 0;
    if (!n || !dv || !f || !rho) return BSL6D_EINVAL;
    for (int d = 0; d < 6; ++d)
        if (n[d] < 1) return BSL6D_EINVAL;
    for (int d = 0; d < 3; ++d)
        if (!(dv[d] > 0.0) || !std::isfinite(dv[d])) return BSL6D_EINVAL;
    const size_t seg = (size_t)n[3] * (size_t)n[4] * (size_t)n[5];
    const size_t nx = (size_t)n[0] * (size_t)n[1] * (size_t)n[2];

    // the split of bsl6d_create: chunks of <= 32768 doubles, even length so that chunks stay 16-byte aligned
    const size_t target = 32768;
    size_t G = (seg + target - 1) / target;
    size_t chunk = (seg + G - 1) / G;
    chunk = (chunk + 1) & ~(size_t)1;
    G = (seg + chunk - 1) / chunk;
    if (nx > 0x7FFFFFFFull / G) return BSL6D_EUNSUPPORTED;                       // grid dimension of the first launch
    if (G > 1 && nx * G > (size_t)BSL6D_STATIC_SCRATCH_DOUBLES) return BSL6D_ESCRATCH;

    cudaError_t e = cudaSuccess;
    double* part = nullptr;
    if (G > 1) {
        const int rc = scratch_of_current_device(&part, &e);
        if (rc != BSL6D_OK) {
            if (cuda_error) *cuda_error = (int)e;
            return rc;
        }
    }

    const double dv3 = dv[0] * dv[1] * dv[2];
    const bool vec = (seg % 2 == 0) && (((uintptr_t)f & 15u) == 0);
    double* out = G == 1 ? rho : part;
    constexpr int T = 256;
    cudaStream_t st = (cudaStream_t)stream;
    if (vec) density_static_kernel<T, true><<<(unsigned)(nx * G), T, 0, st>>>(f, out, seg, (uint32_t)G, chunk, dv3);
    else density_static_kernel<T, false><<<(unsigned)(nx * G), T, 0, st>>>(f, out, seg, (uint32_t)G, chunk, dv3);
    e = cudaGetLastError();
    if (e == cudaSuccess && G > 1) {
        density_static_finish_kernel<<<(unsigned)((nx + 255) / 256), 256, 0, st>>>(part, rho, nx, (uint32_t)G, dv3);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        if (cuda_error) *cuda_error = (int)e;
        return BSL6D_ECUDA;
    }
    return BSL6D_OK;
}
