// bsl6d_api.cu -- the C ABI of include/bsl6d.h: argument checks, launch planning, the Strang driver.
// All arithmetic on f happens in the kernels of sweep_kernels.cuh / density_kernels.cuh.
#include "../../include/bsl6d.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "density_kernels.cuh"
#include "field_kernels.cuh"
#include "fused_api.h"
#include "fused_kernels.cuh"
#include "pointwise_kernels.cuh"
#include "ptile_kernels.cuh"
#include "sweep_kernels.cuh"
#include "vblock_kernels.cuh"

using bsl6d::SweepArgs;

struct bsl6d_ctx {
    bsl6d_grid g;
    int q;
    int device;
    size_t npts;
    double* d_nodes;          // 6 node tables back to back (device)
    size_t node_off[6];
    double* d_part;           // density partial sums (device), nx * G
    uint32_t dens_G;
    size_t dens_chunk;
    int last_cuda;
    long long launches;
    double2* fld[5];          // field step: complex work arrays over the x grid (allocated on first use)
    double2* tw[3];           // field step: twiddle tables exp(-2 pi i m / n_d)
    int field_ready;          // field step: every table and work array is allocated
    int fuse_all;             // tuning/testing: ignore the pay-off policy and fuse wherever a kernel exists
    int fusion;               // 1: consecutive sweeps over two dims run as one fused pass where a kernel exists
    int open_x[3];            // 1: this x dim is NOT periodic but zero-extended (a slab with halo planes)
    int fusion_mode;          // as set by bsl6d_set_fusion
    int use_ptile;            // 1: chains over two dims run as persistent TMA-fed tile passes where a kernel exists
    int use_fused;            // 1: round-1 two-dim tile kernels (pairs / triples) where no ptile kernel exists
    int num_sms;
    int vblock_min;           // fewest sweeps a whole-v-block pass is used for
    int use_vblock;           // 1: runs of velocity-space sweeps run as one whole-v-block pass where a kernel exists
    const void* smem_ok[64];  // kernels whose dynamic shared-memory limit has been raised (and to how much)
    size_t smem_ok_bytes[64];
    int n_smem_ok;
    // host-path working set (bsl6d_run_host), allocated on first use
    double* h_f[2];           // device buffer for f, per slot (bsl6d_run_host_begin keeps two steps in flight)
    double* h_small[2];       // device buffer for shift sources / rho, per slot
    size_t h_small_cap[2];
    cudaStream_t h_stream[2];
    double* h_part[2];        // density partial sums per slot (split v-blocks only)
};

namespace {

// dims 0-2 are periodic unless bsl6d_set_boundary opened them (slab decomposition); dims 3-5 are zero-extended
bool is_periodic(const bsl6d_ctx* c, int dim) { return dim < 3 && !c->open_x[dim]; }

typedef void (*sweep_fn)(const SweepArgs);

struct KernelChoice {
    sweep_fn fn;
    int threads;
    size_t smem;
    int kind;                 // 0 strided, 1 unit, 2 generic
    int gen_T;                // generic: threads; unit and strided: segments per pencil S
    sweep_fn fn_oop;          // strided only, may be null: the kernel for f_in != f_out (sweep_stream_kernel)
    int oop_threads;
};

// Launch shape of the strided sweep: T threads per block, at least MINB resident blocks per SM (caps the
// registers ptxas may use: a thread holds its whole pencil, 2*(N [+Q-1]) registers, plus 2*Q for the weights).
// Pencils that fit 128 registers: 4 blocks of 128 threads (16 warps/SM).  Longer pencils (N = 48 with Q = 10, N = 64)
// allow only ~12 warps/SM; they run as blocks of 64 threads, 6 (or 4) per SM.  Measured against 3 blocks of 128
// threads in alternating runs on one box: no difference beyond noise (C5 x sweeps 6.21-6.48 TB/s either way) -- inside a
// long step these kernels are held back by the 1 kW power cap (SM clock ~1.55 GHz), not by the block shape.  Two or
// four threads per pencil (S > 1 below) were slower (6.09 / 5.0-5.6 TB/s): the shared rows are re-read through L1/L2.
template <int N, int Q, bool P>
constexpr int strided_regs_wanted() { return 2 * (N + (P ? 0 : Q - 1)) + 2 * Q + 24; }
constexpr auto kTuneLongT = 64;
constexpr auto kTuneLongMinb = 6;
template <int N, int Q, bool P>
constexpr int strided_threads() { return strided_regs_wanted<N, Q, P>() <= 128 ? 128 : kTuneLongT; }
template <int N, int Q, bool P>
constexpr int strided_minblocks() {
    constexpr int est = strided_regs_wanted<N, Q, P>();
    return est <= 128 ? 4 : (est <= 176 ? kTuneLongMinb : (kTuneLongMinb * 2) / 3);
}

// Segments per pencil: 1 (a thread owns its whole pencil) unless the pencil is too long for 4 blocks per SM.
template <int N, int Q, bool P> constexpr int strided_segments() { return 1; }

template <int N, int Q, bool P>
KernelChoice strided_choice() {
    constexpr int S = strided_segments<N, Q, P>();
    constexpr int T = strided_threads<N, Q, P>();
    constexpr int MINB = S == 1 ? strided_minblocks<N, Q, P>() : 4;
    // Out of place, long periodic pencils stream through a register window instead (sweep_stream_kernel: 96-122 instead
    // of 162-168 registers at N = 48, Q = 10; C5 x sweeps +1.7-2.8 % in alternating runs on one box).  Zero-extended
    // long pencils (N = 64, Q = 6) and the pencils that fit 128 registers anyway measured 0.6-2 % slower that way.
constexpr auto kTuneStreamRegs = 128;
    if constexpr (P && S == 1 && strided_regs_wanted<N, Q, P>() > kTuneStreamRegs) {
        KernelChoice kc{bsl6d::sweep_strided_kernel<N, Q, P, T, MINB, S>, T, 0, 0, S};
        kc.fn_oop = bsl6d::sweep_stream_kernel<N, Q, P, 128, 4, 12>;
        kc.oop_threads = 128;
        return kc;
    }
    return KernelChoice{bsl6d::sweep_strided_kernel<N, Q, P, T, MINB, S>, T, 0, 0, S, nullptr, 0};
}

// Launch shape of the unit-stride sweep: S segments per pencil, T threads (a multiple of 32*S), MINB blocks/SM.
template <int N, int Q> constexpr int unit_segments() { return N >= 48 ? 4 : 1; }
template <int N, int Q> constexpr int unit_minblocks() { return (N >= 48 && Q <= 8) ? 6 : 4; }   // q = 10 at 80 registers spills
// Tile filled by cp.async (true) or by loads staged in registers.  Alternating runs on one box, v3 sweep in-step, GB/s:
// C3 (N = 64, q = 6, with 6 blocks/SM) 6440-6486 -> 6915-6948; C2 (N = 32, q = 8) 6631-6668 -> 6946-7009;
// C5 (N = 32, q = 10) 6715 -> 6600-6612, so the widest stencil on short pencils keeps the register fill.
template <int N, int Q> constexpr bool unit_async() { return unit_segments<N, Q>() > 1 || Q <= 8; }
template <int N, int Q> constexpr int unit_threads() { return 128 % (32 * unit_segments<N, Q>()) == 0 ? 128 : 32 * unit_segments<N, Q>(); }

template <int N, int Q>
KernelChoice unit_choice() {
    constexpr int S = unit_segments<N, Q>();
    constexpr int T = unit_threads<N, Q>();
    constexpr int MINB = unit_minblocks<N, Q>();
    return KernelChoice{bsl6d::sweep_unit_kernel<N, Q, S, T, MINB, unit_async<N, Q>()>, T, sizeof(double) * (T / S) * (N | 1), 1, S, nullptr, 0};
}

template <int N, bool P>
bool strided_by_q(int q, KernelChoice& c) {
    switch (q) {
        case 4: c = strided_choice<N, 4, P>(); return true;
        case 6: c = strided_choice<N, 6, P>(); return true;
        case 8: c = strided_choice<N, 8, P>(); return true;
        case 10: c = strided_choice<N, 10, P>(); return true;
        default: return false;
    }
}

template <bool P>
bool strided_lookup(int n, int q, KernelChoice& c) {
    switch (n) {
        case 8: return strided_by_q<8, P>(q, c);
        case 16: return strided_by_q<16, P>(q, c);
        case 32: return strided_by_q<32, P>(q, c);
        case 37: return strided_by_q<37, P>(q, c);          // the paper's benchmark extent
        case 48: return strided_by_q<48, P>(q, c);
        case 64: return strided_by_q<64, P>(q, c);
        default: return false;
    }
}

template <int N>
bool unit_by_q(int q, KernelChoice& c) {
    switch (q) {
        case 4: c = unit_choice<N, 4>(); return true;
        case 6: c = unit_choice<N, 6>(); return true;
        case 8: c = unit_choice<N, 8>(); return true;
        case 10: c = unit_choice<N, 10>(); return true;
        default: return false;
    }
}

bool unit_lookup(int n, int q, KernelChoice& c) {
    switch (n) {
        case 8: return unit_by_q<8>(q, c);
        case 16: return unit_by_q<16>(q, c);
        case 32: return unit_by_q<32>(q, c);
        case 37: return unit_by_q<37>(q, c);
        case 48: return unit_by_q<48>(q, c);
        case 64: return unit_by_q<64>(q, c);
        default: return false;
    }
}

template <int T>
const void* generic_by_q(int q) {
    switch (q) {
        case 2: return (const void*)bsl6d::sweep_generic_kernel<2, T>;
        case 4: return (const void*)bsl6d::sweep_generic_kernel<4, T>;
        case 6: return (const void*)bsl6d::sweep_generic_kernel<6, T>;
        case 8: return (const void*)bsl6d::sweep_generic_kernel<8, T>;
        case 10: return (const void*)bsl6d::sweep_generic_kernel<10, T>;
        case 12: return (const void*)bsl6d::sweep_generic_kernel<12, T>;
        default: return nullptr;
    }
}
const void* generic_fn(int q, int T) { return T == 64 ? generic_by_q<64>(q) : generic_by_q<32>(q); }

// unit-stride fallback: PB pencils per block, S = ceil(n / RMAX) threads per pencil, RMAX outputs per thread at most
template <int PB, int RMAX>
const void* generic_unit_by_q(int q) {
    switch (q) {
        case 2: return (const void*)bsl6d::sweep_generic_unit_kernel<2, PB, RMAX>;
        case 4: return (const void*)bsl6d::sweep_generic_unit_kernel<4, PB, RMAX>;
        case 6: return (const void*)bsl6d::sweep_generic_unit_kernel<6, PB, RMAX>;
        case 8: return (const void*)bsl6d::sweep_generic_unit_kernel<8, PB, RMAX>;
        case 10: return (const void*)bsl6d::sweep_generic_unit_kernel<10, PB, RMAX>;
        case 12: return (const void*)bsl6d::sweep_generic_unit_kernel<12, PB, RMAX>;
        default: return nullptr;
    }
}
// shape of the unit-stride fallback for extent n: pencils per block, segments per pencil, outputs per thread (0: none)
struct GenericUnitShape { int pb, s, rmax; };
GenericUnitShape generic_unit_shape(int n) {
    const int rmax = n <= 256 ? 16 : 32;
    const int s = (n + rmax - 1) / rmax;
    if (s > 16) return GenericUnitShape{0, 0, 0};            // extent above 512
    const int pb = 64 * s <= 512 ? 64 : 32;
    return GenericUnitShape{pb, s, rmax};
}
const void* generic_unit_fn(int q, int n) {
    const GenericUnitShape g = generic_unit_shape(n);
    if (!g.pb) return nullptr;
    if (g.rmax == 16) return g.pb == 64 ? generic_unit_by_q<64, 16>(q) : generic_unit_by_q<32, 16>(q);
    return generic_unit_by_q<32, 32>(q);
}

template <int T>
const void* peer_by_q(int q) {
    switch (q) {
        case 2: return (const void*)bsl6d::sweep_peer_kernel<2, T>;
        case 4: return (const void*)bsl6d::sweep_peer_kernel<4, T>;
        case 6: return (const void*)bsl6d::sweep_peer_kernel<6, T>;
        case 8: return (const void*)bsl6d::sweep_peer_kernel<8, T>;
        case 10: return (const void*)bsl6d::sweep_peer_kernel<10, T>;
        case 12: return (const void*)bsl6d::sweep_peer_kernel<12, T>;
        default: return nullptr;
    }
}

// The compiled-extent kernel for bsl6d_advect_x1_peer: the streaming sweep with rows taken from the neighbours' arrays.
template <int N>
const void* peer_stream_by_q(int q) {
    switch (q) {
        case 4: return (const void*)bsl6d::sweep_stream_kernel<N, 4, false, 128, 4, 12, true>;
        case 6: return (const void*)bsl6d::sweep_stream_kernel<N, 6, false, 128, 4, 12, true>;
        case 8: return (const void*)bsl6d::sweep_stream_kernel<N, 8, false, 128, 4, 12, true>;
        case 10: return (const void*)bsl6d::sweep_stream_kernel<N, 10, false, 128, 4, 12, true>;
        default: return nullptr;
    }
}
const void* peer_stream_fn(int n, int q) {
    switch (n) {
        case 8: return peer_stream_by_q<8>(q);
        case 16: return peer_stream_by_q<16>(q);
        case 32: return peer_stream_by_q<32>(q);
        case 48: return peer_stream_by_q<48>(q);
        case 64: return peer_stream_by_q<64>(q);
        default: return nullptr;
    }
}

// Which kernel serves a sweep along `dim`?  (Also used by bsl6d_kernel_name.)
int choose_kernel(const bsl6d_ctx* c, int dim, KernelChoice& k) {
    const int n = c->g.n[dim];
    const bool periodic = is_periodic(c, dim);
    size_t inner = 1;
    for (int d = dim + 1; d < 6; ++d) inner *= (size_t)c->g.n[d];
    bool ok;
    if (inner == 1) ok = !periodic && unit_lookup(n, c->q, k);
    else ok = periodic ? strided_lookup<true>(n, c->q, k) : strided_lookup<false>(n, c->q, k);
    if (ok) return BSL6D_OK;
    // fallback: pencils staged in shared memory: n * T doubles (strided), (n|1) * PB doubles (unit stride)
    const size_t cap = 200 * 1024;
    if (inner == 1 && !periodic) {
        const GenericUnitShape g = generic_unit_shape(n);
        if (!g.pb) return BSL6D_EUNSUPPORTED;
        const size_t smem = (size_t)(n | 1) * (size_t)g.pb * sizeof(double);
        if (smem > cap) return BSL6D_EUNSUPPORTED;
        k = KernelChoice{nullptr, g.pb * g.s, smem, 2, g.pb, nullptr, 0};      // gen_T = pencils per block
        return BSL6D_OK;
    }
    const size_t per_thread = (size_t)n * sizeof(double);
    int T = 64;
    if (per_thread * T > cap) T = 32;
    if (per_thread * T > cap) return BSL6D_EUNSUPPORTED;
    k = KernelChoice{nullptr, T, per_thread * T, 2, T, nullptr, 0};
    return BSL6D_OK;
}

int cuda_fail(bsl6d_ctx* c, cudaError_t e) {
    if (c) c->last_cuda = (int)e;
    (void)cudaGetLastError();
    return BSL6D_ECUDA;
}

// Every entry point runs on the device the context was created on (its tables live there).
int check_device(bsl6d_ctx* c) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return dev == c->device ? BSL6D_OK : BSL6D_EINVAL;
}

// Raise a kernel's dynamic shared-memory limit once (the attribute is per function and sticks): remembered per context.
int allow_smem(bsl6d_ctx* c, const void* fn, size_t smem) {
    if (smem <= 48 * 1024) return BSL6D_OK;
    for (int k = 0; k < c->n_smem_ok; ++k)
        if (c->smem_ok[k] == fn && c->smem_ok_bytes[k] >= smem) return BSL6D_OK;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(c, e);
    for (int k = 0; k < c->n_smem_ok; ++k)
        if (c->smem_ok[k] == fn) { c->smem_ok_bytes[k] = smem; return BSL6D_OK; }
    if (c->n_smem_ok < 64) { c->smem_ok[c->n_smem_ok] = fn; c->smem_ok_bytes[c->n_smem_ok++] = smem; }
    return BSL6D_OK;
}

uint32_t ceil_pow2_log2(uint64_t v) {
    uint32_t l = 0;
    while ((1ull << l) < v) ++l;
    return l;
}

// Source-index terms of a sweep along `dim` whose shift source is dense over the dims in `mask`:
// runs of adjacent masked dims inside the outer / inner group of the [outer][N][inner] view.
int build_src_terms(const int32_t* n, int dim, unsigned mask, bsl6d::SrcTerms& t) {
    std::memset(&t, 0, sizeof(t));
    size_t sstride[6];
    {
        size_t s = 1;
        for (int d = 5; d >= 0; --d) {
            if (mask & (1u << d)) { sstride[d] = s; s *= (size_t)n[d]; } else sstride[d] = 0;
        }
        if (s > 0xFFFFFFFFull) return BSL6D_EUNSUPPORTED;
    }
    for (int grp = 0; grp < 2; ++grp) {
        const int dlo = grp == 0 ? 0 : dim + 1, dhi = grp == 0 ? dim : 6;   // [dlo, dhi)
        int d = dhi - 1;
        size_t below = 1;
        while (d >= dlo) {
            if (!(mask & (1u << d))) { below *= (size_t)n[d]; --d; continue; }
            // run of masked dims d, d-1, ... (towards slower dims)
            size_t extent = 1;
            const size_t run_below = below, run_sstride = sstride[d];
            while (d >= dlo && (mask & (1u << d))) { extent *= (size_t)n[d]; below *= (size_t)n[d]; --d; }
            const bool slowest = (d < dlo);
            if (t.nterms >= (uint32_t)bsl6d::kMaxSrcTerms) return BSL6D_EUNSUPPORTED;
            const uint32_t k = t.nterms++;
            t.t_inner[k] = (uint32_t)grp;
            t.t_below[k] = (uint32_t)run_below;
            t.t_extent[k] = slowest ? 0u : (uint32_t)extent;
            t.t_sstride[k] = (uint32_t)run_sstride;
        }
    }
    return BSL6D_OK;
}

// Build the launch arguments and enqueue one sweep.
int launch_sweep(bsl6d_ctx* c, const double* f_in, double* f_out, int dim, const double* src, unsigned mask,
                 double scale, cudaStream_t stream) {
    if (!c || !f_in || !f_out || !src) return BSL6D_EINVAL;
    if (dim < 0 || dim > 5 || (mask & ~0x3Fu) || (mask & (1u << dim))) return BSL6D_EINVAL;
    if (!std::isfinite(scale)) return BSL6D_EINVAL;
    const size_t bytes = c->npts * sizeof(double);
    if (f_in != f_out) {
        const char* a = (const char*)f_in;
        const char* b = (const char*)f_out;
        if (a < b + bytes && b < a + bytes) return BSL6D_EALIAS;
    }
    const int32_t* n = c->g.n;
    size_t inner = 1, outer = 1;
    for (int d = dim + 1; d < 6; ++d) inner *= (size_t)n[d];
    for (int d = 0; d < dim; ++d) outer *= (size_t)n[d];
    if (inner > 0xFFFFFFFFull || outer > 0xFFFFFFFFull || inner * outer > 0xFFFFFFFFull) return BSL6D_EUNSUPPORTED;

    KernelChoice kc;
    int rc = check_device(c);
    if (rc) return rc;
    rc = choose_kernel(c, dim, kc);
    if (rc) return rc;
    if (kc.fn_oop && f_in != f_out) {                      // out of place: the streaming variant where there is one
        kc.fn = kc.fn_oop;
        kc.threads = kc.oop_threads;
    }

    SweepArgs a;
    std::memset(&a, 0, sizeof(a));
    a.in = f_in;
    a.out = f_out;
    a.src = src;
    a.scale = scale;
    a.inner = (uint32_t)inner;
    a.outer = (uint32_t)outer;
    a.n = (uint32_t)n[dim];

    rc = build_src_terms(n, dim, mask, a.terms);
    if (rc) return rc;

    // ---- grid -------------------------------------------------------------------------------------------
    unsigned grid;
    if (kc.kind == 1) {
        const size_t pb = (size_t)kc.threads / (size_t)kc.gen_T;      // pencils per block = T / S
        grid = (unsigned)((outer + pb - 1) / pb);
    } else {
        // strided: kc.gen_T = segments per pencil (threads / segments pencils per block); generic: gen_T = threads
        const uint64_t pencils = kc.kind == 0 ? (uint64_t)kc.threads / (uint64_t)kc.gen_T : (uint64_t)kc.threads;
        if (kc.kind == 0 && kc.gen_T == 1 && inner % 32 != 0 && inner > 1) {
            // odd inner extents (37^k): flattened pencil index, every lane busy
            a.ti_log2 = bsl6d::kFlatPencils;
            a.nib = (uint32_t)(inner * outer);
            grid = (unsigned)((inner * outer + pencils - 1) / pencils);
        } else {
            const uint64_t lim = inner < pencils ? inner : pencils;
            a.ti_log2 = ceil_pow2_log2(lim);
            const uint32_t TI = 1u << a.ti_log2, TO = (uint32_t)pencils / TI;
            a.nib = (uint32_t)((inner + TI - 1) / TI);
            const uint64_t nbo = (outer + TO - 1) / TO;
            if ((uint64_t)a.nib * nbo > 0x7FFFFFFFull) return BSL6D_EUNSUPPORTED;
            grid = (unsigned)((uint64_t)a.nib * nbo);
        }
    }

    cudaError_t e;
    if (kc.kind == 2) {
        const void* gfn = (inner == 1 && !is_periodic(c, dim)) ? generic_unit_fn(c->q, n[dim]) : generic_fn(c->q, kc.gen_T);
        if (!gfn) return BSL6D_EUNSUPPORTED;
        rc = allow_smem(c, gfn, kc.smem);
        if (rc) return rc;
        int per = is_periodic(c, dim) ? 1 : 0;
        void* gargs[] = {(void*)&a, (void*)&per};                  // the unit-stride kernel takes only `a`
        grid = (unsigned)((inner * outer + (size_t)kc.gen_T - 1) / (size_t)kc.gen_T);
        e = cudaLaunchKernel(gfn, dim3(grid), dim3(kc.threads), gargs, kc.smem, stream);
        if (e != cudaSuccess) return cuda_fail(c, e);
    } else {
        rc = allow_smem(c, (const void*)kc.fn, kc.smem);
        if (rc) return rc;
        void* args[] = {(void*)&a};
        e = cudaLaunchKernel((const void*)kc.fn, dim3(grid), dim3(kc.threads), args, kc.smem, stream);
        if (e != cudaSuccess) return cuda_fail(c, e);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->launches += 1;
    return BSL6D_OK;
}

// ---- sequences of sweeps: planning into passes ---------------------------------------------
struct SweepDesc { int dim; const double* src; unsigned mask; double scale; };

struct Pass {
    int first, count;         // sweeps [first, first+count)
    bool fused;               // two-dim tile pass (fused_kernels.cuh)
    bsl6d::FusedChoice fc;
    int pattern;
    bool vblock;              // whole-v-block pass (vblock_kernels.cuh)
    bsl6d::VBlockChoice vc;
    bool ptile;               // persistent TMA-fed two-dim tile pass (ptile_kernels.cuh)
    bsl6d::PTileChoice pc;
    int dim_a, dim_b;
};

bool fused_lookup(int q, int na, int nb, bool pa, bool pb, int pattern, bsl6d::FusedChoice& fc) {
    switch (q) {
        case 6: return bsl6d::fused_lookup_q6(na, nb, pa, pb, pattern, fc);
        case 8: return bsl6d::fused_lookup_q8(na, nb, pa, pb, pattern, fc);
        case 10: return bsl6d::fused_lookup_q10(na, nb, pa, pb, pattern, fc);
        default: return false;
    }
}

int check_sweep_desc(const bsl6d_ctx* c, const SweepDesc& s) {
    if (!s.src) return BSL6D_EINVAL;
    if (s.dim < 0 || s.dim > 5 || (s.mask & ~0x3Fu) || (s.mask & (1u << s.dim))) return BSL6D_EINVAL;
    if (!std::isfinite(s.scale)) return BSL6D_EINVAL;
    (void)c;
    return BSL6D_OK;
}

// Can sweeps [i, i+cnt) run as one fused pass?  cnt = 2: dims (a, b); cnt = 3: dims (a, b, a); a < b, b not unit-stride.
bool try_fuse(const bsl6d_ctx* c, const SweepDesc* sw, int i, int cnt, Pass& p) {
    const int a = sw[i].dim, b = sw[i + 1].dim;
    if (!(a < b)) return false;
    if (cnt == 3 && sw[i + 2].dim != a) return false;
    const int32_t* n = c->g.n;
    size_t inner_b = 1, mid = 1, outer = 1;
    for (int d = b + 1; d < 6; ++d) inner_b *= (size_t)n[d];
    for (int d = a + 1; d < b; ++d) mid *= (size_t)n[d];
    for (int d = 0; d < a; ++d) outer *= (size_t)n[d];
    if (inner_b < 2) return false;
    const int pattern = cnt == 2 ? bsl6d::kPatAB : bsl6d::kPatABA;
    bsl6d::FusedChoice fc;
    if (!fused_lookup(c->q, n[a], n[b], is_periodic(c, a), is_periodic(c, b), pattern, fc)) return false;
    if (inner_b % (size_t)fc.C) return false;
    if (c->npts > 0xFFFFFFFFull) return false;                        // 32-bit pencil indices in the kernel
    // Policy from measurement: a pair only pays with >= 64-byte row segments and a tile whose
    // rows are not spread over hundreds of MB (x1 on the big grids); the three-sweep rotation always pays.
    if (cnt == 2 && !c->fuse_all) {
        const size_t strideA_bytes = mid * (size_t)n[b] * inner_b * sizeof(double);
        if (fc.C < 8 || strideA_bytes >= ((size_t)64 << 20)) return false;
    }
    const size_t blocks = outer * mid * (inner_b / (size_t)fc.C);
    if (blocks > 0x7FFFFFFFull) return false;
    p.first = i; p.count = cnt; p.fused = true; p.fc = fc; p.pattern = pattern; p.vblock = false; p.ptile = false;
    return true;
}

bool ptile_lookup(int q, int na, int nb, bool pa, bool pb, bsl6d::PTileChoice& pc) {
    switch (q) {
        case 6: return bsl6d::ptile_lookup_q6(na, nb, pa, pb, pc);
        case 8: return bsl6d::ptile_lookup_q8(na, nb, pa, pb, pc);
        case 10: return bsl6d::ptile_lookup_q10(na, nb, pa, pb, pc);
        default: return false;
    }
}

// Can sweeps [i, i+cnt) -- any order of sweeps along exactly two dims a < b, b not the unit-stride dim -- run as one
// persistent tile pass?
bool try_ptile(const bsl6d_ctx* c, const SweepDesc* sw, int i, int cnt, Pass& p) {
    if (cnt < 2 || cnt > bsl6d::kMaxPSweeps) return false;
    int a = sw[i].dim, b = -1;
    for (int k = 1; k < cnt; ++k) {
        const int d = sw[i + k].dim;
        if (d == a || d == b) continue;
        if (b >= 0) return false;
        b = d;
    }
    if (b < 0) return false;
    if (a > b) { const int t = a; a = b; b = t; }
    const int32_t* n = c->g.n;
    size_t inner_b = 1, mid = 1, outer = 1;
    for (int d = b + 1; d < 6; ++d) inner_b *= (size_t)n[d];
    for (int d = a + 1; d < b; ++d) mid *= (size_t)n[d];
    for (int d = 0; d < a; ++d) outer *= (size_t)n[d];
    if (inner_b < (size_t)bsl6d::kPTileC || inner_b % (size_t)bsl6d::kPTileC) return false;
    if (c->npts > 0xFFFFFFFFull) return false;                        // 32-bit pencil indices in the kernel
    bsl6d::PTileChoice pc;
    if (!bsl6d::ptile_available() || !ptile_lookup(c->q, n[a], n[b], is_periodic(c, a), is_periodic(c, b), pc)) return false;
    if (!c->fuse_all) {
        // Policy from measurement: one TMA box per tile keeps 64 KB in flight per SM, which is
        // enough when the 64-byte rows of a tile lie close together (v1+v2: 256 B apart; x3+v1: 8 KB) and not when every
        // row sits in its own DRAM page (x2+x3: 256 KB apart -- there the round-1 kernels, which keep 2 x 64 KB of
        // register-staged loads in flight, are faster).
        const size_t strideB_bytes = inner_b * sizeof(double);
        if (strideB_bytes > ((size_t)64 << 10)) return false;
    }
    const size_t tiles = outer * mid * (inner_b / (size_t)bsl6d::kPTileC);
    if (tiles > 0x7FFFFFFFull) return false;
    p.first = i; p.count = cnt; p.fused = false; p.pattern = 0; p.vblock = false; p.ptile = true; p.pc = pc;
    p.dim_a = a; p.dim_b = b;
    return true;
}

// Can sweeps [i, i+cnt) -- all of them along velocity dims -- run as one whole-v-block pass?
bool try_vblock(const bsl6d_ctx* c, const SweepDesc* sw, int i, int cnt, Pass& p) {
    if (cnt < 2 || cnt > bsl6d::kMaxVSweeps) return false;
    for (int k = 0; k < cnt; ++k) {
        if (sw[i + k].dim < 3) return false;
        // Policy from measurement: a v3 sweep inside the pass needs the block in the other cut
        // (re-tiled through L2: store, cluster barrier, reload -- or, slower still, read through distributed shared
        // memory) and costs more than the v3 sweep as a pass of its own; only fusion mode 2 takes it.
        if (sw[i + k].dim == 5 && !c->fuse_all) return false;
    }
    const int32_t* n = c->g.n;
    bsl6d::VBlockChoice vc;
    if (!bsl6d::vblock_lookup(n[3], n[4], n[5], c->q, vc)) return false;
    const size_t nx = (size_t)n[0] * n[1] * n[2];
    if (c->npts > 0xFFFFFFFFull || nx * (size_t)vc.cl > 0x7FFFFFFFull) return false;
    p.first = i; p.count = cnt; p.fused = false; p.pattern = 0; p.vblock = true; p.vc = vc; p.ptile = false;
    return true;
}

// tma_ok = false keeps the TMA-fed passes (persistent tile, whole-v-block) out of the plan: their tensor maps need
// 16-byte aligned arrays, and the header only asks for 8.  Such chains run as round-1 tile passes or single sweeps.
int plan_passes(const bsl6d_ctx* c, const SweepDesc* sw, int ns, std::vector<Pass>& passes, bool tma_ok = true) {
    passes.clear();
    for (int i = 0; i < ns; ++i) {
        int rc = check_sweep_desc(c, sw[i]);
        if (rc) return rc;
        KernelChoice kc;
        rc = choose_kernel(c, sw[i].dim, kc);
        if (rc) return rc;
    }
    // Cheapest plan over the chain (dynamic programme from the back).  Costs are in units of ONE single sweep of the
    // same grid (a 16 B/point pass at HBM speed) and come from the per-pass timings of DESIGN.md section 10
    // (C2: q = 8, C5: q = 10, in-step medians); they only have to rank the alternatives:
    //   single sweep                      1
    //   persistent tile pass, n sweeps    0.45 + (0.035 q + 0.07) n      (+0.3 when an extent exceeds 32: two buffers)
    //   v-block pass, n sweeps            1.10 + (0.020 q + 0.03) n      (+1.3 per switch between v1/v2 sweeps and v3
    //                                                                      sweeps: the block is re-tiled through L2)
    //   round-1 tile kernels              pair 0.7 + 0.10 q,  a-b-a triple 0.7 + 0.13 q
    // Fusion mode 2 ("wherever a kernel exists") counts passes instead: every pass costs 1, ties go to the larger group.
    // pick[i] > 0: a round-1 tile pass over that many sweeps (or a single sweep); pick[i] >= 100: a persistent tile pass
    // over pick[i]-100 sweeps; pick[i] < 0: a v-block pass over -pick[i] sweeps.
    const double q = (double)c->q;
    const bool by_count = c->fuse_all != 0;
    const double eps = 1e-9;
    std::vector<double> best(ns + 1, 0.0);
    std::vector<int> pick(ns + 1, 1);
    std::vector<Pass> cand2(ns), cand3(ns), candv(ns), candp(ns);
    auto better = [&](double total, double cur) { return total < cur - eps || (by_count && total < cur + eps); };
    for (int i = ns - 1; i >= 0; --i) {
        best[i] = 1.0 + best[i + 1];
        pick[i] = 1;
        if (c->fusion && c->use_fused && i + 1 < ns && try_fuse(c, sw, i, 2, cand2[i])) {
            const double total = (by_count ? 1.0 : 0.7 + 0.10 * q) + best[i + 2];
            if (total < best[i] - eps) { best[i] = total; pick[i] = 2; }
        }
        if (c->fusion && c->use_fused && i + 2 < ns && try_fuse(c, sw, i, 3, cand3[i])) {
            const double total = (by_count ? 1.0 : 0.7 + 0.13 * q) + best[i + 3];
            if (total < best[i] - eps) { best[i] = total; pick[i] = 3; }
        }
        if (c->fusion && c->use_ptile && tma_ok) {
            for (int len = 2; len <= bsl6d::kMaxPSweeps && i + len <= ns; ++len) {
                Pass p;
                if (!try_ptile(c, sw, i, len, p)) break;      // a third dim (or the unit-stride dim) ends the chain
                const bool big = p.pc.na > 32 || p.pc.nb > 32;
                const double cost = by_count ? 1.0 : 0.45 + (0.035 * q + 0.07) * len + (big ? 0.3 : 0.0);
                const double total = cost + best[i + len];
                if (better(total, best[i])) { best[i] = total; pick[i] = 100 + len; candp[i] = p; }
            }
        }
        if (c->fusion && c->use_vblock && tma_ok) {
            int run = 0;
            while (i + run < ns && sw[i + run].dim >= 3 && (c->fuse_all || sw[i + run].dim != 5) &&
                   run < bsl6d::kMaxVSweeps)
                ++run;
            int switches = 0;
            for (int len = 1; len <= run; ++len) {
                if (len > 1 && (sw[i + len - 1].dim == 5) != (sw[i + len - 2].dim == 5)) ++switches;
                if (len < c->vblock_min) continue;
                Pass p;
                if (!try_vblock(c, sw, i, len, p)) break;
                const double cost = by_count ? 1.0 : 1.10 + (0.020 * q + 0.03) * len + 1.3 * switches;
                const double total = cost + best[i + len];
                if (better(total, best[i])) { best[i] = total; pick[i] = -len; candv[i] = p; }
            }
        }
    }
    for (int i = 0; i < ns;) {
        if (pick[i] < 0) { passes.push_back(candv[i]); i += -pick[i]; }
        else if (pick[i] >= 100) { passes.push_back(candp[i]); i += pick[i] - 100; }
        else if (pick[i] == 3) { passes.push_back(cand3[i]); i += 3; }
        else if (pick[i] == 2) { passes.push_back(cand2[i]); i += 2; }
        else {
            Pass p;
            std::memset(&p, 0, sizeof(p));
            p.first = i; p.count = 1;
            passes.push_back(p);
            i += 1;
        }
    }
    return BSL6D_OK;
}

int launch_fused(bsl6d_ctx* c, const double* f_in, double* f_out, const SweepDesc* sw, const Pass& p,
                 cudaStream_t stream) {
    const int a = sw[p.first].dim, b = sw[p.first + 1].dim;
    const int32_t* n = c->g.n;
    size_t inner_b = 1, mid = 1, outer = 1;
    for (int d = b + 1; d < 6; ++d) inner_b *= (size_t)n[d];
    for (int d = a + 1; d < b; ++d) mid *= (size_t)n[d];
    for (int d = 0; d < a; ++d) outer *= (size_t)n[d];
    bsl6d::FusedArgs fa;
    std::memset(&fa, 0, sizeof(fa));
    fa.in = f_in;
    fa.out = f_out;
    fa.mid = (uint32_t)mid;
    fa.inner_b = (uint32_t)inner_b;
    fa.nchunks = (uint32_t)(inner_b / (size_t)p.fc.C);
    for (int k = 0; k < p.count; ++k) {
        const SweepDesc& s = sw[p.first + k];
        fa.sw[k].src = s.src;
        fa.sw[k].scale = s.scale;
        int rc = build_src_terms(n, s.dim, s.mask, fa.sw[k].terms);
        if (rc) return rc;
    }
    cudaError_t e;
    if (int rcs = allow_smem(c, p.fc.fn, p.fc.smem)) return rcs;
    const unsigned grid = (unsigned)(outer * mid * (size_t)fa.nchunks);
    void* args[] = {(void*)&fa};
    e = cudaLaunchKernel(p.fc.fn, dim3(grid), dim3(p.fc.threads), args, p.fc.smem, stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->launches += 1;
    return BSL6D_OK;
}

int launch_vblock(bsl6d_ctx* c, const double* f_in, double* f_out, const SweepDesc* sw, const Pass& p,
                  cudaStream_t stream) {
    const int32_t* n = c->g.n;
    bsl6d::VBlockArgs va;
    std::memset(&va, 0, sizeof(va));
    va.nsweeps = (uint32_t)p.count;
    va.nx = (uint32_t)((size_t)n[0] * n[1] * n[2]);
    for (int k = 0; k < p.count; ++k) {
        const SweepDesc& s = sw[p.first + k];
        va.sw[k].src = s.src;
        va.sw[k].scale = s.scale;
        va.sw[k].dim = s.dim;
        int rc = build_src_terms(n, s.dim, s.mask, va.sw[k].terms);
        if (rc) return rc;
    }
    if (int rcs = allow_smem(c, p.vc.fn, p.vc.smem)) return rcs;
    cudaError_t e = bsl6d::vblock_launch(p.vc, f_in, f_out, va.nx, n[3], va, stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->launches += 1;
    return BSL6D_OK;
}

int launch_ptile(bsl6d_ctx* c, const double* f_in, double* f_out, const SweepDesc* sw, const Pass& p,
                 cudaStream_t stream) {
    const int a = p.dim_a, b = p.dim_b;
    const int32_t* n = c->g.n;
    size_t inner_b = 1, mid = 1, outer = 1;
    for (int d = b + 1; d < 6; ++d) inner_b *= (size_t)n[d];
    for (int d = a + 1; d < b; ++d) mid *= (size_t)n[d];
    for (int d = 0; d < a; ++d) outer *= (size_t)n[d];
    bsl6d::PTileArgs pa;
    std::memset(&pa, 0, sizeof(pa));
    pa.nsweeps = (uint32_t)p.count;
    pa.mid = (uint32_t)mid;
    pa.inner_b = (uint32_t)inner_b;
    pa.nchunks = (uint32_t)(inner_b / (size_t)bsl6d::kPTileC);
    pa.ntiles = (uint32_t)(outer * mid * (size_t)pa.nchunks);
    for (int k = 0; k < p.count; ++k) {
        const SweepDesc& s = sw[p.first + k];
        pa.sw[k].src = s.src;
        pa.sw[k].scale = s.scale;
        pa.sw[k].along_b = s.dim == b ? 1 : 0;
        int rc = build_src_terms(n, s.dim, s.mask, pa.sw[k].terms);
        if (rc) return rc;
    }
    if (int rcs = allow_smem(c, p.pc.fn, p.pc.smem)) return rcs;
    cudaError_t e = bsl6d::ptile_launch(p.pc, f_in, f_out, outer, mid, inner_b, pa, c->num_sms, stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->launches += 1;
    return BSL6D_OK;
}

int launch_pass(bsl6d_ctx* c, const double* src, double* dst, const SweepDesc* sw, const Pass& p, cudaStream_t st) {
    if (p.ptile) return launch_ptile(c, src, dst, sw, p, st);
    if (p.vblock) return launch_vblock(c, src, dst, sw, p, st);
    if (p.fused) return launch_fused(c, src, dst, sw, p, st);
    const SweepDesc& s = sw[p.first];
    return launch_sweep(c, src, dst, s.dim, s.src, s.mask, s.scale, st);
}

bool partial_overlap(const bsl6d_ctx* c, const void* x, const void* y) {
    if (x == y) return false;
    const size_t bytes = c->npts * sizeof(double);
    const char* a = (const char*)x;
    const char* b = (const char*)y;
    return a < b + bytes && b < a + bytes;
}

// Both arrays on 16-byte boundaries (what a TMA tensor map needs)?  A null pointer counts as aligned.
bool aligned16(const void* x, const void* y) { return (((uintptr_t)x | (uintptr_t)y) & 15u) == 0; }

// f_in -> f_out: the first pass reads f_in and writes f_out, the others run in place on f_out.
int run_sequence_in_out(bsl6d_ctx* c, const double* f_in, double* f_out, const SweepDesc* sw, int ns,
                        cudaStream_t st) {
    if (!c || !f_in || !f_out || ns < 0 || (ns > 0 && !sw)) return BSL6D_EINVAL;
    if (partial_overlap(c, f_in, f_out)) return BSL6D_EALIAS;
    std::vector<Pass> passes;
    int rc = check_device(c);
    if (rc) return rc;
    rc = plan_passes(c, sw, ns, passes, aligned16(f_in, f_out));
    if (rc) return rc;
    if (passes.empty()) {
        if (f_in != f_out) {
            cudaError_t e = cudaMemcpyAsync(f_out, f_in, c->npts * sizeof(double), cudaMemcpyDeviceToDevice, st);
            if (e != cudaSuccess) return cuda_fail(c, e);
        }
        return BSL6D_OK;
    }
    const double* cur = f_in;
    for (const Pass& p : passes) {
        rc = launch_pass(c, cur, f_out, sw, p, st);
        if (rc) return rc;
        cur = f_out;
    }
    return BSL6D_OK;
}

// In place on f, ping-ponging with f_tmp when given; the result always lands in f.
int run_sequence_pingpong(bsl6d_ctx* c, double* f, double* f_tmp, const SweepDesc* sw, int ns, cudaStream_t st) {
    if (!c || !f) return BSL6D_EINVAL;
    if (f_tmp && (f_tmp == f || partial_overlap(c, f, f_tmp))) return BSL6D_EALIAS;
    std::vector<Pass> passes;
    int rc = check_device(c);
    if (rc) return rc;
    rc = plan_passes(c, sw, ns, passes, aligned16(f, f_tmp));
    if (rc) return rc;
    const int np = (int)passes.size();
    double* cur = f;
    double* other = f_tmp;
    for (int s = 0; s < np; ++s) {
        double* dst = cur;
        if (other && !((np & 1) && s == 0)) dst = other;     // odd count: the first pass runs in place
        rc = launch_pass(c, cur, dst, sw, passes[s], st);
        if (rc) return rc;
        if (dst != cur) { other = cur; cur = dst; }
    }
    return BSL6D_OK;
}

struct Shear { int dim; int src_dim; double scale; };

constexpr int kMaxShears = 48;                               // 16 axis rotations x 3 shears

// Three shears of a rotation about coordinate axis `ax` by `theta` (see bsl6d_rotate in the header).
void axis_shears(const bsl6d_ctx* c, int ax, double theta, Shear* out) {
    const int a = (ax + 1) % 3, b = (ax + 2) % 3;
    const double t = std::tan(0.5 * theta), s = std::sin(theta);
    out[0] = Shear{3 + a, 3 + b, t / c->g.dx[3 + a]};       // foot displacement -v_b tan(theta/2)
    out[1] = Shear{3 + b, 3 + a, -s / c->g.dx[3 + b]};      // foot displacement +v_a sin(theta)
    out[2] = out[0];
}

// The shear sequence of the rotation by B*dt.  B along one coordinate axis: three shears.  B in general position
// (reading R1): with B/|B| = (sin vt cos ph, sin vt sin ph, cos vt) and theta = |B| dt,
// R(b, theta) = Rz(ph) Ry(vt) Rz(theta) Ry(-vt) Rz(-ph); the factors are applied left to right, each as three shears,
// a factor above pi/2 in ceil(|angle| / (pi/2)) equal pieces.  |theta| <= 2 pi.  `out` holds kMaxShears entries.
int plan_rotation(const bsl6d_ctx* c, const double B[3], double dt, Shear* out, int* count) {
    *count = 0;
    if (!std::isfinite(dt)) return BSL6D_EINVAL;
    int ax = -1, nz = 0;
    for (int i = 0; i < 3; ++i) {
        if (!std::isfinite(B[i])) return BSL6D_EINVAL;
        if (B[i] != 0.0) { ax = i; ++nz; }
    }
    if (nz == 0) return BSL6D_OK;
    const double half_pi = 1.5707963267948966;
    if (nz == 1) {
        // reading R2: above pi/2 in equal pieces (tan(theta/2) diverges at pi); one piece = the plain three shears
        const double theta = B[ax] * dt;
        if (std::fabs(theta) > 6.283185307179586477) return BSL6D_EUNSUPPORTED;
        int pieces = (int)std::ceil(std::fabs(theta) / half_pi);
        if (pieces < 1) pieces = 1;
        for (int k = 0; k < pieces; ++k) axis_shears(c, ax, theta / (double)pieces, out + 3 * k);
        *count = 3 * pieces;
        return BSL6D_OK;
    }
    const double bn = std::sqrt(B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
    const double theta = bn * dt;
    if (std::fabs(theta) > 6.283185307179586477) return BSL6D_EUNSUPPORTED;
    const double vt = std::acos(B[2] / bn);
    const double ph = std::atan2(B[1], B[0]);
    const int axes[5] = {2, 1, 2, 1, 2};
    const double ang[5] = {ph, vt, theta, -vt, -ph};
    int n = 0;
    for (int i = 0; i < 5; ++i) {
        if (ang[i] == 0.0) continue;
        const int pieces = (int)std::ceil(std::fabs(ang[i]) / half_pi);
        for (int k = 0; k < pieces && n + 3 <= kMaxShears; ++k) {
            axis_shears(c, axes[i], ang[i] / (double)pieces, out + n);
            n += 3;
        }
    }
    *count = n;
    return BSL6D_OK;
}

// ---- field step ------------------------------------------------------------------------------
int field_setup(bsl6d_ctx* c) {
    if (c->field_ready) return BSL6D_OK;
    const size_t nx = (size_t)c->g.n[0] * c->g.n[1] * c->g.n[2];
    if (nx > 0x7FFFFFFFull) return BSL6D_EUNSUPPORTED;
    // A buffer that an earlier, failed attempt already allocated is kept and reused (nothing is allocated twice).
    for (int d = 0; d < 3; ++d) {
        const int n = c->g.n[d];
        std::vector<double2> w((size_t)n);
        for (int m = 0; m < n; ++m) {
            const double ang = -2.0 * 3.14159265358979323846 * (double)m / (double)n;
            w[(size_t)m] = make_double2(std::cos(ang), std::sin(ang));
        }
        if (!c->tw[d] && cudaMalloc((void**)&c->tw[d], (size_t)n * sizeof(double2)) != cudaSuccess) {
            (void)cudaGetLastError();
            c->tw[d] = nullptr;
            return BSL6D_ENOMEM;
        }
        cudaError_t e = cudaMemcpy(c->tw[d], w.data(), (size_t)n * sizeof(double2), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) return cuda_fail(c, e);
    }
    for (int k = 0; k < 5; ++k)
        if (!c->fld[k] && cudaMalloc((void**)&c->fld[k], nx * sizeof(double2)) != cudaSuccess) {
            (void)cudaGetLastError();
            c->fld[k] = nullptr;
            return BSL6D_ENOMEM;
        }
    c->field_ready = 1;
    return BSL6D_OK;
}

int field_solve(bsl6d_ctx* c, const double* rho, int adiabatic, double c1, double e_fac, double* const E[3],
                cudaStream_t st) {
    if (!c || !rho || !E || !E[0] || !E[1] || !E[2]) return BSL6D_EINVAL;
    if (!std::isfinite(c1) || !std::isfinite(e_fac)) return BSL6D_EINVAL;
    if (c->open_x[0] || c->open_x[1] || c->open_x[2]) return BSL6D_EUNSUPPORTED;   // spectral solve: periodic x only
    int rc = check_device(c);
    if (rc) return rc;
    rc = field_setup(c);
    if (rc) return rc;
    const uint32_t n0 = (uint32_t)c->g.n[0], n1 = (uint32_t)c->g.n[1], n2 = (uint32_t)c->g.n[2];
    const uint32_t total = n0 * n1 * n2;
    const unsigned T = 128, grid = (total + T - 1) / T;
    double2 *A = c->fld[0], *B = c->fld[1];
    using namespace bsl6d;
    // forward: axis 2 (real in), axis 1, axis 0
    dft_axis_kernel<true, false><<<grid, T, 0, st>>>(rho, A, c->tw[2], n2, 1u, total, 0, 1.0);
    {   // every later launch has the same shape on the same stream: if this one was accepted the others are too,
        // and if it was not, nothing has been enqueued
        cudaError_t e0 = cudaGetLastError();
        if (e0 != cudaSuccess) return cuda_fail(c, e0);
    }
    dft_axis_kernel<false, false><<<grid, T, 0, st>>>(A, B, c->tw[1], n1, n2, total, 0, 1.0);
    dft_axis_kernel<false, false><<<grid, T, 0, st>>>(B, A, c->tw[0], n0, n1 * n2, total, 0, 1.0);
    FieldArgs fa;
    for (int d = 0; d < 3; ++d) { fa.n[d] = (uint32_t)c->g.n[d]; fa.L[d] = (double)c->g.n[d] * c->g.dx[d]; }
    fa.adiabatic = adiabatic;
    fa.c1 = c1;
    spectral_field_kernel<<<grid, T, 0, st>>>(A, c->fld[2], c->fld[3], c->fld[4], fa);
    const double scale = e_fac / (double)total;
    for (int d = 0; d < 3; ++d) {
        dft_axis_kernel<false, false><<<grid, T, 0, st>>>(c->fld[2 + d], A, c->tw[0], n0, n1 * n2, total, 1, 1.0);
        dft_axis_kernel<false, false><<<grid, T, 0, st>>>(A, B, c->tw[1], n1, n2, total, 1, 1.0);
        dft_axis_kernel<false, true><<<grid, T, 0, st>>>(B, E[d], c->tw[2], n2, 1u, total, 1, scale);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->launches += 13;
    return BSL6D_OK;
}

}  // namespace

extern "C" {

int bsl6d_version(void) { return BSL6D_VERSION; }

const char* bsl6d_strerror(int code) {
    switch (code) {
        case BSL6D_OK: return "ok";
        case BSL6D_EINVAL: return "invalid argument";
        case BSL6D_EALIAS: return "f_in and f_out overlap partially";
        case BSL6D_EUNSUPPORTED: return "unsupported configuration";
        case BSL6D_ECUDA: return "CUDA runtime error";
        case BSL6D_ENOMEM: return "out of memory";
        case BSL6D_ESCRATCH: return "needs more scratch than the library's static device array holds";
        default: return "unknown error";
    }
}

int bsl6d_create(const bsl6d_grid* grid, int degree, bsl6d_ctx** out) {
    if (!grid || !out) return BSL6D_EINVAL;
    *out = nullptr;
    if (degree < 1 || degree > 11 || !(degree & 1)) return BSL6D_EINVAL;
    size_t npts = 1, nn = 0;
    for (int d = 0; d < 6; ++d) {
        if (grid->n[d] < 1 || !(grid->dx[d] > 0.0) || !std::isfinite(grid->dx[d]) || !std::isfinite(grid->lo[d]))
            return BSL6D_EINVAL;
        if (npts > (size_t)1 << 40) return BSL6D_EUNSUPPORTED;
        npts *= (size_t)grid->n[d];
        nn += (size_t)grid->n[d];
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return BSL6D_ECUDA; }
    bsl6d_ctx* c = new (std::nothrow) bsl6d_ctx();
    if (!c) return BSL6D_ENOMEM;
    std::memset(c, 0, sizeof(*c));
    c->g = *grid;
    c->q = degree + 1;
    c->device = dev;
    c->npts = npts;
    c->fusion = 1;
    c->fuse_all = 0;
    c->use_vblock = 1;
    c->use_ptile = 1;
    c->use_fused = 1;
    c->fusion_mode = 1;
    c->vblock_min = 2;
    {
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
            (void)cudaGetLastError();
            sms = 148;
        }
        c->num_sms = sms;
    }

    std::vector<double> nodes(nn);
    size_t off = 0;
    for (int d = 0; d < 6; ++d) {
        c->node_off[d] = off;
        for (int i = 0; i < grid->n[d]; ++i) {
            const double step = (double)i * grid->dx[d];      // one multiply, one add (no contraction: see build flags)
            nodes[off + i] = grid->lo[d] + step;
        }
        off += (size_t)grid->n[d];
    }
    e = cudaMalloc((void**)&c->d_nodes, nn * sizeof(double));
    if (e != cudaSuccess) { delete c; (void)cudaGetLastError(); return e == cudaErrorMemoryAllocation ? BSL6D_ENOMEM : BSL6D_ECUDA; }
    e = cudaMemcpy(c->d_nodes, nodes.data(), nn * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(c->d_nodes); delete c; (void)cudaGetLastError(); return BSL6D_ECUDA; }

    // density plan: chunks of <= 32768 doubles (256 KB) per block
    const size_t seg = (size_t)grid->n[3] * grid->n[4] * grid->n[5];
    const size_t nx = (size_t)grid->n[0] * grid->n[1] * grid->n[2];
    const size_t target = 32768;
    size_t G = (seg + target - 1) / target;
    size_t chunk = (seg + G - 1) / G;
    chunk = (chunk + 1) & ~(size_t)1;                           // even => 16-byte aligned chunks
    G = (seg + chunk - 1) / chunk;
    c->dens_G = (uint32_t)G;
    c->dens_chunk = chunk;
    if (G > 1) {
        e = cudaMalloc((void**)&c->d_part, nx * G * sizeof(double));
        if (e != cudaSuccess) { cudaFree(c->d_nodes); delete c; (void)cudaGetLastError(); return BSL6D_ENOMEM; }
    }
    *out = c;
    return BSL6D_OK;
}

void bsl6d_destroy(bsl6d_ctx* c) {
    if (!c) return;
    for (int sl = 0; sl < 2; ++sl) {
        if (c->h_stream[sl]) { cudaStreamSynchronize(c->h_stream[sl]); cudaStreamDestroy(c->h_stream[sl]); }
        cudaFree(c->h_f[sl]);
        cudaFree(c->h_small[sl]);
        cudaFree(c->h_part[sl]);
    }
    for (int k = 0; k < 5; ++k) cudaFree(c->fld[k]);
    for (int k = 0; k < 3; ++k) cudaFree(c->tw[k]);
    cudaFree(c->d_part);
    cudaFree(c->d_nodes);
    (void)cudaGetLastError();
    delete c;
}

int bsl6d_last_cuda_error(const bsl6d_ctx* c) { return c ? c->last_cuda : 0; }
long long bsl6d_launch_count(const bsl6d_ctx* c) { return c ? c->launches : 0; }

int bsl6d_kernel_name(const bsl6d_ctx* c, int dim, char* buf, int buflen) {
    if (!c || !buf || buflen < 1 || dim < 0 || dim > 5) return BSL6D_EINVAL;
    KernelChoice k;
    int rc = choose_kernel(c, dim, k);
    if (rc) return rc;
    const char* kind = k.kind == 0 ? "strided" : (k.kind == 1 ? "unit" : "generic");
    if (k.kind == 1)
        std::snprintf(buf, (size_t)buflen, "%s<N=%d,Q=%d,S=%d,T=%d>", kind, (int)c->g.n[dim], c->q, k.gen_T, k.threads);
    else if (k.kind == 0 && k.gen_T > 1)
        std::snprintf(buf, (size_t)buflen, "%s<N=%d,Q=%d,%s,S=%d,T=%d>", kind, (int)c->g.n[dim], c->q,
                      is_periodic(c, dim) ? "periodic" : "zero", k.gen_T, k.threads);
    else if (k.kind == 0 && k.fn_oop)                         // f_in != f_out runs the streaming variant
        std::snprintf(buf, (size_t)buflen, "stream<N=%d,Q=%d,%s,T=%d> (in place: strided<T=%d>)", (int)c->g.n[dim], c->q,
                      is_periodic(c, dim) ? "periodic" : "zero", k.oop_threads, k.threads);
    else
        std::snprintf(buf, (size_t)buflen, "%s<N=%d,Q=%d,%s,T=%d>", kind, (int)c->g.n[dim], c->q,
                      is_periodic(c, dim) ? "periodic" : "zero", k.threads);
    return BSL6D_OK;
}

int bsl6d_advect_generic(bsl6d_ctx* c, const double* f_in, double* f_out, int dim, const double* src,
                         unsigned src_dim_mask, double scale, void* stream) {
    return launch_sweep(c, f_in, f_out, dim, src, src_dim_mask, scale, (cudaStream_t)stream);
}

int bsl6d_advect(bsl6d_ctx* c, const double* f_in, double* f_out, int dim, const double* shift_source, double dt,
                 void* stream) {
    if (!c || dim < 0 || dim > 5 || !std::isfinite(dt)) return BSL6D_EINVAL;
    const double scale = dt / c->g.dx[dim];
    if (dim < 3) {
        const double* s = shift_source ? shift_source : c->d_nodes + c->node_off[dim + 3];
        return launch_sweep(c, f_in, f_out, dim, s, 1u << (dim + 3), scale, (cudaStream_t)stream);
    }
    if (!shift_source) return BSL6D_EINVAL;
    return launch_sweep(c, f_in, f_out, dim, shift_source, 0x7u, scale, (cudaStream_t)stream);
}

int bsl6d_advect_x1_peer(bsl6d_ctx* c, const double* f_in, const double* f_left, const double* f_right, double* f_out,
                         int halo_planes, const double* shift_source, double dt, void* stream) {
    if (!c || !f_in || !f_left || !f_right || !f_out || !std::isfinite(dt)) return BSL6D_EINVAL;
    const int32_t* n = c->g.n;
    if (halo_planes < c->q / 2 || halo_planes > n[0]) return BSL6D_EINVAL;
    if (int rcd = check_device(c)) return rcd;
    // out of place against all three inputs: the neighbours read this slab's input while it is swept
    if (f_out == f_in || f_out == f_left || f_out == f_right || partial_overlap(c, f_in, f_out) ||
        partial_overlap(c, f_left, f_out) || partial_overlap(c, f_right, f_out))
        return BSL6D_EALIAS;
    size_t inner = 1;
    for (int d = 1; d < 6; ++d) inner *= (size_t)n[d];
    if (inner > 0xFFFFFFFFull) return BSL6D_EUNSUPPORTED;
    const double* ssrc = shift_source ? shift_source : c->d_nodes + c->node_off[3];
    if (const void* sfn = peer_stream_fn(n[0], c->q)) {
        // compiled extent: the streaming register kernel, rows beyond the slab loaded from the neighbours' arrays
        SweepArgs sa;
        std::memset(&sa, 0, sizeof(sa));
        sa.in = f_in;
        sa.left = f_left;
        sa.right = f_right;
        sa.out = f_out;
        sa.src = ssrc;
        sa.scale = dt / c->g.dx[0];
        sa.inner = (uint32_t)inner;
        sa.outer = 1u;
        sa.n = (uint32_t)n[0];
        int rcs = build_src_terms(n, 0, 1u << 3, sa.terms);
        if (rcs) return rcs;
        const unsigned T = 128;
        unsigned grid;
        if (inner % 32 != 0) {
            sa.ti_log2 = bsl6d::kFlatPencils;
            sa.nib = (uint32_t)inner;
            grid = (unsigned)((inner + T - 1) / T);
        } else {
            sa.ti_log2 = ceil_pow2_log2(inner < T ? inner : T);
            const uint32_t TI = 1u << sa.ti_log2, TO = T / TI;
            sa.nib = (uint32_t)((inner + TI - 1) / TI);
            grid = sa.nib * ((1u + TO - 1) / TO);
        }
        void* sargs[] = {(void*)&sa};
        cudaError_t es = cudaLaunchKernel(sfn, dim3(grid), dim3(T), sargs, 0, (cudaStream_t)stream);
        if (es != cudaSuccess) return cuda_fail(c, es);
        es = cudaGetLastError();
        if (es != cudaSuccess) return cuda_fail(c, es);
        c->launches += 1;
        return BSL6D_OK;
    }
    const size_t rows = (size_t)n[0] + 2 * (size_t)halo_planes;
    int T = 64;
    if (rows * T * sizeof(double) > 200 * 1024) T = 32;
    if (rows * T * sizeof(double) > 200 * 1024) return BSL6D_EUNSUPPORTED;
    const void* fn = T == 64 ? peer_by_q<64>(c->q) : peer_by_q<32>(c->q);
    if (!fn) return BSL6D_EUNSUPPORTED;
    bsl6d::PeerArgs a;
    std::memset(&a, 0, sizeof(a));
    a.in = f_in;
    a.left = f_left;
    a.right = f_right;
    a.out = f_out;
    a.src = ssrc;
    a.scale = dt / c->g.dx[0];
    a.inner = (uint32_t)inner;
    a.n = (uint32_t)n[0];
    a.w = (uint32_t)halo_planes;
    int rc = build_src_terms(n, 0, 1u << 3, a.terms);
    if (rc) return rc;
    const size_t smem = rows * T * sizeof(double);
    rc = allow_smem(c, fn, smem);
    if (rc) return rc;
    void* args[] = {(void*)&a};
    const unsigned grid = (unsigned)((inner + (size_t)T - 1) / (size_t)T);
    cudaError_t e = cudaLaunchKernel(fn, dim3(grid), dim3((unsigned)T), args, smem, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->launches += 1;
    return BSL6D_OK;
}

int bsl6d_rotate(bsl6d_ctx* c, const double* f_in, double* f_out, const double B[3], double dt, void* stream) {
    if (!c || !f_in || !f_out || !B) return BSL6D_EINVAL;
    Shear sh[kMaxShears];
    int cnt = 0;
    int rc = plan_rotation(c, B, dt, sh, &cnt);
    if (rc) return rc;
    SweepDesc sw[kMaxShears];
    for (int i = 0; i < cnt; ++i)
        sw[i] = SweepDesc{sh[i].dim, c->d_nodes + c->node_off[sh[i].src_dim], 1u << sh[i].src_dim, sh[i].scale};
    return run_sequence_in_out(c, f_in, f_out, sw, cnt, (cudaStream_t)stream);
}

int bsl6d_strang_step(bsl6d_ctx* c, double* f, double* f_tmp, const double* const E[3], const double B[3], double dt,
                      void* stream) {
    if (!c || !f || !std::isfinite(dt)) return BSL6D_EINVAL;
    SweepDesc steps[9 + kMaxShears];
    int ns = 0;
    const double half = 0.5 * dt;
    for (int d = 0; d < 3; ++d)
        steps[ns++] = SweepDesc{d, c->d_nodes + c->node_off[d + 3], 1u << (d + 3), half / c->g.dx[d]};
    if (E)
        for (int d = 0; d < 3; ++d)
            if (E[d]) steps[ns++] = SweepDesc{3 + d, E[d], 0x7u, dt / c->g.dx[3 + d]};
    if (B) {
        Shear sh[kMaxShears];
        int cnt = 0;
        int rc = plan_rotation(c, B, dt, sh, &cnt);
        if (rc) return rc;
        for (int i = 0; i < cnt; ++i)
            steps[ns++] = SweepDesc{sh[i].dim, c->d_nodes + c->node_off[sh[i].src_dim], 1u << sh[i].src_dim, sh[i].scale};
    }
    for (int d = 0; d < 3; ++d)
        steps[ns++] = SweepDesc{d, c->d_nodes + c->node_off[d + 3], 1u << (d + 3), half / c->g.dx[d]};
    return run_sequence_pingpong(c, f, f_tmp, steps, ns, (cudaStream_t)stream);
}

int bsl6d_advect_seq(bsl6d_ctx* c, const double* f_in, double* f_out, const bsl6d_sweep* sweeps, int nsweeps,
                     void* stream) {
    if (!c || nsweeps < 0 || nsweeps > 64 || (nsweeps > 0 && !sweeps)) return BSL6D_EINVAL;
    SweepDesc sw[64];
    for (int i = 0; i < nsweeps; ++i) {
        const bsl6d_sweep& s = sweeps[i];
        if (s.dim < 0 || s.dim > 5) return BSL6D_EINVAL;
        if (!s.src && s.dim < 3)
            sw[i] = SweepDesc{s.dim, c->d_nodes + c->node_off[s.dim + 3], 1u << (s.dim + 3), s.scale};
        else
            sw[i] = SweepDesc{s.dim, s.src, s.src_dim_mask, s.scale};
    }
    return run_sequence_in_out(c, f_in, f_out, sw, nsweeps, (cudaStream_t)stream);
}

int bsl6d_seq_passes(bsl6d_ctx* c, const bsl6d_sweep* sweeps, int nsweeps) {
    if (!c || nsweeps < 0 || nsweeps > 64 || (nsweeps > 0 && !sweeps)) return BSL6D_EINVAL;
    SweepDesc sw[64];
    static const double dummy = 0.0;
    for (int i = 0; i < nsweeps; ++i) {
        const bsl6d_sweep& s = sweeps[i];
        if (s.dim < 0 || s.dim > 5) return BSL6D_EINVAL;
        if (!s.src && s.dim < 3) sw[i] = SweepDesc{s.dim, &dummy, 1u << (s.dim + 3), s.scale};
        else sw[i] = SweepDesc{s.dim, s.src ? s.src : &dummy, s.src_dim_mask, s.scale};
    }
    std::vector<Pass> passes;
    int rc = plan_passes(c, sw, nsweeps, passes);
    return rc ? rc : (int)passes.size();
}

int bsl6d_set_boundary(bsl6d_ctx* c, int dim, int open) {
    if (!c || dim < 0 || dim > 2 || (open != 0 && open != 1)) return BSL6D_EINVAL;
    const int old = c->open_x[dim];
    c->open_x[dim] = open;
    return old;
}

int bsl6d_set_fusion(bsl6d_ctx* c, int enable) {
    if (!c) return BSL6D_EINVAL;
    if (enable < 0 || enable > 5) return BSL6D_EINVAL;
    const int old = c->fusion_mode;
    c->fusion_mode = enable;
    c->fusion = enable ? 1 : 0;
    c->fuse_all = enable == 2 ? 1 : 0;
    c->use_ptile = (enable == 1 || enable == 2 || enable == 5) ? 1 : 0;   // 3: round-1 tile kernels only; 4: those + v-block passes
    c->use_vblock = (enable == 3 || enable == 5) ? 0 : 1;               // 5: planner without v-block passes
    c->use_fused = 1;
    return old;
}

int bsl6d_advect_pointwise(bsl6d_ctx* c, const double* f_in, double* f_out, int dim, const double* alpha_cells,
                           int q, void* stream) {
    if (!c || !f_in || !f_out || !alpha_cells || dim < 0 || dim > 5) return BSL6D_EINVAL;
    if (q < 1 || !(q & 1)) return BSL6D_EINVAL;
    if (partial_overlap(c, f_in, f_out)) return BSL6D_EALIAS;
    if (alpha_cells == f_out || partial_overlap(c, alpha_cells, f_out)) return BSL6D_EALIAS;
    if (int rcd = check_device(c)) return rcd;
    const int32_t* n = c->g.n;
    size_t inner = 1, outer = 1;
    for (int d = dim + 1; d < 6; ++d) inner *= (size_t)n[d];
    for (int d = 0; d < dim; ++d) outer *= (size_t)n[d];
    if (inner * outer > 0xFFFFFFFFull) return BSL6D_EUNSUPPORTED;
    bsl6d::PointwiseChoice pc;
    if (!bsl6d::pointwise_lookup(n[dim], q, is_periodic(c, dim), inner == 1, pc)) return BSL6D_EUNSUPPORTED;
    bsl6d::PointwiseArgs a;
    std::memset(&a, 0, sizeof(a));
    a.in = f_in;
    a.out = f_out;
    a.alpha = alpha_cells;
    a.inner = (uint32_t)inner;
    a.outer = (uint32_t)outer;
    a.n = (uint32_t)n[dim];
    a.periodic = is_periodic(c, dim) ? 1u : 0u;
    a.pb = (uint32_t)pc.unit;
    a.ld = (uint32_t)(n[dim] | 1);
    unsigned grid;
    if (pc.unit) {
        grid = (unsigned)((outer + (size_t)pc.unit - 1) / (size_t)pc.unit);
    } else {
        a.npencil = (uint32_t)(inner * outer);
        grid = (unsigned)((inner * outer + (size_t)pc.threads - 1) / (size_t)pc.threads);
    }
    cudaError_t e;
    if (int rcs = allow_smem(c, pc.fn, pc.smem)) return rcs;
    void* args[] = {(void*)&a};
    e = cudaLaunchKernel(pc.fn, dim3(grid), dim3(pc.threads), args, pc.smem, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(c, e);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->launches += 1;
    return BSL6D_OK;
}

int bsl6d_field_poisson(bsl6d_ctx* c, const double* rho, double rho_fac, double e_fac, double* const E[3],
                        void* stream) {
    return field_solve(c, rho, 0, rho_fac, e_fac, E, (cudaStream_t)stream);
}

int bsl6d_field_adiabatic(bsl6d_ctx* c, const double* rho, double phi_fac, double e_fac, double* const E[3],
                          void* stream) {
    return field_solve(c, rho, 1, phi_fac, e_fac, E, (cudaStream_t)stream);
}

int bsl6d_vp_step(bsl6d_ctx* c, double* f, double* f_tmp, double* rho, double* const E[3], const double B[3],
                  double dt, int closure, double c1, double e_fac, void* stream) {
    if (!c || !f || !rho || !E || !E[0] || !E[1] || !E[2] || !std::isfinite(dt)) return BSL6D_EINVAL;
    if (closure != 0 && closure != 1) return BSL6D_EINVAL;
    if (!std::isfinite(c1) || !std::isfinite(e_fac)) return BSL6D_EINVAL;
    if (int rcd = check_device(c)) return rcd;
    // the field solve in the middle of the step needs a periodic x grid: say so before the first sweep is enqueued
    if (c->open_x[0] || c->open_x[1] || c->open_x[2]) return BSL6D_EUNSUPPORTED;
    Shear sh[kMaxShears];
    int cnt = 0;
    if (B) {
        int rc = plan_rotation(c, B, dt, sh, &cnt);
        if (rc) return rc;
    }
    int rc = field_setup(c);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const double half = 0.5 * dt;
    SweepDesc xs[3], vs[6 + kMaxShears];
    for (int d = 0; d < 3; ++d) xs[d] = SweepDesc{d, c->d_nodes + c->node_off[d + 3], 1u << (d + 3), half / c->g.dx[d]};
    int nv = 0;
    for (int d = 0; d < 3; ++d) vs[nv++] = SweepDesc{3 + d, E[d], 0x7u, dt / c->g.dx[3 + d]};
    for (int i = 0; i < cnt; ++i)
        vs[nv++] = SweepDesc{sh[i].dim, c->d_nodes + c->node_off[sh[i].src_dim], 1u << sh[i].src_dim, sh[i].scale};
    for (int d = 0; d < 3; ++d) vs[nv++] = xs[d];
    {   // plan both halves before the first launch: a failed call must not leave f half-advanced
        if (f_tmp && (f_tmp == f || partial_overlap(c, f, f_tmp))) return BSL6D_EALIAS;
        std::vector<Pass> dry;
        rc = plan_passes(c, xs, 3, dry);
        if (rc) return rc;
        rc = plan_passes(c, vs, nv, dry);
        if (rc) return rc;
    }
    rc = run_sequence_pingpong(c, f, f_tmp, xs, 3, st);
    if (rc) return rc;
    rc = bsl6d_density(c, f, rho, stream);
    if (rc) return rc;
    rc = field_solve(c, rho, closure, c1, e_fac, E, st);
    if (rc) return rc;
    return run_sequence_pingpong(c, f, f_tmp, vs, nv, st);
}

static int density_impl(bsl6d_ctx* c, const double* f, double* rho, double* part, void* stream);

int bsl6d_density(bsl6d_ctx* c, const double* f, double* rho, void* stream) {
    if (!c || !f || !rho) return BSL6D_EINVAL;
    if (int rcd = check_device(c)) return rcd;
    return density_impl(c, f, rho, c->d_part, stream);
}

int bsl6d_density_scratch(bsl6d_ctx* c, const double* f, double* rho, double* scratch, void* stream) {
    if (!c || !f || !rho || (c->dens_G > 1 && !scratch)) return BSL6D_EINVAL;
    if (int rcd = check_device(c)) return rcd;
    return density_impl(c, f, rho, scratch, stream);
}

long long bsl6d_density_scratch_doubles(const bsl6d_ctx* c) {
    if (!c) return BSL6D_EINVAL;
    if (c->dens_G <= 1) return 0;
    return (long long)((size_t)c->g.n[0] * c->g.n[1] * c->g.n[2] * c->dens_G);
}

// part: nx * G doubles of scratch for the partial sums of split v-blocks (unused when G == 1)
static int density_impl(bsl6d_ctx* c, const double* f, double* rho, double* part, void* stream) {
    const bsl6d_grid& g = c->g;
    const size_t seg = (size_t)g.n[3] * g.n[4] * g.n[5];
    const size_t nx = (size_t)g.n[0] * g.n[1] * g.n[2];
    const double dv3 = g.dx[3] * g.dx[4] * g.dx[5];
    const uint32_t G = c->dens_G;
    if (nx * G > 0x7FFFFFFFull) return BSL6D_EUNSUPPORTED;
    const bool vec = (seg % 2 == 0) && (((uintptr_t)f & 15u) == 0);
    double* out = G == 1 ? rho : part;
    constexpr int T = 256;
    cudaStream_t st = (cudaStream_t)stream;
    if (vec) bsl6d::density_kernel<T, true><<<(unsigned)(nx * G), T, 0, st>>>(f, out, seg, G, c->dens_chunk, dv3);
    else bsl6d::density_kernel<T, false><<<(unsigned)(nx * G), T, 0, st>>>(f, out, seg, G, c->dens_chunk, dv3);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e);
    c->launches += 1;
    if (G > 1) {
        bsl6d::density_finish_kernel<<<(unsigned)((nx + 255) / 256), 256, 0, st>>>(part, rho, nx, G, dv3);
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(c, e);
        c->launches += 1;
    }
    return BSL6D_OK;
}

int bsl6d_run_host_begin(bsl6d_ctx* c, const double* f_in_host, double* f_out_host, const bsl6d_host_op* ops, int nops,
                         int slot) {
    if (!c || !f_in_host || !f_out_host || nops < 0 || (nops > 0 && !ops) || slot < 0 || slot > 1) return BSL6D_EINVAL;
    if (int rcd = check_device(c)) return rcd;
    const bsl6d_grid& g = c->g;
    const size_t nx = (size_t)g.n[0] * g.n[1] * g.n[2];
    const size_t bytes = c->npts * sizeof(double);
    // validate + size the small-buffer arena (one slot per op so that nothing in flight is overwritten)
    size_t small = 0;
    for (int i = 0; i < nops; ++i) {
        const bsl6d_host_op& op = ops[i];
        if (op.kind == 0) {
            if (op.dim < 0 || op.dim > 5 || !std::isfinite(op.dt)) return BSL6D_EINVAL;
            if (op.dim >= 3 && !op.shift_source) return BSL6D_EINVAL;
            if (op.shift_source) small += op.dim < 3 ? (size_t)g.n[op.dim + 3] : nx;
        } else if (op.kind == 1) {
            Shear sh[kMaxShears];
            int cnt;
            int rc = plan_rotation(c, op.B, op.dt, sh, &cnt);
            if (rc) return rc;
        } else if (op.kind == 2) {
            if (!op.rho_host) return BSL6D_EINVAL;
            small += nx;
        } else {
            return BSL6D_EINVAL;
        }
    }
    cudaError_t e;
    if (!c->h_stream[slot]) {
        e = cudaStreamCreateWithFlags(&c->h_stream[slot], cudaStreamNonBlocking);
        if (e != cudaSuccess) return cuda_fail(c, e);
    }
    if (!c->h_f[slot]) {
        e = cudaMalloc((void**)&c->h_f[slot], bytes);
        if (e != cudaSuccess) { (void)cudaGetLastError(); c->h_f[slot] = nullptr; return BSL6D_ENOMEM; }
    }
    if (small > c->h_small_cap[slot]) {
        cudaFree(c->h_small[slot]);
        c->h_small[slot] = nullptr;
        c->h_small_cap[slot] = 0;
        e = cudaMalloc((void**)&c->h_small[slot], small * sizeof(double));
        if (e != cudaSuccess) { (void)cudaGetLastError(); return BSL6D_ENOMEM; }
        c->h_small_cap[slot] = small;
    }
    if (c->dens_G > 1 && !c->h_part[slot]) {                // each slot reduces through scratch of its own
        e = cudaMalloc((void**)&c->h_part[slot], nx * c->dens_G * sizeof(double));
        if (e != cudaSuccess) { (void)cudaGetLastError(); c->h_part[slot] = nullptr; return BSL6D_ENOMEM; }
    }
    cudaStream_t st = c->h_stream[slot];
    e = cudaMemcpyAsync(c->h_f[slot], f_in_host, bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(c, e);
    size_t off = 0;
    int rc = BSL6D_OK;
    for (int i = 0; i < nops && rc == BSL6D_OK; ++i) {
        const bsl6d_host_op& op = ops[i];
        if (op.kind == 0) {
            const double* dsrc = nullptr;
            if (op.shift_source) {
                const size_t cnt = op.dim < 3 ? (size_t)g.n[op.dim + 3] : nx;
                e = cudaMemcpyAsync(c->h_small[slot] + off, op.shift_source, cnt * sizeof(double), cudaMemcpyHostToDevice, st);
                if (e != cudaSuccess) { rc = cuda_fail(c, e); break; }
                dsrc = c->h_small[slot] + off;
                off += cnt;
            }
            rc = bsl6d_advect(c, c->h_f[slot], c->h_f[slot], op.dim, dsrc, op.dt, st);
        } else if (op.kind == 1) {
            rc = bsl6d_rotate(c, c->h_f[slot], c->h_f[slot], op.B, op.dt, st);
        } else {
            rc = density_impl(c, c->h_f[slot], c->h_small[slot] + off, c->h_part[slot], st);
            if (rc == BSL6D_OK) {
                e = cudaMemcpyAsync(op.rho_host, c->h_small[slot] + off, nx * sizeof(double), cudaMemcpyDeviceToHost, st);
                if (e != cudaSuccess) rc = cuda_fail(c, e);
            }
            off += nx;
        }
    }
    if (rc == BSL6D_OK) {
        e = cudaMemcpyAsync(f_out_host, c->h_f[slot], bytes, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) rc = cuda_fail(c, e);
    }
    if (rc != BSL6D_OK) (void)cudaStreamSynchronize(st);    // leave nothing of a failed call in flight
    return rc;
}

int bsl6d_run_host_end(bsl6d_ctx* c, int slot) {
    if (!c || slot < 0 || slot > 1) return BSL6D_EINVAL;
    if (int rcd = check_device(c)) return rcd;
    if (!c->h_stream[slot]) return BSL6D_OK;               // nothing was ever begun on this slot
    cudaError_t e = cudaStreamSynchronize(c->h_stream[slot]);
    if (e != cudaSuccess) return cuda_fail(c, e);
    return BSL6D_OK;
}

int bsl6d_run_host(bsl6d_ctx* c, const double* f_in_host, double* f_out_host, const bsl6d_host_op* ops, int nops) {
    int rc = bsl6d_run_host_begin(c, f_in_host, f_out_host, ops, nops, 0);
    if (rc != BSL6D_OK) return rc;
    return bsl6d_run_host_end(c, 0);
}

}  // extern "C"
