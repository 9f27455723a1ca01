/* bsl6d.h -- C ABI of libbsl6d.so: the split 1-D advection sweep of the 6-D backward semi-Lagrangian
 * Vlasov method of arXiv 2303.05994 ("BSL6D"), hand-written for NVIDIA B200 (sm_100a).
 *
 * Citations are lines of the paper text plus the section / equation they fall in; "reading Sx"
 * refers to the table of readings in DESIGN.md.
 *
 * Data model
 *   f        fp64 distribution function on a 6-D tensor grid, dims d = 0..5 = (x1,x2,x3,v1,v2,v3), extents
 *            n[d], C order: v3 has unit stride, lin = ((((i1*n1+i2)*n2+i3)*n3+j1)*n4+j2)*n5+j3.  This is a
 *            contiguous torch tensor of shape (n0,..,n5) and the paper's on-disk / CPU layout.
 *   nodes    node i of dim d sits at lo[d] + i*dx[d].
 *   bounds   dims 0-2 are periodic with period n[d]*dx[d]; dims 3-5 are extended by zero outside the grid
 *            (BASELINE.json north_star; the paper is silent on the v boundary, reading S6).
 *   stencil  centred Lagrange interpolation of odd degree p on q = p+1 (even) nodes around the foot of the
 *            characteristic, eq (7), for any displacement (integer part + fraction, reading S2).
 *
 * Ownership and execution
 *   Unless a function says HOST, every f / rho / shift-source pointer is a DEVICE pointer owned by the caller,
 *   8-byte aligned (16-byte for best speed: an f / f_tmp / f_out that is not on a 16-byte boundary runs without the
 *   TMA-fed fused passes -- more passes, the same numbers); the library neither allocates nor frees them.  The context owns
 *   only small device tables.  Work is enqueued on the caller's stream (`stream` is a cudaStream_t passed as
 *   void*, NULL = legacy default stream) and the call returns without synchronising.  Functions return 0 or
 *   a negative BSL6D_E* code; a failed call has enqueued nothing.  No exceptions, no printing, no aborts.
 *   There is no CPU fallback anywhere: without a CUDA device bsl6d_create fails with BSL6D_ECUDA.
 *   Preconditions not checked: f finite; |displacement| < 2^30 cells.
 *   Size limits (32-bit index arithmetic in the kernels): a sweep along dim d needs (number of pencils) =
 *   npts / n[d] < 2^32, else BSL6D_EUNSUPPORTED; the fused passes need npts = n0*..*n5 <= 2^32 - 1 -- a larger grid
 *   (48^6 = 98 GB would still fit one B200) is NOT refused: every chain then runs as single sweeps, correct but with
 *   one pass per sweep, and bsl6d_seq_passes reports that count.  bsl6d_density needs n0*n1*n2 * G < 2^31.
 *   A context is not thread-safe: one host thread at a time per context.  Sweeps and rotations of one context may be in
 *   flight on several streams; bsl6d_density with v-blocks above 32768 points (bsl6d_density_scratch lifts that),
 *   bsl6d_field_* and bsl6d_vp_step use work arrays of the context and must not overlap each other in time; each bsl6d_run_host slot is one queue with work
 *   arrays of its own.
 */
#ifndef BSL6D_H
#define BSL6D_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BSL6D_VERSION 100

#if defined(__GNUC__)
#define BSL6D_API __attribute__((visibility("default")))
#else
#define BSL6D_API
#endif

typedef struct bsl6d_ctx bsl6d_ctx;

typedef struct bsl6d_grid {
    int32_t n[6];   /* extents, each >= 1 */
    double lo[6];   /* coordinate of node 0 */
    double dx[6];   /* node spacing, > 0 */
} bsl6d_grid;

enum {
    BSL6D_OK = 0,
    BSL6D_EINVAL = -1,        /* null pointer, bad extent / spacing / degree / dim / mask, non-finite dt */
    BSL6D_EALIAS = -2,        /* f_in and f_out overlap partially (exact aliasing f_in == f_out is legal) */
    BSL6D_EUNSUPPORTED = -3,  /* oblique B turning more than 2 pi; extent without a kernel / too large for on-chip staging */
    BSL6D_ECUDA = -4,         /* CUDA runtime failure; see bsl6d_last_cuda_error */
    BSL6D_ENOMEM = -5,        /* host or device allocation failed */
    BSL6D_ESCRATCH = -6       /* bsl6d_density_static: the problem needs more than BSL6D_STATIC_SCRATCH_DOUBLES of scratch */
};

/* Create a context for `grid` and Lagrange degree `degree` (odd, 1..11; stencil width q = degree+1).
 * Uses the current CUDA device.  *out receives the context (HOST pointer, opaque). */
BSL6D_API int bsl6d_create(const bsl6d_grid* grid, int degree, bsl6d_ctx** out);
BSL6D_API void bsl6d_destroy(bsl6d_ctx* ctx);

/* One 1-D advection sweep along `dim` (eq (5), 74-76: one factor of the split step):
 *     f_out[p, j] = sum_{m=-q/2+1..q/2} l_m(theta_p) * f_in[p, j + k_p + m],
 *     alpha_p = -(shift_source[p] * (dt/dx[dim])) cells,  k_p = floor(alpha_p),  theta_p = alpha_p - k_p
 * for every pencil p (all index combinations of the other five dims).  The foot of the characteristic of
 * output node j is j + alpha_p (reading S1).
 *   dim 0..2 (x_d advection, dX/dt = V): shift_source = n[dim+3] doubles, the velocity of each
 *            v_d node; NULL selects the grid's own nodes lo[dim+3] + i*dx[dim+3].
 *   dim 3..5 (v_d advection by the electric field, dV/dt = (q/m)E): shift_source = n0*n1*n2 doubles, C order,
 *            (q/m)*E_{dim-3}(x); NULL is BSL6D_EINVAL.
 * f_in == f_out is legal (in place). */
BSL6D_API int bsl6d_advect(bsl6d_ctx* ctx, const double* f_in, double* f_out, int dim,
                 const double* shift_source, double dt, void* stream);

/* The primitive behind every named sweep: src is a dense C-order DEVICE array over the dims whose bit is set
 * in src_dim_mask (bit d = dim d; the mask must not contain `dim`; mask 0 = one scalar);
 * alpha_p = -(src[p] * scale) cells (the shift is a function of a subset D of the coordinates). */
BSL6D_API int bsl6d_advect_generic(bsl6d_ctx* ctx, const double* f_in, double* f_out, int dim,
                         const double* src, unsigned src_dim_mask, double scale, void* stream);

/* Rotation of velocity space by the background field, dV/dt = V x B (eq (3)), as velocity shears
 * (BASELINE.json configs[3], reading S7).  B: HOST, 3 doubles, = (q/m)*B0.  Result: f_out(v) = f_in(R(B*dt) v).
 *   B along one coordinate axis c, (a,b,c) cyclic, theta = B[c]*dt: shear v_a by foot displacement -v_b*tan(theta/2),
 *     shear v_b by +v_a*sin(theta), shear v_a again -- three sweeps, ONE fused pass f_in -> f_out where a fused kernel
 *     exists, else f_in -> f_out and two sweeps in place.  |theta| > pi/2 is applied in ceil(|theta|/(pi/2)) equal
 *     pieces of three shears each (tan(theta/2) diverges at pi; reading R2); |theta| > 2 pi is BSL6D_EUNSUPPORTED.
 *   B in general position (reading R1): with B/|B| = (sin vt cos ph, sin vt sin ph, cos vt) and
 *     theta = |B|*dt, R = Rz(ph) Ry(vt) Rz(theta) Ry(-vt) Rz(-ph), the five factors applied left to right, each as
 *     three shears (a factor above pi/2 in equal pieces): 15 or more sweeps, the Rz factors fused.  |theta| <= 2 pi,
 *     else BSL6D_EUNSUPPORTED.
 *   B == 0 copies f_in to f_out. */
BSL6D_API int bsl6d_rotate(bsl6d_ctx* ctx, const double* f_in, double* f_out, const double B[3], double dt, void* stream);

/* One Strang-split time step (order per BASELINE.json configs[4], reading S8), result in f:
 *   x1,x2,x3 with dt/2  ->  v1,v2,v3 with E (dt)  ->  rotation (theta = B_c*dt)  ->  x1,x2,x3 with dt/2.
 * E: HOST array of three DEVICE pointers ((q/m)E_d over x, C order); a NULL entry skips that sweep, E == NULL
 * skips all three.  B: HOST, may be NULL (no rotation).  f_tmp: optional second DEVICE buffer of the size of f;
 * if given the sweeps ping-pong between f and f_tmp, if NULL they run in place.  The numbers are identical. */
BSL6D_API int bsl6d_strang_step(bsl6d_ctx* ctx, double* f, double* f_tmp, const double* const E[3], const double B[3],
                      double dt, void* stream);

/* ---- sequences of sweeps, fused on chip ------------------------------------------------
 * The Lie-split step is a chain of 1-D sweeps.  Wherever consecutive sweeps of a chain act along
 * only two dims a < b (b not the unit-stride dim) -- x1 then x2, x3 then v1, the three shears v_a, v_b, v_a of a
 * rotation -- the library stages tiles [n_a][n_b][C contiguous doubles] in shared memory and applies the two or
 * three sweeps in ONE pass over f: 16 B/point of HBM traffic per pass instead of per sweep.  Per sweep the
 * arithmetic is unchanged, so the numbers are bit-identical to issuing the sweeps one by one.
 * bsl6d_rotate, bsl6d_strang_step and bsl6d_advect_seq all go through this planner; a group without a fused
 * kernel (extent not in {8,16,32,48,64}, degree not in {5,7,9}, inner extent not a multiple of C) silently runs
 * as single sweeps, and so does a PAIR that measurement says does not pay (row segments under 64 bytes, or a tile
 * whose rows lie >= 64 MB apart).  The planner picks the grouping with the fewest passes.
 * bsl6d_set_fusion(ctx, 0) turns grouping off (every sweep its own pass), 1 is the default policy, 2 fuses
 * wherever a kernel exists; for tests and tuning also 3 (round-1 tile kernels only), 4 (those + whole-v-block
 * passes), 5 (the default policy without whole-v-block passes); returns the old setting. */
typedef struct bsl6d_sweep {
    int32_t dim;             /* swept dim 0..5 */
    uint32_t src_dim_mask;   /* dims the shift source is dense over (bit d), must not contain `dim` */
    const double* src;       /* DEVICE; NULL with dim < 3 selects the grid's v_dim nodes (mask is then ignored) */
    double scale;            /* alpha_cells = -(src[p] * scale), as in bsl6d_advect_generic */
} bsl6d_sweep;
/* Apply sweeps[0..nsweeps) in order: the first pass reads f_in and writes f_out, later passes run in place on
 * f_out (f_in == f_out is legal).  nsweeps <= 64; nsweeps == 0 copies. */
BSL6D_API int bsl6d_advect_seq(bsl6d_ctx* ctx, const double* f_in, double* f_out, const bsl6d_sweep* sweeps,
                     int nsweeps, void* stream);
/* Number of passes (kernel launches) bsl6d_advect_seq would use for this chain on 16-byte aligned arrays, or a
 * negative error code. */
BSL6D_API int bsl6d_seq_passes(bsl6d_ctx* ctx, const bsl6d_sweep* sweeps, int nsweeps);
BSL6D_API int bsl6d_set_fusion(bsl6d_ctx* ctx, int enable);

/* ---- slab decomposition along x1 (section 3.3, 323) --------------------
 * The paper distributes f over MPI ranks and gives every rank halo cells around its sub-domain:
 * the interpolation along a distributed dim then reads the neighbour's points from the halo instead of wrapping.
 * Here the slowest dim x1 is the one to distribute (each rank then owns one contiguous slab, and every sweep but
 * the x1 sweep, the rotation and the density moment stay local).  A rank keeps its L = n0/R planes plus w halo planes
 * on either side in ONE array of (L + 2w) x n1 x ... x n5 doubles and uses two contexts on it:
 *   - a context for the grid (L, n1, .., n5) on the interior pointer f + w*n1*..*n5: all sweeps along dims 1-5,
 *     bsl6d_rotate, bsl6d_density (x2, x3 stay periodic, they are not distributed);
 *   - a context for the grid (L + 2w, n1, .., n5) with bsl6d_set_boundary(ctx, 0, 1): the x1 sweep over the whole
 *     array.  Dim 0 is then zero-extended instead of periodic, and with w >= q/2 + max|displacement in cells| no
 *     interior output ever reads beyond the halo; halo outputs are meaningless and are overwritten by the next
 *     exchange.  The interior outputs are bit-identical to those of the periodic sweep on the undivided grid.
 * The halo exchange itself (the neighbour's w boundary planes, contiguous: one copy or one send/recv per side) is
 * plumbing and lives in the Python layer (torch.distributed over NCCL); see paper_2303_05994_b200/slab.py.
 * open = 1 opens dim 0, 1 or 2; open = 0 makes it periodic again.  Returns the old setting or BSL6D_EINVAL.
 * bsl6d_field_* and bsl6d_vp_step need a fully periodic x grid and return BSL6D_EUNSUPPORTED on an opened context. */
BSL6D_API int bsl6d_set_boundary(bsl6d_ctx* ctx, int dim, int open);

/* The x1 sweep of a slab WITHOUT halo planes and without an exchange step: the planes a pencil needs from the
 * neighbouring slabs are read where they are.  ctx describes the slab (grid (L, n1, .., n5)); f_in is the slab's own
 * array, f_left / f_right the arrays of the ring neighbours below and above -- same shape, DEVICE pointers this GPU
 * can dereference: peer memory of another GPU mapped into this process (the loads then travel over NVLink: compute
 * and "collective" are one kernel), arrays of other slabs on the same device, or f_in itself (a ring of one: plain
 * periodic sweep).  halo_planes = w >= q/2 + the largest |displacement| in cells, rounded up, and <= L: the
 * neighbours' nearest w planes are guaranteed to be used; a foot further away may read zeros (the caller's promise,
 * as for halo planes).  Slab thicknesses 8/16/32/48/64 run a compiled streaming register kernel, any other thickness
 * a run-time-extent kernel that stages the pencil and 2w neighbour planes in shared memory.  Out of place only (f_out must not overlap any input: the neighbours are reading f_in meanwhile), and
 * the neighbours' arrays must hold the state of the same step: synchronise the ring before the call and before
 * anyone overwrites an input (one barrier per x1 sweep; paper_2303_05994_b200/slab.py PeerSlab).
 * shift_source as for bsl6d_advect with dim = 0.  Results are bit-identical to the periodic sweep on the undivided
 * grid (PAPER.md:150-152, 323 describe the halo version this replaces; eq (9) its cost). */
BSL6D_API int bsl6d_advect_x1_peer(bsl6d_ctx* ctx, const double* f_in, const double* f_left, const double* f_right,
                         double* f_out, int halo_planes, const double* shift_source, double dt, void* stream);

/* Density moment rho[x] = dv1*dv2*dv3 * sum_{j1,j2,j3} f[x, j]   (eq (2); bare moment, reading S9).
 * rho: n0*n1*n2 doubles.  The summation order is fixed (deterministic, tree-shaped). */
BSL6D_API int bsl6d_density(bsl6d_ctx* ctx, const double* f, double* rho, void* stream);
/* The same moment with the work array given by the caller, so that several moments of one context can be in flight on
 * different streams at once (bsl6d_density keeps the partial sums of split v-blocks in ONE array of the context; two
 * overlapping calls race on it).  scratch: DEVICE, bsl6d_density_scratch_doubles(ctx) doubles = n0*n1*n2 * G when a
 * v-block is cut into G > 1 chunks of <= 32768 doubles, else 0 (scratch may then be NULL).  One scratch array per
 * stream in flight; contents on entry do not matter.  Same bits as bsl6d_density. */
BSL6D_API int bsl6d_density_scratch(bsl6d_ctx* ctx, const double* f, double* rho, double* scratch, void* stream);
BSL6D_API long long bsl6d_density_scratch_doubles(const bsl6d_ctx* ctx);

/* ---- the density moment without any allocation ----------------------------------------------------------------
 * For callers that may not call cudaMalloc / cudaFree (or anything that does): code living inside a host application
 * that owns all device memory through a pool or caching allocator of its own, diagnostics that run between time steps
 * and cannot afford the device-wide synchronisation an allocation or a free may bring, jobs so close to the memory
 * limit that an allocation in mid-run may fail.  Every other entry point needs a context, and bsl6d_create allocates;
 * this one needs none: it computes the same moment as bsl6d_density (same chunking, same order of additions, the same
 * bits) from plain arguments, and the scratch that split v-blocks need -- the partial sums, nx*G doubles with
 * nx = n0*n1*n2 and G = the number of chunks of <= 32768 doubles one v-block n3*n4*n5 is cut into -- sits in a
 * __device__ array compiled into the library: BSL6D_STATIC_SCRATCH_DOUBLES doubles = 2 MiB, held by every GPU the
 * library's code is loaded on, from load until the process exits.
 *   n      HOST, the six extents (each >= 1);   dv: HOST, the spacings of v1, v2, v3 (finite, > 0)
 *   f      DEVICE, n0*..*n5 doubles, C order, 8-byte aligned (16 for full speed);   rho: DEVICE, n0*n1*n2 doubles
 *   stream cudaStream_t as void*; the launches (one, or two when G > 1) are enqueued there, no synchronisation
 *   cuda_error  HOST, may be NULL: receives the cudaError_t when the call returns BSL6D_ECUDA, else 0
 * f and rho must live on the CURRENT device.  Returns BSL6D_ESCRATCH -- and launches nothing -- when G > 1 and
 * nx*G > BSL6D_STATIC_SCRATCH_DOUBLES (BASELINE config C3, 16^3 x 64^3, needs 32768; blocks of <= 32768 velocity
 * points need no scratch at any nx); BSL6D_EUNSUPPORTED when nx*G >= 2^31 or the device ordinal is >= 64.
 * It calls no cudaMalloc, cudaFree or allocating library routine.
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress, which may make the runtime load
 * the library's code onto that device); make that first call outside any stream capture.
 * Sharing: all calls on a device use the one array and find the previous call's partial sums in it.  Nothing needs
 * clearing -- a call overwrites each slot it later reads -- but two calls whose kernels may run at the same time
 * (different streams with no ordering between them, from one host thread or several) race on it and return garbage.
 * Calls on one stream, or ordered by events, are safe; the address look-up itself is guarded by a mutex. */
#define BSL6D_STATIC_SCRATCH_DOUBLES 262144
BSL6D_API int bsl6d_density_static(const int32_t n[6], const double dv[3], const double* f, double* rho, void* stream,
                         int* cuda_error);

/* ---- odd stencil width, one displacement per point ------------------------------------------
 * PAPER.md:86-89 eq (6): for odd q the stencil stays centred on the grid point,
 *     f_out[p, j] = sum_{m=-(q-1)/2..(q-1)/2} l_m(alpha[p, j]) * f_in[p, j + m]        (periodic in x, zero fill in v)
 * with l_m the Lagrange basis on the integer nodes m evaluated at alpha (in cells; the paper assumes |alpha| < 1,
 * PAPER.md:84).  alpha_cells is a DEVICE array with the shape and layout of f: "the most general way to define the
 * interpolation shift is as a function of the full phase space" -- this is the kernel of the paper's
 * own section-5 benchmark (random alpha/dx in [-1,1], widths 3/5/7/9, 37^6 points).  A sweep moves
 * 24 B/point.  q odd, 1..11 (else BSL6D_EUNSUPPORTED); any extent: kernels compiled per extent for q in {3,5,7,9} and
 * extents {8,16,32,37,48,64}, run-time-extent kernels otherwise (unit-stride dim: extent <= ~400, else
 * BSL6D_EUNSUPPORTED).  f_in == f_out is legal; alpha_cells must not overlap f_out. */
BSL6D_API int bsl6d_advect_pointwise(bsl6d_ctx* ctx, const double* f_in, double* f_out, int dim,
                           const double* alpha_cells, int q, void* stream);

/* ---- field step: the self-consistent electric field ------------------------------------------
 * PAPER.md:44-48 eq (2): rho_c = q (int f dv - n0), -Laplace(phi) = rho_c, E = -grad(phi), solved pseudo-spectrally on
 * the periodic x grid; eq (11): the adiabatic-electron closure (n0 q^2/T_e) phi = rho_c.
 * rho is the bare moment of bsl6d_density (n0*n1*n2 doubles, DEVICE).  The neutralising background n0 is the mean of
 * the moment (the k = 0 mode is dropped, reading F1); Nyquist modes have no first derivative (reading F2).
 *   poisson:    E_d <- e_fac * ( -d/dx_d phi ),   -Laplace(phi) = rho_fac * (rho - mean)
 *   adiabatic:  E_d <- e_fac * ( -d/dx_d phi ),    phi = phi_fac * (rho - mean)
 * E: HOST array of three DEVICE pointers (outputs, n0*n1*n2 doubles each).  With e_fac = q/m the outputs are exactly
 * the shift sources bsl6d_advect wants for dims 3..5.  The transform is a hand-written separable DFT (any extent);
 * 13 small launches on the caller's stream. */
BSL6D_API int bsl6d_field_poisson(bsl6d_ctx* ctx, const double* rho, double rho_fac, double e_fac, double* const E[3],
                        void* stream);
BSL6D_API int bsl6d_field_adiabatic(bsl6d_ctx* ctx, const double* rho, double phi_fac, double e_fac, double* const E[3],
                          void* stream);
/* One self-consistent Strang step (Fig. 1 caption at 114), result in f:
 *   x1,x2,x3 (dt/2) -> rho = moment(f) -> field solve -> v1,v2,v3 with E (dt) -> rotation (B may be NULL) -> x1,x2,x3 (dt/2).
 * closure 0 = Poisson (c1 = rho_fac), 1 = adiabatic (c1 = phi_fac).  rho and E[0..2] are caller-owned DEVICE work
 * buffers and hold the mid-step moment and field on return.  f_tmp as in bsl6d_strang_step. */
BSL6D_API int bsl6d_vp_step(bsl6d_ctx* ctx, double* f, double* f_tmp, double* rho, double* const E[3], const double B[3],
                  double dt, int closure, double c1, double e_fac, void* stream);

/* ---- end-to-end entry point on HOST buffers -------------------------------------------------------------
 * Runs a sequence of operations on a distribution function that lives in HOST memory (pinned for full speed):
 * copies f_in_host to the device, runs the ops back to back on an internal stream, copies the result to
 * f_out_host (may equal f_in_host) and, for density ops, rho to op.rho_host; synchronises before returning.
 * Device working buffers are allocated on first use and kept by the context. */
typedef struct bsl6d_host_op {
    int32_t kind;                /* 0 = advect, 1 = rotate, 2 = density (of the current state) */
    int32_t dim;                 /* advect: sweep dim */
    const double* shift_source;  /* advect: HOST pointer or NULL, sizes as in bsl6d_advect */
    double dt;                   /* advect, rotate */
    double B[3];                 /* rotate */
    double* rho_host;            /* density: HOST output, n0*n1*n2 doubles */
} bsl6d_host_op;
BSL6D_API int bsl6d_run_host(bsl6d_ctx* ctx, const double* f_in_host, double* f_out_host,
                   const bsl6d_host_op* ops, int nops);
/* The same in two halves, so that two independent problems can be in flight at once: bsl6d_run_host_begin enqueues
 * upload, ops and download on the internal stream of `slot` (0 or 1; each slot has its own device buffers) and returns
 * without waiting; bsl6d_run_host_end(ctx, slot) waits for everything begun on that slot.  With two slots the upload
 * of one problem overlaps the download of the other (the host link is full duplex) and the kernels of either -- for a
 * stream of problems the step time drops from upload + compute + download to about max(upload, download).  Until
 * bsl6d_run_host_end returns, f_in_host, f_out_host, every shift_source and rho_host of the call must stay valid and
 * untouched (the ops array itself is consumed before _begin returns).  A second _begin on a slot queues behind the
 * first.  bsl6d_run_host(...) == _begin(..., 0) followed by _end(ctx, 0). */
BSL6D_API int bsl6d_run_host_begin(bsl6d_ctx* ctx, const double* f_in_host, double* f_out_host,
                         const bsl6d_host_op* ops, int nops, int slot);
BSL6D_API int bsl6d_run_host_end(bsl6d_ctx* ctx, int slot);

/* ---- introspection ------------------------------------------------------------------------------------ */
BSL6D_API const char* bsl6d_strerror(int code);
BSL6D_API int bsl6d_last_cuda_error(const bsl6d_ctx* ctx);          /* cudaError_t of the last BSL6D_ECUDA, else 0 */
BSL6D_API long long bsl6d_launch_count(const bsl6d_ctx* ctx);       /* kernels launched by this context so far */
/* Name of the kernel variant bsl6d_advect* would launch for `dim` ("strided<N,Q,..>", "unit<N,Q,..>", "generic<..>";
 * "stream<N,Q,..> (in place: strided<..>)" where an out-of-place sweep streams its pencils through a register window
 * and the in-place sweep holds them whole -- bit-identical results either way). */
BSL6D_API int bsl6d_kernel_name(const bsl6d_ctx* ctx, int dim, char* buf, int buflen);
BSL6D_API int bsl6d_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BSL6D_H */
