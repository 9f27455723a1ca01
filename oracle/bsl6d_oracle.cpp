// bsl6d_oracle.cpp -- ORACLE: TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU implementation of the split 1-D advection
// sweep of the 6-D backward semi-Lagrangian method of arXiv 2303.05994
// (PAPER.md = /root/reference/PAPER.md).  It exists only so that tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// can check and time the CUDA path against something written straight from the
// paper.  It shares no code, header, table or helper with the CUDA library in
// paper_2303_05994_b200/csrc and must never be called from the product path.
//
// Everything is fp64 ("double"), loops are plain and un-blocked, OpenMP is used
// for one thing only: `parallel for` over independent pencils.  Compile with
//     g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC
// (-ffp-contract=off: every a*b+c below is two IEEE roundings, as written).
//
// Conventions:
//   dims d = 0..5 = (x1,x2,x3,v1,v2,v3), extents n[d], C-order (v3 unit stride);
//   dims 0-2 periodic, dims 3-5 zero-extended (BASELINE.json north_star);
//   stencil width q = degree+1 is EVEN, nodes m = -q/2+1 .. q/2  (eq (7)).
//
// Pin status (tests/test_oracle_pins.py, all run with -m "not gpu"):
//   lagrange weights   pinned (Vandermonde moment solve in exact rationals, textbook midpoint values)
//   pencil / sweep     pinned (np.roll permutation, polynomial reproduction, mass, scipy
//                      BarycentricInterpolator on every stencil, exact-rational matrix, free streaming)
//   rotate             pinned (2x2 shear product = rotation matrix, closed-form rotated Gaussian, 2*pi return)
//   density            pinned (math.fsum brute force, Maxwellian closed form)
//   strang_step        pinned compositionally + E=0,B=0 free-streaming closed form + E-only closed form
//   sweep_pointwise    pinned (odd-q weights: closed forms and exact rationals; polynomial reproduction with
//                      per-point alpha; whole-cell alpha = exact roll; numpy polynomial interpolation per point)
//
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int kMaxQ = 16;

// Lagrange basis values l_m(theta) on the integer nodes m = -q/2+1 .. q/2
// (eq (7): even q, stencil centred on the foot of the characteristic).
//   w[m] = prod_{n != m} (theta - n) / prod_{n != m} (m - n)
// numerator: n ascending; denominator: exact small integer; ONE division.
void lagrange_weights(int q, double theta, double* w) {
    const int m_lo = -q / 2 + 1;
    for (int mi = 0; mi < q; ++mi) {
        const int m = m_lo + mi;
        double num = 1.0;
        double den = 1.0;
        for (int ni = 0; ni < q; ++ni) {
            const int n = m_lo + ni;
            if (n == m) continue;
            num = num * (theta - (double)n);
            den = den * (double)(m - n);
        }
        w[mi] = num / den;
    }
}

// One pencil (eq (5) with the 1-D interpolant of eq (7)), generalised to
// |alpha| >= 1 cell by the split alpha = k + theta, k = floor(alpha) (reading S2).
//   out[j] = sum_m l_m(theta) * g[j + k + m]
// g is periodic (x dims) or zero outside [0,n) (v dims).  `g` and `out` must not overlap.
void pencil_update(int n, int q, bool periodic, const double* g, double a, double scale, double* out) {
    const double alpha = -(a * scale);            // foot (in cells) = j + alpha  (reading S1)
    const double kf = std::floor(alpha);
    const long long k = (long long)kf;
    const double theta = alpha - kf;              // in [0,1]
    double w[kMaxQ];
    lagrange_weights(q, theta, w);
    const int m_lo = -q / 2 + 1;
    for (int j = 0; j < n; ++j) {
        double acc = 0.0;
        for (int mi = 0; mi < q; ++mi) {
            const long long jj = (long long)j + k + (long long)(m_lo + mi);
            double val;
            if (periodic) {
                val = g[((jj % n) + n) % n];
            } else {
                val = (jj >= 0 && jj < n) ? g[jj] : 0.0;
            }
            acc = acc + w[mi] * val;
        }
        out[j] = acc;
    }
}

// ---- NEXT row N3: odd stencil width, per-point displacement (the paper's own section-5 benchmark kernel) -------
// PAPER.md:86-89 eq (6): for odd q the stencil stays centred on the grid point,
//   f(x_j + alpha) = sum_{i=j-(q-1)/2}^{j+(q-1)/2} l_i(alpha) f(x_i),   |alpha| < dx,
// with l_m the Lagrange basis on the integer nodes m = -(q-1)/2 .. (q-1)/2 evaluated at alpha (in cells).
// the displacement may be a function of all six coordinates ("random shifts alpha/dx in [-1,1]").
void lagrange_weights_odd(int q, double alpha, double* w) {
    const int h = (q - 1) / 2;
    for (int mi = 0; mi < q; ++mi) {
        const int m = mi - h;
        double num = 1.0, den = 1.0;
        for (int ni = 0; ni < q; ++ni) {
            const int n = ni - h;
            if (n == m) continue;
            num = num * (alpha - (double)n);
            den = den * (double)(m - n);
        }
        w[mi] = num / den;
    }
}

// out[j] = sum_m l_m(alpha[j]) g[j+m]; g periodic (x dims) or zero outside [0,n) (v dims).
void pencil_update_pointwise(int n, int q, bool periodic, const double* g, const double* alpha, double* out) {
    const int h = (q - 1) / 2;
    double w[kMaxQ];
    for (int j = 0; j < n; ++j) {
        lagrange_weights_odd(q, alpha[j], w);
        double acc = 0.0;
        for (int mi = 0; mi < q; ++mi) {
            const long long jj = (long long)j + (long long)(mi - h);
            double val;
            if (periodic) val = g[((jj % n) + n) % n];
            else val = (jj >= 0 && jj < n) ? g[jj] : 0.0;
            acc = acc + w[mi] * val;
        }
        out[j] = acc;
    }
}

struct Grid {            // the oracle's own description of the phase-space grid
    int32_t n[6];
    double lo[6];
    double dx[6];        // node i of dim d sits at lo[d] + i*dx[d]
};

long long total_points(const int32_t n[6]) {
    long long t = 1;
    for (int d = 0; d < 6; ++d) t *= n[d];
    return t;
}

// Sweep along `dim` over the whole 6-D array.  src is a dense C-order array over the dims
// whose bit is set in src_mask (ascending dim order); alpha_cells = -(src[p] * scale).
// f_in == f_out is legal: every pencil is copied to a local buffer first.
void sweep(const int32_t n[6], const double* f_in, double* f_out, int dim,
           const double* src, unsigned src_mask, double scale, int q) {
    long long stride[6];
    stride[5] = 1;
    for (int d = 4; d >= 0; --d) stride[d] = stride[d + 1] * n[d + 1];
    long long sstride[6];                          // strides of the src array (0 if dim not in mask)
    {
        long long s = 1;
        for (int d = 5; d >= 0; --d) {
            if (src_mask & (1u << d)) { sstride[d] = s; s *= n[d]; } else sstride[d] = 0;
        }
    }
    const int nd = n[dim];
    const bool periodic = dim < 3;
    const long long npencil = total_points(n) / nd;
#pragma omp parallel
    {
        std::vector<double> g(nd), o(nd);
#pragma omp for schedule(static)
        for (long long p = 0; p < npencil; ++p) {
            // decode p -> the five indices other than `dim` (C-order over those dims)
            long long rem = p, base = 0, soff = 0;
            for (int d = 5; d >= 0; --d) {
                if (d == dim) continue;
                const long long id = rem % n[d];
                rem /= n[d];
                base += id * stride[d];
                soff += id * sstride[d];
            }
            for (int j = 0; j < nd; ++j) g[j] = f_in[base + (long long)j * stride[dim]];
            pencil_update(nd, q, periodic, g.data(), src[soff], scale, o.data());
            for (int j = 0; j < nd; ++j) f_out[base + (long long)j * stride[dim]] = o[j];
        }
    }
}

std::vector<double> nodes(const Grid& g, int d) {
    std::vector<double> v(g.n[d]);
    for (int i = 0; i < g.n[d]; ++i) v[i] = g.lo[d] + (double)i * g.dx[d];
    return v;
}

// v x B0 rotation as three velocity shears (BASELINE.json configs[3]; reading S7).
// B = (q/m) B0 has exactly one non-zero component c; (a,b,c) cyclic; theta = B_c * dt.
//   f_new(v) = f_old(R(theta) v),  R = Sa(-tan(theta/2)) Sb(sin theta) Sa(-tan(theta/2)),
// the backward foot of dV/dt = V x B (eq (3)).
// Rotation about ONE coordinate axis c by `theta` as three shears (BASELINE.json configs[3], reading S7):
// (a,b,c) cyclic; foot displacement along v_a: -v_b*tan(theta/2); along v_b: +v_a*sin(theta); along v_a again.
// Result: f_out(v) = f_in(R_c(theta) v), R_c the right-handed rotation about axis c.
void rotate_axis(const Grid& g, int q, const double* f_in, double* f_out, int c, double theta) {
    const int a = (c + 1) % 3, b = (c + 2) % 3;
    const double t = std::tan(0.5 * theta), s = std::sin(theta);
    const std::vector<double> va = nodes(g, 3 + a), vb = nodes(g, 3 + b);
    sweep(g.n, f_in,  f_out, 3 + a, vb.data(), 1u << (3 + b), t / g.dx[3 + a], q);
    sweep(g.n, f_out, f_out, 3 + b, va.data(), 1u << (3 + a), -s / g.dx[3 + b], q);
    sweep(g.n, f_out, f_out, 3 + a, vb.data(), 1u << (3 + b), t / g.dx[3 + a], q);
}

// NEXT row N4 (oblique B): the axis-rotation sequence for a field B in general position (reading R1):
// with b = B/|B| = (sin(vt)cos(ph), sin(vt)sin(ph), cos(vt)) and theta = |B| dt,
//     R(b, theta) = Rz(ph) Ry(vt) Rz(theta) Ry(-vt) Rz(-ph),
// and since (T_M f)(v) = f(M v) composes as T_A T_B = T_{BA}, the factors are APPLIED left to right:
//     Rz(ph), Ry(vt), Rz(theta), Ry(-vt), Rz(-ph).
// An axis rotation by more than pi/2 is applied in ceil(|angle| / (pi/2)) equal pieces (tan(piece/2) stays <= 1).
// |theta| <= 2 pi is required (at most 4 + 4*2 = 12 entries... 16 reserved).
int rotation_plan(const double B[3], double dt, int* axes, double* angles) {
    const double bn = std::sqrt(B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
    const double theta = bn * dt;
    const double vt = std::acos(B[2] / bn);
    const double ph = std::atan2(B[1], B[0]);
    const int ax[5] = {2, 1, 2, 1, 2};
    const double an[5] = {ph, vt, theta, -vt, -ph};
    const double half_pi = 1.5707963267948966;
    int cnt = 0;
    for (int i = 0; i < 5; ++i) {
        if (an[i] == 0.0) continue;
        const int pieces = (int)std::ceil(std::fabs(an[i]) / half_pi);
        for (int k = 0; k < pieces && cnt < 16; ++k) { axes[cnt] = ax[i]; angles[cnt++] = an[i] / (double)pieces; }
    }
    return cnt;
}

int rotate(const Grid& g, int q, const double* f_in, double* f_out, const double B[3], double dt) {
    int c = -1, nz = 0;
    for (int i = 0; i < 3; ++i)
        if (B[i] != 0.0) { c = i; ++nz; }
    const long long npts = total_points(g.n);
    if (nz == 0) { if (f_in != f_out) std::memcpy(f_out, f_in, sizeof(double) * npts); return 0; }
    if (nz == 1) {
        // Reading R2: tan(theta/2) diverges at theta = pi, so an axis rotation above pi/2 is applied in
        // ceil(|theta| / (pi/2)) equal pieces of three shears (one piece for |theta| <= pi/2: the plain three shears);
        // more than a full turn is rejected, as for an oblique axis.
        const double theta = B[c] * dt;
        if (std::fabs(theta) > 6.283185307179586477) return -1;
        int pieces = (int)std::ceil(std::fabs(theta) / 1.5707963267948966);
        if (pieces < 1) pieces = 1;
        const double* cur = f_in;
        for (int k = 0; k < pieces; ++k) { rotate_axis(g, q, cur, f_out, c, theta / (double)pieces); cur = f_out; }
        return 0;
    }
    int axes[16];
    double angles[16];
    if (std::sqrt(B[0] * B[0] + B[1] * B[1] + B[2] * B[2]) * std::fabs(dt) > 6.283185307179586477) return -1;
    const int cnt = rotation_plan(B, dt, axes, angles);
    const double* cur = f_in;
    for (int i = 0; i < cnt; ++i) { rotate_axis(g, q, cur, f_out, axes[i], angles[i]); cur = f_out; }
    if (cnt == 0 && f_in != f_out) std::memcpy(f_out, f_in, sizeof(double) * npts);
    return 0;
}

}  // namespace

extern "C" {

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// w[q] <- l_m(theta), m = -q/2+1 .. q/2.   q even, 2 <= q <= 16.
int oracle_lagrange_weights(int q, double theta, double* w) {
    if (q < 2 || q > kMaxQ || (q & 1)) return -1;
    lagrange_weights(q, theta, w);
    return 0;
}

// P independent pencils of length n: g_in[P][n], a[P] (shift-source value per pencil).
int oracle_sweep_pencils(int n, int q, int periodic, long long P, const double* g_in,
                         const double* a, double scale, double* g_out) {
    if (q < 2 || q > kMaxQ || (q & 1) || n < 1) return -1;
#pragma omp parallel for schedule(static)
    for (long long p = 0; p < P; ++p)
        pencil_update(n, q, periodic != 0, g_in + p * n, a[p], scale, g_out + p * n);
    return 0;
}

// General sweep (the primitive): alpha_cells = -(src * scale), src dense over the dims in src_mask.
int oracle_sweep(const int32_t* n, const double* f_in, double* f_out, int dim,
                 const double* src, unsigned src_mask, double scale, int q) {
    if (q < 2 || q > kMaxQ || (q & 1) || dim < 0 || dim > 5) return -1;
    if (src_mask & (1u << dim)) return -1;
    sweep(n, f_in, f_out, dim, src, src_mask, scale, q);
    return 0;
}

// Named sweep.  dim 0-2: x_d advection, shift_source = v_d node values (n[dim+3] doubles) or NULL
// for the grid's own nodes; dim 3-5: shift_source = (q/m) E_{dim-3}(x), n0*n1*n2 doubles.
// foot (cells) of output point j: j - shift_source[p] * (dt/dx[dim])     (eq (3))
int oracle_advect(const int32_t* n, const double* lo, const double* dx, int degree,
                  const double* f_in, double* f_out, int dim, const double* shift_source, double dt) {
    Grid g;
    for (int d = 0; d < 6; ++d) { g.n[d] = n[d]; g.lo[d] = lo[d]; g.dx[d] = dx[d]; }
    const int q = degree + 1;
    if (dim < 0 || dim > 5) return -1;
    const double scale = dt / g.dx[dim];
    if (dim < 3) {
        std::vector<double> v;
        const double* s = shift_source;
        if (!s) { v = nodes(g, dim + 3); s = v.data(); }
        return oracle_sweep(g.n, f_in, f_out, dim, s, 1u << (dim + 3), scale, q);
    }
    if (!shift_source) return -1;
    return oracle_sweep(g.n, f_in, f_out, dim, shift_source, 0x7u, scale, q);
}

int oracle_rotate(const int32_t* n, const double* lo, const double* dx, int degree,
                  const double* f_in, double* f_out, const double* B, double dt) {
    Grid g;
    for (int d = 0; d < 6; ++d) { g.n[d] = n[d]; g.lo[d] = lo[d]; g.dx[d] = dx[d]; }
    return rotate(g, degree + 1, f_in, f_out, B, dt);
}

// rho[x] = dv1*dv2*dv3 * sum_j f[x,j]   (eq (2), bare moment: reading S9).
// Accumulated in long double so the result is the correctly rounded sum for all practical purposes.
int oracle_density(const int32_t* n, const double* dx, const double* f, double* rho) {
    const long long nx = (long long)n[0] * n[1] * n[2];
    const long long nv = (long long)n[3] * n[4] * n[5];
    const double dv3 = dx[3] * dx[4] * dx[5];
#pragma omp parallel for schedule(static)
    for (long long x = 0; x < nx; ++x) {
        long double acc = 0.0L;
        const double* p = f + x * nv;
        for (long long j = 0; j < nv; ++j) acc += (long double)p[j];
        rho[x] = dv3 * (double)acc;
    }
    return 0;
}

// One Strang step, in place (order fixed by BASELINE.json configs[4], reading S8):
//   x1,x2,x3 (dt/2)  ->  E-sweeps v1,v2,v3 (dt)  ->  rotation (theta = B_c dt)  ->  x1,x2,x3 (dt/2)
// E0/E1/E2: (q/m) E_d(x) over the x grid (C-order), any may be NULL (that sweep is skipped).
int oracle_strang_step(const int32_t* n, const double* lo, const double* dx, int degree, double* f,
                       const double* E0, const double* E1, const double* E2, const double* B, double dt) {
    const double* E[3] = {E0, E1, E2};
    const double half = 0.5 * dt;
    int rc;
    for (int d = 0; d < 3; ++d)
        if ((rc = oracle_advect(n, lo, dx, degree, f, f, d, nullptr, half))) return rc;
    for (int d = 0; d < 3; ++d)
        if (E[d] && (rc = oracle_advect(n, lo, dx, degree, f, f, 3 + d, E[d], dt))) return rc;
    if (B && (B[0] != 0.0 || B[1] != 0.0 || B[2] != 0.0))
        if ((rc = oracle_rotate(n, lo, dx, degree, f, f, B, dt))) return rc;
    for (int d = 0; d < 3; ++d)
        if ((rc = oracle_advect(n, lo, dx, degree, f, f, d, nullptr, half))) return rc;
    return 0;
}

// The (axis, angle) list rotate() applies for an oblique B (up to 16 entries); returns the count.
int oracle_rotation_plan(const double* B, double dt, int* axes, double* angles) {
    if (!B || !axes || !angles) return -1;
    int nz = 0;
    for (int i = 0; i < 3; ++i) nz += B[i] != 0.0;
    if (nz < 2) return -1;
    return rotation_plan(B, dt, axes, angles);
}

int oracle_lagrange_weights_odd(int q, double alpha, double* w) {
    if (q < 1 || q > kMaxQ || !(q & 1) || !w) return -1;
    lagrange_weights_odd(q, alpha, w);
    return 0;
}

// Sweep along `dim` with one displacement per POINT: alpha has the shape and layout of f (in cells).
int oracle_sweep_pointwise(const int32_t* n, const double* f_in, double* f_out, int dim, const double* alpha, int q) {
    if (!n || !f_in || !f_out || !alpha || dim < 0 || dim > 5 || q < 1 || q > kMaxQ || !(q & 1)) return -1;
    long long stride[6];
    stride[5] = 1;
    for (int d = 4; d >= 0; --d) stride[d] = stride[d + 1] * n[d + 1];
    const int nd = n[dim];
    const bool periodic = dim < 3;
    const long long npencil = total_points(n) / nd;
#pragma omp parallel
    {
        std::vector<double> g(nd), a(nd), o(nd);
#pragma omp for schedule(static)
        for (long long p = 0; p < npencil; ++p) {
            long long rem = p, base = 0;
            for (int d = 5; d >= 0; --d) {
                if (d == dim) continue;
                base += (rem % n[d]) * stride[d];
                rem /= n[d];
            }
            for (int j = 0; j < nd; ++j) {
                g[j] = f_in[base + (long long)j * stride[dim]];
                a[j] = alpha[base + (long long)j * stride[dim]];
            }
            pencil_update_pointwise(nd, q, periodic, g.data(), a.data(), o.data());
            for (int j = 0; j < nd; ++j) f_out[base + (long long)j * stride[dim]] = o[j];
        }
    }
    return 0;
}

}  // extern "C"
