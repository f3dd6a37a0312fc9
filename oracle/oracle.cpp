// oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU implementation of what the hot path of
// arxiv/paper_2602_03857 computes: the closed-form vertical gravity of right
// rectangular prisms (Sec. 2.1 Eq. 1-3), the dense operator
// d = G m (Eq. 4-6), its transpose, the depth weighting
// (formula from BASELINE.json north_star), and the data-space
// solve (Eq. 9-11) by conjugate gradients
// and, on tiny inputs, by Cholesky (data space) and via the model-space normal
// equations (Eq. 8).
//
// Rules this file keeps:
//   * per prism, 8 corners, no node sharing, no tiling, no reordering beyond
//     what the equations state; rows / columns are independent loops;
//   * Psi in `double` (prec=0) with sums accumulated in `long double`, or
//     everything in `long double` (prec=1, the "truth" build used to measure
//     the FP64 cancellation floor on subsamples);
//   * shares NO code, header, table or constant with the CUDA path
//     (paper_2602_03857_b200/csrc). Only tests/, __graft_entry__.smoke() and
//     bench.py's cpu_baseline / --impl reference legs may load this library.
//
// Readings of the paper taken here:
//   C1 coordinates are corner - station;  C2 p=1 lower / p=2 upper bound,
//   z positive down;  C3 principal-value atan of the quotient;  C6 guards:
//   Z==0 -> Z*atan(.)=0, X==0 -> X*ln(.)=0, Y==0 -> Y*ln(.)=0;
//   C5 w=(zc+z0)^(-beta/2), zc = cell-centre depth below the mesh top;
//   C8 textbook CG, x0=0, exactly `iters` iterations.
//
// Pins: tests/test_oracle_pins.py (worked values, superposition, point mass,
// Bouguer slab, mirror, row sums, dot-product test, push-through, direct-vs-CG,
// Jacobi-PCG against scipy and the symmetrically scaled system, the outer loop's
// step halving against a brute-force scan and its tolerance stops).
// PARITY UNPINNED against the PAPER: orc_invert, the outer model-update loop with
// step backtracking.  The paper prints neither the
// residual norm nor the backtracking rule; orc_invert follows readings R1-R4 of
// DESIGN.md 5.7 step by step and is pinned to what the algebra fixes, not to a
// value the paper prints.

#include <cmath>
#include <cstddef>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>
#include <algorithm>

namespace {

typedef long double ld;

// ---- Eq. 2-3 ------------------------------------------------
template <class T>
T psi(T X, T Y, T Z) {
    T R = std::sqrt(X * X + Y * Y + Z * Z);              // Eq. 3
    T t_atan = T(0), t_lx = T(0), t_ly = T(0);
    if (Z != T(0)) t_atan = Z * std::atan((X * Y) / (Z * R));   // C3, C6
    if (X != T(0)) t_lx = X * std::log(R + Y);                   // C6
    if (Y != T(0)) t_ly = Y * std::log(R + X);                   // C6
    return t_atan - t_lx - t_ly;                                 // Eq. 2
}

// ---- Eq. 1: coefficient of one prism at one station, without gamma*rho
template <class T>
T prism_coeff(T xo, T yo, T zo, T x1, T x2, T y1, T y2, T z1, T z2) {
    const T xs[2] = {x1 - xo, x2 - xo};   // C1: corner - station; index 0 <-> p=1
    const T ys[2] = {y1 - yo, y2 - yo};
    const T zs[2] = {z1 - zo, z2 - zo};
    T s = T(0);
    for (int p = 1; p <= 2; ++p)
        for (int q = 1; q <= 2; ++q)
            for (int r = 1; r <= 2; ++r) {
                T sigma = ((p + q + r) % 2 == 0) ? T(1) : T(-1);   // (-1)^(p+q+r)
                s += sigma * psi<T>(xs[p - 1], ys[q - 1], zs[r - 1]);
            }
    return s;
}

struct Mesh {
    int nx, ny, nz;
    const double *xn, *yn, *zn;   // node coordinates, nx+1 / ny+1 / nz+1
    long long M() const { return (long long)nx * ny * nz; }
};

// cell (i,j,k) <-> index (i*ny + j)*nz + k  (z fastest; SURVEY.md 8(a) layout note, C11)
inline void cell_ijk(const Mesh& m, long long c, int& i, int& j, int& k) {
    k = (int)(c % m.nz);
    long long t = c / m.nz;
    j = (int)(t % m.ny);
    i = (int)(t / m.ny);
}

template <class T>
T g_entry(const Mesh& m, long long c, double xo, double yo, double zo) {
    int i, j, k;
    cell_ijk(m, c, i, j, k);
    return prism_coeff<T>((T)xo, (T)yo, (T)zo, (T)m.xn[i], (T)m.xn[i + 1], (T)m.yn[j], (T)m.yn[j + 1],
                          (T)m.zn[k], (T)m.zn[k + 1]);
}

template <class F>
void parallel_for(long long n, int nthreads, F f) {
    if (nthreads <= 1 || n <= 1) {
        for (long long i = 0; i < n; ++i) f(i);
        return;
    }
    std::vector<std::thread> th;
    nthreads = (int)std::min<long long>(nthreads, n);
    for (int t = 0; t < nthreads; ++t)
        th.emplace_back([=]() {
            for (long long i = t; i < n; i += nthreads) f(i);
        });
    for (auto& x : th) x.join();
}

// ---- Eq. 5: d_i = sum_k g_ik u_k -------------------------------
template <class T>
void forward_t(const Mesh& m, long long nobs, const double* xo, const double* yo, const double* zo, double gamma,
               const double* u, double* d, int nthreads) {
    const long long M = m.M();
    parallel_for(nobs, nthreads, [&](long long i) {
        ld acc = 0;
        for (long long c = 0; c < M; ++c) acc += (ld)g_entry<T>(m, c, xo[i], yo[i], zo[i]) * (ld)u[c];
        d[i] = (double)((ld)gamma * acc);
    });
}

// ---- transpose of Eq. 5: (G^T v)_k = sum_i g_ik v_i, for selected cells ------
template <class T>
void adjoint_t(const Mesh& m, long long nobs, const double* xo, const double* yo, const double* zo, double gamma,
               const double* v, long long ncells, const long long* cells, double* g, int nthreads) {
    parallel_for(ncells, nthreads, [&](long long cc) {
        long long c = cells ? cells[cc] : cc;
        ld acc = 0;
        for (long long i = 0; i < nobs; ++i) acc += (ld)g_entry<T>(m, c, xo[i], yo[i], zo[i]) * (ld)v[i];
        g[cc] = (double)((ld)gamma * acc);
    });
}

}  // namespace

extern "C" {

// Psi of Eq. 2 in double (prec=0) or long double rounded to double (prec=1).
double orc_psi(double X, double Y, double Z, int prec) {
    return prec ? (double)psi<ld>(X, Y, Z) : psi<double>(X, Y, Z);
}

// gz (same units as gamma*rho*length) of one prism at one station, Eq. 1.
double orc_prism_gz(double xo, double yo, double zo, double x1, double x2, double y1, double y2, double z1,
                    double z2, double rho, double gamma, int prec) {
    if (prec) return (double)((ld)gamma * (ld)rho * prism_coeff<ld>(xo, yo, zo, x1, x2, y1, y2, z1, z2));
    return gamma * rho * prism_coeff<double>(xo, yo, zo, x1, x2, y1, y2, z1, z2);
}

// d = G u (Eq. 5-6). All pointers HOST. u[M], d[nobs].
void orc_forward(int nx, int ny, int nz, const double* xn, const double* yn, const double* zn, long long nobs,
                 const double* xo, const double* yo, const double* zo, double gamma, const double* u, double* d,
                 int prec, int nthreads) {
    Mesh m{nx, ny, nz, xn, yn, zn};
    if (prec) forward_t<ld>(m, nobs, xo, yo, zo, gamma, u, d, nthreads);
    else forward_t<double>(m, nobs, xo, yo, zo, gamma, u, d, nthreads);
}

// g = G^T v restricted to `ncells` cells (cells==NULL: all M cells, ncells must be M).
void orc_adjoint(int nx, int ny, int nz, const double* xn, const double* yn, const double* zn, long long nobs,
                 const double* xo, const double* yo, const double* zo, double gamma, const double* v,
                 long long ncells, const long long* cells, double* g, int prec, int nthreads) {
    Mesh m{nx, ny, nz, xn, yn, zn};
    if (prec) adjoint_t<ld>(m, nobs, xo, yo, zo, gamma, v, ncells, cells, g, nthreads);
    else adjoint_t<double>(m, nobs, xo, yo, zo, gamma, v, ncells, cells, g, nthreads);
}

// Dense G (nobs x M, row-major, prism index fastest), gamma included. Eq. 6.
void orc_tabulate(int nx, int ny, int nz, const double* xn, const double* yn, const double* zn, long long nobs,
                  const double* xo, const double* yo, const double* zo, double gamma, double* G, int nthreads) {
    Mesh m{nx, ny, nz, xn, yn, zn};
    const long long M = m.M();
    parallel_for(nobs, nthreads, [&](long long i) {
        for (long long c = 0; c < M; ++c) G[i * M + c] = gamma * g_entry<double>(m, c, xo[i], yo[i], zo[i]);
    });
}

// Depth weights w_k = (zc_k + z0)^(-beta/2), zc_k = depth of the cell centre below the mesh top zn[0]
// (BASELINE.json north_star; reading C5).
void orc_depth_weights(int nx, int ny, int nz, const double* zn, double beta, double z0, double* w) {
    for (int i = 0; i < nx; ++i)
        for (int j = 0; j < ny; ++j)
            for (int k = 0; k < nz; ++k) {
                double zc = 0.5 * (zn[k] + zn[k + 1]) - zn[0];
                w[((long long)i * ny + j) * nz + k] = std::pow(zc + z0, -0.5 * beta);
            }
}

// ---- dense-matrix helpers (G given, nobs x M row-major) ------------------------
// d = G u
void orc_dense_matvec(long long N, long long M, const double* G, const double* u, double* d, int nthreads) {
    parallel_for(N, nthreads, [&](long long i) {
        ld acc = 0;
        for (long long c = 0; c < M; ++c) acc += (ld)G[i * M + c] * (ld)u[c];
        d[i] = (double)acc;
    });
}
// g = G^T v
void orc_dense_rmatvec(long long N, long long M, const double* G, const double* v, double* g, int nthreads) {
    parallel_for(M, nthreads, [&](long long c) {
        ld acc = 0;
        for (long long i = 0; i < N; ++i) acc += (ld)G[i * M + c] * (ld)v[i];
        g[c] = (double)acc;
    });
}

// diag_i = sum_k G_ik^2 w_k^-2  (diagonal of G W^-2 G^T); trace = sum_i diag_i (reading C7).
void orc_gram_diag(long long N, long long M, const double* G, const double* w, double* diag, int nthreads) {
    parallel_for(N, nthreads, [&](long long i) {
        ld acc = 0;
        for (long long c = 0; c < M; ++c) {
            ld g = G[i * M + c];
            acc += g * g / ((ld)w[c] * (ld)w[c]);
        }
        diag[i] = (double)acc;
    });
}

// Explicit A = G W^-2 G^T + lambda I (N x N, row-major).  PAPER.md:114 "construct the N x N data space system".
void orc_form_A(long long N, long long M, const double* G, const double* w, double lambda, double* A, int nthreads) {
    std::vector<double> iw2(M);
    for (long long c = 0; c < M; ++c) iw2[c] = 1.0 / (w[c] * w[c]);
    parallel_for(N, nthreads, [&](long long i) {
        for (long long j = 0; j <= i; ++j) {
            ld acc = 0;
            for (long long c = 0; c < M; ++c) acc += (ld)G[i * M + c] * (ld)iw2[c] * (ld)G[j * M + c];
            A[i * N + j] = (double)acc;
        }
    });
    for (long long i = 0; i < N; ++i) {
        for (long long j = 0; j < i; ++j) A[j * N + i] = A[i * N + j];
        A[i * N + i] += lambda;
    }
}

// Plain Cholesky A = L L^T (lower, in place, long-double accumulation), then solve A x = b.
// Returns 0, or k+1 if the k-th pivot is not positive.
int orc_cholesky_solve(long long n, double* A, const double* b, double* x) {
    for (long long j = 0; j < n; ++j) {
        ld s = A[j * n + j];
        for (long long k = 0; k < j; ++k) s -= (ld)A[j * n + k] * (ld)A[j * n + k];
        if (!(s > 0)) return (int)j + 1;
        double ljj = (double)std::sqrt(s);
        A[j * n + j] = ljj;
        for (long long i = j + 1; i < n; ++i) {
            ld t = A[i * n + j];
            for (long long k = 0; k < j; ++k) t -= (ld)A[i * n + k] * (ld)A[j * n + k];
            A[i * n + j] = (double)(t / ljj);
        }
    }
    std::vector<double> y(n);
    for (long long i = 0; i < n; ++i) {
        ld t = b[i];
        for (long long k = 0; k < i; ++k) t -= (ld)A[i * n + k] * (ld)y[k];
        y[i] = (double)(t / A[i * n + i]);
    }
    for (long long i = n - 1; i >= 0; --i) {
        ld t = y[i];
        for (long long k = i + 1; k < n; ++k) t -= (ld)A[k * n + i] * (ld)x[k];
        x[i] = (double)(t / A[i * n + i]);
    }
    return 0;
}

// Data-space direct solve (Eq. 11 with W_m = W^-2, W_d = lambda I, m_ref = 0):
// alpha = (G W^-2 G^T + lambda I)^-1 d ;  m = W^-2 G^T alpha.
int orc_dataspace_direct(long long N, long long M, const double* G, const double* w, double lambda,
                         const double* dobs, double* alpha, double* m, int nthreads) {
    std::vector<double> A((size_t)N * N);
    orc_form_A(N, M, G, w, lambda, A.data(), nthreads);
    int rc = orc_cholesky_solve(N, A.data(), dobs, alpha);
    if (rc) return rc;
    if (m) {
        orc_dense_rmatvec(N, M, G, alpha, m, nthreads);
        for (long long c = 0; c < M; ++c) m[c] /= (w[c] * w[c]);
    }
    return 0;
}

// Model-space Tikhonov solve (Eq. 8 with W_d = lambda I, W_m^-1 = W^2, m_ref = 0):
// (G^T G + lambda W^2) m = G^T d.   Tiny inputs only (M x M Cholesky).
int orc_modelspace_direct(long long N, long long M, const double* G, const double* w, double lambda,
                          const double* dobs, double* m, int nthreads) {
    std::vector<double> B((size_t)M * M);
    parallel_for(M, nthreads, [&](long long a) {
        for (long long b = 0; b <= a; ++b) {
            ld acc = 0;
            for (long long i = 0; i < N; ++i) acc += (ld)G[i * M + a] * (ld)G[i * M + b];
            B[a * M + b] = (double)acc;
        }
    });
    for (long long a = 0; a < M; ++a) {
        for (long long b = 0; b < a; ++b) B[b * M + a] = B[a * M + b];
        B[a * M + a] += lambda * w[a] * w[a];
    }
    std::vector<double> rhs(M);
    orc_dense_rmatvec(N, M, G, dobs, rhs.data(), nthreads);
    return orc_cholesky_solve(M, B.data(), rhs.data(), m);
}

// Variant of the two dense products used ONLY for the self-sensitivity figure of protocol P4:
// the same sums in reversed index order with a plain `double` accumulator -- a second, equally valid FP64
// evaluation order whose results differ from the long-double-accumulated ones by ~sqrt(n)*2^-53.
static void dense_matvec_alt(long long N, long long M, const double* G, const double* u, double* d, int nthreads) {
    parallel_for(N, nthreads, [&](long long i) {
        double acc = 0;
        for (long long c = M - 1; c >= 0; --c) acc += G[i * M + c] * u[c];
        d[i] = acc;
    });
}
static void dense_rmatvec_alt(long long N, long long M, const double* G, const double* v, double* g, int nthreads) {
    parallel_for(M, nthreads, [&](long long c) {
        double acc = 0;
        for (long long i = N - 1; i >= 0; --i) acc += G[i * M + c] * v[i];
        g[c] = acc;
    });
}

// ---- conjugate gradients on A = G W^-2 G^T + lambda I (reading C8) ----------
// State (x, r, p, rho) is in/out so that single steps can be injected (SURVEY.md 8(c) protocol P1).
// If `start` != 0 the state is initialised to x=0, r=p=dobs, rho=r.r first.
// G may be NULL: then the operator is applied matrix-free through the per-prism loops above
// (mesh/station arrays required); otherwise the tabulated G is reused.
// hist (may be NULL) receives ||r||_2 after each iteration at hist[it+1]; hist[0] = initial ||r||.
// ab (may be NULL) receives the step scalars a_j, b_j at ab[2*it], ab[2*it+1].
// reverse != 0 (needs G): every sum (the two dense products and the dot products) runs in reversed index order
// with a plain double accumulator -- a second valid FP64 evaluation of the same iteration.  The distance between
// the reverse=0 and reverse=1 iterates is the oracle's own reorder sensitivity (protocol P4).
void orc_cg(long long N, long long M, const double* G, int nx, int ny, int nz, const double* xn, const double* yn,
            const double* zn, const double* xo, const double* yo, const double* zo, double gamma, const double* w,
            double lambda, const double* dobs, int iters, int start, double* x, double* r, double* p, double* rho_io,
            double* hist, double* ab, int reverse, int nthreads) {
    Mesh mesh{nx, ny, nz, xn, yn, zn};
    std::vector<double> g(M), q(N);
    auto dot = [&](const double* a, const double* b) {
        ld acc = 0;
        if (!reverse) {
            for (long long i = 0; i < N; ++i) acc += (ld)a[i] * (ld)b[i];
            return (double)acc;
        }
        double accd = 0;
        for (long long i = N - 1; i >= 0; --i) accd += a[i] * b[i];
        return accd;
    };
    auto applyA = [&](const double* pin, double* qout) {
        if (G && reverse) dense_rmatvec_alt(N, M, G, pin, g.data(), nthreads);
        else if (G) orc_dense_rmatvec(N, M, G, pin, g.data(), nthreads);
        else adjoint_t<double>(mesh, N, xo, yo, zo, gamma, pin, M, nullptr, g.data(), nthreads);
        for (long long c = 0; c < M; ++c) g[c] /= (w[c] * w[c]);
        if (G && reverse) dense_matvec_alt(N, M, G, g.data(), qout, nthreads);
        else if (G) orc_dense_matvec(N, M, G, g.data(), qout, nthreads);
        else forward_t<double>(mesh, N, xo, yo, zo, gamma, g.data(), qout, nthreads);
        for (long long i = 0; i < N; ++i) qout[i] += lambda * pin[i];
    };
    double rho;
    if (start) {
        for (long long i = 0; i < N; ++i) { x[i] = 0.0; r[i] = dobs[i]; p[i] = dobs[i]; }
        rho = dot(r, r);
    } else rho = *rho_io;
    if (hist) hist[0] = std::sqrt(rho);
    for (int it = 0; it < iters; ++it) {
        applyA(p, q.data());
        double delta = dot(p, q.data());
        double a = rho / delta;
        for (long long i = 0; i < N; ++i) { x[i] += a * p[i]; r[i] -= a * q[i]; }
        double rho_new = dot(r, r);
        double b = rho_new / rho;
        for (long long i = 0; i < N; ++i) p[i] = r[i] + b * p[i];
        rho = rho_new;
        if (hist) hist[it + 1] = std::sqrt(rho);
        if (ab) { ab[2 * it] = a; ab[2 * it + 1] = b; }
    }
    *rho_io = rho;
}

// ---- Jacobi-preconditioned CG on A = G W^-2 G^T + lambda I ("CG solver") ----
// Textbook preconditioned CG (Hestenes-Stiefel with M = diag(A) = diag + lambda, `diag` = diag(G W^-2 G^T) as
// written by orc_gram_diag; diag == NULL: M = I, which IS the iteration of orc_cg):
//   r0 = d, z0 = M^-1 r0, p0 = z0, rho0 = r0.z0;
//   q = A p;  a = rho / p.q;  x += a p;  r -= a q;  z = M^-1 r;  rho' = r.z;  b = rho'/rho;  p = z + b p.
// Stops after the iteration whose recursive residual satisfies ||r||_2 <= rtol ||d||_2 (rtol = 0: exactly `iters`
// iterations), before anything else if ||r0|| already does.  Returns the number of iterations performed.
// State (x, r, p, rho = r.z) in/out as in orc_cg; hist[it+1] = ||r||_2 (not the M-norm); ab as in orc_cg.
int orc_pcg(long long N, long long M, const double* G, const double* w, double lambda, const double* diag,
            const double* dobs, int iters, double rtol, int start, double* x, double* r, double* p, double* rho_io,
            double* hist, double* ab, int nthreads) {
    std::vector<double> g(M), q(N), z(N);
    auto dot = [&](const double* a, const double* b) {
        ld acc = 0;
        for (long long i = 0; i < N; ++i) acc += (ld)a[i] * (ld)b[i];
        return (double)acc;
    };
    auto applyMinv = [&](const double* rin, double* zout) {
        for (long long i = 0; i < N; ++i) zout[i] = diag ? rin[i] / (diag[i] + lambda) : rin[i];
    };
    auto applyA = [&](const double* pin, double* qout) {
        orc_dense_rmatvec(N, M, G, pin, g.data(), nthreads);
        for (long long c = 0; c < M; ++c) g[c] /= (w[c] * w[c]);
        orc_dense_matvec(N, M, G, g.data(), qout, nthreads);
        for (long long i = 0; i < N; ++i) qout[i] += lambda * pin[i];
    };
    const double tol2 = rtol * rtol * dot(dobs, dobs);
    double rho;
    if (start) {
        for (long long i = 0; i < N; ++i) { x[i] = 0.0; r[i] = dobs[i]; }
        applyMinv(r, z.data());
        for (long long i = 0; i < N; ++i) p[i] = z[i];
        rho = dot(r, z.data());
    } else rho = *rho_io;
    double rr = dot(r, r);
    if (hist) hist[0] = std::sqrt(rr);
    int it = 0;
    for (; it < iters; ++it) {
        if (rtol > 0.0 && rr <= tol2) break;
        applyA(p, q.data());
        double delta = dot(p, q.data());
        double a = rho / delta;
        for (long long i = 0; i < N; ++i) { x[i] += a * p[i]; r[i] -= a * q[i]; }
        applyMinv(r, z.data());
        double rho_new = dot(r, z.data());
        rr = dot(r, r);
        double b = rho_new / rho;
        for (long long i = 0; i < N; ++i) p[i] = z[i] + b * p[i];
        rho = rho_new;
        if (hist) hist[it + 1] = std::sqrt(rr);
        if (ab) { ab[2 * it] = a; ab[2 * it + 1] = b; }
    }
    *rho_io = rho;
    return it;
}

// ---- the paper's outer model-update loop around Eq. 10-11 ----------
// PARITY UNPINNED against the paper (see the header).  Readings R1-R4, step by step:
//   R1  m_0 = m_ref (NULL = 0);  r_k = d_obs - G m_k;  delta_m from Eq. 10-11 applied to r_k;  m_{k+1} = m_k + s delta_m
//   R2  outer "res" = ||r_k||_2 / ||d_obs||_2, stop when <= tol_outer or after max_outer updates;
//       inner: orc_pcg on (G W^-2 G^T + lambda I) alpha = r_k from 0, <= max_inner iterations, rtol = tol_inner
//       (diag = NULL: plain CG)
//   R3  s = 1, halved at most 10 times until ||r_k - s G delta_m||_2 < ||r_k||_2; no decrease: stop with m_k
//   R4  G is linear: G delta_m is formed once per update, every trial residual is r_k - s G delta_m
// Outputs: m[M]; dpred[N] = d_obs - r (= G m); hist[max_outer+1] = ||r_k|| / ||d_obs||; steps[max_outer] = accepted s;
// inner[max_outer] = CG iterations of each update; trials[max_outer*11] = ||r_k - 2^-h G delta_m||^2 of every trial
// made (NaN where none was made; for the margin checks of the parity tests).  The last three may be NULL.
// Returns the number of updates applied.
int orc_invert(long long N, long long M, const double* G, const double* w, double lambda, const double* diag,
               const double* dobs, const double* mref, int max_outer, int max_inner, double tol_outer,
               double tol_inner, double* m, double* dpred, double* hist, double* steps, int* inner, double* trials,
               int nthreads) {
    std::vector<double> r(N), dd(N), rt(N), alpha(N), cr(N), cp(N), dm(M);
    auto norm2 = [&](const double* a) {
        ld acc = 0;
        for (long long i = 0; i < N; ++i) acc += (ld)a[i] * (ld)a[i];
        return (double)acc;
    };
    if (trials) for (int i = 0; i < max_outer * 11; ++i) trials[i] = std::nan("");
    if (mref) {
        for (long long c = 0; c < M; ++c) m[c] = mref[c];
        orc_dense_matvec(N, M, G, m, dd.data(), nthreads);
        for (long long i = 0; i < N; ++i) r[i] = dobs[i] - dd[i];                       // R1
    } else {
        for (long long c = 0; c < M; ++c) m[c] = 0.0;
        for (long long i = 0; i < N; ++i) r[i] = dobs[i];
    }
    const double nd2 = norm2(dobs);
    const double dn = nd2 > 0.0 ? std::sqrt(nd2) : 1.0;
    double nr2 = norm2(r.data());
    hist[0] = std::sqrt(nr2) / dn;
    int k = 0;
    for (; k < max_outer; ++k) {
        if (std::sqrt(nr2) / dn <= tol_outer) break;                                    // R2 (outer)
        double rho = 0.0;
        int its = orc_pcg(N, M, G, w, lambda, diag, r.data(), max_inner, tol_inner, 1, alpha.data(), cr.data(),
                          cp.data(), &rho, nullptr, nullptr, nthreads);                 // R2 (inner)
        if (inner) inner[k] = its;
        orc_dense_rmatvec(N, M, G, alpha.data(), dm.data(), nthreads);                  // Eq. 11: delta_m = W^-2 G^T alpha
        for (long long c = 0; c < M; ++c) dm[c] /= (w[c] * w[c]);
        orc_dense_matvec(N, M, G, dm.data(), dd.data(), nthreads);                      // R4
        double s = 1.0, n2 = 0.0;
        bool ok = false;
        for (int h = 0; h <= 10; ++h, s *= 0.5) {                                       // R3
            for (long long i = 0; i < N; ++i) rt[i] = r[i] - s * dd[i];
            n2 = norm2(rt.data());
            if (trials) trials[k * 11 + h] = n2;
            if (n2 < nr2) { ok = true; break; }
        }
        if (steps) steps[k] = ok ? s : 0.0;
        if (!ok) break;
        for (long long c = 0; c < M; ++c) m[c] += s * dm[c];
        r = rt;
        nr2 = n2;
        hist[k + 1] = std::sqrt(nr2) / dn;
    }
    for (long long i = 0; i < N; ++i) dpred[i] = dobs[i] - r[i];
    return k;
}

int orc_hardware_threads() { return (int)std::thread::hardware_concurrency(); }

}  // extern "C"
