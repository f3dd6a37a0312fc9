/* grav.h -- C ABI of libgrav.so: matrix-free FP64 prism-gravity operator and data-space CG on one B200 (sm_100a).
 *
 * What is computed (citations: P:nn = PAPER.md line nn of arxiv/paper_2602_03857; BJ = BASELINE.json north_star):
 *   G_ik = gamma * sum_{p,q,r in {1,2}} (-1)^(p+q+r) Psi(x_p - xo_i, y_q - yo_i, z_r - zo_i)        P:49-52  Eq. 1
 *   Psi(X,Y,Z) = Z atan(XY/(ZR)) - X ln(R+Y) - Y ln(R+X),  R = sqrt(X^2+Y^2+Z^2)                     P:54-58  Eq. 2-3
 *   d = G u                                                                                           P:68-74  Eq. 5-6
 *   g = G^T v                                                                                         P:98-110 (G^T of Eq. 9-11)
 *   w_k = (zc_k + z0)^(-beta/2), zc_k = depth of the cell centre below the mesh top                   P:85; BJ
 *   (G W^-2 G^T + lambda I) alpha = d_obs by CG,  m = W^-2 G^T alpha                                  P:101-118 Eq. 10-11; BJ
 *
 * Conventions.  z is positive DOWN.  Cell (i,j,k), 0-based, has flat index (i*ny + j)*nz + k (z fastest) and
 * bounds [xn[i],xn[i+1]] x [yn[j],yn[j+1]] x [zn[k],zn[k+1]].  Stations are SoA (obs_x, obs_y, obs_z).
 * gamma = 6.674e-6 gives gz in mGal for densities in kg/m^3 and lengths in m.  All arithmetic is FP64.
 *
 * Pointers.  Names ending in _host are HOST pointers (pageable or pinned), names ending in _dev are DEVICE pointers
 * on the context's device.  `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *
 * Ownership.  grav_mesh_create copies the node and station coordinates and the Psi tables to the device (its only
 * allocation, <= 4.6 MB at 178,797 stations; freed by grav_mesh_destroy).  EVERY other device byte belongs to the caller:
 * inputs, outputs and one workspace block (grav_workspace_bytes / grav_set_workspace) that must stay alive and
 * must not be touched by the caller while a call that uses it is in flight.
 *
 * Execution.  *_dev entry points enqueue kernels on `stream` and return without synchronising (CG scalars stay
 * on the device).  Exceptions: grav_invert synchronises once per trial step (it reads one scalar back), and
 * grav_depth_weights does one blocking 16-byte copy when z0 < 0.  *_host entry points copy in, compute, copy out and
 * synchronise `stream` before returning.
 * Results are deterministic (fixed reduction orders, no atomics on data).
 *
 * Errors.  Every call returns a grav_status; no exception crosses the ABI; grav_last_error() returns a
 * thread-local message for the last non-OK status.  There is no CPU fallback anywhere in this library.
 */
#ifndef GRAV_H_
#define GRAV_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct grav_ctx grav_ctx; /* opaque */

typedef enum {
    GRAV_OK = 0,
    GRAV_EINVAL = -1,  /* NULL pointer, non-positive size, non-increasing node coordinates, bad mode */
    GRAV_ENOMEM = -2,  /* host or device allocation of the geometry copy failed */
    GRAV_ECUDA = -3,   /* a CUDA runtime call or kernel launch failed (message has the CUDA error string) */
    GRAV_ESTATE = -4,  /* workspace not set / too small, or stored G requested before grav_store_g */
    GRAV_ENOTFIT = -5  /* stored G does not fit in the workspace given */
} grav_status;

/* operator modes */
enum {
    GRAV_MATRIX_FREE = 0, /* closed form evaluated on the fly for every station x node pair (BJ kernels 1, 2) */
    GRAV_STORED_F64 = 1,  /* G tabulated once as N x M doubles, products are HBM-bound GEMV (BJ kernel 4) */
    GRAV_STORED_F32 = 2   /* G stored as float (the paper's precision), accumulated in FP64 */
};

/* Device-resident CG state for resuming / single-step injection (SURVEY.md 8(c) protocol P1).
 * x, r, p: N doubles each; rho: 1 double (= r.r).  resume = 0: the solver initialises x=0, r=p=d_obs and
 * overwrites the state on return; resume != 0: the solver continues from the state given. */
typedef struct {
    double* x_dev;
    double* r_dev;
    double* p_dev;
    double* rho_dev;
    int resume;
} grav_cg_state;

/* Create a context for a rectilinear nx x ny x nz prism mesh and nobs stations (mesh of prisms
 * defined by their vertices; stations (x0_i, y0_i[, z0_i])).
 * xn_host[nx+1], yn_host[ny+1], zn_host[nz+1]: node coordinates, strictly increasing; z down.
 * obs_*_host[nobs]: station coordinates.  gamma: gravitational constant in the caller's units.
 * device: CUDA device ordinal.  Errors: GRAV_EINVAL, GRAV_ENOMEM, GRAV_ECUDA. */
grav_status grav_mesh_create(grav_ctx** out, int nx, int ny, int nz, const double* xn_host, const double* yn_host,
                             const double* zn_host, long long nobs, const double* obs_x_host,
                             const double* obs_y_host, const double* obs_z_host, double gamma, int device);
void grav_mesh_destroy(grav_ctx* ctx);

/* Problem sizes: out[0]=N stations, out[1]=M prisms, out[2]=number of mesh nodes (nx+1)(ny+1)(nz+1). */
grav_status grav_sizes(const grav_ctx* ctx, long long out[3]);

/* Bytes of caller-owned device workspace needed for `mode` (GRAV_MATRIX_FREE, or the matrix-free block plus the
 * N x M stored G in FP64 / FP32).  0 on error. */
size_t grav_workspace_bytes(const grav_ctx* ctx, int mode);
/* Hand the workspace to the context (256-byte aligned).  Invalidates a previously stored G.
 * Errors: GRAV_EINVAL (NULL / misaligned), GRAV_ESTATE (smaller than the matrix-free block). */
grav_status grav_set_workspace(grav_ctx* ctx, void* ws_dev, size_t bytes);

/* d = G u, matrix-free (Eq. 5-6; BJ kernel 1).  u_dev[M] -> d_dev[N]. */
grav_status grav_forward(grav_ctx* ctx, const double* u_dev, double* d_dev, void* stream);
/* g = G^T v, matrix-free (BJ kernel 2).  v_dev[N] -> g_dev[M]. */
grav_status grav_adjoint(grav_ctx* ctx, const double* v_dev, double* g_dev, void* stream);
/* w_k = (zc_k + z0)^(-beta/2) (BJ).  w_dev[M].  Requires zc_k + z0 > 0 for every layer (else GRAV_EINVAL). */
grav_status grav_depth_weights(grav_ctx* ctx, double beta, double z0, double* w_dev, void* stream);

/* Conjugate gradients on (G W^-2 G^T + lambda I) alpha = d_obs (Eq. 10-11 with W_m = W^-2,
 * W_d = lambda I, m_ref = 0; textbook Hestenes-Stiefel, x0 = 0).  Runs exactly `iters` iterations when rtol = 0;
 * with rtol > 0 the iteration freezes (remaining launches become no-ops) once ||r||_2 <= rtol * ||d_obs||_2.
 * mode: operator used for the products (stored modes need grav_store_g first).
 * precond_dev[N] or NULL: Jacobi preconditioning ("CG solver with depth-weighted
 *   regularization").  Pass diag(G W^-2 G^T) as written by grav_gram_diag; the solver applies z = r / (precond + lambda),
 *   rho = r.z, p = z + b p.  NULL: plain CG (z = r).
 * state: NULL or see grav_cg_state (with a preconditioner rho is r.z).   alpha_dev[N]: solution.
 * m_dev[M] or NULL: m = W^-2 G^T alpha.
 * hist_dev[iters+1] or NULL: ||r||_2 before the first and after every iteration (recursive residual).
 * ab_dev[2*iters] or NULL: step scalars a_j (step length), b_j (direction update) of every iteration. */
grav_status grav_dataspace_cg(grav_ctx* ctx, const double* dobs_dev, const double* w_dev, double lambda, int iters,
                              double rtol, int mode, const double* precond_dev, grav_cg_state* state,
                              double* alpha_dev, double* m_dev, double* hist_dev, double* ab_dev, void* stream);

/* Tabulate G (N x M row-major, prism index fastest; "global memory (sensitivity matrix)", Listing 1)
 * into the workspace in FP64 (fp32 = 0) or FP32 (fp32 != 0).  GRAV_ENOTFIT if the workspace is too small. */
grav_status grav_store_g(grav_ctx* ctx, int fp32, void* stream);
/* d = G u and g = G^T v with the stored G (HBM-bound GEMV, BJ kernel 4; "matrix multiplications"). */
grav_status grav_forward_stored(grav_ctx* ctx, const double* u_dev, double* d_dev, void* stream);
grav_status grav_adjoint_stored(grav_ctx* ctx, const double* v_dev, double* g_dev, void* stream);
/* Device pointer / element size (8 or 4; 0 if none) of the stored G, for inspection by tests. */
grav_status grav_stored_g(const grav_ctx* ctx, const void** g_dev, int* elem_bytes);

/* diag_dev[N] = diag(G W^-2 G^T)_ii = sum_k G_ik^2 / w_k^2, matrix-free per-pair evaluation (its sum is the
 * trace that fixes lambda = 1e-2 * trace / N, BJ config 1; diag + lambda is the Jacobi preconditioner of
 * grav_dataspace_cg).  Needs the workspace. */
grav_status grav_gram_diag(grav_ctx* ctx, const double* w_dev, double* diag_dev, void* stream);

/* Small problems (N <= 1024, needs a stored FP64 G): form A = G W^-2 G^T + lambda I explicitly and solve
 * A alpha = d_obs by Cholesky on the device (BJ config 1 "solved both directly and by CG").
 * A_dev: N*N doubles of caller scratch (holds the factor on return).  m_dev[M] or NULL. */
grav_status grav_direct_solve(grav_ctx* ctx, const double* dobs_dev, const double* w_dev, double lambda,
                              double* A_dev, double* alpha_dev, double* m_dev, void* stream);

/* The paper's outer model-update loop around the data-space CG (<= 30 outer updates, <= 20 inner CG
 * iterations, both stopped at res <= 1e-4; "Gauss-Newton-style update loop with step-size backtracking";
 * Eq. 10-11, for the update itself).  The paper prints neither the residual norm nor the backtracking
 * rule; DESIGN.md 2 (R1-R4) fixes them, and parity with the PAPER's loop is therefore unpinned (the oracle restates
 * the same readings):
 *   m_0 = m_ref (NULL = 0);  r_k = d_obs - G m_k;  stop when ||r_k||_2 / ||d_obs||_2 <= tol_outer or k = max_outer;
 *   alpha = CG on (G W^-2 G^T + lambda I) alpha = r_k, <= max_inner iterations, stopped at ||res|| <= tol_inner ||r_k||;
 *   delta_m = W^-2 G^T alpha;  s = 1, halved at most 10 times until ||r_k - s G delta_m|| < ||r_k||
 *   (no decrease: stop with m_k);  m_{k+1} = m_k + s delta_m.
 * dobs_dev[N], w_dev[M], mref_dev[M] or NULL, precond_dev[N] or NULL (Jacobi preconditioner of the inner solves, as in
 * grav_dataspace_cg), m_dev[M] out, dpred_dev[N] out or NULL (= G m): DEVICE.
 * hist_host[max_outer + 1] (||r_k|| / ||d_obs||, entries 0..*n_outer_host), step_host[max_outer] (accepted s per
 * update, 0 = rejected), inner_host[max_outer] (CG iterations each update performed before its tolerance stop),
 * n_outer_host (updates applied): HOST, each may be NULL.  mode as in grav_dataspace_cg.
 * SYNCHRONISES the stream once per trial step (one scalar read back); needs the workspace. */
grav_status grav_invert(grav_ctx* ctx, const double* dobs_dev, const double* w_dev, double lambda,
                        const double* mref_dev, const double* precond_dev, int max_outer, int max_inner,
                        double tol_outer, double tol_inner, int mode, double* m_dev, double* dpred_dev,
                        double* hist_host, double* step_host, int* inner_host, int* n_outer_host, void* stream);

/* End-to-end variants with HOST buffers: host->device copy of the inputs, the same kernels, device->host copy
 * of the result, then cudaStreamSynchronize(stream).  Staging buffers live in the workspace. */
grav_status grav_forward_host(grav_ctx* ctx, const double* u_host, double* d_host, void* stream);
grav_status grav_adjoint_host(grav_ctx* ctx, const double* v_host, double* g_host, void* stream);
grav_status grav_dataspace_cg_host(grav_ctx* ctx, const double* dobs_host, double beta, double z0, double lambda,
                                   int iters, double rtol, int mode, double* alpha_host, double* m_host,
                                   double* hist_host, void* stream);

/* Observation-sharded operation over several GPUs ("observation domain partitioned across devices, model-space
 * variables replicated and synchronised").  Each rank creates its context on ITS OWN station shard (same mesh) and
 * registers two collectives over the `world` ranks, both ordered on the `stream` they are handed (e.g. NCCL; return 0
 * on success).  The library calls them exactly where the method exchanges data:
 *   - allgather of the local node sums T (2 N_n doubles: [hi | lo] planes of the compensated sums) after the local
 *     adjoint kernel; the ranks' (hi, lo) pairs are then combined error-free, in rank order, by the same kernel that
 *     combines station chunks, so the sharded G^T v equals the single-rank one to rounding and is bit-identical on
 *     every rank -> grav_adjoint / CG / model recovery return the GLOBAL G^T v, m;
 *   - allreduce_sum of the 256-entry block partials of the CG dot products (d.d, p.q, r.z, r.r), of the norms of
 *     grav_invert, and (stored modes) of the M-vector after the local G^T product.
 * grav_forward, grav_gram_diag and alpha stay local to the rank's stations; there is no other communication.
 * grav_set_comm changes the workspace layout (the gather buffer needs world x 2 N_n doubles): call it BEFORE
 * grav_workspace_bytes / grav_set_workspace; it detaches a workspace set earlier.  comm = NULL or world = 1 restores
 * single-rank operation.  grav_direct_solve is not available on a sharded context. */
typedef struct {
    int world; /* number of ranks, >= 1 */
    int rank;  /* this rank, 0 <= rank < world */
    /* buf_dev[k] = sum over ranks of buf_dev[k], k < count, in place, every rank receives the same bits */
    int (*allreduce_sum)(double* buf_dev, long long count, void* stream, void* user);
    /* recv_dev[r * count + k] = send_dev[k] of rank r, k < count (recv_dev holds world * count doubles) */
    int (*allgather)(const double* send_dev, double* recv_dev, long long count, void* stream, void* user);
    void* user;
} grav_comm;
grav_status grav_set_comm(grav_ctx* ctx, const grav_comm* comm);

/* Precision of the matrix-free evaluation ("using Float32 precision").
 * GRAV_PREC_F64 (default): everything in FP64 (BJ).  GRAV_PREC_F32: grav_forward, grav_adjoint and the GRAV_MATRIX_FREE
 * products inside grav_dataspace_cg / grav_invert evaluate Psi in Float32 - from coordinate differences formed in FP64,
 * with the cancellation-free form of R + Y for Y < 0 - and accumulate in FP64; vectors stay FP64.  The per-pair family
 * (grav_store_g, grav_gram_diag) always evaluates in FP64.  The Float32 closed form has a cancellation floor of
 * ~(|X| + |Y| + |Z|) 2^-24 per corner term (~1e-3 m at 10 km, where far-field coefficients are 1e-5..1e-3 m): this mode
 * reproduces the paper's precision for comparison, its error is reported by bench.py and it is NOT held to the 1e-10
 * operator tolerance.  Errors: GRAV_EINVAL. */
enum { GRAV_PREC_F64 = 0, GRAV_PREC_F32 = 1 };
grav_status grav_set_precision(grav_ctx* ctx, int precision);

/* Allocation-free stored-G adjoint product (for callers that cannot call cudaMalloc or hold a workspace: code under
 * CUDA graph capture, serving loops, harnesses that forbid allocation):
 *     g[m] = sum_i G[i][m] v[i]          (w_dev == NULL)        -- what grav_adjoint_stored computes (Eq. 10's G^T)
 *     g[m] = sum_i G[i][m] v[i] / w[m]^2 (w_dev != NULL)        -- W^-2 G^T v, the model recovery of Eq. 10-11
 * with the same kernels, row chunking and summation order as grav_adjoint_stored, so the results are bit-identical.
 * Needs no context and no workspace: the per-chunk column sums go to a file-scope device array of
 * GRAV_NOALLOC_MAX_DOUBLES doubles (16 MiB) that every GPU loading the library holds until exit.  The call makes no
 * cudaMalloc / cudaFree and calls no allocating library routine; it enqueues 2 kernels on `stream` and returns.
 * G_dev: N x M row-major on `device`, elem_bytes = 8 (double) or 4 (float; accumulated in FP64).  v_dev[N], w_dev[M] or
 * NULL, g_dev[M]: device doubles, caller-owned.  Limit: min(16, ceil(N / 256)) * M <= GRAV_NOALLOC_MAX_DOUBLES (e.g.
 * M <= 131,072 for N >= 3,841; M <= 2,097,152 for N <= 256); beyond it the call returns GRAV_EINVAL with a message
 * stating the limit and launches nothing.
 * The array is shared by all calls and keeps the last call's contents; nothing in it has to start at zero (every entry
 * the reduction reads is written by the same call first).  Calls that overlap on the GPU (different streams, or
 * different threads without ordering) race on it: serialise them on one stream or with events.
 * The first call on a device looks up the array's address (cudaGetSymbolAddress, once per device; not an allocation):
 * call grav_noalloc_setup(device) beforehand where that must not happen inside the critical region (e.g. before
 * beginning a capture).  Errors: GRAV_EINVAL (NULL pointer, N or M < 1, elem_bytes, size beyond the limit, device
 * index), GRAV_ECUDA. */
#define GRAV_NOALLOC_MAX_DOUBLES (2ll << 20)
grav_status grav_noalloc_setup(int device);
grav_status grav_gemvt_noalloc(int device, const void* G_dev, int elem_bytes, long long N, long long M,
                               const double* v_dev, const double* w_dev, double* g_dev, void* stream);

/* Launch accounting: number of kernels this context has launched since creation (for bench.py's gpu_launches). */
long long grav_launch_count(const grav_ctx* ctx);
/* FP64 DFMA-only microbenchmark: runs `iters` dependent-chain-free DFMA per thread on the whole device and
 * returns the number of FP64 thread-instructions executed in *ninstr and the elapsed ms in *ms (synchronises).
 * Used to confirm the FP64 pipe peak in the same run as the roofline numbers. */
grav_status grav_fp64_peak_probe(int device, int iters, double* ninstr, double* ms);
/* Diagnostics.  variant 0 (default): hand-built Psi evaluator (table-driven ln, reduced-argument atan2, MUFU-seeded
 * sqrt / reciprocal; csrc/psi.cuh); variant 1: the same tilings with CUDA libm (sqrt, /, atan, log).  Both are tested
 * against the oracle; variant 1 exists for cross-checks and A/B timing. */
grav_status grav_debug_set_psi_variant(grav_ctx* ctx, int variant);
/* One Psi evaluation per argument triple with a device evaluator (tests compare them with the oracle's Psi argument by
 * argument): variant 0 = hand-built FP64 evaluator with the 256-entry log table, 1 = CUDA libm FP64, 2 = Float32
 * evaluator, 3 = hand-built FP64 evaluator with the exponent-and-mantissa log table (GRAV_ESTATE when the context has
 * none; arguments of the logarithms must then lie in its range).  X_dev, Y_dev, Z_dev, out_dev: n doubles each.
 * Variants 0, 2, 3 return Psi + (X + Y) k0 ln 2 with k0 = grav_debug_k0(ctx) (clamped to +-100 for variant 2): the
 * offset that cancels exactly in every signed sum of the library.  Needs no workspace. */
grav_status grav_debug_psi_eval_device(grav_ctx* ctx, int variant, long long n, const double* X_dev, const double* Y_dev,
                                       const double* Z_dev, double* out_dev, void* stream);
/* Which log table the variant-0 kernels use: -1 the context's default (grav_debug_log2d_default), 0 the 256-entry
 * table with explicit exponent handling, 1 the exponent-and-mantissa table (GRAV_ESTATE when the geometry does not
 * admit it).  Both form the same sums in the same order; they differ by rounding only.  For tests and A/B timing. */
grav_status grav_debug_set_log2d(grav_ctx* ctx, int mode);
/* Host-side evaluation of the variant-0 algorithm (same source, MUFU seeds emulated at 2^-20 accuracy) so that
 * CPU-only tests can check it: returns Psi(X,Y,Z) + (X+Y)*k0*ln2 (the offset cancels in every signed sum, see
 * csrc/psi.cuh).  log2d = 0: 256-entry log table; 1: exponent-and-mantissa table, valid for arguments of the
 * logarithms in [2^-80, 2^80).  Caches its tables per k0: not thread-safe. */
double grav_debug_psi_eval_host(double X, double Y, double Z, int k0, int log2d);
/* The global exponent offset k0 chosen for this context (2^k0 ~ survey scale). */
int grav_debug_k0(const grav_ctx* ctx);
/* Number of binades of the exponent-and-mantissa log table built for this context, or 0 when the geometry does not
 * bound the arguments of the logarithms (a station level with or inside the mesh, or a ratio above 2^40): then the
 * kernels use the 256-entry table with explicit exponent handling. */
int grav_debug_log2d_binades(const grav_ctx* ctx);
/* 1 when the default kernels of this context use that table: it exists AND the problem is large enough to amortise
 * filling it per block (stations x nodes >= 5e7). */
int grav_debug_log2d_default(const grav_ctx* ctx);

/* Thread-local message of the last failure on this thread ("" if none). */
const char* grav_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GRAV_H_ */
