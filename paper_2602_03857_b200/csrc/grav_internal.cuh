// grav_internal.cuh -- shared declarations of the CUDA path (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/grav.h"
#include "psi.cuh"

namespace grav {

// Geometry handed to every kernel by value.  Node (a,b,c) <-> flat index (a*nyp + b)*nzp + c (z fastest), so a
// vertical node column is contiguous; "column" col = a*nyp + b.
struct Geom {
    int nx, ny, nz;        // cells
    int nxp, nyp, nzp;     // nodes per axis = cells + 1
    int ncol;              // nxp * nyp node columns
    long long N, M, Nn;    // stations, prisms, nodes
    const double* xn;      // device, nxp
    const double* yn;      // device, nyp
    const double* zn;      // device, nzp
    const double* xo;      // device, N
    const double* yo;
    const double* zo;
    double gamma;
};

// Launch plans fixed at context creation (deterministic reduction orders).
struct Plan {
    // forward: grid (obs tiles, node-column chunks)
    int log2d;             // 1: kernels use the 2-D log table (psi.cuh LOG2D)
    int persistent;        // 1: node kernels launch one block per SM slot that draws work items from a counter
    int sms;               // multiprocessors of the device
    int fwd_reduce_rx;     // stations per block of forward_reduce (32, or 8 when stations are few and chunks many)
    int fwd_tpb, fwd_tiles, fwd_nchunk, fwd_cols_per_chunk;
    // adjoint: grid (node-thread blocks, station chunks)
    int adj_tpb, adj_kc, adj_ncg, adj_blocks, adj_nchunk, adj_obs_per_chunk;
    int adj_kt;            // > 0: the column is covered by whole groups of adj_kc nodes and one tail group of adj_kt (adjoint.cu)
    // per-pair family (stored.cu): node tile of pair_tnx x pair_tny node columns per block
    int pair_tnx, pair_tny, pair_tiles_x, pair_tiles_y;
};

constexpr int kDotBlocks = 256;     // block partials of the fused CG dot products
constexpr int kDotThreads = 256;

// CG scalar block (device): see cg.cu.  rho is double-buffered by iteration parity so that no kernel reads a
// scalar another block of the same launch writes.
struct CgScalars {
    double rho[2];
    double delta, a, b, dnorm2, tol2, rr;     // rr = ||r||^2 of the last finished iteration
    int done[2], iters_done;                  // done: frozen flag (rtol reached), by iteration parity like rho
};

struct WsLayout {
    size_t cnode, tnode, fwd_partial, adj_partial, gcell, cg_x, cg_r, cg_p, cg_q, cg_z, cg_w, dot_partial, scalars,
        stage_m, stage_n, stage_hist, work, inv_dm, inv_r, inv_dd, inv_try, inv_scal, gram_partial, comm_gather, matfree_end,
        gemvt_partial, gstore;
};

// (hi_out, lo_out) = (hi_in, lo_in) + x with the rounding error of hi_in + x captured exactly (Knuth TwoSum).
__device__ __forceinline__ void two_sum_acc(double hi_in, double lo_in, double x, double& hi_out, double& lo_out) {
    const double s = hi_in + x;
    const double bb = s - hi_in;
    const double err = (hi_in - (s - bb)) + (x - bb);
    hi_out = s;
    lo_out = lo_in + err;
}

}  // namespace grav

struct grav_ctx {
    grav::Geom g;
    grav::Plan plan;
    grav::WsLayout lay;
    int device;
    void* geom_dev;          // one allocation holding xn,yn,zn,xo,yo,zo and the Psi tables
    char* ws;                // caller's workspace
    size_t ws_bytes;
    int stored_elem;         // 0 none, 8 FP64, 4 FP32
    grav::PsiDev pd;         // Psi tables (inside geom_dev), constants and the global exponent offset k0
    int psi_variant;         // 0 hand-built FP64 evaluator, 1 CUDA libm FP64, 2 Float32 evaluator (grav_set_precision)
    int log2d_force;         // -1: the plan's choice; 0 / 1: force the 256-entry / the 2-D log table (diagnostic)
    grav_comm comm;          // observation-sharded operation (world == 1: single rank, no callbacks)
    long long launches;
};

namespace grav {

inline bool use_log2d(const grav_ctx* c) {
    if (!c->pd.tab2d) return false;
    return c->log2d_force < 0 ? c->plan.log2d != 0 : c->log2d_force != 0;
}

// Opt a kernel into > 48 KB of dynamic shared memory once per (kernel, device); thread-safe (the attribute is per
// device, and setting it twice is harmless).
template <class Kernel>
inline cudaError_t ensure_dynamic_smem(Kernel kernel, size_t bytes, int device, unsigned long long* done_mask) {
    const unsigned long long bit = 1ull << (device & 63);
    if (__atomic_load_n(done_mask, __ATOMIC_ACQUIRE) & bit) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) __atomic_fetch_or(done_mask, bit, __ATOMIC_RELEASE);
    return e;
}

// every launcher returns cudaGetLastError() of its launches and bumps ctx->launches
// --- nodeops.cu
cudaError_t launch_cell_to_node(grav_ctx* c, const double* u, const double* w_or_null, double* cnode, cudaStream_t s);
cudaError_t launch_node_to_cell(grav_ctx* c, const double* tnode, const double* w_or_null, double scale, double* gcell,
                                cudaStream_t s);
cudaError_t launch_depth_weights(grav_ctx* c, double beta, double z0, double* w, cudaStream_t s);
// --- forward.cu : partial sums of sum_n cnode[n] Psi(node_n - obs_i) into fwd_partial
// work: one int of device scratch (the item counter of a persistent launch, plan.persistent)
cudaError_t launch_forward_nodes(grav_ctx* c, const double* cnode, double* partial, const int* done, int* work,
                                 cudaStream_t s);
// d = scale * sum_chunks partial (+ lam * p if p != NULL); if dot_partial != NULL also block partials of p.d
cudaError_t launch_forward_reduce(grav_ctx* c, const double* partial, double scale, double lam, const double* p,
                                  double* d, double* dot_partial, const int* done, cudaStream_t s);
// --- adjoint.cu : tnode[n] = sum_i v_i Psi(node_n - obs_i)
cudaError_t launch_adjoint_nodes(grav_ctx* c, const double* v, double* partial, const int* done, int* work,
                                 cudaStream_t s);
cudaError_t launch_adjoint_reduce(grav_ctx* c, const double* partial, int nchunk, double* tnode, cudaStream_t s);
// --- cg.cu
cudaError_t launch_cg_init(grav_ctx* c, const double* dobs, const double* minv, double lam, double* x, double* r,
                           double* z, double* p, double* dotp, int resume, cudaStream_t s);
cudaError_t launch_cg_init_finish(grav_ctx* c, const double* dotp, CgScalars* sc, double rtol, int resume,
                                  const double* rho_in, double* hist, cudaStream_t s);
cudaError_t launch_dot_pq(grav_ctx* c, const double* p, double lam, double* q, double* dotp, const CgScalars* sc,
                          int it, cudaStream_t s);
cudaError_t launch_cg_update_xr(grav_ctx* c, double* x, double* r, const double* p, const double* q,
                                const double* minv, double lam, double* z, const double* dotp_in, double* dotp_out,
                                CgScalars* sc, int it, cudaStream_t s);
cudaError_t launch_cg_update_p(grav_ctx* c, const double* z, double* p, const double* dotp, CgScalars* sc, double* hist,
                               double* ab, int it, cudaStream_t s);
// --- stored.cu
cudaError_t launch_tabulate(grav_ctx* c, void* G, int elem, cudaStream_t s);
cudaError_t launch_gemv(grav_ctx* c, const void* G, int elem, const double* u, double* d, cudaStream_t s);
cudaError_t launch_gemvt(grav_ctx* c, const void* G, int elem, const double* v, const double* w_or_null, double* g,
                         double* partial, cudaStream_t s);
// winv2: M doubles of scratch (1 / w^2)
cudaError_t launch_gram_diag(grav_ctx* c, const double* w, double* winv2, double* partial, double* diag,
                             cudaStream_t s);
cudaError_t launch_form_A(grav_ctx* c, const double* G, const double* w, double lam, double* A, cudaStream_t s);
cudaError_t launch_cholesky_solve(grav_ctx* c, double* A, const double* b, double* x, int n, cudaStream_t s);
int gemvt_chunks(long long N);
// no-allocation variant of gemvt: per-chunk sums in a file-scope device array of kNoAllocMaxDoubles (16 MiB)
constexpr long long kNoAllocMaxDoubles = 2ll << 20;
cudaError_t noalloc_setup(int device, double** ptr_or_null);
long long noalloc_gemvt_doubles(long long N, long long M);
cudaError_t launch_gemvt_noalloc(int device, const void* G, int elem, long long N, long long M, const double* v,
                                 const double* w_or_null, double* g, cudaStream_t s);
void make_pair_plan(const Geom& g, const PsiDev& pd, bool log2d, Plan& p);
size_t gram_partial_doubles(const Geom& g, const Plan& p);
// --- psi_check.cu : one Psi evaluation per argument triple with the chosen device evaluator (diagnostic)
cudaError_t launch_psi_check(grav_ctx* c, int variant, long long n, const double* X, const double* Y, const double* Z,
                             double* out, cudaStream_t s);
// --- invert.cu : vector kernels of the outer model-update loop
cudaError_t launch_inv_residual(grav_ctx* c, const double* r, double s, const double* dd, double* out, double* partial,
                                cudaStream_t st);
cudaError_t launch_inv_finish(grav_ctx* c, const double* partial, double* scalar, cudaStream_t st);
cudaError_t launch_inv_axpy(grav_ctx* c, double a, const double* x, double* y, cudaStream_t st);

}  // namespace grav
