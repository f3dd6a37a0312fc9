// cg.cu -- fused vector operations of the data-space conjugate-gradient solve (BASELINE.json north_star kernel 3).
//
// Textbook Hestenes-Stiefel CG on A = G W^-2 G^T + lambda I (Eq. 10-11; reading C8):
//     q = A p;  delta = p.q;  a = rho/delta;  x += a p;  r -= a q;  rho' = r.r;  b = rho'/rho;  p = r + b p.
// All scalars stay on the device (CgScalars); dot products are two-stage with a fixed tree order, every block
// re-reduces the same kDotBlocks partials, so all blocks see bit-identical scalars and the result is
// deterministic.  q = G(.) + lambda p and the p.q partials are produced by forward_reduce (forward.cu) or
// dot_pq (stored-G mode).
#include "grav_internal.cuh"

namespace grav {

__device__ __forceinline__ double block_sum(double v, double* sh) {
    sh[threadIdx.x] = v;
    __syncthreads();
#pragma unroll
    for (int s = kDotThreads / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    double r = sh[0];
    __syncthreads();
    return r;
}

__device__ __forceinline__ double sum_partials(const double* __restrict__ dotp, double* sh) {
    static_assert(kDotBlocks == kDotThreads, "one partial per thread");
    return block_sum(dotp[threadIdx.x], sh);
}

__global__ void __launch_bounds__(kDotThreads) cg_init_kernel(long long N, const double* __restrict__ dobs,
                                                               double* __restrict__ x, double* __restrict__ r,
                                                               double* __restrict__ p, double* __restrict__ dotp,
                                                               int resume) {
    __shared__ double sh[kDotThreads];
    double loc = 0.0;
    for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < N; i += (long long)gridDim.x * kDotThreads) {
        double d = dobs[i];
        loc = fma(d, d, loc);
        if (!resume) { x[i] = 0.0; r[i] = d; p[i] = d; }
    }
    double s = block_sum(loc, sh);
    if (threadIdx.x == 0) dotp[blockIdx.x] = s;
}

__global__ void __launch_bounds__(kDotThreads) cg_init_finish_kernel(const double* __restrict__ dotp, CgScalars* sc,
                                                                      double rtol, int resume,
                                                                      const double* __restrict__ rho_in,
                                                                      double* __restrict__ hist) {
    __shared__ double sh[kDotThreads];
    double dn2 = sum_partials(dotp, sh);
    if (threadIdx.x == 0) {
        double rho = resume ? *rho_in : dn2;
        sc->rho[0] = rho;
        sc->rho[1] = rho;
        sc->dnorm2 = dn2;
        sc->tol2 = rtol * rtol * dn2;
        sc->delta = 0.0; sc->a = 0.0; sc->b = 0.0;
        sc->done = (rtol > 0.0 && rho <= sc->tol2) ? 1 : 0;
        sc->iters_done = 0;
        if (hist) hist[0] = sqrt(rho);
    }
}

// stored-G mode: q arrives without the lambda term; add it and form the p.q partials.
__global__ void __launch_bounds__(kDotThreads) dot_pq_kernel(long long N, const double* __restrict__ p,
                                                              const double* __restrict__ q, double lam,
                                                              double* __restrict__ q_out, double* __restrict__ dotp,
                                                              const int* __restrict__ done) {
    if (*done) return;
    __shared__ double sh[kDotThreads];
    double loc = 0.0;
    for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < N; i += (long long)gridDim.x * kDotThreads) {
        double pi = p[i];
        double val = fma(lam, pi, q[i]);
        q_out[i] = val;
        loc = fma(pi, val, loc);
    }
    double s = block_sum(loc, sh);
    if (threadIdx.x == 0) dotp[blockIdx.x] = s;
}

__global__ void __launch_bounds__(kDotThreads) cg_update_xr_kernel(long long N, double* __restrict__ x,
                                                                    double* __restrict__ r, const double* __restrict__ p,
                                                                    const double* __restrict__ q,
                                                                    const double* __restrict__ dotp_in,
                                                                    double* __restrict__ dotp_out, CgScalars* sc, int it) {
    if (sc->done) return;
    __shared__ double sh[kDotThreads];
    const double delta = sum_partials(dotp_in, sh);
    const double a = sc->rho[it & 1] / delta;
    double loc = 0.0;
    for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < N; i += (long long)gridDim.x * kDotThreads) {
        x[i] = fma(a, p[i], x[i]);
        double ri = fma(-a, q[i], r[i]);
        r[i] = ri;
        loc = fma(ri, ri, loc);
    }
    double s = block_sum(loc, sh);
    if (threadIdx.x == 0) {
        dotp_out[blockIdx.x] = s;
        if (blockIdx.x == 0) { sc->delta = delta; sc->a = a; }
    }
}

__global__ void __launch_bounds__(kDotThreads) cg_update_p_kernel(long long N, const double* __restrict__ r,
                                                                   double* __restrict__ p, const double* __restrict__ dotp,
                                                                   CgScalars* sc, int it, double* __restrict__ hist_slot,
                                                                   double* __restrict__ ab_slot) {
    __shared__ double sh[kDotThreads];
    if (sc->done) {   // frozen: carry rho forward so that the parity bookkeeping stays valid
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            double rho = sc->rho[it & 1];
            sc->rho[(it + 1) & 1] = rho;
            if (hist_slot) *hist_slot = sqrt(rho);
            if (ab_slot) { ab_slot[0] = 0.0; ab_slot[1] = 0.0; }
        }
        return;
    }
    const double rho_new = sum_partials(dotp, sh);
    const double b = rho_new / sc->rho[it & 1];
    for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < N; i += (long long)gridDim.x * kDotThreads)
        p[i] = fma(b, p[i], r[i]);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        sc->rho[(it + 1) & 1] = rho_new;
        sc->b = b;
        if (hist_slot) *hist_slot = sqrt(rho_new);
        if (ab_slot) { ab_slot[0] = sc->a; ab_slot[1] = b; }
        sc->iters_done = it + 1;
    }
}

// `done` must be raised only after every block of update_p has read it: separate 1-thread kernel.
__global__ void cg_check_done_kernel(CgScalars* sc, int it) {
    if (!sc->done && sc->tol2 > 0.0 && sc->rho[(it + 1) & 1] <= sc->tol2) sc->done = 1;
}

cudaError_t launch_cg_init(grav_ctx* c, const double* dobs, double* x, double* r, double* p, double* dotp, int resume,
                           cudaStream_t s) {
    cg_init_kernel<<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, dobs, x, r, p, dotp, resume);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_cg_init_finish(grav_ctx* c, const double* dotp, CgScalars* sc, double rtol, int resume,
                                  const double* rho_in, double* hist, cudaStream_t s) {
    cg_init_finish_kernel<<<1, kDotThreads, 0, s>>>(dotp, sc, rtol, resume, rho_in, hist);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_dot_pq(grav_ctx* c, const double* p, const double* q, double lam, double* q_out, double* dotp,
                          const CgScalars* sc, cudaStream_t s) {
    dot_pq_kernel<<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, p, q, lam, q_out, dotp, &sc->done);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_cg_update_xr(grav_ctx* c, double* x, double* r, const double* p, const double* q,
                                const double* dotp_in, double* dotp_out, CgScalars* sc, int it, cudaStream_t s) {
    cg_update_xr_kernel<<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, x, r, p, q, dotp_in, dotp_out, sc, it);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_cg_update_p(grav_ctx* c, const double* r, double* p, const double* dotp, CgScalars* sc, int it,
                               double rtol, double* hist_slot, double* ab_slot, cudaStream_t s) {
    cg_update_p_kernel<<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, r, p, dotp, sc, it, hist_slot, ab_slot);
    c->launches++;
    if (rtol > 0.0) {
        cg_check_done_kernel<<<1, 1, 0, s>>>(sc, it);
        c->launches++;
    }
    return cudaGetLastError();
}

}  // namespace grav
