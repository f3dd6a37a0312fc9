// cg.cu -- fused vector operations of the data-space conjugate-gradient solve (BASELINE.json north_star kernel 3).
//
// Textbook Hestenes-Stiefel CG on A = G W^-2 G^T + lambda I (Eq. 10-11; reading C8), optionally
// with the Jacobi preconditioner M = diag(A) ("CG solver"):
//     q = A p;  delta = p.q;  a = rho/delta;  x += a p;  r -= a q;  z = M^-1 r;  rho' = r.z;  b = rho'/rho;  p = z + b p.
// Without a preconditioner z IS r (the same buffer) and rho = r.r.  All scalars stay on the device (CgScalars); dot
// products are two-stage with a fixed tree order, every block re-reduces the same kDotBlocks partials, so all blocks see
// bit-identical scalars and the result is deterministic.  rho and the frozen flag are double-buffered by iteration parity.  q = G(.) + lambda p and the p.q partials are produced by
// forward_reduce (forward.cu) or dot_pq (stored-G mode).  Dot partial layout: [A: p.q | B: r.z | C: r.r].
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

// Start (resume == 0): x = 0, r = d, z = M^-1 d, p = z.  Resume: the state (x, r, p) is the caller's.
// Partials: dotp[0..) of r.z (start only), dotp[kDotBlocks..) of d.d, dotp[2 kDotBlocks..) of r.r.
__global__ void __launch_bounds__(kDotThreads) cg_init_kernel(long long N, const double* __restrict__ dobs,
                                                               const double* __restrict__ minv, double lam, double* x,
                                                               double* r, double* z, double* p,
                                                               double* __restrict__ dotp, int resume) {
    __shared__ double sh[kDotThreads];
    double locd = 0.0, locz = 0.0, locr = 0.0;
    for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < N; i += (long long)gridDim.x * kDotThreads) {
        const double d = dobs[i];
        locd = fma(d, d, locd);
        if (resume) {
            const double ri = r[i];
            locr = fma(ri, ri, locr);
        } else {
            const double zi = minv ? d / (minv[i] + lam) : d;
            locz = fma(d, zi, locz);
            x[i] = 0.0; r[i] = d; p[i] = zi;
            if (minv) z[i] = zi;
        }
    }
    const double sd = block_sum(locd, sh);
    const double sz = block_sum(locz, sh);
    const double sr = resume ? block_sum(locr, sh) : sd;
    if (threadIdx.x == 0) {
        dotp[blockIdx.x] = sz;
        dotp[kDotBlocks + blockIdx.x] = sd;
        dotp[2 * kDotBlocks + blockIdx.x] = sr;
    }
}

__global__ void __launch_bounds__(kDotThreads) cg_init_finish_kernel(const double* __restrict__ dotp, CgScalars* sc,
                                                                      double rtol, int resume,
                                                                      const double* __restrict__ rho_in,
                                                                      double* __restrict__ hist) {
    __shared__ double sh[kDotThreads];
    const double dz = sum_partials(dotp, sh);
    const double dn2 = sum_partials(dotp + kDotBlocks, sh);
    const double rr = sum_partials(dotp + 2 * kDotBlocks, sh);
    if (threadIdx.x == 0) {
        const double rho = resume ? *rho_in : dz;
        sc->rho[0] = rho;
        sc->rho[1] = rho;
        sc->dnorm2 = dn2;
        sc->tol2 = rtol * rtol * dn2;
        sc->delta = 0.0; sc->a = 0.0; sc->b = 0.0;
        sc->rr = rr;
        sc->done[0] = (rtol > 0.0 && rr <= sc->tol2) ? 1 : 0;
        sc->done[1] = 0;
        sc->iters_done = 0;
        if (hist) hist[0] = sqrt(rr);
    }
}

// stored-G mode: q arrives without the lambda term; add it in place and form the p.q partials.
__global__ void __launch_bounds__(kDotThreads) dot_pq_kernel(long long N, const double* __restrict__ p, double lam,
                                                              double* q, double* __restrict__ dotp,
                                                              const int* __restrict__ done) {
    if (*done) {      // frozen: keep the exchanged partials finite (a sharded run all-reduces them every iteration)
        if (threadIdx.x == 0) dotp[blockIdx.x] = 0.0;
        return;
    }
    __shared__ double sh[kDotThreads];
    double loc = 0.0;
    for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < N; i += (long long)gridDim.x * kDotThreads) {
        const double pi = p[i];
        const double val = fma(lam, pi, q[i]);
        q[i] = val;
        loc = fma(pi, val, loc);
    }
    const double s = block_sum(loc, sh);
    if (threadIdx.x == 0) dotp[blockIdx.x] = s;
}

// minv != NULL: z (its own buffer) = r / (minv + lam); minv == NULL: z is r.  dotp_out: [r.z | r.r] partials.
__global__ void __launch_bounds__(kDotThreads) cg_update_xr_kernel(long long N, double* __restrict__ x, double* r,
                                                                    const double* __restrict__ p,
                                                                    const double* __restrict__ q,
                                                                    const double* __restrict__ minv, double lam,
                                                                    double* z, const double* __restrict__ dotp_in,
                                                                    double* __restrict__ dotp_out, CgScalars* sc,
                                                                    int it) {
    if (sc->done[it & 1]) {
        if (threadIdx.x == 0) { dotp_out[blockIdx.x] = 0.0; dotp_out[kDotBlocks + blockIdx.x] = 0.0; }
        return;
    }
    __shared__ double sh[kDotThreads];
    const double delta = sum_partials(dotp_in, sh);
    const double a = sc->rho[it & 1] / delta;
    double loc = 0.0, locz = 0.0;
    for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < N; i += (long long)gridDim.x * kDotThreads) {
        x[i] = fma(a, p[i], x[i]);
        const double ri = fma(-a, q[i], r[i]);
        r[i] = ri;
        loc = fma(ri, ri, loc);
        if (minv) {
            const double zi = ri / (minv[i] + lam);
            z[i] = zi;
            locz = fma(ri, zi, locz);
        }
    }
    const double s = block_sum(loc, sh);
    const double sz = minv ? block_sum(locz, sh) : s;
    if (threadIdx.x == 0) {
        dotp_out[blockIdx.x] = sz;
        dotp_out[kDotBlocks + blockIdx.x] = s;
        if (blockIdx.x == 0) { sc->delta = delta; sc->a = a; }
    }
}

// `it` is the iteration index of this call (a kernel argument).  rho and the frozen flag are double-buffered by its
// parity: iteration it reads slot it & 1 and block 0 writes slot (it + 1) & 1, so no kernel reads a scalar that another
// block of the same launch writes, and no separate "advance" launch is needed.
__global__ void __launch_bounds__(kDotThreads) cg_update_p_kernel(long long N, const double* z, double* p,
                                                                   const double* __restrict__ dotp, CgScalars* sc,
                                                                   double* __restrict__ hist, double* __restrict__ ab,
                                                                   int it) {
    __shared__ double sh[kDotThreads];
    double* hist_slot = hist ? hist + it + 1 : nullptr;
    double* ab_slot = ab ? ab + 2 * it : nullptr;
    if (sc->done[it & 1]) {   // frozen: carry rho and the flag forward so that the parity bookkeeping stays valid
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            sc->rho[(it + 1) & 1] = sc->rho[it & 1];
            sc->done[(it + 1) & 1] = 1;
            if (hist_slot) *hist_slot = hist_slot[-1];
            if (ab_slot) { ab_slot[0] = 0.0; ab_slot[1] = 0.0; }
        }
        return;
    }
    const double rho_new = sum_partials(dotp, sh);
    const double rr = sum_partials(dotp + kDotBlocks, sh);
    const double b = rho_new / sc->rho[it & 1];
    for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < N; i += (long long)gridDim.x * kDotThreads)
        p[i] = fma(b, p[i], z[i]);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        sc->rho[(it + 1) & 1] = rho_new;
        sc->b = b;
        sc->rr = rr;
        if (hist_slot) *hist_slot = sqrt(rr);
        if (ab_slot) { ab_slot[0] = sc->a; ab_slot[1] = b; }
        sc->iters_done = it + 1;
        sc->done[(it + 1) & 1] = (sc->tol2 > 0.0 && rr <= sc->tol2) ? 1 : 0;
    }
}

cudaError_t launch_cg_init(grav_ctx* c, const double* dobs, const double* minv, double lam, double* x, double* r,
                           double* z, double* p, double* dotp, int resume, cudaStream_t s) {
    cg_init_kernel<<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, dobs, minv, lam, x, r, z, p, dotp, resume);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_cg_init_finish(grav_ctx* c, const double* dotp, CgScalars* sc, double rtol, int resume,
                                  const double* rho_in, double* hist, cudaStream_t s) {
    cg_init_finish_kernel<<<1, kDotThreads, 0, s>>>(dotp, sc, rtol, resume, rho_in, hist);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_dot_pq(grav_ctx* c, const double* p, double lam, double* q, double* dotp, const CgScalars* sc,
                          int it, cudaStream_t s) {
    dot_pq_kernel<<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, p, lam, q, dotp, &sc->done[it & 1]);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_cg_update_xr(grav_ctx* c, double* x, double* r, const double* p, const double* q,
                                const double* minv, double lam, double* z, const double* dotp_in, double* dotp_out,
                                CgScalars* sc, int it, cudaStream_t s) {
    cg_update_xr_kernel<<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, x, r, p, q, minv, lam, z, dotp_in, dotp_out, sc, it);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_cg_update_p(grav_ctx* c, const double* z, double* p, const double* dotp, CgScalars* sc, double* hist,
                               double* ab, int it, cudaStream_t s) {
    cg_update_p_kernel<<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, z, p, dotp, sc, hist, ab, it);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace grav
