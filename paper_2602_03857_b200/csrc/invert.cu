// invert.cu -- the paper's outer model-update loop around the data-space CG.
//
//   PAPER.md:101-114 (Eq. 10-11): delta_m = W_m G^T (G W_m G^T + W_d)^-1 delta_d,  delta_d = d_obs - G m_ref
//   <= 30 outer model updates, <= 20 inner CG iterations each, both stopped at res <= 1e-4
//   "outer Gauss-Newton-style update loop with step-size backtracking"
//
// The paper prints neither the residual norm nor the backtracking rule; DESIGN.md 2 (readings R1-R4) fixes them:
//   m_0 = m_ref; r_k = d_obs - G m_k; stop when ||r_k||_2 / ||d_obs||_2 <= tol_outer;
//   alpha_k = CG on (G W^-2 G^T + lambda I) alpha = r_k, <= max_inner iterations, stopped at ||.|| <= tol_inner ||r_k||;
//   delta_m = W^-2 G^T alpha_k;  s = 1, halved (<= 10 times) until ||r_k - s G delta_m|| < ||r_k||;
//   m_{k+1} = m_k + s delta_m.   G is linear, so backtracking costs no operator application: G delta_m is formed once.
// Every norm is a fixed-order two-stage reduction; the host reads one scalar per trial step (the only
// synchronisation: an outer iteration is 2 * max_inner + 2 operator applications, seconds at config 5).
#include "grav_internal.cuh"

namespace grav {

// out = r - s * dd (dd == NULL: out = r); partial[block] = sum of out^2 over the block's elements
__global__ void __launch_bounds__(kDotThreads) inv_residual_kernel(long long N, const double* __restrict__ r, double s,
                                                                    const double* __restrict__ dd,
                                                                    double* __restrict__ out,
                                                                    double* __restrict__ partial) {
    __shared__ double sh[kDotThreads];
    double loc = 0.0;
    for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < N; i += (long long)gridDim.x * kDotThreads) {
        const double v = dd ? fma(-s, dd[i], r[i]) : r[i];
        if (out) out[i] = v;
        loc = fma(v, v, loc);
    }
    sh[threadIdx.x] = loc;
    __syncthreads();
    for (int k = kDotThreads / 2; k > 0; k >>= 1) {
        if (threadIdx.x < k) sh[threadIdx.x] += sh[threadIdx.x + k];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

__global__ void __launch_bounds__(kDotBlocks) inv_finish_kernel(const double* __restrict__ partial,
                                                                 double* __restrict__ scalar) {
    __shared__ double sh[kDotBlocks];
    sh[threadIdx.x] = partial[threadIdx.x];
    __syncthreads();
    for (int k = kDotBlocks / 2; k > 0; k >>= 1) {
        if (threadIdx.x < k) sh[threadIdx.x] += sh[threadIdx.x + k];
        __syncthreads();
    }
    if (threadIdx.x == 0) *scalar = sh[0];
}

// y += a * x   (elementwise, M-vectors, in place)
__global__ void inv_axpy_kernel(long long M, double a, const double* __restrict__ x, double* __restrict__ y) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) y[i] = fma(a, x[i], y[i]);
}

cudaError_t launch_inv_residual(grav_ctx* c, const double* r, double s, const double* dd, double* out, double* partial,
                                cudaStream_t st) {
    inv_residual_kernel<<<kDotBlocks, kDotThreads, 0, st>>>(c->g.N, r, s, dd, out, partial);
    c->launches++;
    return cudaGetLastError();
}
cudaError_t launch_inv_finish(grav_ctx* c, const double* partial, double* scalar, cudaStream_t st) {
    inv_finish_kernel<<<1, kDotBlocks, 0, st>>>(partial, scalar);
    c->launches++;
    return cudaGetLastError();
}
cudaError_t launch_inv_axpy(grav_ctx* c, double a, const double* x, double* y, cudaStream_t st) {
    inv_axpy_kernel<<<(unsigned)((c->g.M + 255) / 256), 256, 0, st>>>(c->g.M, a, x, y);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace grav
