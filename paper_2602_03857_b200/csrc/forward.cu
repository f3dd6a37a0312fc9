// forward.cu -- matrix-free d = G u in node-shared form (BASELINE.json north_star kernel 1).
//
//   d_i = gamma * sum_n c_n Psi(node_n - obs_i),   c = S^T u  (nodeops.cu)          PAPER.md:49-74, Eq. 1-6
//
// Tiling: one thread owns one station (coordinates and accumulator in registers); a block owns a tile of
// stations and a chunk of node columns; the node coefficients c_n of the chunk are read by every thread at the
// same address (broadcast).  X, Y, |XY| and X^2+Y^2 are constant down a node column and hoisted out of the
// z-loop.  Chunk partial sums go to partial[chunk][N]; forward_reduce adds them in fixed order (deterministic).
// Bound: FP64 pipe: ~49 FP64 instructions per evaluation, 8 bytes of c_n per warp.
#include "grav_internal.cuh"
#include "psi.cuh"
#include "psi2.cuh"

namespace grav {

// EV: 0 = CUDA libm (cross-check), 1 = psi_fast (psi.cuh), 2 = psi2_fast (psi2.cuh, the default)
template <int TPB, int UNROLL, int MINB, int EV>
__global__ void __launch_bounds__(TPB, MINB) forward_nodes_kernel(Geom g, PsiDev pd, Psi2Dev pd2,
                                                                        const double2* __restrict__ cnode,
                                                                        double* __restrict__ partial, int cols_per_chunk,
                                                                        const int* __restrict__ done) {
    extern __shared__ double2 s_tab[];
    if (done && *done) return;
    PsiTabView tb;
    Psi2TabView tb2;
    if (EV == 1) tb = psi_tables_to_smem(s_tab, pd);
    if (EV == 2) tb2 = psi2_tables_to_smem(s_tab, pd2);
    const long long i = (long long)blockIdx.x * TPB + threadIdx.x;
    const long long il = i < g.N ? i : g.N - 1;
    const double xo = g.xo[il], yo = g.yo[il], zo = g.zo[il];
    const int col0 = blockIdx.y * cols_per_chunk;
    const int col1 = min(col0 + cols_per_chunk, g.ncol);
    double acc = 0.0;
    int a = col0 / g.nyp, b = col0 - a * g.nyp;
    double X = __ldg(g.xn + a) - xo;
    for (int col = col0; col < col1; ++col) {
        const double Y = __ldg(g.yn + b) - yo;
        const double2* __restrict__ cc = cnode + (long long)col * g.nzp;   // (c_n, zn[c]) pairs: one LDG.128
        double colacc = 0.0;
        if (EV != 0) {
            const PsiColumn pc = psi_column(X, Y);
#pragma unroll UNROLL
            for (int c = 0; c < g.nzp; ++c) {
                const double2 cz = __ldg(cc + c);
                const double Z = cz.y - zo;
                const double coef = cz.x;
                colacc = fma(coef, EV == 1 ? psi_fast(tb, pc, Z) : psi2_fast(tb2, pc, Z), colacc);
            }
            colacc *= pc.s;
        } else {
            const double XY = X * Y;
            const double Q = fma(Y, Y, X * X);
            for (int c = 0; c < g.nzp; ++c) {
                const double2 cz = __ldg(cc + c);
                const double Z = cz.y - zo;
                const double coef = cz.x;
                colacc = fma(coef, psi_libm(X, Y, Z, XY, Q), colacc);
            }
        }
        acc += colacc;
        if (++b == g.nyp) {
            b = 0;
            ++a;
            if (a < g.nxp) X = __ldg(g.xn + a) - xo;
        }
    }
    if (i < g.N) partial[(long long)blockIdx.y * g.N + i] = acc;
}

// d = scale * sum_chunks partial (+ lam * p).  With dotp != NULL also writes block partials of p . d (CG: delta).
__global__ void __launch_bounds__(kDotThreads) forward_reduce_kernel(long long N, int nchunk,
                                                                      const double* __restrict__ partial, double scale,
                                                                      double lam, const double* __restrict__ p,
                                                                      double* __restrict__ d, double* __restrict__ dotp,
                                                                      const int* __restrict__ done) {
    if (done && *done) return;
    __shared__ double sh[kDotThreads];
    double loc = 0.0;
    for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < N; i += (long long)gridDim.x * kDotThreads) {
        double s = 0.0;
        for (int ch = 0; ch < nchunk; ++ch) s += partial[(long long)ch * N + i];
        double val = scale * s;
        if (p) {
            double pi = p[i];
            val = fma(lam, pi, val);
            loc = fma(pi, val, loc);
        }
        d[i] = val;
    }
    if (dotp) {
        sh[threadIdx.x] = loc;
        __syncthreads();
        for (int s = kDotThreads / 2; s > 0; s >>= 1) {
            if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
            __syncthreads();
        }
        if (threadIdx.x == 0) dotp[blockIdx.x] = sh[0];
    }
}

// Launch variants (grav_debug_set_tuning(ctx, 0, v)); the default is the one measured fastest (profiles/).
template <int TPB, int UNROLL, int MINB, int EV = 1>
static cudaError_t fwd_launch_fast(grav_ctx* c, const double2* cnode, double* partial, const int* done, cudaStream_t s) {
    static bool inited = false;
    constexpr size_t smem = EV == 2 ? kTab2SmemBytes : kTabSmemBytes;
    if (!inited) {
        cudaError_t e = cudaFuncSetAttribute(forward_nodes_kernel<TPB, UNROLL, MINB, EV>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        inited = true;
    }
    const Plan& p = c->plan;
    dim3 grid((unsigned)((c->g.N + TPB - 1) / TPB), p.fwd_nchunk);
    forward_nodes_kernel<TPB, UNROLL, MINB, EV><<<grid, TPB, smem, s>>>(c->g, c->pd, c->pd2, cnode, partial,
                                                                        p.fwd_cols_per_chunk, done);
    return cudaGetLastError();
}

cudaError_t init_forward_kernels() { return cudaSuccess; }

cudaError_t launch_forward_nodes(grav_ctx* c, const double* cnode_, double* partial, const int* done, cudaStream_t s) {
    const Plan& p = c->plan;
    const double2* cnode = reinterpret_cast<const double2*>(cnode_);
    cudaError_t e;
    if (c->psi_variant == 0) {
        switch (c->tune[0]) {
            default:
            case 0: e = fwd_launch_fast<256, 4, 2, 2>(c, cnode, partial, done, s); break;
            case 12: e = fwd_launch_fast<128, 2, 4>(c, cnode, partial, done, s); break;
            case 1: e = fwd_launch_fast<256, 1, 3>(c, cnode, partial, done, s); break;
            case 2: e = fwd_launch_fast<256, 2, 2>(c, cnode, partial, done, s); break;
            case 3: e = fwd_launch_fast<128, 1, 4>(c, cnode, partial, done, s); break;
            case 4: e = fwd_launch_fast<256, 1, 4>(c, cnode, partial, done, s); break;
            case 5: e = fwd_launch_fast<256, 4, 2>(c, cnode, partial, done, s); break;
            case 6: e = fwd_launch_fast<512, 2, 1>(c, cnode, partial, done, s); break;
            case 7: e = fwd_launch_fast<128, 4, 3>(c, cnode, partial, done, s); break;
            case 8: e = fwd_launch_fast<128, 4, 2>(c, cnode, partial, done, s); break;
            case 9: e = fwd_launch_fast<128, 3, 3>(c, cnode, partial, done, s); break;
            case 10: e = fwd_launch_fast<128, 2, 3>(c, cnode, partial, done, s); break;
            case 11: e = fwd_launch_fast<128, 8, 2>(c, cnode, partial, done, s); break;
            case 20: e = fwd_launch_fast<256, 2, 2, 2>(c, cnode, partial, done, s); break;
            case 22: e = fwd_launch_fast<128, 2, 3, 2>(c, cnode, partial, done, s); break;
            case 23: e = fwd_launch_fast<128, 4, 3, 2>(c, cnode, partial, done, s); break;
            case 24: e = fwd_launch_fast<256, 1, 3, 2>(c, cnode, partial, done, s); break;
            case 25: e = fwd_launch_fast<512, 2, 1, 2>(c, cnode, partial, done, s); break;
            case 26: e = fwd_launch_fast<256, 3, 2, 2>(c, cnode, partial, done, s); break;
        }
    } else {
        dim3 grid((unsigned)((c->g.N + 127) / 128), p.fwd_nchunk);
        forward_nodes_kernel<128, 1, 4, 0><<<grid, 128, 0, s>>>(c->g, c->pd, c->pd2, cnode, partial, p.fwd_cols_per_chunk, done);
        e = cudaGetLastError();
    }
    c->launches++;
    return e;
}

cudaError_t launch_forward_reduce(grav_ctx* c, const double* partial, double scale, double lam, const double* p,
                                  double* d, double* dot_partial, const CgScalars* sc, cudaStream_t s) {
    const int* done = sc ? &sc->done : nullptr;
    forward_reduce_kernel<<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, c->plan.fwd_nchunk, partial, scale, lam, p, d,
                                                             dot_partial, done);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace grav
