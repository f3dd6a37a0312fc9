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


// Staged variant (the default): the (c_n, zn[c]) stream of the block's column chunk is copied to shared memory in
// column-aligned tiles of <= kFwdStage nodes with cp.async, double-buffered, so the z-loop reads it with a
// broadcast LDS.128 (short, fixed latency) instead of an LDG that exposes the L2 latency to 4 warps per scheduler
// (ncu: 0.95 warps per issue stalled on long_scoreboard before, profiles/r1_ncu_full_cfg3.md).
constexpr int kFwdStage = 1024;   // nodes per buffer (16 KB); columns deeper than this use the unstaged kernel

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

template <int TPB, int UNROLL, int MINB, int EV>
__global__ void __launch_bounds__(TPB, MINB) forward_nodes_staged_kernel(Geom g, PsiDev pd, Psi2Dev pd2,
                                                                               const double2* __restrict__ cnode,
                                                                               double* __restrict__ partial,
                                                                               int cols_per_chunk,
                                                                               const int* __restrict__ done) {
    extern __shared__ double2 s_tab[];
    if (done && *done) return;
    PsiTabView tb;
    Psi2TabView tb2;
    double2* s_stage;
    if (EV == 1) { tb = psi_tables_to_smem(s_tab, pd); s_stage = s_tab + kTabEntries * kRep; }
    else if (EV == 3) { tb2 = psi2_tables_to_smem_2d(s_tab, pd2); s_stage = s_tab + psi2_log2d_smem_entries(pd2); }
    else { tb2 = psi2_tables_to_smem(s_tab, pd2); s_stage = s_tab + kTab2Entries * kRep; }
    const long long i = (long long)blockIdx.x * TPB + threadIdx.x;
    const long long il = i < g.N ? i : g.N - 1;
    const double xo = g.xo[il], yo = g.yo[il], zo = g.zo[il];
    const int col0 = blockIdx.y * cols_per_chunk;
    const int col1 = min(col0 + cols_per_chunk, g.ncol);
    const int cpt = kFwdStage / g.nzp;                       // whole columns per tile (>= 1, checked by the launcher)
    const int ntile = (col1 - col0 + cpt - 1) / cpt;
    auto prefetch = [&](int t) {
        const int c0 = col0 + t * cpt;
        const int nn = (min(c0 + cpt, col1) - c0) * g.nzp;
        const double2* src = cnode + (long long)c0 * g.nzp;
        double2* dst = s_stage + (t & 1) * kFwdStage;
        for (int e = threadIdx.x; e < nn; e += TPB) cp_async16(dst + e, src + e);
        cp_async_commit();
    };
    double acc = 0.0;
    int a = col0 / g.nyp, b = col0 - a * g.nyp;
    double X = __ldg(g.xn + a) - xo;
    if (ntile > 0) prefetch(0);
    for (int t = 0; t < ntile; ++t) {
        if (t + 1 < ntile) { prefetch(t + 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        __syncthreads();
        const int tc0 = col0 + t * cpt;
        const int tc1 = min(tc0 + cpt, col1);
        const double2* sc = s_stage + (t & 1) * kFwdStage;
        for (int col = tc0; col < tc1; ++col, sc += g.nzp) {
            const double Y = __ldg(g.yn + b) - yo;
            const PsiColumn pc = psi_column(X, Y);
            double colacc = 0.0;
#pragma unroll UNROLL
            for (int c = 0; c < g.nzp; ++c) {
                const double2 cz = sc[c];
                const double Z = cz.y - zo;
                colacc = fma(cz.x, EV == 1 ? psi_fast(tb, pc, Z)
                                           : (EV == 3 ? psi2_fast_t<true>(tb2, pc, Z) : psi2_fast(tb2, pc, Z)), colacc);
            }
            acc = fma(colacc, pc.s, acc);
            if (++b == g.nyp) {
                b = 0;
                ++a;
                if (a < g.nxp) X = __ldg(g.xn + a) - xo;
            }
        }
        __syncthreads();      // everyone is done with buffer t&1 before tile t+2 is copied into it
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
    constexpr size_t smem = EV == 2 ? kTab2SmemBytes : kTabSmemBytes;
    static unsigned long long smem_set = 0;
    {
        cudaError_t e = ensure_dynamic_smem(forward_nodes_kernel<TPB, UNROLL, MINB, EV>, smem, c->device, &smem_set);
        if (e != cudaSuccess) return e;
    }
    const Plan& p = c->plan;
    dim3 grid((unsigned)((c->g.N + TPB - 1) / TPB), p.fwd_nchunk);
    forward_nodes_kernel<TPB, UNROLL, MINB, EV><<<grid, TPB, smem, s>>>(c->g, c->pd, c->pd2, cnode, partial,
                                                                        p.fwd_cols_per_chunk, done);
    return cudaGetLastError();
}

template <int TPB, int UNROLL, int MINB, int EV = 2>
static cudaError_t fwd_launch_staged(grav_ctx* c, const double2* cnode, double* partial, const int* done, cudaStream_t s) {
    if (c->g.nzp > kFwdStage) return fwd_launch_fast<TPB, UNROLL, MINB, EV == 3 ? 2 : EV>(c, cnode, partial, done, s);
    if (EV == 3 && !c->pd2.tab2d) return cudaErrorInvalidValue;      // geometry outside the 2-D log table
    constexpr size_t stage = 2 * kFwdStage * sizeof(double2);
    // EV == 3: the opt-in is sized for the largest 2-D table, the launch for this context's table
    constexpr size_t smem_max = EV == 3 ? kAtan2SmemBytes + (size_t)kLog2dMaxBinades * 4096 + stage
                                        : (EV == 2 ? kTab2SmemBytes : kTabSmemBytes) + stage;
    const size_t smem = EV == 3 ? kAtan2SmemBytes + (size_t)c->pd2.nb2d * 4096 + stage : smem_max;
    static unsigned long long smem_set = 0;
    {
        cudaError_t e = ensure_dynamic_smem(forward_nodes_staged_kernel<TPB, UNROLL, MINB, EV>, smem_max, c->device, &smem_set);
        if (e != cudaSuccess) return e;
    }
    const Plan& p = c->plan;
    dim3 grid((unsigned)((c->g.N + TPB - 1) / TPB), p.fwd_nchunk);
    forward_nodes_staged_kernel<TPB, UNROLL, MINB, EV><<<grid, TPB, smem, s>>>(c->g, c->pd, c->pd2, cnode, partial,
                                                                               p.fwd_cols_per_chunk, done);
    return cudaGetLastError();
}

cudaError_t init_forward_kernels() { return cudaSuccess; }

cudaError_t launch_forward_nodes(grav_ctx* c, const double* cnode_, double* partial, const int* done, cudaStream_t s) {
    const Plan& p = c->plan;
    const double2* cnode = reinterpret_cast<const double2*>(cnode_);
    cudaError_t e;
    if (c->psi_variant == 0) {
        switch (c->tune[0]) {   // A/B variants measured in profiles/r1_tail_and_variants.md
            default:
            case 0:   // shipped: 2-D log table when the geometry admits it (grav_api.cu), else the 256-entry table
                if (p.log2d) e = fwd_launch_staged<512, 12, 1, 3>(c, cnode, partial, done, s);
                else e = fwd_launch_staged<256, 8, 2>(c, cnode, partial, done, s);
                break;
            case 8: e = fwd_launch_staged<256, 8, 2>(c, cnode, partial, done, s); break;
            case 1: e = fwd_launch_staged<256, 4, 2>(c, cnode, partial, done, s); break;
            case 2: e = fwd_launch_fast<256, 4, 2, 2>(c, cnode, partial, done, s); break;     // psi2, unstaged
            case 3: e = fwd_launch_fast<256, 8, 2, 2>(c, cnode, partial, done, s); break;
            case 4: e = fwd_launch_fast<128, 2, 4, 1>(c, cnode, partial, done, s); break;     // first generation
            case 5: e = fwd_launch_staged<512, 8, 1>(c, cnode, partial, done, s); break;
            case 6: e = fwd_launch_staged<512, 8, 1, 3>(c, cnode, partial, done, s); break;     // 2-D log table
            case 7: e = fwd_launch_staged<512, 4, 1, 3>(c, cnode, partial, done, s); break;
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
