// forward.cu -- matrix-free d = G u in node-shared form (BASELINE.json north_star kernel 1).
//
//   d_i = gamma * sum_n c_n Psi(node_n - obs_i),   c = S^T u  (nodeops.cu)          PAPER.md:49-74, Eq. 1-6
//
// Tiling: one thread owns one station (coordinates and accumulator in registers); a block owns a tile of
// stations and a chunk of node columns; the node coefficients c_n of the chunk are read by every thread at the
// same address (broadcast).  X, Y, |XY| and X^2+Y^2 are constant down a node column and hoisted out of the
// z-loop.  Chunk partial sums go to partial[chunk][N]; forward_reduce adds them in fixed order (deterministic).
// Bound: FP64 pipe: 43 FP64 instructions per evaluation, 16 bytes of (c_n, z_n) per warp.
#include "grav_internal.cuh"
#include "psi.cuh"

namespace grav {

// Unstaged kernel: the (c_n, z_n) stream is read with LDG.  EVAL 0: psi_eval with the 256-entry log table (fallback for
// node columns deeper than the stage buffer of the staged kernel below); 1: CUDA libm in FP64 (cross-check); 2: the
// Float32 evaluator psi_f32 with FP64 accumulation (grav_set_precision).
template <int TPB, int UNROLL, int MINB, int EVAL>
__global__ void __launch_bounds__(TPB, MINB) forward_nodes_kernel(Geom g, PsiDev pd, const double2* __restrict__ cnode,
                                                                  double* __restrict__ partial, int cols_per_chunk,
                                                                  const int* __restrict__ done) {
    extern __shared__ double2 s_tab[];
    __shared__ float s_at[kAtanN32];
    if (done && *done) return;
    PsiTabView tb;
    if (EVAL == 0) tb = psi_tables_to_smem(s_tab, pd);
    if (EVAL == 2) psi_f32_atan_table(s_at, pd);
    const long long i = (long long)blockIdx.x * TPB + threadIdx.x;
    const long long il = i < g.N ? i : g.N - 1;
    const double xo = g.xo[il], yo = g.yo[il], zo = g.zo[il];
    const int col0 = blockIdx.y * cols_per_chunk;
    const int col1 = min(col0 + cols_per_chunk, g.ncol);
    const float inv_scale = psi_f32_inv_scale(pd.k0);
    double acc = 0.0;
    int a = col0 / g.nyp, b = col0 - a * g.nyp;
    double X = __ldg(g.xn + a) - xo;
    for (int col = col0; col < col1; ++col) {
        const double Y = __ldg(g.yn + b) - yo;
        const double2* __restrict__ cc = cnode + (long long)col * g.nzp;   // (c_n, zn[c]) pairs: one LDG.128
        double colacc = 0.0;
        if (EVAL == 0) {
            const PsiColumn pc = psi_column(X, Y);
#pragma unroll UNROLL
            for (int c = 0; c < g.nzp; ++c) {
                const double2 cz = __ldg(cc + c);
                colacc = fma(cz.x, psi_eval<false>(tb, pc, cz.y - zo), colacc);
            }
            colacc *= pc.s;
        } else if (EVAL == 1) {
            const double XY = X * Y;
            const double Q = fma(Y, Y, X * X);
            for (int c = 0; c < g.nzp; ++c) {
                const double2 cz = __ldg(cc + c);
                colacc = fma(cz.x, psi_libm(X, Y, cz.y - zo, XY, Q), colacc);
            }
        } else {
            const float Xf = (float)X, Yf = (float)Y;
#pragma unroll UNROLL
            for (int c = 0; c < g.nzp; ++c) {
                const double2 cz = __ldg(cc + c);
                colacc = fma(cz.x, (double)psi_f32(Xf, Yf, (float)(cz.y - zo), inv_scale, s_at), colacc);
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

// Staged kernel (the default): the (c_n, zn[c]) stream of the block's column chunk is copied to shared memory in
// column-aligned tiles of <= kFwdStage nodes with cp.async, double-buffered, so the z-loop reads it with a
// broadcast LDS.128 (short, fixed latency) instead of an LDG that exposes the L2 latency to 4 warps per scheduler
// (ncu: 0.95 warps per issue stalled on long_scoreboard before).
constexpr int kFwdStage = 1024;   // nodes per buffer (16 KB); columns deeper than this use the unstaged kernel

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// work != NULL: persistent launch for small problems - a block copies the Psi tables (up to 140 KB) ONCE and then draws
// (station tile, column chunk) items from the counter *work until none is left, instead of one block per item; which
// block computes an item does not change what is written, so the result stays deterministic.
// PERSIST: compiled with the item loop (else one item per block, from blockIdx); TAIL 1: column remainders in groups of 4
// after the UNROLL-wide groups, 0: a plain unrolled loop.
template <int TPB, int UNROLL, int MINB, bool LOG2D, bool PERSIST, int TAIL>
__global__ void __launch_bounds__(TPB, MINB) forward_nodes_staged_kernel(Geom g, PsiDev pd,
                                                                         const double2* __restrict__ cnode,
                                                                         double* __restrict__ partial,
                                                                         int cols_per_chunk,
                                                                         const int* __restrict__ done,
                                                                         int* __restrict__ work, int ntiles,
                                                                         int nitems) {
    extern __shared__ double2 s_tab[];
    __shared__ int s_item;
    if (done && *done) return;
    const PsiTabView tb = psi_tables_load<LOG2D>(s_tab, pd);
    double2* s_stage = s_tab + (LOG2D ? psi_log2d_smem_entries(pd) : (size_t)kTabEntries * kRep);
    const int cpt = kFwdStage / g.nzp;                       // whole columns per tile (>= 1, checked by the launcher)
    for (;;) {
        int bx = blockIdx.x, by = blockIdx.y;
        if (PERSIST && work) {
            __syncthreads();                                 // the previous item's s_item and stage buffers are done with
            if (threadIdx.x == 0) s_item = atomicAdd(work, 1);
            __syncthreads();
            const int item = s_item;
            if (item >= nitems) break;
            by = item / ntiles;                              // tile index fastest: neighbours in time share a chunk's stream
            bx = item - by * ntiles;
        }
        const long long i = (long long)bx * TPB + threadIdx.x;
        const long long il = i < g.N ? i : g.N - 1;
        const double xo = g.xo[il], yo = g.yo[il], zo = g.zo[il];
        const int col0 = by * cols_per_chunk;
        const int col1 = min(col0 + cols_per_chunk, g.ncol);
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
                // UNROLL independent evaluations in flight; the column's remainder in groups of 4 and then singly (a
                // plain `#pragma unroll UNROLL` leaves up to UNROLL - 1 nodes per column - 9 of 33 at config 2 - to a
                // one-at-a-time loop)
                int c = 0;
                if (TAIL == 0) {
#pragma unroll UNROLL
                    for (; c < g.nzp; ++c) {
                        const double2 cz = sc[c];
                        colacc = fma(cz.x, psi_eval<LOG2D>(tb, pc, cz.y - zo), colacc);
                    }
                }
                for (; c + UNROLL <= g.nzp; c += UNROLL) {
#pragma unroll
                    for (int u = 0; u < UNROLL; ++u) {
                        const double2 cz = sc[c + u];
                        colacc = fma(cz.x, psi_eval<LOG2D>(tb, pc, cz.y - zo), colacc);
                    }
                }
                for (; c + 4 <= g.nzp; c += 4) {
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const double2 cz = sc[c + u];
                        colacc = fma(cz.x, psi_eval<LOG2D>(tb, pc, cz.y - zo), colacc);
                    }
                }
#pragma unroll 1
                for (; c < g.nzp; ++c) {
                    const double2 cz = sc[c];
                    colacc = fma(cz.x, psi_eval<LOG2D>(tb, pc, cz.y - zo), colacc);
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
        if (i < g.N) partial[(long long)by * g.N + i] = acc;
        if (!PERSIST || !work) break;
    }
}

// d = scale * sum_chunks partial (+ lam * p).  With dotp != NULL also writes kDotBlocks block partials of p . d (CG:
// delta).  A block is kRedX stations x kRedY chunk lanes: lane y adds chunks y, y + kRedY, ... in increasing order and
// the kRedY lane sums are added in a fixed tree, so the result does not depend on the launch; blocks stride over the
// station tiles.
// RX = 32 stations per block (8 chunk lanes) for the large problems, 8 stations x 32 lanes where the stations are few and
// the chunks many (config 1: 256 stations, 289 one-column chunks) - a property of the context, fixed at its creation.
template <int RX>
__global__ void __launch_bounds__(kDotThreads) forward_reduce_kernel(long long N, int nchunk,
                                                                      const double* __restrict__ partial, double scale,
                                                                      double lam, const double* __restrict__ p,
                                                                      double* __restrict__ d, double* __restrict__ dotp,
                                                                      const int* __restrict__ done) {
    constexpr int RY = kDotThreads / RX;
    if (done && *done) {      // frozen CG: keep the exchanged partials finite
        if (dotp && threadIdx.x == 0) dotp[blockIdx.x] = 0.0;
        return;
    }
    __shared__ double sh[RY][RX + 1];
    __shared__ double shd[RX];
    const int tx = threadIdx.x & (RX - 1), ty = threadIdx.x / RX;
    double loc = 0.0;        // dot partial of the stations this thread finishes (ty == 0 only)
    for (long long i0 = (long long)blockIdx.x * RX; i0 < N; i0 += (long long)gridDim.x * RX) {
        const long long i = i0 + tx;
        double s = 0.0;
        if (i < N) {
#pragma unroll 4
            for (int ch = ty; ch < nchunk; ch += RY) s += partial[(long long)ch * N + i];
        }
        sh[ty][tx] = s;
        __syncthreads();
#pragma unroll
        for (int h = RY / 2; h > 0; h >>= 1) {
            if (ty < h) sh[ty][tx] += sh[ty + h][tx];
            __syncthreads();
        }
        if (ty == 0 && i < N) {
            double val = scale * sh[0][tx];
            if (p) {
                const double pi = p[i];
                val = fma(lam, pi, val);
                loc = fma(pi, val, loc);
            }
            d[i] = val;
        }
        __syncthreads();
    }
    if (dotp) {
        if (ty == 0) shd[tx] = loc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
#pragma unroll
            for (int k = 0; k < RX; ++k) t += shd[k];
            dotp[blockIdx.x] = t;
        }
    }
}

template <int TPB, int UNROLL, int MINB, int EVAL>
static cudaError_t fwd_launch_unstaged(grav_ctx* c, const double2* cnode, double* partial, const int* done,
                                       cudaStream_t s) {
    constexpr size_t smem = EVAL == 0 ? kTabSmemBytes : 0;
    static unsigned long long smem_set = 0;
    if (smem > 48 * 1024) {
        cudaError_t e = ensure_dynamic_smem(forward_nodes_kernel<TPB, UNROLL, MINB, EVAL>, smem, c->device, &smem_set);
        if (e != cudaSuccess) return e;
    }
    dim3 grid((unsigned)((c->g.N + TPB - 1) / TPB), c->plan.fwd_nchunk);
    forward_nodes_kernel<TPB, UNROLL, MINB, EVAL><<<grid, TPB, smem, s>>>(c->g, c->pd, cnode, partial,
                                                                          c->plan.fwd_cols_per_chunk, done);
    return cudaGetLastError();
}

template <int TPB, int UNROLL, int MINB, bool LOG2D, bool PERSIST, int TAIL>
static cudaError_t fwd_launch_staged(grav_ctx* c, const double2* cnode, double* partial, const int* done, int* work,
                                     cudaStream_t s) {
    if (c->g.nzp > kFwdStage) return fwd_launch_unstaged<256, 8, 2, 0>(c, cnode, partial, done, s);
    constexpr size_t stage = 2 * kFwdStage * sizeof(double2);
    // the opt-in is sized for the largest 2-D table, the launch for this context's table
    const size_t smem = psi_smem_bytes<LOG2D>(c->pd) + stage;
    static unsigned long long smem_set = 0;
    {
        cudaError_t e = ensure_dynamic_smem(forward_nodes_staged_kernel<TPB, UNROLL, MINB, LOG2D, PERSIST, TAIL>,
                                            psi_smem_max<LOG2D>() + stage, c->device, &smem_set);
        if (e != cudaSuccess) return e;
    }
    const int ntiles = (int)((c->g.N + TPB - 1) / TPB);
    const long long nitems = (long long)ntiles * c->plan.fwd_nchunk;
    dim3 grid((unsigned)ntiles, c->plan.fwd_nchunk);
    if (PERSIST && c->plan.persistent && nitems < (1ll << 31)) {
        cudaError_t e = cudaMemsetAsync(work, 0, sizeof(int), s);
        if (e != cudaSuccess) return e;
        const long long resident = (long long)c->plan.sms * MINB;
        grid = dim3((unsigned)(nitems < resident ? nitems : resident), 1);
    } else {
        work = nullptr;
    }
    forward_nodes_staged_kernel<TPB, UNROLL, MINB, LOG2D, PERSIST, TAIL><<<grid, TPB, smem, s>>>(c->g, c->pd, cnode, partial,
                                                                                  c->plan.fwd_cols_per_chunk, done,
                                                                                  work, ntiles, (int)nitems);
    return cudaGetLastError();
}

cudaError_t launch_forward_nodes(grav_ctx* c, const double* cnode_, double* partial, const int* done, int* work,
                                 cudaStream_t s) {
    const double2* cnode = reinterpret_cast<const double2*>(cnode_);
    cudaError_t e;
    if (c->psi_variant == 1) e = fwd_launch_unstaged<128, 1, 4, 1>(c, cnode, partial, done, s);
    else if (c->psi_variant == 2) e = fwd_launch_unstaged<256, 8, 4, 2>(c, cnode, partial, done, s);
    // two instantiations of the 2-D-table kernel: the persistent one for small problems (column remainders in groups of
    // 4: +3 % at config 2), the plain grid with a plain unrolled z-loop for the rest (0.5 % faster at configs 3-5)
    else if (use_log2d(c) && c->plan.persistent) e = fwd_launch_staged<512, 12, 1, true, true, 1>(c, cnode, partial, done, work, s);
    else if (use_log2d(c)) e = fwd_launch_staged<512, 12, 1, true, false, 0>(c, cnode, partial, done, work, s);
    else e = fwd_launch_staged<256, 8, 2, false, false, 0>(c, cnode, partial, done, work, s);
    c->launches++;
    return e;
}

cudaError_t launch_forward_reduce(grav_ctx* c, const double* partial, double scale, double lam, const double* p,
                                  double* d, double* dot_partial, const int* done, cudaStream_t s) {
    if (c->plan.fwd_reduce_rx == 8)
        forward_reduce_kernel<8><<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, c->plan.fwd_nchunk, partial, scale, lam, p, d,
                                                                    dot_partial, done);
    else
        forward_reduce_kernel<32><<<kDotBlocks, kDotThreads, 0, s>>>(c->g.N, c->plan.fwd_nchunk, partial, scale, lam, p,
                                                                     d, dot_partial, done);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace grav
