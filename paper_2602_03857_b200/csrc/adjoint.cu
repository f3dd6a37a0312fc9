// adjoint.cu -- matrix-free g = G^T v in node-shared form (BASELINE.json north_star kernel 2).
//
//   T_n = sum_i v_i Psi(node_n - obs_i);   g_k = gamma * sum_pqr sigma T[corner_pqr(k)]   (nodeops.cu)
//
// Transposed tiling: one thread owns KC consecutive nodes of one node column (their z and accumulators live in
// registers); stations are staged through shared memory, kAdjObsStage per block-wide barrier, and read at the same
// address by every thread (broadcast).  X, Y, X*Y, X^2+Y^2 are computed once per (thread, station) and shared by the KC nodes.
// Every node is owned by exactly one thread: no atomics.
//
// Accumulation.  T_n is a sum of up to N same-sign terms of size |v Psi| ~ 1e4..1e5 m whose 8-corner signed
// difference (node_to_cell) is 1e6..1e7 times smaller, so a plain running sum over all stations loses the result
// (measured 7e-9 of max at config 5 with a smooth v).  The sum is therefore two-level: a plain FP64 running sum
// over one tile of kAdjObsTile stations, then an error-free TwoSum (Knuth) of the tile sum into a (hi, lo) pair
// kept in the output buffer (L2-resident; read-modify-written once per tile by the owning thread).  T is handed on
// as two planes [hi | lo] of Nn doubles each; station chunks give partial[chunk][2][Nn], combined in fixed order
// by adjoint_reduce with the same TwoSum.
#include "grav_internal.cuh"
#include "psi.cuh"

namespace grav {

constexpr int kAdjObsTile = 256;     // stations per plain running sum (accuracy: 1024 loses 1.1e-10 of max at config 3)
constexpr int kAdjObsStage = 1024;   // stations staged in shared memory per block-wide barrier

// EV: 0 = CUDA libm (cross-check), 1 = psi_eval with the 256-entry log table, 2 = psi_eval with the 2-D log table,
// 3 = the Float32 evaluator psi_f32 with FP64 accumulation (grav_set_precision)
//
// One item = one block of TPB threads x one station chunk: thread t of node-thread block bx owns the K nodes
// zbeg + cg K ... of node column col, (cg, col) = (t / ncol, t % ncol), t < ncol * ncg.
template <int TPB, int K, int EV>
__device__ __forceinline__ void adjoint_item(const Geom& g, const PsiTabView& tb, const float* s_at, float inv_scale,
                                             double4* s_obs, const double* __restrict__ v, double* __restrict__ partial,
                                             int bx, int by, int zbeg, int ncg, int obs_per_chunk) {
    const long long nthreads = (long long)g.ncol * ncg;
    const long long t = (long long)bx * TPB + threadIdx.x;
    const bool valid = t < nthreads;
    const long long tl = valid ? t : nthreads - 1;
    const int cg = (int)(tl / g.ncol);        // column index fastest: lanes of a warp are neighbouring columns
    const int col = (int)(tl - (long long)cg * g.ncol);
    const int a = col / g.nyp, b = col - a * g.nyp;
    const int c0 = zbeg + cg * K;
    const double xa = g.xn[a], yb = g.yn[b];
    double zc[K], acc[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        zc[k] = g.zn[min(c0 + k, g.nzp - 1)];
        acc[k] = 0.0;
    }
    const long long i0 = (long long)by * obs_per_chunk;
    const long long i1 = min(i0 + (long long)obs_per_chunk, g.N);
    double* out_hi = partial + (long long)by * 2 * g.Nn + (long long)col * g.nzp + c0;
    double* out_lo = out_hi + g.Nn;
    for (long long sbase = i0; sbase < i1; sbase += kAdjObsStage) {
        const int scnt = (int)min((long long)kAdjObsStage, i1 - sbase);
        __syncthreads();
        for (int j = threadIdx.x; j < scnt; j += TPB)
            s_obs[j] = make_double4(g.xo[sbase + j], g.yo[sbase + j], g.zo[sbase + j], v[sbase + j]);
        __syncthreads();
        for (int j0 = 0; j0 < scnt; j0 += kAdjObsTile) {
            const int j1 = min(j0 + kAdjObsTile, scnt);
            for (int j = j0; j < j1; ++j) {
                const double4 o = s_obs[j];
                const double X = xa - o.x, Y = yb - o.y;
                if (EV == 1 || EV == 2) {
                    const PsiColumn pc = psi_column(X, Y);
                    const double vs = o.w * pc.s;
#pragma unroll
                    for (int k = 0; k < K; ++k) acc[k] = fma(vs, psi_eval<EV == 2>(tb, pc, zc[k] - o.z), acc[k]);
                } else if (EV == 3) {
                    const float Xf = (float)X, Yf = (float)Y;
#pragma unroll
                    for (int k = 0; k < K; ++k)
                        acc[k] = fma(o.w, (double)psi_f32(Xf, Yf, (float)(zc[k] - o.z), inv_scale, s_at), acc[k]);
                } else {
                    const double XY = X * Y;
                    const double Q = fma(Y, Y, X * X);
#pragma unroll
                    for (int k = 0; k < K; ++k) acc[k] = fma(o.w, psi_libm(X, Y, zc[k] - o.z, XY, Q), acc[k]);
                }
            }
            // fold the tile sum into the (hi, lo) pair of each owned node and restart the running sum
            if (valid) {
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    if (c0 + k < g.nzp) {
                        double hi = acc[k], lo = 0.0;
                        if (sbase + j0 != i0) two_sum_acc(out_hi[k], out_lo[k], acc[k], hi, lo);
                        out_hi[k] = hi;
                        out_lo[k] = lo;
                    }
                    acc[k] = 0.0;
                }
            }
        }
    }
}

// KT > 0: the column is cut into ncg_main groups of KC nodes and ONE tail group of KT nodes (the nodes from
// ncg_main * KC on), instead of padding the last group of KC: node-thread blocks bx < nblocks_main run the KC body,
// the others the KT body (prime column lengths - config 5 has 151 nodes - otherwise pay up to KC - 1 wasted
// evaluations per column and station).  KT = 0: ncg_main groups of KC cover the column, the last one padded.
// work != NULL: persistent launch for small problems (see forward.cu): the block fills the tables once and draws
// (node-thread block, station chunk) items from the counter.
template <int TPB, int KC, int MINB, int EV, int KT>
__global__ void __launch_bounds__(TPB, MINB) adjoint_nodes_kernel(Geom g, PsiDev pd, const double* __restrict__ v,
                                                                  double* __restrict__ partial, int ncg_main,
                                                                  int nblocks_main, int obs_per_chunk,
                                                                  const int* __restrict__ done,
                                                                  int* __restrict__ work, int nblocks, int nitems) {
    extern __shared__ double2 s_tab[];
    if (done && *done) return;
    __shared__ double4 s_obs[kAdjObsStage];   // (xo, yo, zo, v)
    __shared__ int s_item;
    __shared__ float s_at[kAtanN32];
    PsiTabView tb;
    if (EV == 1 || EV == 2) tb = psi_tables_load<EV == 2>(s_tab, pd);
    if (EV == 3) psi_f32_atan_table(s_at, pd);
    const float inv_scale = psi_f32_inv_scale(pd.k0);
    for (;;) {
        int bx = blockIdx.x, by = blockIdx.y;
        if (work) {
            __syncthreads();                             // the previous item's s_item is done with
            if (threadIdx.x == 0) s_item = atomicAdd(work, 1);
            __syncthreads();
            const int item = s_item;
            if (item >= nitems) break;
            by = item / nblocks;                         // node block fastest: neighbours in time share a station chunk
            bx = item - by * nblocks;
        }
        if (KT == 0 || bx < nblocks_main)
            adjoint_item<TPB, KC, EV>(g, tb, s_at, inv_scale, s_obs, v, partial, bx, by, 0, ncg_main, obs_per_chunk);
        else
            adjoint_item<TPB, (KT > 0 ? KT : 1), EV>(g, tb, s_at, inv_scale, s_obs, v, partial, bx - nblocks_main, by,
                                                     ncg_main * KC, 1, obs_per_chunk);
        if (!work) break;
    }
}

// tnode[2][Nn] = sum over station chunks (or over ranks) of partial[chunk][2][Nn], (hi, lo) pairs combined in chunk
// order.
__global__ void adjoint_reduce_kernel(long long Nn, int nchunk, const double* __restrict__ partial,
                                      double* __restrict__ tnode) {
    long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= Nn) return;
    double hi = partial[n], lo = partial[Nn + n];
    constexpr int U = 8;          // the loads of U chunks are issued together, the TwoSum chain follows in chunk order
    for (int ch0 = 1; ch0 < nchunk; ch0 += U) {
        double h[U], l[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const double* pc = partial + (long long)min(ch0 + u, nchunk - 1) * 2 * Nn;
            h[u] = pc[n];
            l[u] = pc[Nn + n];
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (ch0 + u < nchunk) {
                two_sum_acc(hi, lo, h[u], hi, lo);
                lo += l[u];
            }
    }
    tnode[n] = hi;
    tnode[Nn + n] = lo;
}

template <int TPB, int KC, int MINB, int EV, int KT = 0>
static cudaError_t adj_launch(grav_ctx* c, const double* v, double* partial, const int* done, int* work,
                              cudaStream_t s) {
    // the opt-in is sized for the largest 2-D table, the launch for this context's table
    const size_t smem = (EV == 1 || EV == 2) ? psi_smem_bytes<EV == 2>(c->pd) : 0;
    static unsigned long long smem_set = 0;
    if (EV == 1 || EV == 2) {
        cudaError_t e = ensure_dynamic_smem(adjoint_nodes_kernel<TPB, KC, MINB, EV, KT>, psi_smem_max<EV == 2>(),
                                            c->device, &smem_set);
        if (e != cudaSuccess) return e;
    }
    // KT > 0: whole groups of KC, then one tail group of KT covering the rest of the column (make_plan guarantees it does)
    const int ncg = KT > 0 ? (c->g.nzp - 1) / KC : (c->g.nzp + KC - 1) / KC;
    const int nblocks_main = (int)(((long long)c->g.ncol * ncg + TPB - 1) / TPB);
    const int nblocks = nblocks_main + (KT > 0 ? (int)((c->g.ncol + TPB - 1) / TPB) : 0);
    const long long nitems = (long long)nblocks * c->plan.adj_nchunk;
    dim3 grid((unsigned)nblocks, c->plan.adj_nchunk);
    if (c->plan.persistent && (EV == 1 || EV == 2) && nitems < (1ll << 31)) {
        cudaError_t e = cudaMemsetAsync(work, 0, sizeof(int), s);
        if (e != cudaSuccess) return e;
        const long long resident = (long long)c->plan.sms * MINB;
        grid = dim3((unsigned)(nitems < resident ? nitems : resident), 1);
    } else {
        work = nullptr;
    }
    adjoint_nodes_kernel<TPB, KC, MINB, EV, KT><<<grid, TPB, smem, s>>>(c->g, c->pd, v, partial, ncg, nblocks_main,
                                                                        c->plan.adj_obs_per_chunk, done, work, nblocks,
                                                                        (int)nitems);
    return cudaGetLastError();
}

cudaError_t launch_adjoint_nodes(grav_ctx* c, const double* v, double* partial, const int* done, int* work,
                                 cudaStream_t s) {
    const int kc = c->plan.adj_kc;           // the plan's choice of KC (grav_api.cu make_plan)
    cudaError_t e;
    if (c->psi_variant == 1) e = adj_launch<128, 4, 4, 0>(c, v, partial, done, work, s);
    else if (c->psi_variant == 2) {      // Float32 evaluator: no tables, several blocks per SM
        if (kc <= 4) e = adj_launch<256, 4, 4, 3>(c, v, partial, done, work, s);
        else if (kc == 5) e = adj_launch<256, 5, 4, 3>(c, v, partial, done, work, s);
        else if (kc == 6) e = adj_launch<256, 6, 4, 3>(c, v, partial, done, work, s);
        else e = adj_launch<256, 8, 4, 3>(c, v, partial, done, work, s);      // any larger KC of the plan
    }
    else if (use_log2d(c)) {      // (threads, KC) pairs of make_plan's table
        switch (kc) {
            case 4: e = adj_launch<512, 4, 1, 2>(c, v, partial, done, work, s); break;
            case 5: e = adj_launch<384, 5, 1, 2>(c, v, partial, done, work, s); break;
            case 6: e = adj_launch<384, 6, 1, 2>(c, v, partial, done, work, s); break;
            case 7:
                if (c->plan.adj_kt == 4) e = adj_launch<384, 7, 1, 2, 4>(c, v, partial, done, work, s);
                else if (c->plan.adj_kt == 5) e = adj_launch<384, 7, 1, 2, 5>(c, v, partial, done, work, s);
                else if (c->plan.adj_kt == 6) e = adj_launch<384, 7, 1, 2, 6>(c, v, partial, done, work, s);
                else e = adj_launch<384, 7, 1, 2>(c, v, partial, done, work, s);
                break;
            case 11: e = adj_launch<256, 11, 1, 2>(c, v, partial, done, work, s); break;
            case 13: e = adj_launch<256, 13, 1, 2>(c, v, partial, done, work, s); break;
            case 17: e = adj_launch<256, 17, 1, 2>(c, v, partial, done, work, s); break;
            default: e = adj_launch<256, 8, 1, 2>(c, v, partial, done, work, s); break;
        }
    } else {
        if (kc == 4) e = adj_launch<256, 4, 2, 1>(c, v, partial, done, work, s);
        else if (kc == 5) e = adj_launch<256, 5, 2, 1>(c, v, partial, done, work, s);
        else if (kc == 6) e = adj_launch<128, 6, 3, 1>(c, v, partial, done, work, s);
        else e = adj_launch<128, 8, 2, 1>(c, v, partial, done, work, s);
    }
    c->launches++;
    return e;
}

cudaError_t launch_adjoint_reduce(grav_ctx* c, const double* partial, int nchunk, double* tnode, cudaStream_t s) {
    adjoint_reduce_kernel<<<(unsigned)((c->g.Nn + 255) / 256), 256, 0, s>>>(c->g.Nn, nchunk, partial, tnode);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace grav
