// stored.cu -- the per-pair kernel family and the stored-G path (BASELINE.json north_star kernel 4).
//
// tabulate:  G[i][m] = gamma * sum_pqr sigma Psi(corner_pqr(m) - obs_i)   (Eq. 1; the paper's
//            Listing 1, one thread per entry).  Here one thread evaluates the 4 corners of one
//            horizontal node layer of a prism column, L(c) = sum_{da,db} (-1)^(da+db) Psi(X_da, Y_db, Z_c), and
//            the prism between layers c and c+1 is gamma*(L(c+1) - L(c)) with L(c+1) taken from the next lane
//            (warp shuffle): 4 evaluations per pair instead of 8, stores coalesced along the prism index.
// gemv / gemvt: d = G u (row dots), g = G^T v (column sums), one streaming read of G each, FP64 accumulation
//            ("matrix multiplications"); HBM-bound.
// gram_diag: diag_i = sum_k G_ik^2 / w_k^2 with the same per-pair evaluation, nothing stored (reading C7).
// form_A / cholesky: explicit N x N data-space system for tiny N (BASELINE.json config 1).
#include "grav_internal.cuh"
#include "psi.cuh"
#include "psi2.cuh"

namespace grav {

// ---- per-pair evaluation ---------------------------------------------------------------------------------
// Flattened "layer" index q = cc*nzp + c over cell columns cc = i*ny + j and node layers c = 0..nz.
// A warp owns 32 consecutive q starting at 31*warp; lane l < 31 outputs the prism (cc, k=c) if c < nz.
template <bool FAST>
__device__ __forceinline__ double layer_value(const Geom& g, const Psi2TabView& tb, long long q, long long nq, double xo,
                                              double yo, double zo, int& cc, int& c) {
    q = q < nq ? q : nq - 1;
    cc = (int)(q / g.nzp);
    c = (int)(q - (long long)cc * g.nzp);
    const int i = cc / g.ny, j = cc - i * g.ny;
    const double X1 = g.xn[i] - xo, X2 = g.xn[i + 1] - xo;
    const double Y1 = g.yn[j] - yo, Y2 = g.yn[j + 1] - yo;
    const double Z = g.zn[c] - zo;
    // (-1)^(da+db): (0,0)+, (1,0)-, (0,1)-, (1,1)+
    double v;
    if (FAST) {
        const PsiColumn c11 = psi_column(X1, Y1), c21 = psi_column(X2, Y1), c12 = psi_column(X1, Y2),
                        c22 = psi_column(X2, Y2);
        v = c11.s * psi2_fast(tb, c11, Z);
        v = fma(-c21.s, psi2_fast(tb, c21, Z), v);
        v = fma(-c12.s, psi2_fast(tb, c12, Z), v);
        v = fma(c22.s, psi2_fast(tb, c22, Z), v);
    } else {
        v = psi_libm(X1, Y1, Z, X1 * Y1, fma(Y1, Y1, X1 * X1));
        v -= psi_libm(X2, Y1, Z, X2 * Y1, fma(Y1, Y1, X2 * X2));
        v -= psi_libm(X1, Y2, Z, X1 * Y2, fma(Y2, Y2, X1 * X1));
        v += psi_libm(X2, Y2, Z, X2 * Y2, fma(Y2, Y2, X2 * X2));
    }
    return v;
}

template <typename T, int TPB, bool FAST>
__global__ void __launch_bounds__(TPB) tabulate_kernel(Geom g, Psi2Dev pd, T* __restrict__ G) {
    extern __shared__ double2 s_tab[];
    Psi2TabView tb;
    if (FAST) tb = psi2_tables_to_smem(s_tab, pd);
    const long long nq = (long long)g.nx * g.ny * g.nzp;
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * TPB + threadIdx.x) >> 5;
    const long long q = warp * 31 + lane;
    if (warp * 31 >= nq) return;
    for (long long i = blockIdx.y; i < g.N; i += gridDim.y) {
        int cc, c;
        const double L = layer_value<FAST>(g, tb, q, nq, g.xo[i], g.yo[i], g.zo[i], cc, c);
        const double Lnext = __shfl_down_sync(0xffffffffu, L, 1);
        if (lane < 31 && q < nq && c < g.nz) {
            const long long m = (long long)cc * g.nz + c;
            G[i * g.M + m] = (T)(g.gamma * (Lnext - L));
        }
    }
}


// Column-walking tabulation (the default): one thread owns one cell column (i, j) and walks down its nz + 1 node
// layers for one station after another.  Everything that depends only on (station, corner column) - the four
// PsiColumn hoists - is computed once per column instead of once per layer, the four corner evaluations of a layer
// are independent (4 evaluations in flight per thread), and the entry of prism k is gamma (L(k+1) - L(k)) with both
// layer values formed by the same thread: 4 evaluations per pair, no shuffles, no 64-bit index divisions.
// Lanes are neighbouring cell columns, so a warp's stores of one layer are nz elements apart; consecutive layers
// fill the same 32-byte sectors, which L2 merges before they reach DRAM.
template <typename T, int TPB, int EV>   // EV 2: 256-entry log table, 3: exponent-and-mantissa log table
__global__ void __launch_bounds__(TPB) tabulate_cols_kernel(Geom g, Psi2Dev pd, T* __restrict__ G) {
    extern __shared__ double2 s_tab[];
    const Psi2TabView tb = EV == 3 ? psi2_tables_to_smem_2d(s_tab, pd) : psi2_tables_to_smem(s_tab, pd);
    const int ncc = g.nx * g.ny;
    const int cc = blockIdx.x * TPB + threadIdx.x;
    const int ccl = cc < ncc ? cc : ncc - 1;
    const int i = ccl / g.ny, j = ccl - i * g.ny;
    const double x1 = g.xn[i], x2 = g.xn[i + 1], y1 = g.yn[j], y2 = g.yn[j + 1];
    for (long long st = blockIdx.y; st < g.N; st += gridDim.y) {
        const double xo = g.xo[st], yo = g.yo[st], zo = g.zo[st];
        const PsiColumn c11 = psi_column(x1 - xo, y1 - yo), c21 = psi_column(x2 - xo, y1 - yo),
                        c12 = psi_column(x1 - xo, y2 - yo), c22 = psi_column(x2 - xo, y2 - yo);
        T* __restrict__ out = G + st * g.M + (long long)ccl * g.nz;
        double Lprev = 0.0;
#pragma unroll 2
        for (int c = 0; c < g.nzp; ++c) {
            const double Z = __ldg(g.zn + c) - zo;
            // (-1)^(da+db): (0,0)+, (1,0)-, (0,1)-, (1,1)+   (same order as layer_value)
            double L = c11.s * psi2_fast_t<EV == 3>(tb, c11, Z);
            L = fma(-c21.s, psi2_fast_t<EV == 3>(tb, c21, Z), L);
            L = fma(-c12.s, psi2_fast_t<EV == 3>(tb, c12, Z), L);
            L = fma(c22.s, psi2_fast_t<EV == 3>(tb, c22, Z), L);
            if (c > 0 && cc < ncc) out[c - 1] = (T)(g.gamma * (L - Lprev));
            Lprev = L;
        }
    }
}

template <typename T, int EV>
static cudaError_t tabulate_cols_launch(grav_ctx* c, T* G, cudaStream_t s) {
    constexpr int TPB = 512;
    constexpr size_t smem_max = EV == 3 ? kAtan2SmemBytes + (size_t)kLog2dMaxBinades * 4096 : kTab2SmemBytes;
    const size_t smem = EV == 3 ? kAtan2SmemBytes + (size_t)c->pd2.nb2d * 4096 : smem_max;
    static unsigned long long smem_set = 0;
    cudaError_t e = ensure_dynamic_smem(tabulate_cols_kernel<T, TPB, EV>, smem_max, c->device, &smem_set);
    if (e != cudaSuccess) return e;
    const int ncc = c->g.nx * c->g.ny;
    const unsigned gx = (unsigned)((ncc + TPB - 1) / TPB);
    // every block fills the tables once and then loops over its stations: ~16 blocks per SM in total
    long long gy = (148LL * 16 + gx - 1) / gx;
    if (gy > c->g.N) gy = c->g.N;
    if (gy > 65535) gy = 65535;
    if (gy < 1) gy = 1;
    tabulate_cols_kernel<T, TPB, EV><<<dim3(gx, (unsigned)gy), TPB, smem, s>>>(c->g, c->pd2, G);
    return cudaGetLastError();
}

template <int TPB, bool FAST>
__global__ void __launch_bounds__(TPB) gram_diag_kernel(Geom g, Psi2Dev pd, const double* __restrict__ w,
                                                         double* __restrict__ diag) {
    extern __shared__ double2 s_tab[];
    __shared__ double sh[TPB];
    Psi2TabView tb;
    if (FAST) tb = psi2_tables_to_smem(s_tab, pd);
    const long long nq = (long long)g.nx * g.ny * g.nzp;
    const int lane = threadIdx.x & 31;
    const int warp_in_block = threadIdx.x >> 5;
    constexpr int WPB = TPB / 32;
    const long long nwarp_tasks = (nq + 30) / 31;
    for (long long i = blockIdx.x; i < g.N; i += gridDim.x) {
        const double xo = g.xo[i], yo = g.yo[i], zo = g.zo[i];
        double acc = 0.0;
        for (long long wt = warp_in_block; wt < nwarp_tasks; wt += WPB) {
            const long long q = wt * 31 + lane;
            int cc, c;
            const double L = layer_value<FAST>(g, tb, q, nq, xo, yo, zo, cc, c);
            const double Lnext = __shfl_down_sync(0xffffffffu, L, 1);
            if (lane < 31 && q < nq && c < g.nz) {
                const double gv = g.gamma * (Lnext - L);
                const double ww = w[(long long)cc * g.nz + c];
                acc = fma(gv / ww, gv / ww, acc);
            }
        }
        sh[threadIdx.x] = acc;
        __syncthreads();
        for (int s = TPB / 2; s > 0; s >>= 1) {
            if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
            __syncthreads();
        }
        if (threadIdx.x == 0) diag[i] = sh[0];
        __syncthreads();
    }
}


// Gram diagonal with the same column walk: one block per station (grid-stride), its threads stride over the cell
// columns, every thread accumulates G_ik^2 / w_k^2 down its columns; fixed-order block reduction.
template <int TPB, int EV>
__global__ void __launch_bounds__(TPB) gram_cols_kernel(Geom g, Psi2Dev pd, const double* __restrict__ w,
                                                         double* __restrict__ diag) {
    extern __shared__ double2 s_tab[];
    __shared__ double sh[TPB];
    const Psi2TabView tb = EV == 3 ? psi2_tables_to_smem_2d(s_tab, pd) : psi2_tables_to_smem(s_tab, pd);
    const int ncc = g.nx * g.ny;
    for (long long st = blockIdx.x; st < g.N; st += gridDim.x) {
        const double xo = g.xo[st], yo = g.yo[st], zo = g.zo[st];
        double acc = 0.0;
        for (int cc = threadIdx.x; cc < ncc; cc += TPB) {
            const int i = cc / g.ny, j = cc - i * g.ny;
            const double x1 = g.xn[i] - xo, x2 = g.xn[i + 1] - xo, y1 = g.yn[j] - yo, y2 = g.yn[j + 1] - yo;
            const PsiColumn c11 = psi_column(x1, y1), c21 = psi_column(x2, y1), c12 = psi_column(x1, y2),
                            c22 = psi_column(x2, y2);
            const double* __restrict__ wc = w + (long long)cc * g.nz;
            double Lprev = 0.0;
#pragma unroll 2
            for (int c = 0; c < g.nzp; ++c) {
                const double Z = __ldg(g.zn + c) - zo;
                double L = c11.s * psi2_fast_t<EV == 3>(tb, c11, Z);
                L = fma(-c21.s, psi2_fast_t<EV == 3>(tb, c21, Z), L);
                L = fma(-c12.s, psi2_fast_t<EV == 3>(tb, c12, Z), L);
                L = fma(c22.s, psi2_fast_t<EV == 3>(tb, c22, Z), L);
                if (c > 0) {
                    const double gv = g.gamma * (L - Lprev) / wc[c - 1];
                    acc = fma(gv, gv, acc);
                }
                Lprev = L;
            }
        }
        sh[threadIdx.x] = acc;
        __syncthreads();
        for (int k = TPB / 2; k > 0; k >>= 1) {
            if (threadIdx.x < k) sh[threadIdx.x] += sh[threadIdx.x + k];
            __syncthreads();
        }
        if (threadIdx.x == 0) diag[st] = sh[0];
        __syncthreads();
    }
}

template <int EV>
static cudaError_t gram_cols_launch(grav_ctx* c, const double* w, double* diag, cudaStream_t s) {
    constexpr int TPB = 512;
    constexpr size_t smem_max = EV == 3 ? kAtan2SmemBytes + (size_t)kLog2dMaxBinades * 4096 : kTab2SmemBytes;
    const size_t smem = EV == 3 ? kAtan2SmemBytes + (size_t)c->pd2.nb2d * 4096 : smem_max;
    static unsigned long long smem_set = 0;
    cudaError_t e = ensure_dynamic_smem(gram_cols_kernel<TPB, EV>, smem_max, c->device, &smem_set);
    if (e != cudaSuccess) return e;
    const unsigned blocks = (unsigned)(c->g.N < 148 * 16 ? c->g.N : 148 * 16);
    gram_cols_kernel<TPB, EV><<<blocks, TPB, smem, s>>>(c->g, c->pd2, w, diag);
    return cudaGetLastError();
}

// ---- GEMV: d = G u ----------------------------------------------------------------------------------------
template <typename T> struct Vec2;
template <> struct Vec2<double> { typedef double2 type; };
template <> struct Vec2<float> { typedef float2 type; };

template <typename T, int TPB, int ROWS>
__global__ void __launch_bounds__(TPB) gemv_kernel(long long N, long long M, const T* __restrict__ G,
                                                    const double* __restrict__ u, double* __restrict__ d) {
    __shared__ double sh[ROWS][TPB / 32];
    typedef typename Vec2<T>::type V2;
    const long long row0 = (long long)blockIdx.x * ROWS;
    double acc[ROWS];
#pragma unroll
    for (int r = 0; r < ROWS; ++r) acc[r] = 0.0;
    if ((M & 1) == 0) {   // rows stay 16-byte (8-byte for float) aligned only when M is even
        const long long M2 = M >> 1;
        for (long long m2 = threadIdx.x; m2 < M2; m2 += TPB) {
            const double2 uu = reinterpret_cast<const double2*>(u)[m2];
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const long long row = min(row0 + r, N - 1);
                const V2 gg = __ldcs(reinterpret_cast<const V2*>(G + row * M) + m2);
                acc[r] = fma((double)gg.x, uu.x, acc[r]);
                acc[r] = fma((double)gg.y, uu.y, acc[r]);
            }
        }
    } else {
        for (long long m = threadIdx.x; m < M; m += TPB) {
            const double uu = u[m];
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const long long row = min(row0 + r, N - 1);
                acc[r] = fma((double)G[row * M + m], uu, acc[r]);
            }
        }
    }
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
        double v = acc[r];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) sh[r][threadIdx.x >> 5] = v;
    }
    __syncthreads();
    if (threadIdx.x < ROWS) {
        double v = 0.0;
#pragma unroll
        for (int wv = 0; wv < TPB / 32; ++wv) v += sh[threadIdx.x][wv];
        if (row0 + threadIdx.x < N) d[row0 + threadIdx.x] = v;
    }
}

// ---- GEMV^T: g = G^T v, partial over row chunks -----------------------------------------------------------
template <typename T, int TPB>
__global__ void __launch_bounds__(TPB) gemvt_kernel(long long N, long long M, const T* __restrict__ G,
                                                     const double* __restrict__ v, double* __restrict__ partial,
                                                     int rows_per_chunk) {
    typedef typename Vec2<T>::type V2;
    const long long m2 = (long long)blockIdx.x * TPB + threadIdx.x;     // column pair
    const long long M2 = (M + 1) >> 1;
    const long long r0 = (long long)blockIdx.y * rows_per_chunk;
    const long long r1 = min(r0 + (long long)rows_per_chunk, N);
    if (m2 >= M2) return;
    const bool pair = (2 * m2 + 1 < M) && ((M & 1) == 0);
    double a0 = 0.0, a1 = 0.0;
    if (pair) {
        long long r = r0;
        for (; r + 4 <= r1; r += 4) {
            V2 g0 = __ldcs(reinterpret_cast<const V2*>(G + (r + 0) * M) + m2);
            V2 g1 = __ldcs(reinterpret_cast<const V2*>(G + (r + 1) * M) + m2);
            V2 g2 = __ldcs(reinterpret_cast<const V2*>(G + (r + 2) * M) + m2);
            V2 g3 = __ldcs(reinterpret_cast<const V2*>(G + (r + 3) * M) + m2);
            const double v0 = v[r], v1 = v[r + 1], v2 = v[r + 2], v3 = v[r + 3];
            a0 = fma((double)g0.x, v0, a0); a1 = fma((double)g0.y, v0, a1);
            a0 = fma((double)g1.x, v1, a0); a1 = fma((double)g1.y, v1, a1);
            a0 = fma((double)g2.x, v2, a0); a1 = fma((double)g2.y, v2, a1);
            a0 = fma((double)g3.x, v3, a0); a1 = fma((double)g3.y, v3, a1);
        }
        for (; r < r1; ++r) {
            V2 g0 = __ldcs(reinterpret_cast<const V2*>(G + r * M) + m2);
            a0 = fma((double)g0.x, v[r], a0); a1 = fma((double)g0.y, v[r], a1);
        }
        reinterpret_cast<double2*>(partial + (long long)blockIdx.y * M)[m2] = make_double2(a0, a1);
    } else {   // odd M: scalar columns
        for (long long r = r0; r < r1; ++r) {
            a0 = fma((double)G[r * M + 2 * m2], v[r], a0);
            if (2 * m2 + 1 < M) a1 = fma((double)G[r * M + 2 * m2 + 1], v[r], a1);
        }
        partial[(long long)blockIdx.y * M + 2 * m2] = a0;
        if (2 * m2 + 1 < M) partial[(long long)blockIdx.y * M + 2 * m2 + 1] = a1;
    }
}

__global__ void gemvt_reduce_kernel(long long M, int nchunk, const double* __restrict__ partial,
                                    const double* __restrict__ w, double* __restrict__ g) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= M) return;
    double s = 0.0;
    for (int ch = 0; ch < nchunk; ++ch) s += partial[(long long)ch * M + m];
    if (w) { double ww = w[m]; s = s / (ww * ww); }
    g[m] = s;
}

// ---- explicit data-space matrix and Cholesky (tiny N) ------------------------------------------------------
__global__ void __launch_bounds__(256) form_A_kernel(long long N, long long M, const double* __restrict__ G,
                                                      const double* __restrict__ w, double lam, double* __restrict__ A) {
    __shared__ double sh[256];
    const int i = blockIdx.x, j = blockIdx.y;
    if (j > i) return;
    double acc = 0.0;
    for (long long k = threadIdx.x; k < M; k += 256) {
        double ww = w[k];
        acc = fma(G[i * M + k] / (ww * ww), G[j * M + k], acc);
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        double v = sh[0] + (i == j ? lam : 0.0);
        A[(long long)i * N + j] = v;
        A[(long long)j * N + i] = v;
    }
}

// One block; right-looking Cholesky (lower), then forward / back substitution.  n <= 1024.
__global__ void __launch_bounds__(1024) cholesky_solve_kernel(double* __restrict__ A, const double* __restrict__ b,
                                                               double* __restrict__ x, int n) {
    const int tid = threadIdx.x, nt = blockDim.x;
    for (int j = 0; j < n; ++j) {
        if (tid == 0) A[(long long)j * n + j] = sqrt(A[(long long)j * n + j]);
        __syncthreads();
        const double ljj = A[(long long)j * n + j];
        for (int i = j + 1 + tid; i < n; i += nt) A[(long long)i * n + j] /= ljj;
        __syncthreads();
        const int rem = n - j - 1;
        for (long long e = tid; e < (long long)rem * rem; e += nt) {
            const int i = j + 1 + (int)(e / rem), k = j + 1 + (int)(e % rem);
            if (k <= i) A[(long long)i * n + k] -= A[(long long)i * n + j] * A[(long long)k * n + j];
        }
        __syncthreads();
    }
    // L y = b  (y kept in x)
    for (int i = tid; i < n; i += nt) x[i] = b[i];
    __syncthreads();
    for (int j = 0; j < n; ++j) {
        if (tid == 0) x[j] /= A[(long long)j * n + j];
        __syncthreads();
        const double yj = x[j];
        for (int i = j + 1 + tid; i < n; i += nt) x[i] -= A[(long long)i * n + j] * yj;
        __syncthreads();
    }
    // L^T x = y
    for (int j = n - 1; j >= 0; --j) {
        if (tid == 0) x[j] /= A[(long long)j * n + j];
        __syncthreads();
        const double xj = x[j];
        for (int i = tid; i < j; i += nt) x[i] -= A[(long long)j * n + i] * xj;
        __syncthreads();
    }
}

// ---- launchers --------------------------------------------------------------------------------------------
static unsigned pair_blocks(const Geom& g, int tpb) {
    const long long nq = (long long)g.nx * g.ny * g.nzp;
    const long long nwarps = (nq + 30) / 31;
    return (unsigned)((nwarps * 32 + tpb - 1) / tpb);
}

cudaError_t init_stored_kernels() {
    cudaError_t e = cudaFuncSetAttribute(tabulate_kernel<double, 256, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTab2SmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(tabulate_kernel<float, 256, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTab2SmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(gram_diag_kernel<256, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTab2SmemBytes);
    return e;
}

cudaError_t launch_tabulate(grav_ctx* c, void* G, int elem, cudaStream_t s) {
    dim3 grid(pair_blocks(c->g, 256), (unsigned)(c->g.N < 65535 ? c->g.N : 65535));
    if (c->psi_variant == 0 && c->tune[2] == 0) {          // default: column-walking kernel
        cudaError_t e;
        if (c->plan.log2d) e = elem == 8 ? tabulate_cols_launch<double, 3>(c, (double*)G, s) : tabulate_cols_launch<float, 3>(c, (float*)G, s);
        else e = elem == 8 ? tabulate_cols_launch<double, 2>(c, (double*)G, s) : tabulate_cols_launch<float, 2>(c, (float*)G, s);
        c->launches++;
        return e;
    }
    if (c->psi_variant == 0) {                              // tune[2] = 1: layer-per-thread kernel (A/B)
        if (elem == 8) tabulate_kernel<double, 256, true><<<grid, 256, kTab2SmemBytes, s>>>(c->g, c->pd2, (double*)G);
        else tabulate_kernel<float, 256, true><<<grid, 256, kTab2SmemBytes, s>>>(c->g, c->pd2, (float*)G);
    } else {
        if (elem == 8) tabulate_kernel<double, 256, false><<<grid, 256, 0, s>>>(c->g, c->pd2, (double*)G);
        else tabulate_kernel<float, 256, false><<<grid, 256, 0, s>>>(c->g, c->pd2, (float*)G);
    }
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_gram_diag(grav_ctx* c, const double* w, double* diag, cudaStream_t s) {
    unsigned blocks = (unsigned)(c->g.N < (1 << 20) ? c->g.N : (1 << 20));
    if (c->psi_variant == 0 && c->tune[2] == 0) {          // default: column-walking kernel
        cudaError_t e = c->plan.log2d ? gram_cols_launch<3>(c, w, diag, s) : gram_cols_launch<2>(c, w, diag, s);
        c->launches++;
        return e;
    }
    if (c->psi_variant == 0) gram_diag_kernel<256, true><<<blocks, 256, kTab2SmemBytes, s>>>(c->g, c->pd2, w, diag);
    else gram_diag_kernel<256, false><<<blocks, 256, 0, s>>>(c->g, c->pd2, w, diag);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_gemv(grav_ctx* c, const void* G, int elem, const double* u, double* d, cudaStream_t s) {
    constexpr int ROWS = 4;
    unsigned blocks = (unsigned)((c->g.N + ROWS - 1) / ROWS);
    if (elem == 8) gemv_kernel<double, 256, ROWS><<<blocks, 256, 0, s>>>(c->g.N, c->g.M, (const double*)G, u, d);
    else gemv_kernel<float, 256, ROWS><<<blocks, 256, 0, s>>>(c->g.N, c->g.M, (const float*)G, u, d);
    c->launches++;
    return cudaGetLastError();
}

int gemvt_chunks(long long N) {
    int nchunk = (int)((N + 255) / 256);
    if (nchunk > 16) nchunk = 16;
    if (nchunk < 1) nchunk = 1;
    return nchunk;
}

cudaError_t launch_gemvt(grav_ctx* c, const void* G, int elem, const double* v, const double* w, double* g,
                         double* partial, cudaStream_t s) {
    const long long N = c->g.N, M = c->g.M;
    const int nchunk = gemvt_chunks(N);
    const int rpc = (int)((N + nchunk - 1) / nchunk);
    const long long M2 = (M + 1) >> 1;
    dim3 grid((unsigned)((M2 + 127) / 128), nchunk);
    if (elem == 8) gemvt_kernel<double, 128><<<grid, 128, 0, s>>>(N, M, (const double*)G, v, partial, rpc);
    else gemvt_kernel<float, 128><<<grid, 128, 0, s>>>(N, M, (const float*)G, v, partial, rpc);
    gemvt_reduce_kernel<<<(unsigned)((M + 255) / 256), 256, 0, s>>>(M, nchunk, partial, w, g);
    c->launches += 2;
    return cudaGetLastError();
}

cudaError_t launch_form_A(grav_ctx* c, const double* G, const double* w, double lam, double* A, cudaStream_t s) {
    dim3 grid((unsigned)c->g.N, (unsigned)c->g.N);
    form_A_kernel<<<grid, 256, 0, s>>>(c->g.N, c->g.M, G, w, lam, A);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_cholesky_solve(grav_ctx* c, double* A, const double* b, double* x, int n, cudaStream_t s) {
    cholesky_solve_kernel<<<1, 1024, 0, s>>>(A, b, x, n);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace grav
