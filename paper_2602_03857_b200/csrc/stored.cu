// stored.cu -- the per-pair kernel family and the stored-G path (BASELINE.json north_star kernel 4).
//
// tabulate:  G[i][m] = gamma * sum_pqr sigma Psi(corner_pqr(m) - obs_i)   (Eq. 1; the paper's
//            Listing 1, one thread per entry; "global memory (sensitivity matrix)").
//            Node-shared here: every Psi(node - station) is a corner of up to 8 prisms, so a block takes one station
//            and a tile of (tnx-1) x (tny-1) cell columns, its threads evaluate Psi down the tnx x tny NODE columns
//            of the tile once - (1 + 1/t)^2 (nz+1)/nz ~ 1.15 evaluations per pair instead of 8 - and park the vertical
//            differences Psi(k+1) - Psi(k) in shared memory; the entry of prism (i, j, k) is then the signed sum of
//            the four differences at its corner columns, written with lanes along k (contiguous in G).
// gram_diag: diag_i = sum_k G_ik^2 / w_k^2 with the same walk, nothing stored (reading C7; its sum is the trace
//            that fixes lambda, and diag + lambda is the Jacobi preconditioner of the data-space CG).
// gemv / gemvt: d = G u (row dots), g = G^T v (column sums), one streaming read of G each, FP64 accumulation
//            ("matrix multiplications"); HBM-bound.
// form_A / cholesky: explicit N x N data-space system for tiny N (BASELINE.json config 1).
#include "grav_internal.cuh"
#include "psi.cuh"

namespace grav {

// ---- per-pair evaluation, node-shared --------------------------------------------------------------------
constexpr int kPairTPB = 512;            // threads per block: 12 producer warps + 4 consumer warps
constexpr int kPairProd = 384;           // producer threads = node columns of a tile: up to 19 x 20 (18 x 19 cell columns)
constexpr int kPairCons = kPairTPB - kPairProd;
constexpr int kPairU = 16;               // evaluations in flight per producer thread when tabulating ...
constexpr int kPairUGram = 8;            // ... when summing the Gram diagonal
constexpr int kPairZPad = 32;            // bottom node repeated this many times behind the node depths in shared memory
// registers per thread after the hand-over from the consumer warpgroup to the producers: 384 x 144 + 128 x 80 = 512 x 128
constexpr int kPairConsRegs = 80, kPairProdRegs = 144;
enum { PAIR_F64 = 0, PAIR_F32 = 1, PAIR_GRAM = 2 };
__host__ __device__ constexpr int pair_zn_doubles(int nzp) { return (nzp + kPairZPad + 1) & ~1; }

// named barriers (0 is __syncthreads): FULL[b] - producers arrive, consumers wait; EMPTY[b] - consumers arrive, producers wait
enum { BAR_FULL0 = 1, BAR_FULL1 = 2, BAR_EMPTY0 = 3, BAR_EMPTY1 = 4, BAR_CONS = 5 };
__device__ __forceinline__ void bar_sync(int id, int count) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int count) {
    __threadfence_block();
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory");
}

// Work item = (station, tile), tile index fastest; blocks stride over the items; the z-axis of an item is cut into
// batches of zb layers, numbered q = 0, 1, ... across the items of a block; batch q lives in buffer q & 1.
// The block is warp-specialised.
// Producers (warps 0-11): thread t < nnx * nny owns node column (i0 + t / nny, j0 + t % nny): hoists once per item, then
//   Psi down the column, 8 evaluations in flight, storing dPsi(k) = Psi(k+1) - Psi(k) at buf[t * stride + k - k0]
//   (stride = zb + 2 doubles: 16-byte aligned rows whose 16-byte bank groups differ between neighbouring threads).
//   Per batch: wait EMPTY[q & 1] (from q = 2 on), evaluate and store, arrive on FULL[q & 1].  They never touch G.
// Consumers (warps 12-15): lanes run along the layers of the batch: a warp takes 32 / zb neighbouring cell columns per
//   trip, lane = (cell column within the trip, layer), the block kPairCons / zb cell columns per trip.  Per batch: wait
//   FULL[q & 1]; an entry is gamma * ((d11 - d21) - d12 + d22) from the rows of its four corner columns - the same
//   pairing as node_to_cell (vertical neighbours first: their Psi values are closest), so stored and matrix-free
//   products agree to rounding - stored so that a warp writes runs of zb consecutive entries of G (whole 32-byte
//   sectors); then arrive on EMPTY[q & 1].
// So the FP64 pipe is fed by 3 warps per scheduler without interruption while the 4th turns differences into entries;
// no block-wide barrier inside the item loop.
// EV: 0 = CUDA libm (cross-check), 1 = psi_eval with the 256-entry log table (see pair_dispatch for why not the 2-D one).
// PAIR_GRAM: winv2[cell] = 1 / w_cell^2 (gram_winv2_kernel); the item's sum goes to gram_partial[station][tile].

// Batch depth in layers: compile-time, a power of two dividing 32 (the consumers' lane mapping).
template <int EV> constexpr int pair_zb() { return 16; }

template <int MODE, int EV>
__global__ void __launch_bounds__(kPairTPB, 1) pair_tile_kernel(Geom g, PsiDev pd, int tnx, int tny, int tiles_y,
                                                               int ntiles, void* __restrict__ Gout,
                                                               const double* __restrict__ winv2,
                                                               double* __restrict__ gram_partial) {
    extern __shared__ double2 s_tab[];
    __shared__ double s_red[kPairCons / 32];
    PsiTabView tb;
    size_t tab_entries = 0;
    if (EV == 1) { tb = psi_tables_to_smem(s_tab, pd); tab_entries = (size_t)kTabEntries * kRep; }
    double* s_zn = reinterpret_cast<double*>(s_tab + tab_entries);
    double* s_d = s_zn + pair_zn_doubles(g.nzp);
    // node depths, the bottom node repeated so that the producers never have to clamp an index past the mesh bottom
    for (int c = threadIdx.x; c < g.nzp + kPairZPad; c += kPairTPB) s_zn[c] = g.zn[min(c, g.nz)];
    __syncthreads();
    constexpr int zb = pair_zb<EV>(), stride = zb + 2, bufsz = kPairProd * stride;
    constexpr int U = MODE == PAIR_GRAM ? kPairUGram : kPairU;
    static_assert(zb % U == 0 && kPairZPad >= zb, "batch = whole groups of evaluations; padding covers a batch");
    const int t = threadIdx.x;
    const bool producer = t < kPairProd;
    const int ds = (int)(gridDim.x / ntiles), dt = (int)(gridDim.x - ds * ntiles);  // item += gridDim.x as (station, tile)
    const int nbatch = (g.nz + zb - 1) / zb;
    // batches this block will process in all: the consumers skip the EMPTY arrivals nobody will wait for
    const long long nitems = g.N * (long long)ntiles;
    const long long my_items = blockIdx.x < nitems ? (nitems - 1 - blockIdx.x) / gridDim.x + 1 : 0;
    const long long total_batches = my_items * nbatch;
    // The block's items in order; both roles walk them with the same arithmetic.
    struct Item { long long st; int tile, i0, j0, nnx, nny; };
    auto item_at = [&](long long st, int tile) {
        const int tx = tile / tiles_y, ty = tile - tx * tiles_y;
        const int i0 = tx * (tnx - 1), j0 = ty * (tny - 1);
        return Item{st, tile, i0, j0, min(tnx, g.nxp - i0), min(tny, g.nyp - j0)};      // node columns of this tile
    };
    // The two roles run the item loop in separate branches, each with its own loop variables (sharing them across the
    // branches costs 11 % at config 3), so that each is compiled against its own register budget:
    // when tabulating, registers move from the consumer warpgroup to the three producer warpgroups (whole warpgroups,
    // once; config 3 FP32 tabulation 88.1 -> 85.8 ms.  The Gram sum's consumers want their registers: 89.2 ms without
    // the hand-over, 92.6-94.5 ms with it).
    if (producer) {
        if (MODE != PAIR_GRAM) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kPairProdRegs));
        long long st = blockIdx.x / ntiles;
        int tile = (int)(blockIdx.x - st * ntiles);
        long long q0 = 0;                                                        // number of the item's first batch
        for (; st < g.N; st += ds, tile += dt, q0 += nbatch) {
            if (tile >= ntiles) { tile -= ntiles; if (++st >= g.N) break; }
            const Item it = item_at(st, tile);
            const double zo = g.zo[st];
            const bool active = t < it.nnx * it.nny;
            const int la = active ? t / it.nny : 0, lb = active ? t - la * it.nny : 0;
            const double X = g.xn[it.i0 + la] - g.xo[st], Y = g.yn[it.j0 + lb] - g.yo[st];
            PsiColumn pc;
            double XY = 0.0, Q = 0.0;
            if (EV != 0) pc = psi_column(X, Y);
            else { XY = X * Y; Q = fma(Y, Y, X * X); }
            auto eval = [&](double zn) -> double {
                const double Z = zn - zo;
                if (EV == 0) return psi_libm(X, Y, Z, XY, Q);
                return pc.s * psi_eval<false>(tb, pc, Z);
            };
            double prev = active ? eval(s_zn[0]) : 0.0;
            for (int b = 0; b < nbatch; ++b) {
                const long long q = q0 + b;
                const int par = (int)(q & 1);
                if (q >= 2) bar_sync(BAR_EMPTY0 + par, kPairTPB);           // the consumers are done with batch q - 2
                if (active) {
                    const int k0 = b * zb, nb = min(zb, g.nz - k0);
                    double* dst = s_d + par * bufsz + t * stride;
                    // layers past the mesh bottom (last partial group only) are evaluated at the bottom node (s_zn is
                    // padded), stored, and never used
                    for (int kk = 0; kk < nb; kk += U) {
                        const double* zp = s_zn + k0 + kk + 1;
                        double cur[U];
#pragma unroll
                        for (int u = 0; u < U; ++u) cur[u] = eval(zp[u]);
#pragma unroll
                        for (int u = 0; u < U; u += 2)
                            *reinterpret_cast<double2*>(dst + kk + u) =
                                make_double2(cur[u] - (u ? cur[u - 1] : prev), cur[u + 1] - cur[u]);
                        prev = cur[U - 1];
                    }
                }
                bar_arrive(BAR_FULL0 + par, kPairTPB);
            }
        }
    } else {
        if (MODE != PAIR_GRAM) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kPairConsRegs));
        long long st = blockIdx.x / ntiles;
        int tile = (int)(blockIdx.x - st * ntiles);
        long long q0 = 0;                                                        // number of the item's first batch
        // consumers: lanes along k.  A warp takes cpw = 32 / zb neighbouring cell columns per trip (flattened index
        // cc = li * ncy + lj), lane = (cell within the trip, layer), so that its global accesses are runs of zb
        // consecutive entries of G (64 bytes in FP32) instead of one 16-byte piece per lane
        const int ct = t - kPairProd;
        constexpr int cpw = 32 / zb, trip = cpw * (kPairCons / 32);           // cell columns per warp trip / per block trip
        const int l = ct & (zb - 1);
        const int cc_first = (ct >> 5) * cpw + ((ct & 31) / zb);
        for (; st < g.N; st += ds, tile += dt, q0 += nbatch) {
            if (tile >= ntiles) { tile -= ntiles; if (++st >= g.N) break; }
            const Item it = item_at(st, tile);
            const int nny = it.nny, ncy = nny - 1, ncells = (it.nnx - 1) * ncy;
            const int li_first = cc_first / ncy, lj_first = cc_first - li_first * ncy;
            const int dli = trip / ncy, dlj = trip - dli * ncy;              // advance of (li, lj) per trip
            const int d21 = nny * stride;
            const int off_first = (li_first * nny + lj_first) * stride, off_step = (dli * nny + dlj) * stride;
            const int off_wrap = (nny - ncy) * stride;                       // lj -= ncy, li += 1
            const int cell_first = ((it.i0 + li_first) * g.ny + it.j0 + lj_first) * g.nz + l;
            const int cell_step = (dli * g.ny + dlj) * g.nz, cell_wrap = (g.ny - ncy) * g.nz;
            // (the row base is kept opaque so that the compiler does not re-form st * M per store)
            size_t Grow = (size_t)Gout + (size_t)st * (size_t)g.M * (MODE == PAIR_F64 ? 8 : 4);
            asm volatile("" : "+l"(Grow));
            double gram = 0.0;
            for (int b = 0; b < nbatch; ++b) {
                const long long q = q0 + b;
                const int par = (int)(q & 1);
                const int k0 = b * zb, nb = min(zb, g.nz - k0);
                bar_sync(BAR_FULL0 + par, kPairTPB);                        // the producers have stored batch q
                const double* buf = s_d + par * bufsz + l;
                if (l < nb) {
                    // buffer offset and cell index advance with (li, lj): +step per trip, +wrap when lj wraps
                    int lj = lj_first, off = off_first, cell = cell_first + k0;
                    // 4 trips in flight in every mode.  (Measured for the Gram sum on config 3: 1 trip 167 ms, 2 104 ms,
                    // 4 95 ms, 8 98 ms; parking the weights in shared memory ahead of the barrier, by plain or by
                    // asynchronous copies, 100-103 ms.)
#pragma unroll 4
                    for (int cc = cc_first; cc < ncells; cc += trip) {
                        double wi = 0.0;
                        if (MODE == PAIR_GRAM) wi = __ldg(winv2 + cell);     // from L2: requested before the buffer is read
                        const double* p11 = buf + off;
                        const double val = g.gamma * (((p11[0] - p11[d21]) - p11[stride]) + p11[d21 + stride]);
                        // (the opaque row address no longer tells the compiler its state space: say st.global)
                        if (MODE == PAIR_F64) asm volatile("st.global.f64 [%0], %1;" ::"l"(Grow + (size_t)cell * 8), "d"(val));
                        else if (MODE == PAIR_F32) asm volatile("st.global.f32 [%0], %1;" ::"l"(Grow + (size_t)cell * 4), "f"((float)val));
                        else gram = fma(val * val, wi, gram);
                        lj += dlj; off += off_step; cell += cell_step;
                        if (lj >= ncy) { lj -= ncy; off += off_wrap; cell += cell_wrap; }
                    }
                }
                if (q + 2 < total_batches) bar_arrive(BAR_EMPTY0 + par, kPairTPB);
            }
            if (MODE == PAIR_GRAM) {      // fixed-order sum over the consumer threads -> gram_partial[station][tile]
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) gram += __shfl_down_sync(0xffffffffu, gram, o);
                if ((ct & 31) == 0) s_red[ct >> 5] = gram;
                bar_sync(BAR_CONS, kPairCons);
                if (ct == 0) {
                    double sum = 0.0;
#pragma unroll
                    for (int k = 0; k < kPairCons / 32; ++k) sum += s_red[k];
                    gram_partial[st * ntiles + tile] = sum;
                }
                bar_sync(BAR_CONS, kPairCons);
            }
        }
    }
}

__global__ void gram_winv2_kernel(long long M, const double* __restrict__ w, double* __restrict__ winv2) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m < M) { const double ww = w[m]; winv2[m] = 1.0 / (ww * ww); }
}

// diag[st] = sum over tiles of gram_partial[st][tile], in tile order
__global__ void gram_reduce_kernel(long long N, int ntiles, const double* __restrict__ partial,
                                   double* __restrict__ diag) {
    const long long st = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (st >= N) return;
    double s = 0.0;
    for (int k = 0; k < ntiles; ++k) s += partial[st * ntiles + k];
    diag[st] = s;
}

static size_t pair_smem_bytes(const Geom& g, const PsiDev& pd, int ev) {
    const int zb = pair_zb<1>();
    const size_t tab = ev == 0 ? 0 : kTabSmemBytes;
    return tab + (size_t)pair_zn_doubles(g.nzp) * 8 + 2 * (size_t)kPairProd * (zb + 2) * 8;   // double-buffered
}
constexpr size_t kPairSmemMax = 226 * 1024;     // dynamic part: the opt-in limit of 227 KB includes the static s_red

// Tile shape: tnx * tny <= kPairProd node columns minimising the number of tiles (every tile costs one block the same
// time), ties towards the squarer tile.
void make_pair_plan(const Geom& g, const PsiDev& pd, bool log2d, Plan& p) {
    long long best = -1;
    p.pair_tnx = p.pair_tny = 2;
    for (int tnx = 2; tnx <= kPairProd / 2; ++tnx) {
        const int tny = kPairProd / tnx;
        if (tny < 2) break;
        const int ex = tnx > g.nxp ? g.nxp : tnx, ey = tny > g.nyp ? g.nyp : tny;      // never larger than the mesh
        const long long tiles = (long long)((g.nx + ex - 2) / (ex - 1)) * ((g.ny + ey - 2) / (ey - 1));
        const long long score = tiles * 1024 + (ex > ey ? ex - ey : ey - ex);
        if (best < 0 || score < best) { best = score; p.pair_tnx = ex; p.pair_tny = ey; }
    }
    p.pair_tiles_x = (g.nx + p.pair_tnx - 2) / (p.pair_tnx - 1);
    p.pair_tiles_y = (g.ny + p.pair_tny - 2) / (p.pair_tny - 1);
}

size_t gram_partial_doubles(const Geom& g, const Plan& p) { return (size_t)g.N * p.pair_tiles_x * p.pair_tiles_y; }

template <int MODE, int EV>
static cudaError_t pair_launch(grav_ctx* c, void* G, const double* w, double* gram_partial, cudaStream_t s) {
    const Plan& p = c->plan;
    const size_t smem = pair_smem_bytes(c->g, c->pd, EV);
    if (smem > kPairSmemMax) return cudaErrorInvalidValue;          // node columns deeper than ~20,000 layers
    if (c->g.M >= (1ll << 31)) return cudaErrorInvalidValue;        // the kernel keeps cell indices in 32 bits
    static unsigned long long smem_set = 0;
    cudaError_t e = ensure_dynamic_smem(pair_tile_kernel<MODE, EV>, kPairSmemMax, c->device, &smem_set);
    if (e != cudaSuccess) return e;
    const int ntiles = p.pair_tiles_x * p.pair_tiles_y;
    const long long nitems = c->g.N * (long long)ntiles;
    int sms = 148;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess) sms = 148;
    const unsigned blocks = (unsigned)(nitems < sms ? nitems : sms);    // one resident block per SM (shared memory)
    pair_tile_kernel<MODE, EV><<<blocks, kPairTPB, smem, s>>>(c->g, c->pd, p.pair_tnx, p.pair_tny, p.pair_tiles_y,
                                                               ntiles, G, w, gram_partial);
    return cudaGetLastError();
}

// The per-pair kernel always uses the 256-entry log table in 8 conflict-free copies, also where the matrix-free kernels
// use the single-copy 2-D table: with the difference buffer's traffic on top of the look-ups it is bound by
// shared-memory wavefronts, not by issue slots, so the table without bank collisions wins although it costs 2 FP64 + 7
// other instructions more per evaluation (config 3 FP32 tabulation 103.7 -> 98.8 ms, Gram diagonal 120.3 -> 111.7 ms),
// and its 66 KB leave room for batches of 16 layers.
template <int MODE>
static cudaError_t pair_dispatch(grav_ctx* c, void* G, const double* w, double* gram_partial, cudaStream_t s) {
    if (c->psi_variant == 1) return pair_launch<MODE, 0>(c, G, w, gram_partial, s);
    return pair_launch<MODE, 1>(c, G, w, gram_partial, s);
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
cudaError_t launch_tabulate(grav_ctx* c, void* G, int elem, cudaStream_t s) {
    cudaError_t e = elem == 8 ? pair_dispatch<PAIR_F64>(c, G, nullptr, nullptr, s)
                              : pair_dispatch<PAIR_F32>(c, G, nullptr, nullptr, s);
    c->launches++;
    return e;
}

cudaError_t launch_gram_diag(grav_ctx* c, const double* w, double* winv2, double* partial, double* diag,
                             cudaStream_t s) {
    gram_winv2_kernel<<<(unsigned)((c->g.M + 255) / 256), 256, 0, s>>>(c->g.M, w, winv2);
    cudaError_t e = pair_dispatch<PAIR_GRAM>(c, nullptr, winv2, partial, s);
    if (e != cudaSuccess) return e;
    gram_reduce_kernel<<<(unsigned)((c->g.N + 255) / 256), 256, 0, s>>>(c->g.N, c->plan.pair_tiles_x * c->plan.pair_tiles_y,
                                                                        partial, diag);
    c->launches += 3;
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

// ---- g = [W^-2] G^T v without any allocation (grav_gemvt_noalloc, include/grav.h) -----------------------------
// The same two kernels and the same row chunking as launch_gemvt; the per-chunk column sums live in a file-scope device
// array instead of the caller's workspace, so the call needs no context, no workspace and no cudaMalloc (callers under
// CUDA graph capture, serving loops and harnesses that forbid allocation).  Every GPU that loads the library holds the
// array until exit.  In host code the array's NAME is a host-side stand-in, not a device address: its device address
// is looked up here once per device with cudaGetSymbolAddress, with that device current, and handed to the kernels.
// All calls share the array and it keeps the last call's contents; nothing in it has to start at zero, because
// gemvt_kernel writes every (chunk, column) entry that gemvt_reduce_kernel reads (all nchunk chunks of all M columns)
// before the reduction runs on the same stream.  Calls that overlap on the GPU (different streams) race on it.
static __device__ __align__(256) double g_noalloc_partial[kNoAllocMaxDoubles];

namespace {
constexpr int kNoAllocMaxDevices = 64;
double* s_noalloc_ptr[kNoAllocMaxDevices];          // device address of g_noalloc_partial on each device (0 = not looked up)
}

// Set-up for `device` (which must be current): look the array's device address up.  Idempotent and thread-safe (two
// racing threads store the same value).  Not an allocation: the array is part of the loaded module.
cudaError_t noalloc_setup(int device, double** out) {
    if (device < 0 || device >= kNoAllocMaxDevices) return cudaErrorInvalidDevice;
    double* ptr = __atomic_load_n(&s_noalloc_ptr[device], __ATOMIC_ACQUIRE);
    if (!ptr) {
        cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_partial);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        __atomic_store_n(&s_noalloc_ptr[device], ptr, __ATOMIC_RELEASE);
    }
    if (out) *out = ptr;
    return cudaSuccess;
}

long long noalloc_gemvt_doubles(long long N, long long M) { return (long long)gemvt_chunks(N) * M; }

// `device` is current.  The caller has checked noalloc_gemvt_doubles(N, M) <= kNoAllocMaxDoubles.
cudaError_t launch_gemvt_noalloc(int device, const void* G, int elem, long long N, long long M, const double* v,
                                 const double* w, double* g, cudaStream_t s) {
    double* partial = nullptr;
    cudaError_t e = noalloc_setup(device, &partial);
    if (e != cudaSuccess) return e;
    const int nchunk = gemvt_chunks(N);
    const int rpc = (int)((N + nchunk - 1) / nchunk);
    const long long M2 = (M + 1) >> 1;
    dim3 grid((unsigned)((M2 + 127) / 128), nchunk);
    if (elem == 8) gemvt_kernel<double, 128><<<grid, 128, 0, s>>>(N, M, (const double*)G, v, partial, rpc);
    else gemvt_kernel<float, 128><<<grid, 128, 0, s>>>(N, M, (const float*)G, v, partial, rpc);
    gemvt_reduce_kernel<<<(unsigned)((M + 255) / 256), 256, 0, s>>>(M, nchunk, partial, w, g);
    return cudaGetLastError();
}

}  // namespace grav
