// grav_api.cu -- the C ABI of include/grav.h: context, workspace layout, call sequencing.  No arithmetic of the
// method lives here except the order in which kernels are enqueued.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <new>
#include <vector>

#include "grav_internal.cuh"

using namespace grav;

namespace {

thread_local char g_err[512] = "";

grav_status fail(grav_status st, const char* fmt, const char* a = "", const char* b = "") {
    snprintf(g_err, sizeof(g_err), fmt, a, b);
    return st;
}
grav_status cuda_fail(cudaError_t e, const char* where) {
    return fail(GRAV_ECUDA, "%s: %s", where, cudaGetErrorString(e));
}
#define CK(call, where)                                      \
    do {                                                     \
        cudaError_t e__ = (call);                            \
        if (e__ != cudaSuccess) return cuda_fail(e__, where); \
    } while (0)

size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

int ceil_div(long long a, long long b) { return (int)((a + b - 1) / b); }

// Launch plan: enough blocks to fill 148 SMs several times over, fixed per context => deterministic sums.
// log2d: the context's geometry admits the 2-D log table (psi.cuh LOG2D): kernels of 512 / 256 threads, 1 block per SM.
void make_plan(const Geom& g, const PsiDev& pd, bool log2d, int sms, Plan& p) {
    p.log2d = log2d ? 1 : 0;
    p.sms = sms > 0 ? sms : 148;
    // Small problems (configs 1-2) run the node kernels persistently: with ~50 waves of short blocks the per-block table
    // fill (up to 140 KB from L2) and pipeline start cost 15-20 % of a launch there; from ~1e10 evaluations per product the
    // plain grid is as fast or faster.
    p.persistent = (log2d && (double)g.N * (double)g.Nn < 1e10) ? 1 : 0;
    // Blocks of one launch all take the same time, so a grid of W.f waves of resident blocks costs ceil(W.f) waves:
    // with ~5 waves (the first plan) up to 18 % of the launch was tail.  ~100 blocks per SM keeps the tail <= 2-3 %
    // (profiles/r1_tail_and_variants.md); the price is a larger partial buffer (<= 64 MB), read once.
    const int target_blocks = log2d ? 148 * 48 : 148 * 96;      // ~48 waves either way
    // forward: 256 (512) stations per block; split the node columns into chunks when the station tiles are few
    p.fwd_tpb = log2d ? 512 : 256;
    p.fwd_tiles = ceil_div(g.N, p.fwd_tpb);
    int want = ceil_div(target_blocks, p.fwd_tiles);
    if (want > g.ncol) want = g.ncol;
    if (want > 1024) want = 1024;
    while (want > 1 && (double)want * g.N * 8.0 > 64e6) --want;      // partial buffer <= 64 MB
    if (want < 1) want = 1;
    p.fwd_cols_per_chunk = ceil_div(g.ncol, want);
    if (log2d) {
        // One block per SM is resident, every block of a launch takes the same time (cols_per_chunk columns), so the
        // launch costs ceil(blocks / SMs) rounds: among the chunk sizes between `want` chunks and ~8 rounds pick the one
        // with the cheapest rounds x (columns per chunk + per-block overhead).  The overhead - drawing the item, the
        // first copy of node data, the barriers - is ~3 us (persistent launch) or ~1 us, in units of one column's time
        // (config 2: 1.820 -> 1.76 ms; the sweep of chunk counts there is not monotonic: 1.76 to 1.83 ms).
        const double t_col = (double)g.nzp * 4.0 * 109.4 / 1.965e9;
        const double ovh = (p.persistent ? 3e-6 : 1e-6) / t_col;
        const int cols_lo = p.fwd_cols_per_chunk;
        const int cols_hi = std::max(cols_lo, ceil_div((long long)g.ncol * p.fwd_tiles, (long long)sms * 8));
        double best_cost = 1e300;
        for (int cols = cols_lo; cols <= cols_hi; ++cols) {
            const long long blocks = (long long)ceil_div(g.ncol, cols) * p.fwd_tiles;
            const double cost = (double)ceil_div(blocks, sms) * ((double)cols + ovh);
            if (cost < best_cost * (1.0 - 1e-9)) { best_cost = cost; p.fwd_cols_per_chunk = cols; }
        }
    }
    p.fwd_nchunk = ceil_div(g.ncol, p.fwd_cols_per_chunk);
    p.fwd_reduce_rx = g.N < 32 * kDotBlocks ? 8 : 32;      // few stations: 8 per block and 32 chunk lanes (forward.cu)
    // adjoint: one thread per (node column, group of KC layers); split the stations into chunks when few threads
    // KC nodes per thread: the per-(thread, station) set-up is shared by KC evaluations but the column is padded to a
    // multiple of KC.  With the 2-D log table the compiled (threads, KC) variants all measure 111-116 scheduler cycles
    // per warp-evaluation before padding (configs 2-5), so the padding decides: pick the cheapest
    // base x padded column.  Without the table the fit of round 1 stands, (119.5 + 25.6 / KC).
    p.adj_tpb = 256;
    p.adj_kc = 4;
    double best = 1e300;
    if (log2d) {
        const struct { int tpb, kc; double cyc; } var[] = {{512, 4, 116.3}, {384, 5, 114.4}, {384, 6, 113.5}, {384, 7, 111.5},
                                                           {256, 8, 113.5}, {256, 11, 113.0}, {256, 13, 112.3}, {256, 17, 113.6}};
        for (const auto& v : var) {
            const double cost = v.cyc * (double)(ceil_div(g.nzp, v.kc) * v.kc);
            if (cost < best) { best = cost; p.adj_kc = v.kc; p.adj_tpb = v.tpb; }
        }
    } else {
        for (int kc : {4, 5, 6, 8}) {
            const double cost = (119.5 + 25.6 / kc) * (double)(ceil_div(g.nzp, kc) * kc);
            if (cost < best) { best = cost; p.adj_kc = kc; }
        }
        p.adj_tpb = p.adj_kc >= 6 ? 128 : 256;
    }
    p.adj_kt = 0;
    if (log2d) {
        // whole groups of 7 and ONE tail group of 4-6 nodes instead of a padded last group (adjoint.cu, KT): columns
        // whose length no compiled KC divides (config 5: 151 nodes) lose up to 6 evaluations per column and station
        // to the padding otherwise.
        const int nmain = (g.nzp - 1) / 7, rest = g.nzp - nmain * 7;
        if (nmain >= 1 && rest <= 6) {
            const int kt = rest < 4 ? 4 : rest;
            // measured: 133 cycles per warp-evaluation in the tail group (config 5 with KT = 4: 1853 -> 1826 ms; config 2
            // with KT = 5 instead of its (256, 11) variant: 1.883 -> 1.910 ms, so config 2 keeps (256, 11))
            const double tailcyc = 133.0;
            const double cost = 111.5 * 7.0 * nmain + tailcyc * kt;
            if (cost < best) { best = cost; p.adj_kc = 7; p.adj_tpb = 384; p.adj_kt = kt; }
        }
    }
    p.adj_ncg = p.adj_kt ? (g.nzp - 1) / p.adj_kc + 1 : ceil_div(g.nzp, p.adj_kc);
    p.adj_blocks = p.adj_kt ? ceil_div((long long)g.ncol * (p.adj_ncg - 1), p.adj_tpb) + ceil_div(g.ncol, p.adj_tpb)
                            : ceil_div((long long)g.ncol * p.adj_ncg, p.adj_tpb);
    want = ceil_div(log2d ? 148 * 48 : 148 * 128, p.adj_blocks);
    while (want > 1 && (double)want * 2.0 * g.Nn * 8.0 > 256e6) --want;   // [hi|lo] partial planes <= 256 MB
    // a chunk is at least 64 stations (one shared-memory tile is 256); tiny problems, where that leaves fewer blocks
    // than SMs, go down to 16 stations per chunk
    int maxchunk = ceil_div(g.N, 64);
    if ((long long)maxchunk * p.adj_blocks < 148) maxchunk = ceil_div(g.N, 16);
    if ((long long)maxchunk * p.adj_blocks < 148) maxchunk = ceil_div(g.N, 8);
    if (want > maxchunk) want = maxchunk;
    if (want > 256) want = 256;
    if (want < 1) want = 1;
    p.adj_obs_per_chunk = ceil_div(g.N, want);
    if (log2d) {
        // the same fit of rounds to the SM count as for the forward chunks: among 1..want station chunks (at least ~8
        // rounds) the cheapest rounds x (stations per chunk + per-block overhead in stations' time)
        const double t_obs = (double)p.adj_kc * 111.5 * (p.adj_tpb / 128) / 1.965e9;
        const double ovh = (p.persistent ? 3e-6 : 1e-6) / t_obs;
        double best_cost = 1e300;
        for (int nch = want; nch >= 1; --nch) {
            const int obs = ceil_div(g.N, nch);
            const long long blocks = (long long)ceil_div(g.N, obs) * p.adj_blocks;
            if (nch < want && blocks < (long long)sms * 8) break;
            const double cost = (double)ceil_div(blocks, sms) * ((double)obs + ovh);
            if (cost < best_cost * (1.0 - 1e-9)) { best_cost = cost; p.adj_obs_per_chunk = obs; }
        }
    }
    p.adj_nchunk = ceil_div(g.N, p.adj_obs_per_chunk);
    make_pair_plan(g, pd, log2d, p);
}

void make_layout(const Geom& g, const Plan& p, int world, WsLayout& L) {
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    const size_t D = sizeof(double);
    L.cnode = take(2 * g.Nn * D);              // (c_n, zn[c]) pairs
    L.tnode = take(2 * g.Nn * D);              // T as [hi | lo] planes
    L.fwd_partial = take((size_t)p.fwd_nchunk * g.N * D);
    L.adj_partial = take((size_t)p.adj_nchunk * 2 * g.Nn * D);
    L.gcell = take(g.M * D);
    L.cg_x = take(g.N * D);
    L.cg_r = take(g.N * D);
    L.cg_p = take(g.N * D);
    L.cg_q = take(g.N * D);
    L.cg_z = take(g.N * D);
    L.cg_w = take(g.M * D);
    L.dot_partial = take(3 * kDotBlocks * D);
    L.scalars = take(sizeof(CgScalars) + 64);
    L.stage_m = take(g.M * D);
    L.stage_n = take(g.N * D);
    L.stage_hist = take(4096 * D);
    L.work = take(64);                         // item counters of persistent launches (forward, adjoint)
    L.inv_dm = take(g.M * D);
    L.inv_r = take(g.N * D);
    L.inv_dd = take(g.N * D);
    L.inv_try = take(g.N * D);
    L.inv_scal = take(8 * D);
    L.gram_partial = take(gram_partial_doubles(g, p) * D);
    L.comm_gather = take(world > 1 ? (size_t)world * 2 * g.Nn * D : 0);
    L.matfree_end = off;
    L.gemvt_partial = take((size_t)gemvt_chunks(g.N) * g.M * D);
    L.gstore = off;
}

template <class T> T* wsp(grav_ctx* c, size_t off) { return reinterpret_cast<T*>(c->ws + off); }

grav_status check_ready(grav_ctx* c) {
    if (!c) return fail(GRAV_EINVAL, "NULL context");
    if (!c->ws) return fail(GRAV_ESTATE, "workspace not set (grav_set_workspace)");
    return GRAV_OK;
}

struct DeviceGuard {
    int prev;
    bool ok;
    explicit DeviceGuard(int dev) : prev(0), ok(true) {
        if (cudaGetDevice(&prev) != cudaSuccess) ok = false;
        if (ok && prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() { cudaSetDevice(prev); }
};

// Observation-sharded operation (grav_set_comm): sum `count` doubles at `buf` over all ranks, in place, ordered on
// stream `s`.  No-op for a single-rank context.
grav_status exchange(grav_ctx* c, double* buf, long long count, cudaStream_t s) {
    if (c->comm.world <= 1) return GRAV_OK;
    if (c->comm.allreduce_sum(buf, count, (void*)s, c->comm.user) != 0) return fail(GRAV_ECUDA, "all-reduce callback failed");
    return GRAV_OK;
}

// node sums T = sum_i v_i Psi(node - obs_i) into ws.tnode.  Sharded: the ranks' (hi, lo) planes are gathered and
// combined in rank order with the same error-free kernel that combines station chunks (a plain all-reduce would round
// every rank's contribution to one double and put ~1e-10 of max|g| at risk at config 5).
grav_status adjoint_to_tnode(grav_ctx* c, const double* v, const int* done, cudaStream_t s) {
    double* part = wsp<double>(c, c->lay.adj_partial);
    double* tn = wsp<double>(c, c->lay.tnode);
    if (c->plan.adj_nchunk == 1) {
        CK(launch_adjoint_nodes(c, v, tn, done, wsp<int>(c, c->lay.work) + 1, s), "adjoint_nodes");
    } else {
        CK(launch_adjoint_nodes(c, v, part, done, wsp<int>(c, c->lay.work) + 1, s), "adjoint_nodes");
        CK(launch_adjoint_reduce(c, part, c->plan.adj_nchunk, tn, s), "adjoint_reduce");
    }
    if (c->comm.world > 1) {
        double* gat = wsp<double>(c, c->lay.comm_gather);
        if (c->comm.allgather(tn, gat, 2 * c->g.Nn, (void*)s, c->comm.user) != 0)
            return fail(GRAV_ECUDA, "all-gather callback failed");
        CK(launch_adjoint_reduce(c, gat, c->comm.world, tn, s), "adjoint_reduce (ranks)");
    }
    return GRAV_OK;
}

}  // namespace

extern "C" {

const char* grav_last_error(void) { return g_err; }

grav_status grav_mesh_create(grav_ctx** out, int nx, int ny, int nz, const double* xn, const double* yn,
                             const double* zn, long long nobs, const double* ox, const double* oy, const double* oz,
                             double gamma, int device) {
    if (!out) return fail(GRAV_EINVAL, "out is NULL");
    *out = nullptr;
    if (nx <= 0 || ny <= 0 || nz <= 0 || nobs <= 0) return fail(GRAV_EINVAL, "nx, ny, nz, nobs must be positive");
    if (!xn || !yn || !zn || !ox || !oy || !oz) return fail(GRAV_EINVAL, "NULL coordinate array");
    if (!(gamma == gamma)) return fail(GRAV_EINVAL, "gamma is NaN");
    if ((long long)(nx + 1) * (ny + 1) > 2000000000LL) return fail(GRAV_EINVAL, "too many node columns");
    const double* arrs[3] = {xn, yn, zn};
    const int lens[3] = {nx + 1, ny + 1, nz + 1};
    for (int a = 0; a < 3; ++a)
        for (int i = 0; i < lens[a]; ++i) {
            if (!std::isfinite(arrs[a][i])) return fail(GRAV_EINVAL, "non-finite node coordinate");
            if (i && !(arrs[a][i] > arrs[a][i - 1])) return fail(GRAV_EINVAL, "node coordinates must be strictly increasing");
        }
    for (long long i = 0; i < nobs; ++i)
        if (!std::isfinite(ox[i]) || !std::isfinite(oy[i]) || !std::isfinite(oz[i]))
            return fail(GRAV_EINVAL, "non-finite station coordinate");
    int ndev = 0;
    CK(cudaGetDeviceCount(&ndev), "cudaGetDeviceCount");
    if (device < 0 || device >= ndev) return fail(GRAV_EINVAL, "bad device ordinal");
    DeviceGuard dg(device);
    if (!dg.ok) return fail(GRAV_ECUDA, "cudaSetDevice failed");

    grav_ctx* c = new (std::nothrow) grav_ctx();
    if (!c) return fail(GRAV_ENOMEM, "host allocation failed");
    memset(c, 0, sizeof(*c));
    Geom& g = c->g;
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.nxp = nx + 1; g.nyp = ny + 1; g.nzp = nz + 1;
    g.ncol = g.nxp * g.nyp;
    g.N = nobs;
    g.M = (long long)nx * ny * nz;
    g.Nn = (long long)g.ncol * g.nzp;
    g.gamma = gamma;
    c->device = device;

    const size_t ntab = sizeof(PsiTablesHost) / sizeof(double);
    const size_t ntab2d = (size_t)kLog2dMaxBinades * 256 * 2;
    const size_t nd = (size_t)g.nxp + g.nyp + g.nzp + 3 * (size_t)nobs + ntab + ntab2d + kAtanN32 + 9 * 32;   // each array 256-byte aligned
    std::vector<double> host;
    try { host.assign(nd, 0.0); } catch (...) { delete c; return fail(GRAV_ENOMEM, "host allocation failed"); }
    void* dev = nullptr;
    cudaError_t e = cudaMalloc(&dev, nd * sizeof(double));
    if (e != cudaSuccess) { delete c; return fail(GRAV_ENOMEM, "cudaMalloc of geometry failed: %s", cudaGetErrorString(e)); }
    size_t off = 0;
    auto put = [&](const double* src, size_t n) {
        const double* d = reinterpret_cast<const double*>(dev) + off;
        memcpy(host.data() + off, src, n * sizeof(double));
        off = (off + n + 31) & ~(size_t)31;
        return d;
    };
    g.xn = put(xn, g.nxp); g.yn = put(yn, g.nyp); g.zn = put(zn, g.nzp);
    g.xo = put(ox, nobs); g.yo = put(oy, nobs); g.zo = put(oz, nobs);
    {   // Psi tables (csrc/psi.cuh) and the global exponent offset: 2^k0 ~ half the horizontal survey diagonal
        double lox = xn[0], hix = xn[nx], loy = yn[0], hiy = yn[ny];
        for (long long i = 0; i < nobs; ++i) {
            lox = ox[i] < lox ? ox[i] : lox; hix = ox[i] > hix ? ox[i] : hix;
            loy = oy[i] < loy ? oy[i] : loy; hiy = oy[i] > hiy ? oy[i] : hiy;
        }
        const double diag = std::sqrt((hix - lox) * (hix - lox) + (hiy - loy) * (hiy - loy));
        c->pd.k0 = (diag > 0.0 && std::isfinite(diag)) ? (int)std::ilogb(0.5 * diag) : 0;
        if (c->pd.k0 > 900) c->pd.k0 = 900;
        if (c->pd.k0 < -900) c->pd.k0 = -900;
        PsiTablesHost tabs;               // ~8 KB; generated per context (depends on k0)
        psi_tables_generate(&tabs, c->pd.k0);
        c->pd.tab = reinterpret_cast<const double2*>(put(reinterpret_cast<const double*>(&tabs), ntab));
        c->pd.k = psi_consts_make(c->pd.k0);
        double at32[kAtanN32];
        psi_f32_atan_generate(at32);
        c->pd.atan32 = put(at32, kAtanN32);
        // 2-D log table: arguments a = R + Y obey Zmin^2 / (2 Rmax) <= a <= 2 Rmax, with Zmin the smallest vertical
        // station-node distance and Rmax the largest station-node distance
        c->pd.tab2d = nullptr; c->pd.nb2d = 0; c->pd.emin2d_biased = 0;
        double zmin = INFINITY, r2max = 0.0;
        for (long long i = 0; i < nobs; ++i) {
            const double dx = std::max(std::fabs(xn[0] - ox[i]), std::fabs(xn[nx] - ox[i]));
            const double dy = std::max(std::fabs(yn[0] - oy[i]), std::fabs(yn[ny] - oy[i]));
            const double dz = std::max(std::fabs(zn[0] - oz[i]), std::fabs(zn[nz] - oz[i]));
            r2max = std::max(r2max, dx * dx + dy * dy + dz * dz);
            const double* lb = std::lower_bound(zn, zn + nz + 1, oz[i]);
            if (lb != zn + nz + 1) zmin = std::min(zmin, std::fabs(*lb - oz[i]));
            if (lb != zn) zmin = std::min(zmin, std::fabs(*(lb - 1) - oz[i]));
        }
        const double rmax = std::sqrt(r2max);
        if (zmin > 0.0 && std::isfinite(zmin) && rmax > 0.0 && std::isfinite(rmax)) {
            // one binade of slack below for the rounding of R in R + Y (needs zmin^2 / rmax >> rmax 2^-53, implied
            // by the binade limit); the upper bound 2 Rmax is rigorous up to the rounding covered by the 1e-12
            const int elo = (int)std::ilogb(zmin * zmin / (2.0 * rmax)) - 1;
            const int ehi = (int)std::ilogb(2.0 * rmax * (1.0 + 1e-12));
            const int nb = ehi - elo + 1;
            if (nb <= kLog2dMaxBinades && elo > -900 && ehi < 900) {
                std::vector<double2> t2d((size_t)nb * 256);
                psi_log2d_generate(t2d.data(), c->pd.k0, elo, nb);
                c->pd.tab2d = reinterpret_cast<const double2*>(put(reinterpret_cast<const double*>(t2d.data()), (size_t)nb * 512));
                c->pd.nb2d = nb;
                c->pd.emin2d_biased = elo + 1023;
            }
        }
        c->psi_variant = 0;
        c->log2d_force = -1;
    }
    e = cudaMemcpy(dev, host.data(), off * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(dev); delete c; return cuda_fail(e, "cudaMemcpy geometry"); }
    c->geom_dev = dev;
    c->comm.world = 1;
    // tiny problems (config 1) would pay more for filling ~100 KB of table per block than they gain: the table is
    // built whenever the geometry admits it, but it is the default only from 5e7 evaluations per product
    int sms = 148;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) sms = 148;
    make_plan(g, c->pd, c->pd.tab2d != nullptr && (double)g.N * (double)g.Nn >= 5e7, sms, c->plan);
    make_layout(g, c->plan, 1, c->lay);
    *out = c;
    return GRAV_OK;
}

void grav_mesh_destroy(grav_ctx* c) {
    if (!c) return;
    DeviceGuard dg(c->device);
    if (c->geom_dev) cudaFree(c->geom_dev);
    delete c;
}

grav_status grav_sizes(const grav_ctx* c, long long out[3]) {
    if (!c || !out) return fail(GRAV_EINVAL, "NULL argument");
    out[0] = c->g.N; out[1] = c->g.M; out[2] = c->g.Nn;
    return GRAV_OK;
}

size_t grav_workspace_bytes(const grav_ctx* c, int mode) {
    if (!c) return 0;
    if (mode == GRAV_MATRIX_FREE) return c->lay.matfree_end;
    if (mode == GRAV_STORED_F64) return c->lay.gstore + align_up((size_t)c->g.N * c->g.M * 8);
    if (mode == GRAV_STORED_F32) return c->lay.gstore + align_up((size_t)c->g.N * c->g.M * 4);
    return 0;
}

grav_status grav_set_workspace(grav_ctx* c, void* ws, size_t bytes) {
    if (!c || !ws) return fail(GRAV_EINVAL, "NULL argument");
    if ((uintptr_t)ws & 255) return fail(GRAV_EINVAL, "workspace must be 256-byte aligned");
    if (bytes < c->lay.matfree_end) return fail(GRAV_ESTATE, "workspace smaller than grav_workspace_bytes(GRAV_MATRIX_FREE)");
    c->ws = (char*)ws;
    c->ws_bytes = bytes;
    c->stored_elem = 0;
    return GRAV_OK;
}

grav_status grav_set_comm(grav_ctx* c, const grav_comm* comm) {
    if (!c) return fail(GRAV_EINVAL, "NULL context");
    if (comm && comm->world > 1) {
        if (comm->rank < 0 || comm->rank >= comm->world) return fail(GRAV_EINVAL, "rank outside [0, world)");
        if (!comm->allreduce_sum || !comm->allgather) return fail(GRAV_EINVAL, "NULL collective callback");
        c->comm = *comm;
    } else {
        memset(&c->comm, 0, sizeof(c->comm));
        c->comm.world = 1;
    }
    make_layout(c->g, c->plan, c->comm.world, c->lay);      // the gather buffer depends on the number of ranks
    c->ws = nullptr;
    c->ws_bytes = 0;
    c->stored_elem = 0;
    return GRAV_OK;
}

// ---- allocation-free stored-G adjoint (csrc/stored.cu holds the device array and its address look-up) --------
static_assert(GRAV_NOALLOC_MAX_DOUBLES == kNoAllocMaxDoubles, "include/grav.h states the limit of csrc/stored.cu");

grav_status grav_noalloc_setup(int device) {
    DeviceGuard dg(device);
    if (!dg.ok) return fail(GRAV_EINVAL, "grav_noalloc_setup: cannot make the device current");
    CK(noalloc_setup(device, nullptr), "cudaGetSymbolAddress(no-allocation scratch)");
    return GRAV_OK;
}

grav_status grav_gemvt_noalloc(int device, const void* G, int elem_bytes, long long N, long long M, const double* v,
                               const double* w, double* g, void* stream) {
    if (!G || !v || !g) return fail(GRAV_EINVAL, "grav_gemvt_noalloc: NULL pointer");
    if (N < 1 || M < 1) return fail(GRAV_EINVAL, "grav_gemvt_noalloc: N and M must be positive");
    if (elem_bytes != 8 && elem_bytes != 4) return fail(GRAV_EINVAL, "grav_gemvt_noalloc: elem_bytes must be 8 or 4");
    if (M > kNoAllocMaxDoubles || noalloc_gemvt_doubles(N, M) > kNoAllocMaxDoubles) {
        char need[64], have[64];
        snprintf(need, sizeof(need), "%lld", M > kNoAllocMaxDoubles ? M : noalloc_gemvt_doubles(N, M));
        snprintf(have, sizeof(have), "%lld", (long long)kNoAllocMaxDoubles);
        return fail(GRAV_EINVAL, "grav_gemvt_noalloc: min(16, ceil(N/256)) * M = %s doubles of scratch exceed the built-in "
                                 "array of %s doubles (16 MiB); use grav_adjoint_stored with a workspace", need, have);
    }
    DeviceGuard dg(device);
    if (!dg.ok) return fail(GRAV_EINVAL, "grav_gemvt_noalloc: cannot make the device current");
    CK(launch_gemvt_noalloc(device, G, elem_bytes, N, M, v, w, g, (cudaStream_t)stream), "gemvt_noalloc");
    return GRAV_OK;
}

long long grav_launch_count(const grav_ctx* c) { return c ? c->launches : 0; }

grav_status grav_debug_set_psi_variant(grav_ctx* c, int variant) {
    if (!c || (variant != 0 && variant != 1)) return fail(GRAV_EINVAL, "bad context / variant");
    c->psi_variant = variant;
    c->stored_elem = 0;
    return GRAV_OK;
}

grav_status grav_set_precision(grav_ctx* c, int precision) {
    if (!c || (precision != GRAV_PREC_F64 && precision != GRAV_PREC_F32)) return fail(GRAV_EINVAL, "bad context / precision");
    c->psi_variant = precision == GRAV_PREC_F32 ? 2 : 0;
    return GRAV_OK;
}

grav_status grav_debug_psi_eval_device(grav_ctx* c, int variant, long long n, const double* X, const double* Y,
                                       const double* Z, double* out, void* stream) {
    if (!c || !X || !Y || !Z || !out || n <= 0) return fail(GRAV_EINVAL, "NULL argument / n <= 0");
    if (variant < 0 || variant > 3) return fail(GRAV_EINVAL, "variant must be 0..3");
    if (variant == 3 && !c->pd.tab2d) return fail(GRAV_ESTATE, "the geometry does not admit the 2-D log table");
    DeviceGuard dg(c->device);
    CK(launch_psi_check(c, variant, n, X, Y, Z, out, (cudaStream_t)stream), "psi_check");
    return GRAV_OK;
}

grav_status grav_debug_set_log2d(grav_ctx* c, int mode) {
    if (!c || mode < -1 || mode > 1) return fail(GRAV_EINVAL, "bad context / mode");
    if (mode == 1 && !c->pd.tab2d) return fail(GRAV_ESTATE, "the geometry does not admit the 2-D log table");
    c->log2d_force = mode;
    c->stored_elem = 0;
    return GRAV_OK;
}

int grav_debug_k0(const grav_ctx* c) { return c ? c->pd.k0 : 0; }

int grav_debug_log2d_binades(const grav_ctx* c) { return c ? c->pd.nb2d : 0; }

int grav_debug_log2d_default(const grav_ctx* c) { return c ? c->plan.log2d : 0; }

double grav_debug_psi_eval_host(double X, double Y, double Z, int k0, int log2d) {
    static std::map<int, PsiTablesHost> cache;              // per k0
    if (!cache.count(k0)) psi_tables_generate(&cache[k0], k0);
    PsiTablesHost& tabs = cache[k0];
    PsiTabView tb;
    tb.base = tabs.e; tb.shift = 0; tb.k = psi_consts_make(k0); tb.atan_base = tabs.e + kLogN; tb.log2d = nullptr;
    const PsiColumn pc = psi_column(X, Y);
    if (!log2d) return pc.s * psi_eval<false>(tb, pc, Z);
    const int emin = -80, nb = 160;                   // the host has no shared-memory limit: tabulate 2^-80 .. 2^80
    static std::map<int, std::vector<double2>> cache2d;
    std::vector<double2>& t2d = cache2d[k0];
    if (t2d.empty()) { t2d.assign((size_t)nb * 256, double2()); psi_log2d_generate(t2d.data(), k0, emin, nb); }
    tb.log2d = reinterpret_cast<const char*>(t2d.data()) - ((size_t)(emin + 1023) << 12);
    return pc.s * psi_eval<true>(tb, pc, Z);
}

grav_status grav_forward(grav_ctx* c, const double* u, double* d, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!u || !d) return fail(GRAV_EINVAL, "NULL vector");
    DeviceGuard dg(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    double* cn = wsp<double>(c, c->lay.cnode);
    double* part = wsp<double>(c, c->lay.fwd_partial);
    CK(launch_cell_to_node(c, u, nullptr, cn, s), "cell_to_node");
    CK(launch_forward_nodes(c, cn, part, nullptr, wsp<int>(c, c->lay.work), s), "forward_nodes");
    CK(launch_forward_reduce(c, part, c->g.gamma, 0.0, nullptr, d, nullptr, nullptr, s), "forward_reduce");
    return GRAV_OK;
}

grav_status grav_adjoint(grav_ctx* c, const double* v, double* gout, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!v || !gout) return fail(GRAV_EINVAL, "NULL vector");
    DeviceGuard dg(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    st = adjoint_to_tnode(c, v, nullptr, s);
    if (st) return st;
    CK(launch_node_to_cell(c, wsp<double>(c, c->lay.tnode), nullptr, c->g.gamma, gout, s), "node_to_cell");
    return GRAV_OK;
}

grav_status grav_depth_weights(grav_ctx* c, double beta, double z0, double* w, void* stream) {
    if (!c || !w) return fail(GRAV_EINVAL, "NULL argument");
    if (!(beta == beta) || !(z0 == z0)) return fail(GRAV_EINVAL, "NaN parameter");
    DeviceGuard dg(c->device);
    // zc_k + z0 > 0 for the shallowest layer is enough (zc increases with k).  zn is only on the device;
    // the first layer's half-thickness is positive, so z0 > -that.  Conservative host-side check: z0 >= 0 or
    // fetch the two top nodes.
    if (!(z0 >= 0.0)) {
        double z01[2];
        CK(cudaMemcpy(z01, c->g.zn, 2 * sizeof(double), cudaMemcpyDeviceToHost), "cudaMemcpy zn");
        if (!(0.5 * (z01[1] - z01[0]) + z0 > 0.0)) return fail(GRAV_EINVAL, "zc + z0 must be positive");
    }
    CK(launch_depth_weights(c, beta, z0, w, (cudaStream_t)stream), "depth_weights");
    return GRAV_OK;
}

grav_status grav_store_g(grav_ctx* c, int fp32, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    const int elem = fp32 ? 4 : 8;
    const size_t need = c->lay.gstore + (size_t)c->g.N * c->g.M * elem;
    if (c->ws_bytes < need) return fail(GRAV_ENOTFIT, "stored G does not fit in the workspace");
    DeviceGuard dg(c->device);
    c->stored_elem = 0;
    CK(launch_tabulate(c, c->ws + c->lay.gstore, elem, (cudaStream_t)stream), "tabulate");
    c->stored_elem = elem;
    return GRAV_OK;
}

grav_status grav_stored_g(const grav_ctx* c, const void** gdev, int* elem) {
    if (!c || !gdev || !elem) return fail(GRAV_EINVAL, "NULL argument");
    *elem = c->stored_elem;
    *gdev = c->stored_elem ? (const void*)(c->ws + c->lay.gstore) : nullptr;
    return GRAV_OK;
}

grav_status grav_forward_stored(grav_ctx* c, const double* u, double* d, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!u || !d) return fail(GRAV_EINVAL, "NULL vector");
    if (!c->stored_elem) return fail(GRAV_ESTATE, "no stored G (grav_store_g)");
    DeviceGuard dg(c->device);
    CK(launch_gemv(c, c->ws + c->lay.gstore, c->stored_elem, u, d, (cudaStream_t)stream), "gemv");
    return GRAV_OK;
}

grav_status grav_adjoint_stored(grav_ctx* c, const double* v, double* gout, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!v || !gout) return fail(GRAV_EINVAL, "NULL vector");
    if (!c->stored_elem) return fail(GRAV_ESTATE, "no stored G (grav_store_g)");
    DeviceGuard dg(c->device);
    CK(launch_gemvt(c, c->ws + c->lay.gstore, c->stored_elem, v, nullptr, gout, wsp<double>(c, c->lay.gemvt_partial),
                    (cudaStream_t)stream), "gemvt");
    return exchange(c, gout, c->g.M, (cudaStream_t)stream);
}

grav_status grav_gram_diag(grav_ctx* c, const double* w, double* diag, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!w || !diag) return fail(GRAV_EINVAL, "NULL argument");
    DeviceGuard dg(c->device);
    CK(launch_gram_diag(c, w, wsp<double>(c, c->lay.gcell), wsp<double>(c, c->lay.gram_partial), diag,
                        (cudaStream_t)stream), "gram_diag");
    return GRAV_OK;
}

grav_status grav_dataspace_cg(grav_ctx* c, const double* dobs, const double* w, double lambda, int iters, double rtol,
                              int mode, const double* precond, grav_cg_state* state, double* alpha, double* m,
                              double* hist, double* ab, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!dobs || !w || !alpha) return fail(GRAV_EINVAL, "NULL vector");
    if (iters < 0 || !(lambda == lambda) || !(rtol >= 0.0)) return fail(GRAV_EINVAL, "bad iters / lambda / rtol");
    if (mode != GRAV_MATRIX_FREE && mode != GRAV_STORED_F64 && mode != GRAV_STORED_F32)
        return fail(GRAV_EINVAL, "bad mode");
    if (mode != GRAV_MATRIX_FREE && c->stored_elem != (mode == GRAV_STORED_F64 ? 8 : 4))
        return fail(GRAV_ESTATE, "stored G of the requested precision not present (grav_store_g)");
    if (state && (!state->x_dev || !state->r_dev || !state->p_dev || !state->rho_dev))
        return fail(GRAV_EINVAL, "NULL pointer in grav_cg_state");
    DeviceGuard dg(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    const Geom& g = c->g;
    double* x = state ? state->x_dev : wsp<double>(c, c->lay.cg_x);
    double* r = state ? state->r_dev : wsp<double>(c, c->lay.cg_r);
    double* p = state ? state->p_dev : wsp<double>(c, c->lay.cg_p);
    double* q = wsp<double>(c, c->lay.cg_q);
    double* z = precond ? wsp<double>(c, c->lay.cg_z) : r;          // without a preconditioner z IS r
    double* dotA = wsp<double>(c, c->lay.dot_partial);
    double* dotB = dotA + kDotBlocks;                               // [r.z | r.r]
    CgScalars* sc = wsp<CgScalars>(c, c->lay.scalars);
    double* gcell = wsp<double>(c, c->lay.gcell);
    double* cnode = wsp<double>(c, c->lay.cnode);
    double* tnode = wsp<double>(c, c->lay.tnode);
    double* fpart = wsp<double>(c, c->lay.fwd_partial);
    const void* G = c->ws + c->lay.gstore;
    const int resume = state ? state->resume : 0;

    CK(launch_cg_init(c, dobs, precond, lambda, x, r, z, p, dotA, resume, s), "cg_init");
    if ((st = exchange(c, dotA, 3 * kDotBlocks, s))) return st;
    CK(launch_cg_init_finish(c, dotA, sc, rtol, resume, state ? state->rho_dev : nullptr, hist, s), "cg_init_finish");
    for (int it = 0; it < iters; ++it) {
        const int* done = &sc->done[it & 1];
        if (mode == GRAV_MATRIX_FREE) {
            // q = gamma^2 * Fwd( S^T W^-2 S Adj(p) ) + lambda p
            st = adjoint_to_tnode(c, p, done, s);
            if (st) return st;
            CK(launch_node_to_cell(c, tnode, w, g.gamma, gcell, s), "node_to_cell");
            CK(launch_cell_to_node(c, gcell, nullptr, cnode, s), "cell_to_node");
            CK(launch_forward_nodes(c, cnode, fpart, done, wsp<int>(c, c->lay.work), s), "forward_nodes");
            CK(launch_forward_reduce(c, fpart, g.gamma, lambda, p, q, dotA, done, s), "forward_reduce");
        } else {
            CK(launch_gemvt(c, G, c->stored_elem, p, w, gcell, wsp<double>(c, c->lay.gemvt_partial), s), "gemvt");
            if ((st = exchange(c, gcell, g.M, s))) return st;
            CK(launch_gemv(c, G, c->stored_elem, gcell, q, s), "gemv");
            CK(launch_dot_pq(c, p, lambda, q, dotA, sc, it, s), "dot_pq");
        }
        if ((st = exchange(c, dotA, kDotBlocks, s))) return st;
        CK(launch_cg_update_xr(c, x, r, p, q, precond, lambda, z, dotA, dotB, sc, it, s), "cg_update_xr");
        if ((st = exchange(c, dotB, 2 * kDotBlocks, s))) return st;
        CK(launch_cg_update_p(c, z, p, dotB, sc, hist, ab, it, s), "cg_update_p");
    }
    if (alpha != x) CK(cudaMemcpyAsync(alpha, x, g.N * sizeof(double), cudaMemcpyDeviceToDevice, s), "copy alpha");
    if (state) CK(cudaMemcpyAsync(state->rho_dev, &sc->rho[iters & 1], sizeof(double), cudaMemcpyDeviceToDevice, s), "copy rho");
    if (m) {   // m = W^-2 G^T alpha   (Eq. 11)
        if (mode == GRAV_MATRIX_FREE) {
            st = adjoint_to_tnode(c, x, nullptr, s);
            if (st) return st;
            CK(launch_node_to_cell(c, tnode, w, g.gamma, m, s), "node_to_cell");
        } else {
            CK(launch_gemvt(c, G, c->stored_elem, x, w, m, wsp<double>(c, c->lay.gemvt_partial), s), "gemvt");
            if ((st = exchange(c, m, g.M, s))) return st;
        }
    }
    return GRAV_OK;
}

grav_status grav_direct_solve(grav_ctx* c, const double* dobs, const double* w, double lambda, double* A,
                              double* alpha, double* m, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!dobs || !w || !A || !alpha) return fail(GRAV_EINVAL, "NULL argument");
    if (c->g.N > 1024) return fail(GRAV_EINVAL, "direct solve is limited to N <= 1024");
    if (c->stored_elem != 8) return fail(GRAV_ESTATE, "direct solve needs a stored FP64 G (grav_store_g)");
    if (c->comm.world > 1) return fail(GRAV_ESTATE, "direct solve is not available on an observation-sharded context");
    DeviceGuard dg(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    const double* G = reinterpret_cast<const double*>(c->ws + c->lay.gstore);
    CK(launch_form_A(c, G, w, lambda, A, s), "form_A");
    CK(launch_cholesky_solve(c, A, dobs, alpha, (int)c->g.N, s), "cholesky_solve");
    if (m) CK(launch_gemvt(c, G, 8, alpha, w, m, wsp<double>(c, c->lay.gemvt_partial), s), "gemvt");
    return GRAV_OK;
}

// ---- outer model-update loop (csrc/invert.cu has the passage and the readings) -----------------------------
grav_status grav_invert(grav_ctx* c, const double* dobs, const double* w, double lambda, const double* mref,
                        const double* precond, int max_outer, int max_inner, double tol_outer, double tol_inner,
                        int mode, double* m, double* dpred, double* hist_host, double* step_host, int* inner_host,
                        int* n_outer_host, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!dobs || !w || !m) return fail(GRAV_EINVAL, "NULL vector");
    if (max_outer < 0 || max_inner < 1 || !(tol_outer >= 0.0) || !(tol_inner >= 0.0) || !(lambda == lambda))
        return fail(GRAV_EINVAL, "bad max_outer / max_inner / tolerance / lambda");
    if (mode != GRAV_MATRIX_FREE && mode != GRAV_STORED_F64 && mode != GRAV_STORED_F32)
        return fail(GRAV_EINVAL, "bad mode");
    if (mode != GRAV_MATRIX_FREE && c->stored_elem != (mode == GRAV_STORED_F64 ? 8 : 4))
        return fail(GRAV_ESTATE, "stored G of the requested precision not present (grav_store_g)");
    DeviceGuard dg(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    const Geom& g = c->g;
    double* dm = wsp<double>(c, c->lay.inv_dm);
    double* r = wsp<double>(c, c->lay.inv_r);
    double* dd = wsp<double>(c, c->lay.inv_dd);
    double* rtry = wsp<double>(c, c->lay.inv_try);
    double* scal = wsp<double>(c, c->lay.inv_scal);
    double* part = wsp<double>(c, c->lay.dot_partial);
    double* alpha = wsp<double>(c, c->lay.cg_x);
    auto apply_G = [&](const double* u, double* d) {
        return mode == GRAV_MATRIX_FREE ? grav_forward(c, u, d, stream) : grav_forward_stored(c, u, d, stream);
    };
    // ||out||^2 with out = a - t b (b may be NULL), summed over ranks when sharded; synchronises
    auto norm2 = [&](const double* a_, double t, const double* b_, double* out, double* val) -> grav_status {
        CK(launch_inv_residual(c, a_, t, b_, out, part, s), "inv_residual");
        grav_status e = exchange(c, part, kDotBlocks, s);
        if (e) return e;
        CK(launch_inv_finish(c, part, scal, s), "inv_finish");
        CK(cudaMemcpyAsync(val, scal, sizeof(double), cudaMemcpyDeviceToHost, s), "D2H norm");
        CK(cudaStreamSynchronize(s), "sync");
        return GRAV_OK;
    };
    double nd2 = 0.0, nr2 = 0.0;
    if ((st = norm2(dobs, 0.0, nullptr, nullptr, &nd2))) return st;
    if (mref) {
        CK(cudaMemcpyAsync(m, mref, g.M * sizeof(double), cudaMemcpyDeviceToDevice, s), "copy m_ref");
        if ((st = apply_G(m, dd))) return st;
        if ((st = norm2(dobs, 1.0, dd, r, &nr2))) return st;
    } else {
        CK(cudaMemsetAsync(m, 0, g.M * sizeof(double), s), "zero m");
        if ((st = norm2(dobs, 0.0, nullptr, r, &nr2))) return st;
    }
    const double dn = nd2 > 0.0 ? std::sqrt(nd2) : 1.0;
    if (hist_host) hist_host[0] = std::sqrt(nr2) / dn;
    int k = 0;
    for (; k < max_outer; ++k) {
        if (std::sqrt(nr2) / dn <= tol_outer) break;
        st = grav_dataspace_cg(c, r, w, lambda, max_inner, tol_inner, mode, precond, nullptr, alpha, dm, nullptr, nullptr, stream);
        if (st) return st;
        if (inner_host)     // ordered on the stream; read after the first trial's synchronisation
            CK(cudaMemcpyAsync(inner_host + k, &wsp<CgScalars>(c, c->lay.scalars)->iters_done, sizeof(int),
                               cudaMemcpyDeviceToHost, s), "D2H inner iterations");
        if ((st = apply_G(dm, dd))) return st;
        double step = 1.0, n2 = 0.0;
        bool ok = false;
        for (int h = 0; h <= 10; ++h, step *= 0.5) {
            if ((st = norm2(r, step, dd, rtry, &n2))) return st;
            if (n2 < nr2) { ok = true; break; }
        }
        if (step_host) step_host[k] = ok ? step : 0.0;
        if (!ok) break;                                   // no decrease along delta_m: stop with m_k
        CK(launch_inv_axpy(c, step, dm, m, s), "inv_axpy");
        CK(cudaMemcpyAsync(r, rtry, g.N * sizeof(double), cudaMemcpyDeviceToDevice, s), "copy r");
        nr2 = n2;
        if (hist_host) hist_host[k + 1] = std::sqrt(nr2) / dn;
    }
    if (n_outer_host) *n_outer_host = k;
    if (dpred) {    // d_pred = d_obs - r
        CK(launch_inv_residual(c, dobs, 1.0, r, dpred, part, s), "inv_residual");
    }
    return GRAV_OK;
}

// ---- host-buffer (end-to-end) variants ---------------------------------------------------------------------
grav_status grav_forward_host(grav_ctx* c, const double* u_host, double* d_host, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!u_host || !d_host) return fail(GRAV_EINVAL, "NULL vector");
    DeviceGuard dg(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    double* um = wsp<double>(c, c->lay.stage_m);
    double* dn = wsp<double>(c, c->lay.stage_n);
    CK(cudaMemcpyAsync(um, u_host, c->g.M * sizeof(double), cudaMemcpyHostToDevice, s), "H2D u");
    st = grav_forward(c, um, dn, stream);
    if (st) return st;
    CK(cudaMemcpyAsync(d_host, dn, c->g.N * sizeof(double), cudaMemcpyDeviceToHost, s), "D2H d");
    CK(cudaStreamSynchronize(s), "sync");
    return GRAV_OK;
}

grav_status grav_adjoint_host(grav_ctx* c, const double* v_host, double* g_host, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!v_host || !g_host) return fail(GRAV_EINVAL, "NULL vector");
    DeviceGuard dg(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    double* gm = wsp<double>(c, c->lay.stage_m);
    double* vn = wsp<double>(c, c->lay.stage_n);
    CK(cudaMemcpyAsync(vn, v_host, c->g.N * sizeof(double), cudaMemcpyHostToDevice, s), "H2D v");
    st = grav_adjoint(c, vn, gm, stream);
    if (st) return st;
    CK(cudaMemcpyAsync(g_host, gm, c->g.M * sizeof(double), cudaMemcpyDeviceToHost, s), "D2H g");
    CK(cudaStreamSynchronize(s), "sync");
    return GRAV_OK;
}

grav_status grav_dataspace_cg_host(grav_ctx* c, const double* dobs_host, double beta, double z0, double lambda,
                                   int iters, double rtol, int mode, double* alpha_host, double* m_host,
                                   double* hist_host, void* stream) {
    grav_status st = check_ready(c);
    if (st) return st;
    if (!dobs_host || !alpha_host) return fail(GRAV_EINVAL, "NULL vector");
    if (iters < 0 || iters + 1 > 4096) return fail(GRAV_EINVAL, "iters must be in [0, 4095] for the host variant");
    DeviceGuard dg(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    double* w = wsp<double>(c, c->lay.cg_w);
    double* mm = wsp<double>(c, c->lay.stage_m);
    double* dn = wsp<double>(c, c->lay.stage_n);
    double* hh = wsp<double>(c, c->lay.stage_hist);
    CK(cudaMemcpyAsync(dn, dobs_host, c->g.N * sizeof(double), cudaMemcpyHostToDevice, s), "H2D dobs");
    st = grav_depth_weights(c, beta, z0, w, stream);
    if (st) return st;
    // alpha is produced in the CG's own x buffer and copied out from there
    double* x = wsp<double>(c, c->lay.cg_x);
    st = grav_dataspace_cg(c, dn, w, lambda, iters, rtol, mode, nullptr, nullptr, x, m_host ? mm : nullptr,
                           hist_host ? hh : nullptr, nullptr, stream);
    if (st) return st;
    CK(cudaMemcpyAsync(alpha_host, x, c->g.N * sizeof(double), cudaMemcpyDeviceToHost, s), "D2H alpha");
    if (m_host) CK(cudaMemcpyAsync(m_host, mm, c->g.M * sizeof(double), cudaMemcpyDeviceToHost, s), "D2H m");
    if (hist_host) CK(cudaMemcpyAsync(hist_host, hh, (iters + 1) * sizeof(double), cudaMemcpyDeviceToHost, s), "D2H hist");
    CK(cudaStreamSynchronize(s), "sync");
    return GRAV_OK;
}

}  // extern "C"

// ---- FP64 pipe peak probe ----------------------------------------------------------------------------------
namespace {
__global__ void __launch_bounds__(256) dfma_probe_kernel(double* out, int iters, double seed) {
    double a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 1.0000001, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    double sres = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (sres == 12345.678) out[0] = sres;   // never true; keeps the chain alive
}
}  // namespace

extern "C" grav_status grav_fp64_peak_probe(int device, int iters, double* ninstr, double* ms) {
    if (!ninstr || !ms || iters <= 0) return fail(GRAV_EINVAL, "bad argument");
    DeviceGuard dg(device);
    if (!dg.ok) return fail(GRAV_ECUDA, "cudaSetDevice failed");
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, device), "cudaGetDeviceProperties");
    double* out = nullptr;
    CK(cudaMalloc(&out, 8), "cudaMalloc");
    const int blocks = prop.multiProcessorCount * 8;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    dfma_probe_kernel<<<blocks, 256>>>(out, iters / 10 + 1, 1.0);   // warm-up
    cudaEventRecord(e0);
    dfma_probe_kernel<<<blocks, 256>>>(out, iters, 1.0);
    cudaEventRecord(e1);
    cudaError_t e = cudaEventSynchronize(e1);
    float t = 0.f;
    cudaEventElapsedTime(&t, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    if (e != cudaSuccess) return cuda_fail(e, "dfma probe");
    *ninstr = (double)blocks * 256.0 * 8.0 * (double)iters;
    *ms = t;
    return GRAV_OK;
}
