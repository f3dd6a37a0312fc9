// nodeops.cu -- the exact regrouping between prisms and mesh nodes, and the depth weights.
//
// Eq. 1 sums Psi over the 8 corners of every prism with sign sigma = (-1)^(p+q+r).  On a
// rectilinear mesh a corner of one prism is a corner of up to 8 prisms, so
//     d_i = gamma sum_k u_k sum_pqr sigma Psi(corner_pqr(k) - obs_i) = gamma sum_n c_n Psi(node_n - obs_i),
//     c = S^T u,   S = M x Nn signed corner incidence,
// and (G^T v)_k = gamma sum_pqr sigma T[corner_pqr(k)],  T_n = sum_i v_i Psi(node_n - obs_i)   (g = gamma S T).
// These two kernels are S^T (cell_to_node) and S (node_to_cell); both are HBM-trivial gathers.
//
// Corner p=1 is the lower coordinate (node a = i), p=2 the upper (a = i+1):  sigma = (-1)^(p+q+r)
// = -(-1)^(da+db+dc) with d* = node index - cell index in {0,1}.
#include "grav_internal.cuh"

namespace grav {

__global__ void cell_to_node_kernel(Geom g, const double* __restrict__ u, const double* __restrict__ w,
                                    double* __restrict__ cnode) {
    long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= g.Nn) return;
    int c = (int)(n % g.nzp);
    long long t = n / g.nzp;
    int b = (int)(t % g.nyp);
    int a = (int)(t / g.nyp);
    double acc = 0.0;
#pragma unroll
    for (int da = 0; da < 2; ++da) {
        int i = a - da;
        if (i < 0 || i >= g.nx) continue;
#pragma unroll
        for (int db = 0; db < 2; ++db) {
            int j = b - db;
            if (j < 0 || j >= g.ny) continue;
#pragma unroll
            for (int dc = 0; dc < 2; ++dc) {
                int k = c - dc;
                if (k < 0 || k >= g.nz) continue;
                long long cell = ((long long)i * g.ny + j) * g.nz + k;
                double val = u[cell];
                if (w) { double ww = w[cell]; val = val / (ww * ww); }
                // sigma = -(-1)^(da+db+dc)
                acc += ((da + db + dc) & 1) ? val : -val;
            }
        }
    }
    // stored with the node depth beside it, so that the forward z-loop needs ONE 16-byte load per evaluation
    reinterpret_cast<double2*>(cnode)[n] = make_double2(acc, g.zn[c]);
}

// tnode holds T as two planes [hi | lo] of Nn doubles (adjoint.cu).
__global__ void node_to_cell_kernel(Geom g, const double* __restrict__ tnode, const double* __restrict__ w,
                                    double scale, double* __restrict__ gcell) {
    long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= g.M) return;
    int k = (int)(cell % g.nz);
    long long t = cell / g.nz;
    int j = (int)(t % g.ny);
    int i = (int)(t / g.ny);
    // fixed summation order: pair the two z-corners of each (p,q) edge first (their Psi values are closest)
    double acc = 0.0, accl = 0.0;
#pragma unroll
    for (int da = 0; da < 2; ++da)
#pragma unroll
        for (int db = 0; db < 2; ++db) {
            long long base = ((long long)(i + da) * g.nyp + (j + db)) * g.nzp + k;
            // sigma(da,db,dc) = -(-1)^(da+db+dc):  dc=0 -> -(-1)^(da+db), dc=1 -> +(-1)^(da+db)
            double e = tnode[base + 1] - tnode[base];                    // high parts: close values, exact difference
            double el = tnode[g.Nn + base + 1] - tnode[g.Nn + base];      // low parts (adjoint.cu "Accumulation")
            acc += ((da + db) & 1) ? -e : e;
            accl += ((da + db) & 1) ? -el : el;
        }
    double val = scale * (acc + accl);
    if (w) { double ww = w[cell]; val = val / (ww * ww); }
    gcell[cell] = val;
}

// w_k = (zc_k + z0)^(-beta/2)   (BASELINE.json north_star).  Depends on the layer only.
__global__ void depth_weights_kernel(Geom g, double beta, double z0, double* __restrict__ w) {
    long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= g.M) return;
    int k = (int)(cell % g.nz);
    double zc = 0.5 * (g.zn[k] + g.zn[k + 1]) - g.zn[0];
    w[cell] = pow(zc + z0, -0.5 * beta);
}

static inline unsigned blocks_for(long long n, int tpb) { return (unsigned)((n + tpb - 1) / tpb); }

cudaError_t launch_cell_to_node(grav_ctx* c, const double* u, const double* w, double* cnode, cudaStream_t s) {
    cell_to_node_kernel<<<blocks_for(c->g.Nn, 256), 256, 0, s>>>(c->g, u, w, cnode);
    c->launches++;
    return cudaGetLastError();
}
cudaError_t launch_node_to_cell(grav_ctx* c, const double* tnode, const double* w, double scale, double* gcell,
                                cudaStream_t s) {
    node_to_cell_kernel<<<blocks_for(c->g.M, 256), 256, 0, s>>>(c->g, tnode, w, scale, gcell);
    c->launches++;
    return cudaGetLastError();
}
cudaError_t launch_depth_weights(grav_ctx* c, double beta, double z0, double* w, cudaStream_t s) {
    depth_weights_kernel<<<blocks_for(c->g.M, 256), 256, 0, s>>>(c->g, beta, z0, w);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace grav
