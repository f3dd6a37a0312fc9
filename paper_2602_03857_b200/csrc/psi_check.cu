// psi_check.cu -- the device Psi evaluators on caller-supplied arguments, one evaluation per thread (diagnostic).
//
// Lets the tests compare every evaluator that ships in the kernels - table-driven FP64 with either log table, CUDA
// libm FP64, Float32 - with the oracle's Psi(X, Y, Z) (Eq. 2-3) argument by argument ON THE DEVICE,
// MUFU seeds and all, instead of only through sums over a mesh.
#include "grav_internal.cuh"
#include "psi.cuh"

namespace grav {

// variant 0: psi_eval, 256-entry log table; 1: psi_libm; 2: psi_f32; 3: psi_eval, 2-D log table.
// Variants 0, 2 and 3 return Psi + (X + Y) k0' ln 2 (the exactly-cancelling offset; k0' = k0, clamped to +-100 for 2).
template <int VARIANT>
__global__ void __launch_bounds__(256) psi_check_kernel(PsiDev pd, long long n, const double* __restrict__ X,
                                                         const double* __restrict__ Y, const double* __restrict__ Z,
                                                         double* __restrict__ out) {
    extern __shared__ double2 s_tab[];
    __shared__ float s_at[kAtanN32];
    if (VARIANT == 2) psi_f32_atan_table(s_at, pd);
    PsiTabView tb;
    if (VARIANT == 0) tb = psi_tables_to_smem(s_tab, pd);
    if (VARIANT == 3) tb = psi_tables_to_smem_2d(s_tab, pd);
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256) {
        const double x = X[i], y = Y[i], z = Z[i];
        double v;
        if (VARIANT == 1) v = psi_libm(x, y, z, x * y, fma(y, y, x * x));
        else if (VARIANT == 2) v = (double)psi_f32((float)x, (float)y, (float)z, psi_f32_inv_scale(pd.k0), s_at);
        else {
            const PsiColumn pc = psi_column(x, y);
            v = pc.s * psi_eval<VARIANT == 3>(tb, pc, z);
        }
        out[i] = v;
    }
}

cudaError_t launch_psi_check(grav_ctx* c, int variant, long long n, const double* X, const double* Y, const double* Z,
                             double* out, cudaStream_t s) {
    const unsigned blocks = (unsigned)((n + 255) / 256 < 1184 ? (n + 255) / 256 : 1184);
    static unsigned long long set0 = 0, set3 = 0;
    cudaError_t e = cudaSuccess;
    if (variant == 0) {
        e = ensure_dynamic_smem(psi_check_kernel<0>, kTabSmemBytes, c->device, &set0);
        if (e == cudaSuccess) psi_check_kernel<0><<<blocks, 256, kTabSmemBytes, s>>>(c->pd, n, X, Y, Z, out);
    } else if (variant == 1) {
        psi_check_kernel<1><<<blocks, 256, 0, s>>>(c->pd, n, X, Y, Z, out);
    } else if (variant == 2) {
        psi_check_kernel<2><<<blocks, 256, 0, s>>>(c->pd, n, X, Y, Z, out);
    } else {
        e = ensure_dynamic_smem(psi_check_kernel<3>, psi_smem_max<true>(), c->device, &set3);
        if (e == cudaSuccess)
            psi_check_kernel<3><<<blocks, 256, psi_smem_bytes<true>(c->pd), s>>>(c->pd, n, X, Y, Z, out);
    }
    c->launches++;
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace grav
