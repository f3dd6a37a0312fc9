// psi2.cuh -- second-generation device evaluator of Psi(X,Y,Z) = Z atan(XY/(ZR)) - X ln(R+Y) - Y ln(R+X)
// (Eq. 2-3), designed from B200 measurements (profiles/r1_fp64_issue_microbench.md):
//   * a half-rate FP64 instruction costs 2 scheduler cycles and every other instruction ~1 more, even when the
//     FP64 pipe is the only busy pipe, so the evaluator minimises  2 x (#FP64) + (#other)  per evaluation;
//   * DFMA latency is 8 cycles, I2F.F64 and LDS are free next to a DFMA stream, IMAD.HI is quarter rate.
// Same value as psi_fast of psi.cuh (same exactly-cancelling k0 offset, same guards of reading C6), different
// instruction mix:
//   sqrt : MUFU.RSQ64H seed y0, two Newton steps on g ~ sqrt(S) that share h0 = y0/2:
//          g1 = g0 + (S - g0^2) h0, R = g1 + (S - g1^2) h0  (relative error <= 2^-53 + 2^-59).
//   ln   : table entry (invc', logc) indexed by the top 8 mantissa bits; the power of two of the argument is folded
//          into invc by ONE integer multiply-add on its high word (invc 2^-e), so r = fma(a, invc 2^-e, -1) needs no
//          mantissa extraction; the exponent becomes a double by I2F (XU pipe, idle otherwise), not by FP64 adds.
//   atan : angle = atan2(n, d), n = |XY|, d = |Z| R, WITHOUT the min/max swap of psi.cuh:  q = n/(n+d) in [0,1] from
//          a MUFU.RCP64H seed, j = round(K q), direction (c_j, 1-c_j), c_j = j/K exactly, A_j = atan2(c_j, 1-c_j),
//          t = tan(angle - A_j) = (n - c_j (n+d)) / (d + c_j (n-d)),  |angle - A_j| <= 2 |q - c_j| <= 1/K + 2^-19
//          (d angle/dq = (cos + sin)^2 in [1, 2]), one true division, odd Taylor polynomial of atan t.
//          K = 256: |t| <= 2^-8 (1 + 2^-11), Taylor to t^5, truncation t^7/7 <= 2.1e-18.
// The same source compiles for the host with the MUFU seeds emulated (tests/test_fastmath_host.py).
#pragma once
#include "psi.cuh"

namespace grav {

#ifndef GRAV_LOG2BITS
#define GRAV_LOG2BITS 8
#endif
constexpr int kLog2Bits = GRAV_LOG2BITS;        // 8: |r| <= 2^-9, Taylor to r^5;  10: |r| <= 2^-11, Taylor to r^4
constexpr int kLog2N = 1 << kLog2Bits;          // mantissa intervals
constexpr int kAtan2K = 256;                    // c_j = j / 256, j = 0..256
constexpr int kAtan2N = kAtan2K + 2;            // +1 slack entry for the seed's 2^-20 error at q = 1
constexpr int kTab2Entries = kLog2N + kAtan2N;  // log entries first, then atan entries
constexpr size_t kTab2SmemBytes = (size_t)kTab2Entries * kRep * sizeof(double2);

struct Psi2TablesHost {
    double2 e[kTab2Entries];   // [0,256): (invc', logc);  [256, 256+258): (c_j, A_j)
};

// Host-side generator (long double libm); the CUDA path's own, the oracle has none.  The log entries depend on the
// context's exponent offset k0: invc' has its exponent field lowered by k0, so that the device forms
// invc 2^-(e'+k0) = invc' with e' = biased_exponent(a) - 1023 - k0 subtracted from its exponent field.
inline void psi2_tables_generate(Psi2TablesHost* t, int k0) {
    for (int i = 0; i < kLog2N; ++i) {
        long double centre = 1.0L + ((long double)i + 0.5L) / (long double)kLog2N;
        double invc = (double)(1.0L / centre);
        uint64_t u; memcpy(&u, &invc, 8);
        u -= (uint64_t)((int64_t)k0 << 52);
        double invc_b; memcpy(&invc_b, &u, 8);
        t->e[i].x = invc_b;
        t->e[i].y = (double)(-logl((long double)invc));
    }
    const long double half_pi = acosl(-1.0L) / 2.0L;
    for (int j = 0; j < kAtan2N; ++j) {
        int jj = j <= kAtan2K ? j : kAtan2K;      // slack entry repeats the last one
        double c = (double)jj / (double)kAtan2K;
        long double a = (jj == kAtan2K) ? half_pi : atan2l((long double)c, (long double)(1.0 - c));
        t->e[kLog2N + j].x = c;
        t->e[kLog2N + j].y = (double)a;
    }
}

// Constants that are NOT exactly representable in the 32 high bits travel as kernel parameters; the others
// (-1/2, -1/4, 1/2, 1, K, 1.5 2^52) are written as literals and become FP64 immediates.
struct Psi2Consts {
    double ln2;
    double l3, l5;       // 1/3, 1/5       (ln(1+r) Taylor)
    double a3, a5;       // -1/3, 1/5      (atan Taylor)
    int ebias;           // 1023 + k0
    int pad;
};
inline Psi2Consts psi2_consts_make(int k0) {
    Psi2Consts c;
    c.ln2 = 0.69314718055994529;
    c.l3 = 0.33333333333333331; c.l5 = 0.2;
    c.a3 = -0.33333333333333331; c.a5 = 0.2;
    c.ebias = 1023 + k0;
    c.pad = 0;
    return c;
}

struct Psi2TabView {
    const double2* base;   // already offset by the thread's copy; entry i at base[i << shift]
    int shift;
    Psi2Consts k;
    const double2* atan_base;   // first atan entry of the thread's copy; entry j at atan_base[j << shift]
    const char* log2d;     // LOG2D variant: single-copy table indexed by exponent AND mantissa, pre-offset so that
                           // the entry of a sits at log2d + ((hi_word(a) & 0xfffff000) >> 8); NULL otherwise
};

// LOG2D variant (shipped where admissible; profiles/r1_tail_and_variants.md): one table over every binade the
// arguments can reach, entry = (invc 2^-e, logc + (e - k0) ln2): no exponent extraction, no I2F, no scaling of invc,
// one FP64 instruction fewer per logarithm - 44 FP64 + 16 other instructions per evaluation instead of 46 + 23.
// The price is 4 KB of shared memory per binade and a single copy: the lanes of a warp collide on banks (ncu: the L1
// data stage goes from 46 % to 97 % busy in the forward kernel), yet the kernels are 9 % faster overall, also with
// random stations; handing the stations over in Z-curve order changes the forward time by only -0.5 %.
// Valid only when every argument lies in the tabulated binades: a = R + Y obeys Zmin^2 / (2 Rmax) <= a <= 2 Rmax;
// the context checks that from the geometry (grav_api.cu) and otherwise keeps the 256-entry evaluator, whose guards
// (reading C6) also cover Z = 0 and a = 0.
constexpr int kLog2dMaxBinades = 40;          // 160 KB; arguments may span a ratio of 2^40
inline void psi2_log2d_generate(double2* out, int k0, int emin, int nb) {
    const long double ln2 = logl(2.0L);
    for (int b = 0; b < nb; ++b) {
        const int e = emin + b;                       // unbiased exponent of the argument
        for (int i = 0; i < 256; ++i) {
            long double centre = 1.0L + ((long double)i + 0.5L) / 256.0L;
            double invc = (double)(1.0L / centre);
            out[b * 256 + i].x = ldexp(invc, -e);
            out[b * 256 + i].y = (double)(-logl((long double)invc) + (long double)(e - k0) * ln2);
        }
    }
}
GRAV_HOSTDEV double log2d_fast(const Psi2TabView& tb, double a) {
    const unsigned m = (unsigned)hi_word(a) & 0xfffff000u;
#ifdef __CUDA_ARCH__
    const double2 ent = *reinterpret_cast<const double2*>(tb.log2d + __umulhi(m, 1u << 24));
#else
    const double2 ent = *reinterpret_cast<const double2*>(tb.log2d + (m >> 8));
#endif
    const double r = fma(a, ent.x, -1.0);
    const double r2 = r * r;
    double q = fma(r, tb.k.l5, -0.25);
    q = fma(q, r, tb.k.l3);
    q = fma(q, r, -0.5);
    const double p = fma(r2, q, r);
    return ent.y + p;
}

// ln(a / 2^k0) for 0 < a < 2^1000 (finite garbage for a == 0: reading C6, the caller multiplies it by an exact 0).
GRAV_HOSTDEV double log2_fast(const Psi2TabView& tb, double a) {
    const int hw = hi_word(a);
    const unsigned mbits = (unsigned)hw & (0x000fffffu & ~((1u << (20 - kLog2Bits)) - 1u));   // top mantissa bits
#ifdef __CUDA_ARCH__
    // byte offset = idx * (16 << shift) = mbits >> (12 - 4 - shift): one shift-and-add on top of the base address
    // written as a high multiply by a power of two so that ptxas folds shift and base add into one LEA.HI
    const double2 ent = *reinterpret_cast<const double2*>(reinterpret_cast<const char*>(tb.base) +
                                                          __umulhi(mbits, 1u << (32 - (20 - kLog2Bits - 4 - kRepShift))));
#else
    const double2 ent = tb.base[(mbits >> (20 - kLog2Bits)) << tb.shift];
#endif
    const int e = (hw >> 20) - tb.k.ebias;                                   // a > 0: sign bit clear
    const double invc = make_double(hi_word(ent.x) - (e << 20), lo_word(ent.x));   // invc 2^-(e + k0): one IMAD
#ifdef __CUDA_ARCH__
    const double ed = __int2double_rn(e);                                    // I2F.F64.S32
#else
    const double ed = (double)e;
#endif
    const double r = fma(a, invc, -1.0);
    const double r2 = r * r;
    double q;
    if (kLog2Bits >= 10) {
        q = fma(r, -0.25, tb.k.l3);          // truncation r^5/5 <= 2^-55/5 = 5.5e-18
    } else {
        q = fma(r, tb.k.l5, -0.25);          // truncation r^6/6 <= 2^-54/6 = 9.3e-18
        q = fma(q, r, tb.k.l3);
    }
    q = fma(q, r, -0.5);
    const double p = fma(r2, q, r);
    const double base = fma(ed, tb.k.ln2, ent.y);
    return base + p;
}

// Returns s * Psi(X, Y, Z) (+ the exactly-cancelling k0 offset), s = sign(XY); col from psi_column (psi.cuh).
template <bool LOG2D>
GRAV_HOSTDEV double psi2_fast_t(const Psi2TabView& tb, const PsiColumn& col, double Z) {
    // ---- R = sqrt(X^2 + Y^2 + Z^2)
    const double S = fma(Z, Z, col.Q);
    const double y0 = rsqrt_seed(S);
    const double g0 = S * y0;
    const double h0 = y0 * 0.5;
    const double res0 = fma(-g0, g0, S);
    const double g1 = fma(res0, h0, g0);
    const double res1 = fma(-g1, g1, S);
    const double R = fma(res1, h0, g1);
    // ---- logarithms
    const double L1 = LOG2D ? log2d_fast(tb, R + col.Y) : log2_fast(tb, R + col.Y);
    const double L2 = LOG2D ? log2d_fast(tb, R + col.X) : log2_fast(tb, R + col.X);
    // ---- angle = atan2(|XY|, |Z| R) in [0, pi/2]
    const double n = col.nXY;
    const double az = fabs(Z);
    const double d = az * R;
    const double sum = n + d;
    const double dif = n - d;
    const double q0 = n * rcp_seed(sum);
    const double jm = fma(q0, (double)kAtan2K, 6755399441055744.0);   // 1.5 * 2^52: low word = round(K q0)
    const int j = lo_word(jm);
    const double2 ent = tb.atan_base[j << tb.shift];
    const double num = fma(-ent.x, sum, n);
    const double den = fma(ent.x, dif, d);
    // t = num / den = num yd / (1 - e1) = num yd (1 + e1 + e1^2 + O(2^-60)),  e1 = 1 - den yd ~ 2^-20
    const double yd = rcp_seed(den);
    const double e1 = fma(-den, yd, 1.0);
    const double t0 = num * yd;
    const double e2 = fma(e1, e1, e1);
    const double t = fma(t0, e2, t0);
    const double t2 = t * t;
    const double pa = fma(t2, tb.k.a5, tb.k.a3);
    const double w = fma(t * t2, pa, t);
    const double angle = ent.y + w;
    // ---- s Psi = |Z| angle - (sX) L1 - (sY) L2
    double out = az * angle;
    out = fma(-col.sX, L1, out);
    out = fma(-col.sY, L2, out);
    return out;
}

GRAV_HOSTDEV double psi2_fast(const Psi2TabView& tb, const PsiColumn& col, double Z) {
    return psi2_fast_t<false>(tb, col, Z);
}

#ifdef __CUDACC__
struct Psi2Dev {
    const double2* tab;     // kTab2Entries entries in global memory
    Psi2Consts k;
    const double2* tab2d;   // LOG2D variant: nb2d * 256 entries in global memory, or NULL when the geometry rules it out
    int nb2d;               // binades tabulated
    int emin2d_biased;      // biased exponent of the first binade
};
__device__ __forceinline__ Psi2TabView psi2_tables_to_smem(double2* s_tab, const Psi2Dev& pd) {
    for (int e = threadIdx.x; e < kTab2Entries * kRep; e += blockDim.x) s_tab[e] = pd.tab[e >> kRepShift];
    __syncthreads();
    Psi2TabView v;
    v.base = s_tab + (threadIdx.x & (kRep - 1));
    v.shift = kRepShift;
    v.k = pd.k;
    v.atan_base = v.base + (kLog2N << kRepShift);
    v.log2d = nullptr;
    return v;
}
// LOG2D layout: [atan entries, kRep interleaved copies][2-D log table, one copy, pd.nb2d * 256 entries]
constexpr size_t kAtan2SmemBytes = (size_t)kAtan2N * kRep * sizeof(double2);
__device__ __forceinline__ size_t psi2_log2d_smem_entries(const Psi2Dev& pd) {
    return (size_t)kAtan2N * kRep + (size_t)pd.nb2d * 256;
}
__device__ __forceinline__ Psi2TabView psi2_tables_to_smem_2d(double2* s_tab, const Psi2Dev& pd) {
    for (int e = threadIdx.x; e < kAtan2N * kRep; e += blockDim.x) s_tab[e] = pd.tab[kLog2N + (e >> kRepShift)];
    double2* s_2d = s_tab + kAtan2N * kRep;
    for (int e = threadIdx.x; e < pd.nb2d * 256; e += blockDim.x) s_2d[e] = pd.tab2d[e];
    __syncthreads();
    Psi2TabView v;
    v.base = nullptr;
    v.shift = kRepShift;
    v.k = pd.k;
    v.atan_base = s_tab + (threadIdx.x & (kRep - 1));
    v.log2d = reinterpret_cast<const char*>(s_2d) - ((size_t)pd.emin2d_biased << 12);
    return v;
}
#endif

}  // namespace grav
