// fp64_math.cuh -- branch-free FP64 rsqrt and exp(x <= 0) for the Yukawa kernel
//   G_k(r) = exp(-k r) / (4 pi r)        (Eq. (18), north_star)
// tuned for the sm_100a FP64 pipe (64 lanes/SM: one warp-wide DFMA per 2 cycles per SM
// sub-partition, so every non-FP64 instruction -- MUFU seed, LDS table look-up, integer
// exponent insertion -- issues in the FP64 pipe's shadow and is free).
//
// Accuracy target: <= ~1.5 ulp per kernel value (the parity tolerances are 1e-13 / 1e-12
// relative 2-norm on sums of 1e4..1e6 terms).
//
//   rsqrt: MUFU.RSQ64H seed (rel. error <~ 2^-20) + one cubic (Halley-type) step,
//          5 FP64 instructions, residual 5 e^3/16 < 2^-58.
//   exp:   x = 16 n' ... exp(x) = 2^n * 2^(j/16) * p(r),  n16 = rint(x * 16/ln2) = 16 n + j,
//          r = x - n16 ln2/16, |r| <= ln2/32, p = degree-6 near-minimax polynomial
//          (max rel. error 7.6e-18 in exact arithmetic), 2^(j/16) from a 16-entry shared-memory
//          table (16 x 8 B = 32 banks: conflict-free), 2^n by integer add into the exponent field.
//          4 + 6 + 1 = 11 FP64 instructions.  Argument must satisfy -2^30 < x <= 0 (x = -k r);
//          results below 2^-1022 are clamped to ~2^-1022 (absolute error < 1e-307).
//   Coefficients: Chebyshev-node interpolant of exp on [-ln2/32, ln2/32] computed in 60-digit
//   arithmetic and rounded to double; T16[j] = 2^(j/16) correctly rounded.
#pragma once
#include <cuda_runtime.h>

namespace bltc {

__device__ __constant__ const double kExpT16[16] = {
    0x1.0000000000000p+0, 0x1.0b5586cf9890fp+0, 0x1.172b83c7d517bp+0, 0x1.2387a6e756238p+0,
    0x1.306fe0a31b715p+0, 0x1.3dea64c123422p+0, 0x1.4bfdad5362a27p+0, 0x1.5ab07dd485429p+0,
    0x1.6a09e667f3bcdp+0, 0x1.7a11473eb0187p+0, 0x1.8ace5422aa0dbp+0, 0x1.9c49182a3f090p+0,
    0x1.ae89f995ad3adp+0, 0x1.c199bdd85529cp+0, 0x1.d5818dcfba487p+0, 0x1.ea4afa2a490dap+0};

#define BLTC_EXP_16_OVER_LN2 0x1.71547652b82fep+4
#define BLTC_EXP_LN2_OVER_16 0x1.62e42fefa39efp-5
#define BLTC_EXP_MAGIC 6755399441055744.0 /* 1.5 * 2^52 */
#define BLTC_EXP_C1 0x1.000000000000ap+0
#define BLTC_EXP_C2 0x1.0000000000003p-1
#define BLTC_EXP_C3 0x1.5555555405047p-3
#define BLTC_EXP_C4 0x1.55555554ad2d0p-5
#define BLTC_EXP_C5 0x1.11126efea4abcp-7
#define BLTC_EXP_C6 0x1.6c181f5984fddp-10

// Copy the table to shared memory (call from the first 16 threads, then __syncthreads()).
__device__ __forceinline__ void exp_table_init(double* t16_smem, int tid) {
    if (tid < 16) t16_smem[tid] = kExpT16[tid];
}

// MUFU.RSQ64H: approximate 1/sqrt from the high word only.
__device__ __forceinline__ double rsqrt_seed(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}

// rinv = 1/sqrt(r2), r = sqrt(r2).  ZERO_SAFE: r2 == 0 gives rinv = 0, r = 0 (the singular
// term "is skipped") via one integer compare + select on the seed's high word.
template <bool ZERO_SAFE>
__device__ __forceinline__ void rsqrt_sqrt(double r2, double& rinv, double& r) {
    double y0 = rsqrt_seed(r2);
    if (ZERO_SAFE) {
        int hi = __double2hiint(y0);
        hi = (hi == 0x7ff00000) ? 0 : hi;          // +inf (r2 == 0)  ->  +0
        y0 = __hiloint2double(hi, __double2loint(y0));
    }
    double t = r2 * y0;                 // ~ sqrt(r2)
    double e = fma(-t, y0, 1.0);        // 1 - r2 y0^2
    double p = fma(0.375, e, 0.5);
    double ye = y0 * e;
    rinv = fma(ye, p, y0);              // y0 (1 + e/2 + 3 e^2/8)
    r = r2 * rinv;
}

// exp(x) for -2^30 < x <= 0.  t16: shared-memory copy of kExpT16.
__device__ __forceinline__ double exp_neg(double x, const double* __restrict__ t16) {
    double t = fma(x, BLTC_EXP_16_OVER_LN2, BLTC_EXP_MAGIC);
    int n16 = __double2loint(t);                    // rint(x * 16/ln2), two's complement
    double nf = t - BLTC_EXP_MAGIC;
    double r = fma(nf, -BLTC_EXP_LN2_OVER_16, x);
    double tj = t16[n16 & 15];
    double p = fma(BLTC_EXP_C6, r, BLTC_EXP_C5);
    p = fma(p, r, BLTC_EXP_C4);
    p = fma(p, r, BLTC_EXP_C3);
    p = fma(p, r, BLTC_EXP_C2);
    p = fma(p, r, BLTC_EXP_C1);
    double s = tj * r;
    double e = fma(s, p, tj);                       // tj * (1 + r p(r))
    int n = max(n16 >> 4, -1022);                   // clamp: result stays a normal number
    return __hiloint2double(__double2hiint(e) + (n << 20), __double2loint(e));
}

}  // namespace bltc
