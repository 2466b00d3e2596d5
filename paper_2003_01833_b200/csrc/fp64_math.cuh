// fp64_math.cuh -- branch-free FP64 rsqrt and exp(x <= 0) for the Yukawa kernel
//   G_k(r) = exp(-k r) / (4 pi r)        (Eq. (18), north_star)
// tuned for the sm_100a FP64 pipe: 64 lanes/SM, one warp-wide FP64 instruction per 2 cycles per SM
// sub-partition.  Measured on B200: step time ~ 2 x (FP64 instructions) +
// (non-FP64 instructions that do not land in the shadow cycle of an FP64 issue), and FMA-pipe
// instructions (IMAD, IMAD.MOV, IMAD.SHL) cost the FP64 pipe 1-2 cycles each.  So both functions
// minimise the FP64 count AND keep their integer work on the ALU pipe (SHF / LOP3 / ISETP / SEL via
// inline PTX that ptxas cannot turn into IMAD).
//
//   rsqrt: MUFU.RSQ64H seed (XU pipe, rel. error <~ 2^-20) + one cubic step: 5 FP64 instructions,
//          residual 5 e^3/16 < 2^-58; +1 for r = r2 * rinv.
//   exp:   u = r * c,  c = -k T/ln2 (per orbital, host-computed),  T = BLTC_EXP_T = 8192 (exp_table.inc);
//          t = u + (1.5*2^52 + 1023 T)  ->  low word m = rint(u) + 1023 T = T*(n + 1023) + j
//          rho = u - rint(u) in [-1/2, 1/2];   exp(-k r) = 2^n * 2^(j/T) * (1 + rho (C1 + C2 rho))
//          2^(j/T): 64 KB shared-memory table per CTA, read by per-lane LDS.64 (random entries: ~4.4 SM cycles
//          per warp lookup against 2 conflict-free, measured; a 16-copy conflict-free table of 512 entries needs
//          the cubic polynomial again and was measured slower, tuning log);
//          2^n: the table's high words are pre-biased by -(j << 7), so adding (m << 7) -- one shift, one add,
//          both on the ALU pipe -- puts the biased exponent n + 1023 and the mantissa of 2^(j/T) in place.
//          6 FP64 instructions per exp.  Quadratic near-minimax polynomial: relative error <= 6.3e-15 (about 28
//          ulp), odd in rho and therefore of pseudo-random sign from pair to pair; the measured end-to-end parity
//          errors are 3e-16 ... 2.4e-14.  BLTC_EXP_DEG == 3 (T = 2048, cubic, 7 instructions,
//          8.6e-18) remains as a compile-time alternative: python gen_exp_table.py 2048 3 > exp_table.inc.
//          Any u <= 0 is legal: if m < 0 (exp(-k r) < 2^-1023) the high word of t differs from 0x43380000
//          and m is replaced by 0, which gives a subnormal-sized value (absolute error < 1e-307).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "exp_table.inc"

namespace bltc {

constexpr int kExpT = BLTC_EXP_T;
constexpr int kExpLog2T = BLTC_EXP_LOG2T;
constexpr int kExpTableBytes = kExpT * 8;
constexpr double kExpMagic = 6755399441055744.0 + 1023.0 * BLTC_EXP_T;   // 1.5 * 2^52 + 1023 T (exact)

__device__ const double kExpTab[BLTC_EXP_T] = {BLTC_EXP_TABLE};

// Shared-memory table: the caller provides kExpTableBytes of dynamic shared memory at `raw` (shared-window byte
// address, 16-byte aligned); entry addresses are raw + 8 j.  Call with all threads, then __syncthreads().
constexpr int kExpTableSmemBytes = kExpTableBytes;
__device__ __forceinline__ uint32_t exp_table_init(uint32_t raw, int tid, int nthreads) {
    const uint32_t base = raw;
    for (int i = tid; i < kExpT; i += nthreads) {
        const double v = kExpTab[i];
        // entry j holds the mantissa of 2^(j/T) with the high word pre-biased by -(j << (20 - log2 T)):
        // adding (m << (20 - log2 T)), m = T (n + 1023) + j, then yields 2^n 2^(j/T) with one shift-add
        const uint32_t hi = ((uint32_t)__double2hiint(v) & 0x000fffffu) - ((uint32_t)i << (20 - kExpLog2T));
        asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(base + 8u * i), "r"((uint32_t)__double2loint(v)), "r"(hi));
    }
    return base;
}

// Constants that must live in registers (an FP64 instruction takes at most one non-register operand;
// without this ptxas re-materialises them with IMAD.MOV inside the loop).  Loaded once per thread
// from values the compiler cannot see through.
struct MathRegs {
    double c375;    // 0.375
    double c2;      // BLTC_EXP_C2
    double magic;   // kExpMagic
};
__device__ __forceinline__ MathRegs math_regs_init(const double* __restrict__ opaque3) {
    MathRegs m;
    m.c375 = opaque3[0];
    m.c2 = opaque3[1];
    m.magic = opaque3[2];
    return m;
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
__device__ __forceinline__ void rsqrt_sqrt(double r2, double& rinv, double& r, const MathRegs& mr) {
    int hi = __double2hiint(rsqrt_seed(r2));
    if (ZERO_SAFE) hi = (hi == 0x7ff00000) ? 0 : hi;     // +inf (r2 == 0)  ->  +0
    uint32_t lo;
    asm("shr.u32 %0, %1, 31;" : "=r"(lo) : "r"(hi));     // = 0 (the seed is positive); an ALU-pipe "mov"
    const double y0 = __hiloint2double(hi, (int)lo);
    const double t = r2 * y0;                 // ~ sqrt(r2)
    const double e = fma(-t, y0, 1.0);        // 1 - r2 y0^2
    const double p = fma(e, mr.c375, 0.5);
    const double q = e * p;
    rinv = fma(y0, q, y0);                    // y0 (1 + e/2 + 3 e^2/8); two distinct register operands
    r = r2 * rinv;
}

// exp(-k r) given r >= 0 and c = -k T/ln2.  tab = value returned by exp_table_init.
// GUARD = false is legal only when the caller has proved k r < 708 for every pair (no underflow);
// ec = per-launch constants that live in uniform registers (kernel parameter).
struct ExpConst { double c1, c3; };
template <bool GUARD>
__device__ __forceinline__ double exp_neg_kr(double r, double c, uint32_t tab, const MathRegs& mr,
                                             const ExpConst& ec) {
    const double t = fma(r, c, mr.magic);
    const double nf = t - mr.magic;                     // rint(u), exact
    const double rho = fma(r, c, -nf);
    int m = __double2loint(t);
    if (GUARD) m = (__double2hiint(t) == 0x43380000) ? m : 0;
    // table address = tab + 8 j: the mask first, then shift and add -- ptxas fuses the last two into one LEA on the
    // ALU pipe whether `tab` sits in a uniform or (wide orbital tiles) a vector register; masking the shifted index
    // instead leaves an IMAD.IADD on the FMA pipe in the second case
    uint32_t j, j8, lo, hi;
    asm("and.b32 %0, %1, %2;" : "=r"(j) : "r"(m), "n"(BLTC_EXP_T - 1));
    asm("shf.l.wrap.b32 %0, %1, %2, 3;" : "=r"(j8) : "r"(0), "r"(j));
    asm("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(lo), "=r"(hi) : "r"(j8 + tab));
    // exponent n + 1023 merged by a shift and an add, both pinned to the ALU pipe: written as
    // hi + (m << s), ptxas emits one IMAD (m * 2^s + hi) on the FMA pipe, which steals FP64-pipe issue cycles
    uint32_t msh;
    asm("shf.l.wrap.b32 %0, %1, %2, %3;" : "=r"(msh) : "r"(0), "r"(m), "n"(20 - BLTC_EXP_LOG2T));
    const uint32_t hi2 = hi + msh;
    const double tj = __hiloint2double((int)hi2, (int)lo);   // 2^n * 2^(j/T)
#if BLTC_EXP_DEG == 3
    double p = fma(rho, ec.c3, mr.c2);
    p = fma(p, rho, ec.c1);
#else
    const double p = fma(rho, mr.c2, ec.c1);
#endif
    const double q = p * rho;
    return fma(tj, q, tj);                              // tj (1 + rho p(rho)); two distinct register operands
}

// host side: c = -k T / ln2, rounded once from extended precision
inline double exp_scale_of_k(double k) {
    return (double)(-(long double)k * (long double)BLTC_EXP_T / 0.693147180559945309417232121458176568L);
}

}  // namespace bltc
