/*
 * oracle/direct_sum.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain CPU definition of the discrete modified-Helmholtz (Yukawa) convolution of
 * treecode-accelerated Green Iteration (arXiv 2003.01833), written from the paper.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, link or call this file.  It shares no code with the CUDA path.
 *
 * What it computes (one orbital per call), O-1 in DESIGN.md:
 *
 *   S_i   = sum over sources j with r_ij != 0 of  G_k(r_ij) * w_j * (f_j - f_i)   [subtract = 1]
 *         = sum over sources j with r_ij != 0 of  G_k(r_ij) * w_j *  f_j          [subtract = 0]
 *   out_i = -2 * (S_i + f_i / k^2)   [subtract = 1, finalize = 1]
 *   out_i = -2 *  S_i                [subtract = 0, finalize = 1]
 *   out_i =  S_i                     [finalize = 0: the raw quadrature sum of Eq. (32)]
 *
 *   G_k(r) = exp(-k r) / (4 pi r)
 *
 * Citations (PAPER.md line, equation):
 *   - discrete convolution sum u_i = sum_{j != i} G(r_i, r_j) f_j w_j ......... PAPER.md:371  Eq. (32)
 *   - Green Iteration integral, kernel e^{-k r}/(2 pi r), leading minus sign,
 *     k = sqrt(-2 eps)  ==  -2 * G_k with G_k = e^{-kr}/(4 pi r) ............... PAPER.md:193  Eq. (18)
 *   - "The singular r' = r term in the quadrature sums is skipped" ............. PAPER.md:200
 *   - singularity subtraction  int (f(r') - f(r)) K + f(r) int K ............... PAPER.md:204  Eq. (20)
 *   - int e^{-k r}/r = 4 pi / k^2   (so int G_k = 1/k^2) ....................... PAPER.md:208  Eq. (21)
 *
 * Readings: R2 sign/prefactor; R3 "skipped" means r_ij == 0 exactly.
 *
 * Arithmetic: every kernel value in IEEE double with libm sqrt/exp (strict, no fast-math,
 * no FMA contraction); the sum over j is accumulated in long double so that the oracle
 * is the more accurate side of every comparison.
 *
 * kind = 0: Yukawa kernel above.
 * kind = 1: TEST kernel G(x,y) = prod_d (1 + (x_d - y_d)^m), m = (int)k: a polynomial of
 *           per-axis degree m in the source point.  It exists only so that the treecode
 *           oracle's far field can be pinned: barycentric interpolation of degree n >= m
 *           reproduces it exactly (see oracle/bltc_cpu.c and tests/test_oracle_pins.py).
 *           kind = 1 never skips a term and is only meaningful with finalize = 0.
 * kind = 2: Coulomb-type kernel 1/(4 pi r) (k ignored) -- the k -> 0 limit, used for the
 *           order-of-magnitude anchor PAPER.md:500 (Fig. 11, 2.31e-6).  finalize = 0 only.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

static double ipow(double a, int m) { double p = 1.0; for (int i = 0; i < m; ++i) p *= a; return p; }

/* value of the kernel between target (tx,ty,tz) and source (sx,sy,sz); *skip set when the
 * term is the singular one. */
double oracle_kernel(int kind, double k, double tx, double ty, double tz,
                     double sx, double sy, double sz, int* skip)
{
    double dx = tx - sx, dy = ty - sy, dz = tz - sz;
    *skip = 0;
    if (kind == 1) {
        int m = (int)k;
        return (1.0 + ipow(dx, m)) * (1.0 + ipow(dy, m)) * (1.0 + ipow(dz, m));
    }
    double r = sqrt(dx * dx + dy * dy + dz * dz);
    if (r == 0.0) { *skip = 1; return 0.0; }
    if (kind == 2) return 1.0 / (4.0 * M_PI * r);
    return exp(-k * r) / (4.0 * M_PI * r);
}

/* M targets against N sources, one orbital.  tf may be NULL iff subtract == 0.
 * Returns 0, or -1 on bad arguments. */
int oracle_direct(int kind, int64_t M, const double* tx, const double* ty, const double* tz,
                  const double* tf,
                  int64_t N, const double* sx, const double* sy, const double* sz,
                  const double* sw, const double* sf,
                  double k, int subtract, int finalize, double* out)
{
    if (M < 0 || N < 0 || !out) return -1;
    if (subtract && !tf) return -1;
    if (kind == 0 && !(k > 0.0)) return -1;
    int64_t i;
#pragma omp parallel for schedule(dynamic, 16)
    for (i = 0; i < M; ++i) {
        long double S = 0.0L;
        double fi = subtract ? tf[i] : 0.0;
        for (int64_t j = 0; j < N; ++j) {
            int skip;
            double G = oracle_kernel(kind, k, tx[i], ty[i], tz[i], sx[j], sy[j], sz[j], &skip);
            if (skip) continue;
            double df = subtract ? (sf[j] - fi) : sf[j];
            S += (long double)(G * sw[j] * df);
        }
        if (finalize) {
            long double v = S;
            if (subtract) v += (long double)fi / ((long double)k * (long double)k);
            out[i] = (double)(-2.0L * v);
        } else {
            out[i] = (double)S;
        }
    }
    return 0;
}
