/*
 * oracle/coulomb_sum.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain CPU definition of the discrete Hartree-potential (Coulomb) convolution of TAGI with the
 * Gaussian singularity subtraction of arXiv 2003.01833 Section 4.3, written from the paper.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, link or call this file.  It shares no code with the CUDA path.
 *
 * What it computes (one density per call), O-3 in DESIGN.md:
 *
 *   subtract = 1:  V_i = sum over sources j with r_ij != 0 of
 *                          (f_j - f_i * exp(-r_ij^2 / alpha^2)) * w_j / r_ij   +   2 pi alpha^2 f_i
 *   subtract = 0:  V_i = sum over sources j with r_ij != 0 of  f_j * w_j / r_ij
 *
 * Citations (PAPER.md line, equation):
 *   - Hartree potential V_H(r) = int rho(r') / |r - r'| dr' ..................... PAPER.md:197  Eq. (19)
 *   - "The singular r' = r term in the quadrature sums is skipped" .............. PAPER.md:200
 *   - Gaussian singularity subtraction
 *       int f(r')/|r-r'| = int (f(r') - f(r) e^{-|r-r'|^2/alpha^2}) / |r-r'|
 *                          + f(r) int e^{-|r-r'|^2/alpha^2} / |r-r'| ............ PAPER.md:220  Eq. (23)
 *   - int e^{-r^2/alpha^2} / r dr' = 2 pi alpha^2 ............................... PAPER.md:224  Eq. (24)
 *   - "this work uses ... alpha = 1 a.u." ....................................... PAPER.md:229
 *   - discrete convolution sum over the quadrature points ....................... PAPER.md:371  Eq. (32)
 *
 * Reading R3: "skipped" means r_ij == 0 exactly.  There is no 1/(4 pi) and no -2 here:
 * the kernel of Eq. (19) is 1/r as printed.
 *
 * Arithmetic: IEEE double, libm sqrt/exp (strict, no fast-math, no FMA contraction); the sum
 * over j is accumulated in long double.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* one term of the sum: target value fi (used only if subtract), source value fj, weight wj.
 * *skip is set when r == 0. */
double oracle_coulomb_term(double tx, double ty, double tz, double sx, double sy, double sz,
                           double fi, double fj, double wj, double alpha, int subtract, int* skip)
{
    double dx = tx - sx, dy = ty - sy, dz = tz - sz;
    double r2 = dx * dx + dy * dy + dz * dz;
    double r = sqrt(r2);
    *skip = 0;
    if (r == 0.0) { *skip = 1; return 0.0; }
    if (subtract) return (fj - fi * exp(-r2 / (alpha * alpha))) * wj / r;     /* Eq. (23), first integrand */
    return fj * wj / r;                                                       /* Eq. (19) */
}

/* M targets against N sources.  tf may be NULL iff subtract == 0.  Returns 0, or -1 on bad arguments. */
int oracle_coulomb_direct(int64_t M, const double* tx, const double* ty, const double* tz, const double* tf,
                          int64_t N, const double* sx, const double* sy, const double* sz,
                          const double* sw, const double* sf, double alpha, int subtract, double* out)
{
    if (M < 0 || N < 0 || !out) return -1;
    if (subtract && (!tf || !(alpha > 0.0))) return -1;
    int64_t i;
#pragma omp parallel for schedule(dynamic, 16)
    for (i = 0; i < M; ++i) {
        long double S = 0.0L;
        double fi = subtract ? tf[i] : 0.0;
        for (int64_t j = 0; j < N; ++j) {
            int skip;
            double t = oracle_coulomb_term(tx[i], ty[i], tz[i], sx[j], sy[j], sz[j], fi, sf[j], sw[j],
                                           alpha, subtract, &skip);
            if (skip) continue;
            S += (long double)t;
        }
        if (subtract) S += 2.0L * (long double)M_PI * (long double)alpha * (long double)alpha * (long double)fi;   /* Eq. (24) */
        out[i] = (double)S;
    }
    return 0;
}
