/*
 * oracle/fcg_oracle.c -- plain, slow, obviously-correct CPU oracle for the FFT-accelerated CG path
 * of arXiv 1305.3625 (PAPER.md = /root/reference/PAPER.md).
 *
 * TEST INFRASTRUCTURE ONLY: may be called from tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py.  The product (paper_1305_3625_b200/) never
 * imports, links or executes anything in this directory, and this file shares no code, header,
 * table or constant generator with the CUDA path.
 *
 * Contents
 *   oracle_spectrum            closed-form spectrum of BASELINE.json configs[0]
 *   oracle_dft2_brute          the 2D DFT by its definition, O(N^2)          (pins the FFT)
 *   oracle_conv_direct         direct circular convolution, O(N^2)           (pins Listing 4)
 *   oracle_fft2_{f64,f32}      textbook radix-2 FFT, rows then columns
 *   oracle_apply_{f64,f32}     y = k o x + F^-1(s o F x)   (Listing 4)
 *   oracle_cg_{f64,f32}        conjugate gradient          (Listing 2)
 *   oracle_pcg_{f64,f32}       the same with the spectral preconditioner M = kbar I + C
 *   oracle_break_step_*, oracle_fracture_*   break rule + quasi-static loop (PAPER.md:78,
 *                              BASELINE.json configs[3])
 *   oracle_green_function      eq. (1c): real-space Green's function, closed form of the integral
 *   oracle_kernel_spectrum_*   s = Re F G, the static transform of the kernel
 *   oracle_force_{apply,cg,break_step,fracture}_*   the paper's formulation in the bond forces, (I + K G) f = K D
 *                              (eq. (2))
 *   oracle_inverse_spectrum_*, oracle_force_from_displacement_*   the same state through the displacements:
 *                              (K + G^-1) u = K D by oracle_cg / oracle_pcg with s = 1 / g, then eq. (1a) (reading F7)
 * Pins (tests/test_oracle_*.py): none of these functions is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -fPIC -shared fcg_oracle.c -o libfcg_oracle.so -lm
 * (-ffp-contract=off: every multiply and add below rounds once, as written.)
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

#define ORACLE_CAT2(a, b) a##b
#define ORACLE_CAT(a, b) ORACLE_CAT2(a, b)

#define REAL double
#define CPLX cplx_f64
#define FN(name) ORACLE_CAT(name, _f64)
#include "fcg_oracle_impl.h"
#undef REAL
#undef FN
#undef CPLX
#define CPLX cplx_f32
#define REAL float
#define FN(name) ORACLE_CAT(name, _f32)
#include "fcg_oracle_impl.h"
#undef REAL
#undef FN
#undef CPLX

/* Spectrum of BASELINE.json configs[0]:
 *   s[m,n] = 1 / sqrt(4 sin^2(pi m/L) + 4 sin^2(pi n/L))   for (m,n) != (0,0),   s[0,0] = L/(2 pi),
 * row-major [m][n], fp64. */
void oracle_spectrum(int L, double* s)
{
    for (int m = 0; m < L; ++m)
        for (int n = 0; n < L; ++n) {
            if (m == 0 && n == 0) { s[0] = (double)L / (2.0 * M_PI); continue; }
            double sm = sin(M_PI * (double)m / (double)L);
            double sn = sin(M_PI * (double)n / (double)L);
            s[(size_t)m * L + n] = 1.0 / sqrt(4.0 * sm * sm + 4.0 * sn * sn);
        }
}

/* 2D DFT by definition:  X[m,n] = sum_{a,b} x[a,b] exp(-2 pi i (m a + n b)/L).
 * x: L x L real; X: L x L interleaved complex.  inverse != 0: +i and 1/L^2, complex input xin
 * (interleaved), complex output.  O(L^4): tiny L only.  The phase index (m a + n b) mod L is reduced
 * in integers so every cos/sin argument lies in [0, 2 pi). */
void oracle_dft2_brute(int L, const double* x_real, double* X)
{
    for (int m = 0; m < L; ++m)
        for (int n = 0; n < L; ++n) {
            double re = 0.0, im = 0.0;
            for (int a = 0; a < L; ++a)
                for (int b = 0; b < L; ++b) {
                    int ph = (int)(((long long)m * a + (long long)n * b) % L);
                    double ang = -2.0 * M_PI * (double)ph / (double)L;
                    re += x_real[(size_t)a * L + b] * cos(ang);
                    im += x_real[(size_t)a * L + b] * sin(ang);
                }
            X[2 * ((size_t)m * L + n)] = re;
            X[2 * ((size_t)m * L + n) + 1] = im;
        }
}

void oracle_idft2_brute(int L, const double* X, double* x)
{
    double inv = 1.0 / ((double)L * (double)L);
    for (int a = 0; a < L; ++a)
        for (int b = 0; b < L; ++b) {
            double re = 0.0, im = 0.0;
            for (int m = 0; m < L; ++m)
                for (int n = 0; n < L; ++n) {
                    int ph = (int)(((long long)m * a + (long long)n * b) % L);
                    double ang = 2.0 * M_PI * (double)ph / (double)L;
                    double c = cos(ang), sn = sin(ang);
                    double xr = X[2 * ((size_t)m * L + n)], xi = X[2 * ((size_t)m * L + n) + 1];
                    re += xr * c - xi * sn;
                    im += xr * sn + xi * c;
                }
            x[2 * ((size_t)a * L + b)] = re * inv;
            x[2 * ((size_t)a * L + b) + 1] = im * inv;
        }
}

/* Direct circular convolution:
 *   y[a,b] = sum_{a',b'} c[(a-a') mod L, (b-b') mod L] * x[a',b'].   O(L^4): tiny L only. */
void oracle_conv_direct(int L, const double* c, const double* x, double* y)
{
    for (int a = 0; a < L; ++a)
        for (int b = 0; b < L; ++b) {
            double acc = 0.0;
            for (int a2 = 0; a2 < L; ++a2)
                for (int b2 = 0; b2 < L; ++b2) {
                    int da = (a - a2 + L) % L, db = (b - b2 + L) % L;
                    acc += c[(size_t)da * L + db] * x[(size_t)a2 * L + b2];
                }
            y[(size_t)a * L + b] = acc;
        }
}

/* Real-space Green's function of eq. (1c), PAPER.md:63:
 *     G_ij = (1 - nu^2) / (pi E a^2)  *  int int_{-a/2}^{a/2} dx' dy' / | r_i - r_j(x', y') |
 * i.e. the surface displacement at bond i of an elastic half space under a unit force spread uniformly over the a x a
 * square of bond j.  The integral of 1/r over a rectangle has the closed form (antiderivative checked by differentiation:
 * d^2/dxdy [ x asinh(y/|x|) + y asinh(x/|y|) ] = 1/sqrt(x^2+y^2))
 *     I(X, Y) = sum over the four corners (x, y) = (X +- a/2, Y +- a/2) of  sign * ( x asinh(y/|x|) + y asinh(x/|y|) ),
 * sign = + for (+,+) and (-,-), - otherwise.  Corners are odd multiples of a/2, never on an axis.
 * Reading F3 (the paper does not state the boundary condition; Fourier acceleration implies a periodic lattice):
 * r_i - r_j is the minimum-image offset, da -> da - L for da > L/2 (I is even in X and in Y, so da = L/2 is unambiguous).
 * Output: G[da][db], da, db = 0..L-1, row-major, fp64.  G is even, so its transform is real. */
static double oracle_corner(double x, double y) { return x * asinh(y / fabs(x)) + y * asinh(x / fabs(y)); }

void oracle_green_function(int L, double nu, double E, double a, double* G)
{
    double pref = (1.0 - nu * nu) / (M_PI * E * a * a);
    double h = 0.5 * a;
    for (int da = 0; da < L; ++da)
        for (int db = 0; db < L; ++db) {
            double X = a * (double)(da <= L / 2 ? da : da - L);
            double Y = a * (double)(db <= L / 2 ? db : db - L);
            double I = oracle_corner(X + h, Y + h) - oracle_corner(X - h, Y + h)
                     - oracle_corner(X + h, Y - h) + oracle_corner(X - h, Y - h);
            G[(size_t)da * L + db] = pref * I;
        }
}

#ifdef _OPENMP
#include <omp.h>
int oracle_num_threads(void) { return omp_get_max_threads(); }
void oracle_set_num_threads(int n) { if (n > 0) omp_set_num_threads(n); }
#else
int oracle_num_threads(void) { return 1; }
void oracle_set_num_threads(int n) { (void)n; }
#endif
