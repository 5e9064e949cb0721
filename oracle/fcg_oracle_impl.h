/*
 * oracle/fcg_oracle_impl.h -- precision-generic body of the CPU oracle.
 *
 * TEST INFRASTRUCTURE ONLY.  Included twice by fcg_oracle.c, once with REAL=double (SUF=_f64)
 * and once with REAL=float (SUF=_f32).  Shares no code with the CUDA path.
 *
 * Everything here is the plain definition or the paper's algorithm written out in the paper's
 * order (PAPER.md = /root/reference/PAPER.md):
 *   - Listing 4: cpyComplex -> forward 2D FFT -> elementMult with the static
 *     spectrum -> inverse 2D FFT -> cpyReal; normalisation afterwards (Listing 3).
 *   - Listing 2: un-preconditioned conjugate gradient.
 *   - break rule: BASELINE.json configs[3] (the paper only says "bonds break").
 *
 * Precision reading S12: vectors, spectrum, twiddles and FFT arithmetic in
 * REAL; dot-product accumulators and the CG scalars alpha, beta, rho in double for both REAL types.
 */

typedef struct { REAL re, im; } CPLX;

/* ---- textbook iterative radix-2 complex FFT (bit reversal + log2 n butterfly stages) ------------
 * X[k] = sum_j x[j] exp(sign * 2 pi i j k / n); sign = -1 forward, +1 inverse (unnormalised).
 * tw[j] = exp(sign * 2 pi i j / n) for j < n/2, each evaluated with fp64 cos/sin of its own angle
 * (no recurrence) and then rounded to REAL. */
static void FN(make_twiddles)(CPLX* tw, int n, int sign)
{
    for (int j = 0; j < n / 2; ++j) {
        double ang = (double)sign * 2.0 * M_PI * (double)j / (double)n;
        tw[j].re = (REAL)cos(ang);
        tw[j].im = (REAL)sin(ang);
    }
}

static void FN(fft1d)(CPLX* x, int n, const CPLX* tw)
{
    /* bit-reversal permutation */
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { CPLX t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    /* butterfly stages, len = 2, 4, ..., n */
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, step = n / len;
        for (int base = 0; base < n; base += len) {
            for (int j = 0; j < half; ++j) {
                CPLX w = tw[j * step];
                CPLX a = x[base + j], b = x[base + j + half];
                CPLX wb;
                wb.re = w.re * b.re - w.im * b.im;
                wb.im = w.re * b.im + w.im * b.re;
                x[base + j].re = a.re + wb.re;        x[base + j].im = a.im + wb.im;
                x[base + j + half].re = a.re - wb.re; x[base + j + half].im = a.im - wb.im;
            }
        }
    }
}

/* 2D transform of an L x L row-major complex array, in place: all rows, then all columns. */
static void FN(fft2d)(CPLX* buf, int L, int sign)
{
    CPLX* tw = (CPLX*)malloc(sizeof(CPLX) * (size_t)(L / 2 + 1));
    FN(make_twiddles)(tw, L, sign);
#pragma omp parallel
    {
        CPLX* col = (CPLX*)malloc(sizeof(CPLX) * (size_t)L);
#pragma omp for schedule(static)
        for (int a = 0; a < L; ++a) FN(fft1d)(buf + (size_t)a * L, L, tw);
#pragma omp for schedule(static)
        for (int b = 0; b < L; ++b) {
            for (int a = 0; a < L; ++a) col[a] = buf[(size_t)a * L + b];
            FN(fft1d)(col, L, tw);
            for (int a = 0; a < L; ++a) buf[(size_t)a * L + b] = col[a];
        }
        free(col);
    }
    free(tw);
}

/* Public: forward (sign=-1) or inverse (sign=+1, includes the 1/L^2 factor) 2D DFT of an
 * interleaved complex L x L array, in place.  Definition: SURVEY.md 8(c) "DFT". */
int FN(oracle_fft2)(int L, REAL* buf_interleaved, int inverse)
{
    if (L < 1 || (L & (L - 1))) return -1;
    CPLX* buf = (CPLX*)buf_interleaved;
    FN(fft2d)(buf, L, inverse ? +1 : -1);
    if (inverse) {
        REAL scale = (REAL)(1.0 / ((double)L * (double)L)); /* power of two: exact */
        size_t N = (size_t)L * L;
        for (size_t i = 0; i < N; ++i) { buf[i].re *= scale; buf[i].im *= scale; }
    }
    return 0;
}

/* c = C x = F^-1 ( s o F x ), the route of Listing 4. work: N complex. */
static void FN(convolve)(int L, const REAL* s, const REAL* x, REAL* c, CPLX* work)
{
    size_t N = (size_t)L * L;
    REAL scale = (REAL)(1.0 / ((double)L * (double)L));
    for (size_t i = 0; i < N; ++i) { work[i].re = x[i]; work[i].im = (REAL)0; }   /* cpyComplex */
    FN(fft2d)(work, L, -1);                                                        /* cufft2D fwd */
    for (size_t i = 0; i < N; ++i) { work[i].re *= s[i]; work[i].im *= s[i]; }     /* elementMult */
    FN(fft2d)(work, L, +1);                                                        /* cufft2D inv */
    for (size_t i = 0; i < N; ++i) c[i] = work[i].re * scale;                      /* cpyReal + normalise */
}

/* y = A x = k o x + C x   ("one element-by-element multiplication and a call to CUBLAS later",
 * PAPER.md:151; operator of BASELINE.json configs[0]). */
static void FN(apply)(int L, const REAL* s, const REAL* k, const REAL* x, REAL* y, CPLX* work)
{
    size_t N = (size_t)L * L;
    FN(convolve)(L, s, x, y, work);
    for (size_t i = 0; i < N; ++i) y[i] = k[i] * x[i] + y[i];
}

int FN(oracle_apply)(int L, const REAL* s, const REAL* k, const REAL* x, REAL* y)
{
    if (L < 1 || (L & (L - 1))) return -1;
    CPLX* work = (CPLX*)malloc(sizeof(CPLX) * (size_t)L * L);
    FN(apply)(L, s, k, x, y, work);
    free(work);
    return 0;
}

/* dot product with a double accumulator, plain left-to-right sum (reading S12). */
static double FN(dot)(size_t N, const REAL* a, const REAL* b)
{
    double acc = 0.0;
    for (size_t i = 0; i < N; ++i) acc += (double)a[i] * (double)b[i];
    return acc;
}

/* Conjugate gradient, Listing 2 in Hestenes-Stiefel form, step by step as in
 * SURVEY.md 8(c).  Stopping rule (readings S3, S11, S15): first iteration at which the recurrence
 * residual satisfies sqrt(r.r) <= tol * sqrt(f.f).
 *   u        in: initial guess, out: solution
 *   iters    number of operator applications inside the loop (reading S14)
 *   relres   sqrt(rho)/||f|| at exit
 *   hist     optional, capacity maxit+1: relative residual after 0,1,2,... iterations
 *   Phist/Rhist optional, capacity maxit*N each: search direction p_i and residual r_i (before the
 *            update of iteration i) -- used only by the CG-invariant pins on tiny grids
 * returns 0 converged, 1 maxit reached, -4 breakdown (p.Ap <= 0 or not finite), -1 bad argument. */
int FN(oracle_cg)(int L, const REAL* s, const REAL* k, const REAL* f, REAL* u, double tol, int maxit,
                  int* iters, double* relres, double* hist, REAL* Phist, REAL* Rhist)
{
    if (L < 1 || (L & (L - 1)) || maxit < 0 || !(tol >= 0.0)) return -1;
    size_t N = (size_t)L * L;
    int status = 1, it = 0;
    double fn = sqrt(FN(dot)(N, f, f));
    if (fn == 0.0) {
        for (size_t i = 0; i < N; ++i) u[i] = (REAL)0;
        *iters = 0; *relres = 0.0; if (hist) hist[0] = 0.0;
        return 0;
    }
    REAL* r = (REAL*)malloc(sizeof(REAL) * N);
    REAL* p = (REAL*)malloc(sizeof(REAL) * N);
    REAL* q = (REAL*)malloc(sizeof(REAL) * N);
    CPLX* work = (CPLX*)malloc(sizeof(CPLX) * N);

    FN(apply)(L, s, k, u, q, work);                              /* set up initial values */
    for (size_t i = 0; i < N; ++i) { r[i] = f[i] - q[i]; p[i] = r[i]; }
    double rho = FN(dot)(N, r, r);
    if (hist) hist[0] = sqrt(rho) / fn;
    if (sqrt(rho) <= tol * fn) { status = 0; goto done; }

    while (it < maxit) {
        if (Phist) memcpy(Phist + (size_t)it * N, p, sizeof(REAL) * N);
        if (Rhist) memcpy(Rhist + (size_t)it * N, r, sizeof(REAL) * N);
        FN(apply)(L, s, k, p, q, work);                          /* calculate A*x */
        double pq = FN(dot)(N, p, q);                            /* search length (dot product) */
        if (!(pq > 0.0) || !isfinite(pq)) { status = -4; goto done; }
        double alpha = rho / pq;
        REAL al = (REAL)alpha;
        for (size_t i = 0; i < N; ++i) u[i] = u[i] + al * p[i];  /* new x */
        for (size_t i = 0; i < N; ++i) r[i] = r[i] - al * q[i];  /* residue */
        double rho_new = FN(dot)(N, r, r);                       /* residue length */
        ++it;
        if (hist) hist[it] = sqrt(rho_new) / fn;
        if (sqrt(rho_new) <= tol * fn) { rho = rho_new; status = 0; break; }   /* check convergence */
        double beta = rho_new / rho;                             /* update calculation variables */
        REAL be = (REAL)beta;
        for (size_t i = 0; i < N; ++i) p[i] = r[i] + be * p[i];
        rho = rho_new;
    }
done:
    *iters = it;
    *relres = sqrt(rho) / fn;
    free(r); free(p); free(q); free(work);
    return status;
}

/* Preconditioned conjugate gradient (the paper "used [a preconditioner] for a while",
 * PAPER.md:175, without giving one).  Textbook PCG with the spectral preconditioner
 *     M = kbar I + C,   M^-1 = F^-1 diag( 1 / (kbar + s) ) F            (reading D4)
 * i.e. the operator with the stiffnesses replaced by one constant.  m = 1 / (kbar + s) is formed element by element in
 * the working precision (one add, one divide).  Same stopping rule as oracle_cg: first iteration with
 * sqrt(r.r) <= tol sqrt(f.f), r the recurrence residual.
 *   hist    optional, capacity maxit+1: relative residual after 0,1,2,.. iterations
 *   Phist / Zhist / Rhist optional, capacity maxit*N each: p_i, z_i, r_i before the update of iteration i (pins)
 * returns 0 converged, 1 maxit reached, -4 breakdown (p.Ap <= 0, r.z <= 0 or not finite), -1 bad argument. */
int FN(oracle_pcg)(int L, const REAL* s, const REAL* k, const REAL* f, REAL* u, double kbar, double tol, int maxit,
                   int* iters, double* relres, double* hist, REAL* Phist, REAL* Zhist, REAL* Rhist)
{
    if (L < 1 || (L & (L - 1)) || maxit < 0 || !(tol >= 0.0)) return -1;
    size_t N = (size_t)L * L;
    int status = 1, it = 0;
    double fn = sqrt(FN(dot)(N, f, f));
    if (fn == 0.0) {
        for (size_t i = 0; i < N; ++i) u[i] = (REAL)0;
        *iters = 0; *relres = 0.0; if (hist) hist[0] = 0.0;
        return 0;
    }
    REAL* r = (REAL*)malloc(sizeof(REAL) * N);
    REAL* p = (REAL*)malloc(sizeof(REAL) * N);
    REAL* q = (REAL*)malloc(sizeof(REAL) * N);
    REAL* z = (REAL*)malloc(sizeof(REAL) * N);
    REAL* m = (REAL*)malloc(sizeof(REAL) * N);
    CPLX* work = (CPLX*)malloc(sizeof(CPLX) * N);
    for (size_t i = 0; i < N; ++i) m[i] = (REAL)1 / ((REAL)kbar + s[i]);

    FN(apply)(L, s, k, u, q, work);
    for (size_t i = 0; i < N; ++i) r[i] = f[i] - q[i];
    double rr = FN(dot)(N, r, r);
    double rho = 0.0;
    if (hist) hist[0] = sqrt(rr) / fn;
    if (sqrt(rr) <= tol * fn) { status = 0; goto done; }
    FN(convolve)(L, m, r, z, work);                               /* z = M^-1 r */
    for (size_t i = 0; i < N; ++i) p[i] = z[i];
    rho = FN(dot)(N, r, z);
    if (!(rho > 0.0) || !isfinite(rho)) { status = -4; goto done; }

    while (it < maxit) {
        if (Phist) memcpy(Phist + (size_t)it * N, p, sizeof(REAL) * N);
        if (Zhist) memcpy(Zhist + (size_t)it * N, z, sizeof(REAL) * N);
        if (Rhist) memcpy(Rhist + (size_t)it * N, r, sizeof(REAL) * N);
        FN(apply)(L, s, k, p, q, work);
        double pq = FN(dot)(N, p, q);
        if (!(pq > 0.0) || !isfinite(pq)) { status = -4; goto done; }
        double alpha = rho / pq;
        REAL al = (REAL)alpha;
        for (size_t i = 0; i < N; ++i) u[i] = u[i] + al * p[i];
        for (size_t i = 0; i < N; ++i) r[i] = r[i] - al * q[i];
        rr = FN(dot)(N, r, r);
        ++it;
        if (hist) hist[it] = sqrt(rr) / fn;
        if (sqrt(rr) <= tol * fn) { status = 0; break; }
        FN(convolve)(L, m, r, z, work);
        double rho_new = FN(dot)(N, r, z);
        if (!(rho_new > 0.0) || !isfinite(rho_new)) { status = -4; goto done; }
        double beta = rho_new / rho;
        REAL be = (REAL)beta;
        for (size_t i = 0; i < N; ++i) p[i] = z[i] + be * p[i];
        rho = rho_new;
    }
done:
    *iters = it;
    *relres = sqrt(rr) / fn;
    free(r); free(p); free(q); free(z); free(m); free(work);
    return status;
}

/* Break step (BASELINE.json configs[3]; readings S5, S13): over candidates {i : k_i > 0}
 * ratio_i = (k_i * u_i) / t_i  -- one IEEE multiply and one IEEE divide in double -- pick the
 * maximum, ties -> lowest i, NaN skipped; set k_i = 0.  second = runner-up ratio (for the top-2
 * gap of reading S17), -inf if none.  returns 0, or -6 when there is no candidate (index = -1). */
int FN(oracle_break_step)(long long N, REAL* k, const REAL* u, const REAL* t,
                          long long* index, double* ratio, double* second)
{
    long long best = -1;
    double rbest = 0.0, rsecond = -INFINITY;
    for (long long i = 0; i < N; ++i) {
        if (!(k[i] > (REAL)0)) continue;
        double load = (double)k[i] * (double)u[i];
        double rt = load / (double)t[i];
        if (rt != rt) continue;
        if (best < 0) { best = i; rbest = rt; }
        else if (rt > rbest) { rsecond = rbest; rbest = rt; best = i; }
        else if (rt > rsecond) rsecond = rt;
    }
    *index = best; *ratio = rbest; if (second) *second = rsecond;
    if (best < 0) return -6;
    k[best] = (REAL)0;
    return 0;
}

/* Quasi-static loop (BASELINE.json configs[3]; reading S11: warm start from previous u).
 * For each step: solve A u = f by CG from the current u, then break one site.
 * out_index[nsteps], out_iters[nsteps], out_gap[nsteps] (relative top-2 gap, may be NULL).
 * returns the number of completed steps (== nsteps on success), or a negative CG status. */
int FN(oracle_fracture)(int L, const REAL* s, REAL* k, const REAL* f, REAL* u, const REAL* t,
                        int nsteps, double tol, int maxit,
                        long long* out_index, int* out_iters, double* out_gap)
{
    long long N = (long long)L * L;
    for (int step = 0; step < nsteps; ++step) {
        int it; double rr;
        int st = FN(oracle_cg)(L, s, k, f, u, tol, maxit, &it, &rr, NULL, NULL, NULL);
        if (st < 0) return st;
        long long idx; double ratio, second;
        int bs = FN(oracle_break_step)(N, k, u, t, &idx, &ratio, &second);
        if (bs < 0) return step;
        out_index[step] = idx; out_iters[step] = it;
        if (out_gap) out_gap[step] = (ratio - second) / fabs(ratio);
    }
    return nsteps;
}

/* The same quasi-static loop with every solve done by oracle_pcg (preconditioner M = kbar I + C, kbar fixed for the whole
 * loop).  The break sequence is a property of the exact solutions, so it must coincide with
 * oracle_fracture's wherever the top-2 gap exceeds the solver error; only the iteration counts differ. */
int FN(oracle_pcg_fracture)(int L, const REAL* s, REAL* k, const REAL* f, REAL* u, const REAL* t, double kbar,
                            int nsteps, double tol, int maxit,
                            long long* out_index, int* out_iters, double* out_gap)
{
    long long N = (long long)L * L;
    for (int step = 0; step < nsteps; ++step) {
        int it; double rr;
        int st = FN(oracle_pcg)(L, s, k, f, u, kbar, tol, maxit, &it, &rr, NULL, NULL, NULL, NULL);
        if (st < 0) return st;
        long long idx; double ratio, second;
        int bs = FN(oracle_break_step)(N, k, u, t, &idx, &ratio, &second);
        if (bs < 0) return step;
        out_index[step] = idx; out_iters[step] = it;
        if (out_gap) out_gap[step] = (ratio - second) / fabs(ratio);
    }
    return nsteps;
}

/* ================================================================================================
 * The paper's own formulation in the bond forces:
 *     f_i = -k_i (u_i - D)   (1a),      u_i = sum_j G_ij f_j   (1b, with the typo f_i -> f_j: reading G1)
 *     =>  (I + K G) f = K D             (2)
 * solved for f by conjugate gradient as Listing 2 says.  G is applied by Fourier acceleration,
 * G x = F^-1( g o F x ) with g = F G "static and performed during initialization".
 * Reading F1: I + K G is symmetric positive definite on the unbroken bonds when every unbroken bond has the same
 * elastic constant ("For simplicity, all fibers have the same elastic constant"), k_i in {0, kappa}: there
 * it is I + kappa P G P (P = projection on the unbroken bonds), and every CG vector stays in range(P) because b = K D and
 * K G x lie in it and the start vector has f_i = 0 on broken bonds.  That is the case the functions below are for.
 * ------------------------------------------------------------------------------------------------ */

/* s = Re F G: the static transform of a real-space kernel G (L x L, G[da][db], offsets mod L).  For an even kernel
 * (G[-da][-db] = G[da][db]) the transform is real; the imaginary part (rounding) is dropped like cpyReal does. */
int FN(oracle_kernel_spectrum)(int L, const REAL* G, REAL* s)
{
    if (L < 1 || (L & (L - 1))) return -1;
    size_t N = (size_t)L * L;
    CPLX* work = (CPLX*)malloc(sizeof(CPLX) * N);
    for (size_t i = 0; i < N; ++i) { work[i].re = G[i]; work[i].im = (REAL)0; }
    FN(fft2d)(work, L, -1);
    for (size_t i = 0; i < N; ++i) s[i] = work[i].re;
    free(work);
    return 0;
}

/* y = (I + K G) x = x + k o (G x)      (left side of eq. (2)) */
static void FN(force_apply)(int L, const REAL* g, const REAL* k, const REAL* x, REAL* y, CPLX* work)
{
    size_t N = (size_t)L * L;
    FN(convolve)(L, g, x, y, work);
    for (size_t i = 0; i < N; ++i) y[i] = x[i] + k[i] * y[i];
}

int FN(oracle_force_apply)(int L, const REAL* g, const REAL* k, const REAL* x, REAL* y)
{
    if (L < 1 || (L & (L - 1))) return -1;
    CPLX* work = (CPLX*)malloc(sizeof(CPLX) * (size_t)L * L);
    FN(force_apply)(L, g, k, x, y, work);
    free(work);
    return 0;
}

/* Conjugate gradient on (I + K G) f = K D, Listing 2 step by step (same scalars, stopping rule and return values as
 * oracle_cg above; the right-hand side is b_i = k_i * D, one multiply in REAL, and the stop is sqrt(r.r) <= tol sqrt(b.b)).
 *   f   in: initial guess (must be 0 on broken bonds), out: the bond forces */
int FN(oracle_force_cg)(int L, const REAL* g, const REAL* k, double D, REAL* f, double tol, int maxit,
                        int* iters, double* relres, double* hist, REAL* Phist, REAL* Rhist)
{
    if (L < 1 || (L & (L - 1)) || maxit < 0 || !(tol >= 0.0)) return -1;
    size_t N = (size_t)L * L;
    int status = 1, it = 0;
    REAL* b = (REAL*)malloc(sizeof(REAL) * N);
    for (size_t i = 0; i < N; ++i) b[i] = k[i] * (REAL)D;         /* K D */
    double bn = sqrt(FN(dot)(N, b, b));
    if (bn == 0.0) {
        for (size_t i = 0; i < N; ++i) f[i] = (REAL)0;
        *iters = 0; *relres = 0.0; if (hist) hist[0] = 0.0;
        free(b);
        return 0;
    }
    REAL* r = (REAL*)malloc(sizeof(REAL) * N);
    REAL* p = (REAL*)malloc(sizeof(REAL) * N);
    REAL* q = (REAL*)malloc(sizeof(REAL) * N);
    CPLX* work = (CPLX*)malloc(sizeof(CPLX) * N);

    FN(force_apply)(L, g, k, f, q, work);                        /* set up initial values */
    for (size_t i = 0; i < N; ++i) { r[i] = b[i] - q[i]; p[i] = r[i]; }
    double rho = FN(dot)(N, r, r);
    if (hist) hist[0] = sqrt(rho) / bn;
    if (sqrt(rho) <= tol * bn) { status = 0; goto done; }

    while (it < maxit) {
        if (Phist) memcpy(Phist + (size_t)it * N, p, sizeof(REAL) * N);
        if (Rhist) memcpy(Rhist + (size_t)it * N, r, sizeof(REAL) * N);
        FN(force_apply)(L, g, k, p, q, work);                    /* calculate A*x */
        double pq = FN(dot)(N, p, q);                            /* search length (dot product) */
        if (!(pq > 0.0) || !isfinite(pq)) { status = -4; goto done; }
        double alpha = rho / pq;
        REAL al = (REAL)alpha;
        for (size_t i = 0; i < N; ++i) f[i] = f[i] + al * p[i];  /* new x */
        for (size_t i = 0; i < N; ++i) r[i] = r[i] - al * q[i];  /* residue */
        double rho_new = FN(dot)(N, r, r);                       /* residue length */
        ++it;
        if (hist) hist[it] = sqrt(rho_new) / bn;
        if (sqrt(rho_new) <= tol * bn) { rho = rho_new; status = 0; break; }   /* check convergence */
        double beta = rho_new / rho;                             /* update calculation variables */
        REAL be = (REAL)beta;
        for (size_t i = 0; i < N; ++i) p[i] = r[i] + be * p[i];
        rho = rho_new;
    }
done:
    *iters = it;
    *relres = sqrt(rho) / bn;
    free(b); free(r); free(p); free(q); free(work);
    return status;
}

/* The same state through the displacements (reading F7).  Eliminating f instead of u from (1a), (1b): u = G f and f = K (D - u)
 * give G^-1 u = K (D - u), i.e.
 *     (K + G^-1) u = K D,        G^-1 = F^-1 diag(1 / g) F,
 * which is the symmetric system A u = b of BASELINE.json with spectrum s = 1 / g and right-hand side b = K D -- solved by
 * oracle_cg / oracle_pcg as they stand -- followed by eq. (1a) for the forces.  The two functions below are the two
 * element-by-element maps of that route; each is one IEEE operation per step in REAL. */
void FN(oracle_inverse_spectrum)(long long N, const REAL* g, REAL* s)
{
    for (long long i = 0; i < N; ++i) s[i] = (REAL)1 / g[i];
}

/* f_i = -k_i (u_i - D)     eq. (1a), evaluated as k_i * (D - u_i): one subtraction, one multiplication */
void FN(oracle_force_from_displacement)(long long N, const REAL* k, double D, const REAL* u, REAL* f)
{
    for (long long i = 0; i < N; ++i) f[i] = k[i] * ((REAL)D - u[i]);
}

/* Break step in the force formulation (reading F2): the response is linear in D, so the bond that reaches its threshold
 * first as D grows is the one with the largest f_i / t_i (one IEEE divide in double) among the unbroken bonds; ties ->
 * lowest i, NaN skipped.  The bond is removed: k_i = 0 and f_i = 0 (a broken bond carries no force; keeps the warm start
 * inside range(P)).  ratio: with the forces computed at displacement D the bond breaks at D_c = D / ratio.
 * returns 0, or -6 when there is no candidate (index = -1). */
int FN(oracle_force_break_step)(long long N, REAL* k, REAL* f, const REAL* t,
                                long long* index, double* ratio, double* second)
{
    long long best = -1;
    double rbest = 0.0, rsecond = -INFINITY;
    for (long long i = 0; i < N; ++i) {
        if (!(k[i] > (REAL)0)) continue;
        double rt = (double)f[i] / (double)t[i];
        if (rt != rt) continue;
        if (best < 0) { best = i; rbest = rt; }
        else if (rt > rbest) { rsecond = rbest; rbest = rt; best = i; }
        else if (rt > rsecond) rsecond = rt;
    }
    *index = best; *ratio = rbest; if (second) *second = rsecond;
    if (best < 0) return -6;
    k[best] = (REAL)0;
    f[best] = (REAL)0;
    return 0;
}

/* Quasi-static loop in the force formulation ("For each step in the simulation, the displacement is set, and the
 * resulting distribution of forces is calculated.  For large enough local strain, bonds break"):
 * each step solves (I + K G) f = K D from the previous forces and breaks one bond.
 * out_index, out_iters, out_ratio (winning f/t; D_c = D/ratio), out_gap (relative top-2 gap, may be NULL): [nsteps].
 * returns the number of completed steps, or a negative CG status. */
int FN(oracle_force_fracture)(int L, const REAL* g, REAL* k, double D, REAL* f, const REAL* t,
                              int nsteps, double tol, int maxit,
                              long long* out_index, int* out_iters, double* out_ratio, double* out_gap)
{
    long long N = (long long)L * L;
    for (int step = 0; step < nsteps; ++step) {
        int it; double rr;
        int st = FN(oracle_force_cg)(L, g, k, D, f, tol, maxit, &it, &rr, NULL, NULL, NULL);
        if (st < 0) return st;
        long long idx; double ratio, second;
        int bs = FN(oracle_force_break_step)(N, k, f, t, &idx, &ratio, &second);
        if (bs < 0) return step;
        out_index[step] = idx; out_iters[step] = it;
        if (out_ratio) out_ratio[step] = ratio;
        if (out_gap) out_gap[step] = (ratio - second) / fabs(ratio);
    }
    return nsteps;
}

/* The quasi-static loop of the force model through the displacements (reading F7): each step forms b = K D, solves
 * (K + G^-1) u = b from the previous u -- by oracle_cg, or by oracle_pcg when use_pcg (preconditioner M = kbar I + G^-1, kbar
 * fixed for the whole loop) --, evaluates the forces by eq. (1a), f_i = k_i (D - u_i), and breaks the bond with the largest
 * f_i / t_i (reading F2: one IEEE divide in double over {k_i > 0}, ties -> lowest i, NaN skipped; k_i = 0).  u is NOT changed by
 * the break (it is the plate's displacement, and the warm start of the next solve).  The break sequence is a property of the
 * exact solutions, so it coincides with oracle_force_fracture's wherever the top-2 gap exceeds the solver error.
 *   sinv  = 1 / g (oracle_inverse_spectrum);  f: work array of N, on return the forces of the LAST solve with the broken bond zeroed
 * returns the number of completed steps, or a negative solver status. */
int FN(oracle_force_fracture_displacement)(int L, const REAL* sinv, REAL* k, double D, REAL* u, REAL* f, const REAL* t, int use_pcg,
                                           double kbar, int nsteps, double tol, int maxit,
                                           long long* out_index, int* out_iters, double* out_ratio, double* out_gap)
{
    long long N = (long long)L * L;
    REAL* b = (REAL*)malloc(sizeof(REAL) * (size_t)N);
    int step = 0;
    for (; step < nsteps; ++step) {
        int it; double rr;
        for (long long i = 0; i < N; ++i) b[i] = k[i] * (REAL)D;
        int st = use_pcg ? FN(oracle_pcg)(L, sinv, k, b, u, kbar, tol, maxit, &it, &rr, NULL, NULL, NULL, NULL)
                         : FN(oracle_cg)(L, sinv, k, b, u, tol, maxit, &it, &rr, NULL, NULL, NULL);
        if (st < 0) { free(b); return st; }
        FN(oracle_force_from_displacement)(N, k, D, u, f);
        long long idx; double ratio, second;
        int bs = FN(oracle_force_break_step)(N, k, f, t, &idx, &ratio, &second);
        if (bs < 0) break;
        out_index[step] = idx; out_iters[step] = it;
        if (out_ratio) out_ratio[step] = ratio;
        if (out_gap) out_gap[step] = (ratio - second) / fabs(ratio);
    }
    free(b);
    return step;
}
