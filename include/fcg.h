/*
 * fcg.h -- C ABI of libfcg: FFT-accelerated conjugate gradient for the lattice fracture model of
 * arXiv 1305.3625 (Gjerden), hand-written CUDA for NVIDIA B200 (sm_100a).  No cuFFT, no cuBLAS,
 * no CPU fallback.
 *
 * Citations: "PAPER.md:<line>" = /root/reference/PAPER.md; "configs[i]" / "north_star" =
 * BASELINE.json; "S<n>" = reading n in SURVEY.md section 8(c) / DESIGN.md.
 *
 * The problem (north_star, Listings 2 and 4):
 *     solve  A u = f,   A = diag(k) + C,   C x = F^-1 ( s o F x )
 * on a periodic L x L lattice.  F is the 2D DFT
 *     X[m,n] = sum_{a,b} x[a,b] exp(-2 pi i (m a + n b) / L),
 * s is a real spectrum (row-major [m][n]); C x is real because only the even part
 * (s[m,n] + s[-m,-n])/2 of s survives the final "take the real part" step (cpyReal).
 *
 * Conventions for every call
 *   - Site index i = a*L + b (row a, column b fastest).  N = L*L.
 *   - Every array argument is a DEVICE pointer to contiguous memory of the handle's dtype
 *     (float for FCG_F32, double for FCG_F64), 16-byte aligned, owned by the caller (e.g. a
 *     torch tensor).  The library never frees or keeps a caller pointer after the call returns.
 *     Exceptions are spelled out: names ending in _host are HOST pointers.
 *   - All work is enqueued on the stream given to fcg_create.  Calls that fill host out-params
 *     (fcg_solve, fcg_break_step) end with one small device-to-host copy and one stream
 *     synchronisation ("reporting back only a few values to the CPU each time the solver has
 *     completed").  Nothing inside the CG loop synchronises with the host.
 *   - Return value: fcg_status.  >= 0 means the outputs are valid.  On error the outputs are
 *     unspecified unless stated; fcg_last_error() gives a message.  A handle is not thread-safe.
 *   - L must be a power of two, 16 <= L <= 8192 (S8); otherwise FCG_UNSUPPORTED.
 *   - Workspace: fcg_workspace_bytes() ~ 6 N w (T2, two stored spectra, r, p, q, z) + tables.
 */
#ifndef FCG_H
#define FCG_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fcg_handle_s* fcg_handle;

typedef enum { FCG_F32 = 0, FCG_F64 = 1 } fcg_dtype;

typedef enum {
    FCG_OK            =  0,
    FCG_NOT_CONVERGED =  1,  /* maxit reached; u, iters, rel_residual are valid (S16) */
    FCG_INVALID_ARG   = -1,
    FCG_UNSUPPORTED   = -2,
    FCG_CUDA_ERROR    = -3,
    FCG_BREAKDOWN     = -4,  /* p.Ap <= 0 or not finite; u holds the last iterate before the breakdown */
    FCG_NO_SPECTRUM   = -5,  /* fcg_set_spectrum has not been called */
    FCG_NO_CANDIDATE  = -6   /* fcg_break_step: no site with k > 0 (and a non-NaN ratio); index = -1 */
} fcg_status;

/* Options for fcg_set_option. */
typedef enum {
    FCG_OPT_LOOP_MODE    = 0, /* 0 (default): whole solve = one CUDA graph with a device-side WHILE node;
                                 1: kernels enqueued directly, in chunks of FCG_OPT_CHUNK iterations that
                                    exit early on the device flag, host polls once per chunk */
    FCG_OPT_CHUNK        = 1, /* iterations per chunk in loop mode 1 (default 16) */
    FCG_OPT_ROW_VARIANT  = 2, /* -1 (default): tuned rows-per-CTA of the classic row passes; 0,1,..: force variant */
    FCG_OPT_UNROLL       = 4, /* loop mode 0: CG iterations per evaluation of the graph's WHILE condition (1..64; -1, the default: the
                                 measured choice -- 8 for un-preconditioned fp64 solves at L = 1024 and 2048, 4 otherwise);
                                 iterations after the stop are no-op launches, results do not depend on it */
    FCG_OPT_PDL          = 5, /* programmatic dependent launch of the loop kernels.  0: plain stream order; 1: every loop kernel may
                                 start under its predecessor's tail (prologue only: nothing the predecessor writes is read before
                                 griddepcontrol.wait); 2: only the fused last pass starts early and fills its ring of k, p, r strips
                                 (which the column pass does not write) while the column pass drains -- the column pass triggers its
                                 dependents after its own wait, so the early section never runs ahead of the previous iteration;
                                 -1 (default): the measured choice per size (1 at L = 1024 fp64, 2 at L = 1024 fp32, else 0).
                                 Results do not depend on it */
    FCG_OPT_FUSED        = 6, /* 1 (default): for L = 256 and 512 (pipelined engine, loop mode 0) a whole solve is ONE cooperative
                                 kernel with the vectors resident in shared memory and grid barriers between the phases;
                                 0: the graph of four kernels per iteration at every size */
    FCG_OPT_L2_HINTS     = 7, /* bit mask of L2 eviction-priority hints in the pipelined passes (default: all, bit 6
                                 only while one vector is <= 32 MiB; 0..255):
                                 1 u strips (P1 loads) evict-first, 2 u stores evict-first, 4 spectrum rows (P2) evict-first,
                                 8 T2 tiles (P3 loads) evict-first, 16 k strips (P3) evict-first, 32 q loads (P4) evict-first,
                                 64 T2 stores of P1 evict-last, 128 r stores of the fused last pass evict-last (read back by the next P1) */
    FCG_OPT_SPECTRAL_ALPHA = 8, /* 1 (default): fcg_solve evaluates the search length's p.Ap as sum k p^2 (a scalar recurrence fed by the
                                 last pass) + sum shat |P|^2 (Parseval, accumulated in the column pass), so alpha is known before the
                                 last pass and r -= alpha q, r.r ride in it: 3 launches and 13.5 N w bytes per iteration, q never
                                 stored (pipelined engine).  0: p.q as a dot product after the last pass and a
                                 fourth kernel for the residual update (15.5 N w) */
    FCG_OPT_COL_PERSISTENT = 9, /* 1: column pass as persistent CTAs with two column buffers each, the next column's gather in flight
                                 while the current one is transformed (sizes where two buffers fit twice per SM); 0: one CTA per column;
                                 -1 (default): persistent for FCG_F32 and for L <= 1024, where it measured faster */
    FCG_OPT_BARRIER_START = 10, /* testing aid: initial value (taken as unsigned 32-bit) of the arrival counter of the cooperative
                                 kernel's grid barrier; default 0.  A value just below 2^32 makes the counter wrap within a few
                                 iterations (the barrier compares modulo 2^32; tests/test_gpu_robustness.py) */
    FCG_OPT_FFT_DIRECT   = 11, /* 1: fcg_fft_fwd / fcg_fft_inv are two launches, the column pass reading / writing the public layout
                                 X[m][n] itself (a TMA tensor tile per column for FCG_F64; plain 8-byte accesses for FCG_F32, whose
                                 row stride is not a multiple of 16 bytes); 0: three launches, a layout kernel between the internal
                                 T2 and X; -1 (default): two launches where they measured faster -- forward while X is <= 64 MiB
                                 (it then stays in L2 until the neighbouring columns have completed its sectors), inverse for
                                 FCG_F64 at every size and for FCG_F32 while X is <= 64 MiB.  Pipelined engine only (L >= 256) */
    FCG_OPT_FUSED_TWO    = 12, /* 1 (default): the one-launch kernel of FCG_OPT_FUSED runs un-preconditioned CG with TWO grid barriers per
                                 iteration (preconditioned CG with FOUR): it transforms the residual (and z = M^-1 r) instead of the
                                 direction and carries the row-transformed direction by the recurrence of Listing 2 (F_row p' =
                                 F_row r' + beta F_row p, exact in exact arithmetic); 0: three (six)
                                 barriers, the direction itself is transformed */
    FCG_OPT_STAGGER_P1   = 13, /* start offset in ns between the CTAs that share an SM, in the loop's first / column / last pass: CTAs launched */
    FCG_OPT_STAGGER_P2   = 14, /* together otherwise move through their copy and butterfly phases in step and the two do not overlap.  -1 */
    FCG_OPT_STAGGER_P3   = 15, /* (default): the measured value for the size (FCG_F64 L = 2048: 0 / 1500 / 2000; else 0); 0: none; <= 100000 */
    FCG_OPT_ENGINE       = 3  /* 0 (default): pipelined TMA passes where the lattice is large enough (L >= 256), classic
                                 passes otherwise; 1: classic passes only (synchronous loads; kept for A/B measurements).
                                 The stored spectrum's layout belongs to the engine: changing the engine after
                                 fcg_set_spectrum requires calling fcg_set_spectrum again (FCG_NO_SPECTRUM otherwise) */
} fcg_option;

/* Bytes of device workspace a handle of this size needs (0 if the size is unsupported). */
size_t fcg_workspace_bytes(int L, fcg_dtype dt);

/* Lifecycle (allocate -> plan -> execute -> destroy of Listing 3, without cuFFT).
 *   workspace    device memory of at least fcg_workspace_bytes(), 256-byte aligned, caller-owned and kept
 *                alive until fcg_destroy; or NULL: the library allocates and frees its own.
 *   cuda_stream  a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream.
 * Builds twiddle tables and launch plans; may synchronise the stream. */
int fcg_create(int L, fcg_dtype dt, void* workspace, void* cuda_stream, fcg_handle* out);
int fcg_destroy(fcg_handle h);
int fcg_set_option(fcg_handle h, int option, int value);
/* The EFFECTIVE value of an option on this handle, automatic (-1) choices resolved: FCG_OPT_LOOP_MODE, _UNROLL (as an
 * un-preconditioned solve would use it), _PDL, _FUSED, _SPECTRAL_ALPHA, _COL_PERSISTENT, _STAGGER_P1..P3; FCG_INVALID_ARG for the others. */
int fcg_get_option(fcg_handle h, int option, int* value);
/* Later calls enqueue on `cuda_stream` instead of the one given to fcg_create.  The caller orders the two streams (work already
 * enqueued stays where it is); refused (FCG_INVALID_ARG) while a quasi-static loop is pending.  This is what lets a caller
 * record the asynchronous calls (the fcg_slab_* passes, fcg_break_step_static aside) into a CUDA graph of its own: stream
 * capture runs on a stream other than the legacy default one (paper_1305_3625_b200/slab.py does exactly that). */
int fcg_set_stream(fcg_handle h, void* cuda_stream);

/* Static spectrum ("the FFT of G is static and performed during initialization").
 *   s  device, L x L reals, row-major [m][n].  Copied into an internal layout (even part, scaled by
 *      1/L^2 -- exact for power-of-two L, S6 -- permuted to the transform's digit-reversed order);
 *      the caller's array is not referenced afterwards. */
int fcg_set_spectrum(fcg_handle h, const void* s);

/* y = A x = k o x + C x  (Listing 4 + "one element-by-element multiplication and a call to CUBLAS",
 * PAPER.md:141-151).  k, x read-only; y written; y must not alias k or x.  Asynchronous. */
int fcg_apply(fcg_handle h, const void* k, const void* x, void* y);

/* Conjugate gradient, Listing 2, un-preconditioned.
 *   k, f          read-only, N reals each
 *   u             in: initial guess (warm start, configs[3]); out: solution
 *   tol, maxit    stop at the FIRST iteration with ||r||_2 <= tol * ||f||_2, r the recurrence residual
 *                 (S3, S11, S15), or after maxit iterations (status FCG_NOT_CONVERGED)
 *   iters_host    number of operator applications inside the loop (S14)
 *   rel_residual_host   ||r||_2 / ||f||_2 at exit
 * Dot products are accumulated in double and the scalars alpha, beta, rho are double for both dtypes
 * (S12); partial sums are combined in a fixed order, so repeated runs are bit-identical.
 * f == 0 gives u = 0, 0 iterations.  Blocks until the solve has finished. */
int fcg_solve(fcg_handle h, const void* k, const void* f, void* u, double tol, int maxit,
              int* iters_host, double* rel_residual_host);

/* Preconditioned conjugate gradient (the paper "used [a preconditioner] for a while",
 * PAPER.md:175, and gives no formula: reading D4 of DESIGN.md section 10).  Textbook PCG with the spectral preconditioner
 *     M = kbar I + C,    M^-1 r = F^-1 ( 1/(kbar + s) o F r ),
 * the operator with every stiffness replaced by one constant kbar (e.g. the mean of k): one more transform pair per
 * iteration, condition number of M^-1 A bounded by (max k + s_min)/(kbar + s_min) / ((min k + s_min)/(kbar + s_min))
 * independently of L.
 *   fcg_set_preconditioner   s: device, the same L x L spectrum given to fcg_set_spectrum (not referenced afterwards);
 *                            kbar >= 0.  m = 1/(kbar + s) is formed element by element in the handle's dtype (one add,
 *                            one divide) and stored like the operator's spectrum.  Requires fcg_set_spectrum first;
 *                            a later fcg_set_spectrum or engine change invalidates it (FCG_NO_SPECTRUM from fcg_pcg_solve).
 *   fcg_pcg_solve            arguments, stopping rule (||r||_2 <= tol ||f||_2, recurrence residual, first crossing),
 *                            iteration count, scalars in double and determinism as fcg_solve.  FCG_BREAKDOWN also when
 *                            r.z <= 0 or not finite (u then holds the iterate of the completed update).
 * The loop is one CUDA graph with a device-side WHILE node (6 launches per iteration); for L = 256, 512 the whole solve
 * is the one cooperative kernel of FCG_OPT_FUSED, as for fcg_solve. */
int fcg_set_preconditioner(fcg_handle h, const void* s, double kbar);
int fcg_pcg_solve(fcg_handle h, const void* k, const void* f, void* u, double tol, int maxit,
                  int* iters_host, double* rel_residual_host);

/* Same solve with HOST arrays (N reals each): copies k, f, u to library-owned device buffers, solves,
 * copies u back.  This is the end-to-end entry point timed by bench.py ("e2e"). */
int fcg_solve_host(fcg_handle h, const void* k_host, const void* f_host, void* u_host, double tol,
                   int maxit, int* iters_host, double* rel_residual_host);
/* Pipelined form, up to TWO solves outstanding on a handle: _submit stages the inputs on a stream of its own into one of two device
 * buffer sets, enqueues the solve behind them on the handle's stream (where the solve is one graph launch nothing blocks; the
 * one-launch kernel of small lattices and loop mode 1 run to completion inside _submit) and the copy of u back into u_host on a
 * third stream; _wait blocks until the OLDEST outstanding solve has its result in u_host and returns its status (as fcg_solve),
 * count and residual.  So the host<->device copies of solve i+1 and i-1 run under solve i.  k_host, f_host, u_host (pinned memory
 * for real overlap) must stay untouched from _submit until the matching _wait returns; u_host is the initial guess on the way
 * in and the solution on the way out.  A third _submit without a _wait and a _wait with nothing outstanding return
 * FCG_INVALID_ARG.  Between a _submit and its _wait call nothing else on the handle but these two. */
int fcg_solve_host_submit(fcg_handle h, const void* k_host, const void* f_host, void* u_host, double tol, int maxit);
int fcg_solve_host_wait(fcg_handle h, int* iters_host, double* rel_residual_host);

/* Stand-alone transforms (north_star "fcg_fft_fwd/inv").
 *   x  L x L reals;  X  L x (L/2+1) interleaved complex, row-major [m][n], n = 0..L/2
 *   fwd: X = F x (half spectrum; the rest follows from X[-m,-n] = conj X[m,n])
 *   inv: x = F^-1 X including 1/L^2, so inv(fwd(x)) == x.  X must be the spectrum of a real field
 *        (S18); only n = 0..L/2 is read.
 * x and X must not overlap.  Asynchronous. */
int fcg_fft_fwd(fcg_handle h, const void* x, void* X);
int fcg_fft_inv(fcg_handle h, const void* X, void* x);

/* Break step of the quasi-static loop (rule of configs[3], S5, S13):
 * over candidates {i : k_i > 0}: ratio_i = (k_i * u_i) / t_i, one IEEE multiply and one IEEE divide in
 * double; pick the maximum, ties -> lowest i, NaN skipped; set k_i = 0.
 *   k  in/out;  u, t read-only;  index_host = i (or -1);  ratio_host = the winning ratio.
 * Blocks until done. */
int fcg_break_step(fcg_handle h, void* k, const void* u, const void* t,
                   long long* index_host, double* ratio_host);

/* Quasi-static loop (configs[3]): nsteps times { fcg_solve warm-started from the current u;
 * fcg_break_step }.  index_host[nsteps], iters_host[nsteps] are HOST arrays.  Stops early (returning the
 * status) on a negative status; steps_done_host receives the number of completed steps. */
int fcg_fracture(fcg_handle h, void* k, const void* f, void* u, const void* t, int nsteps, double tol,
                 int maxit, long long* index_host, int* iters_host, int* steps_done_host);

/* The same loop with every solve done by fcg_pcg_solve (the preconditioner's kbar stays what fcg_set_preconditioner
 * was given for all steps).  One cooperative launch for L = 256, 512 like fcg_fracture. */
int fcg_pcg_fracture(fcg_handle h, void* k, const void* f, void* u, const void* t, int nsteps, double tol,
                     int maxit, long long* index_host, int* iters_host, int* steps_done_host);

/* Ensembles of independent samples ("good statistics"): the quasi-static loop in two
 * halves, so that ONE host thread can keep several handles busy, each created on its own stream.  For L = 256, 512 (one
 * cooperative kernel of L/2 CTAs per loop) _begin returns as soon as the launch is enqueued and up to three such kernels are
 * resident on a B200 at once; at other sizes _begin runs the loop to its end.  _end blocks and fills the host arrays like
 * fcg_fracture.  k, f, u, t must stay valid and untouched between the two calls; one loop pending per handle.
 *   use_pcg  0: fcg_solve per step, 1: fcg_pcg_solve (fcg_set_preconditioner first). */
int fcg_fracture_begin(fcg_handle h, void* k, const void* f, void* u, const void* t, int nsteps, double tol,
                       int maxit, int use_pcg);
int fcg_fracture_end(fcg_handle h, long long* index_host, int* iters_host, int* steps_done_host);

/* ---- The paper's own formulation in the bond forces ------------------------
 * Model:   f_i = -k_i (u_i - D)  (1a),   u_i = sum_j G_ij f_j  (1b; "f_i" in the print is a typo, reading G1),
 *                          G_ij = (1 - nu^2)/(pi E a^2) * int int_{-a/2}^{a/2} dx' dy' / |r_i - r_j(x', y')|          (1c)
 *                     =>   (I + K G) f = K D                                                                          (2)
 * solved for the forces f by conjugate gradient (Listing 2) with G applied by Fourier acceleration (eq. (3)):
 * G x = F^-1( g o F x ), g = Re F G "static and performed during initialization" and handed to fcg_set_spectrum.
 * Reading F1: I + K G is symmetric positive definite on the unbroken bonds when they all share one elastic constant, k_i in
 * {0, kappa} ("all fibers have the same elastic constant"), and every CG vector then stays zero on broken bonds
 * provided the start vector is; for other k the iteration is not conjugate gradient and the result is unspecified.
 *
 *   fcg_green_function   G[da][db] (L x L, written) = eq. (1c) on the periodic lattice with minimum-image offsets (reading F3),
 *                        the integral in closed form, evaluated in double and rounded once to the handle's dtype.
 *                        E > 0, a > 0.  Asynchronous.
 *   fcg_kernel_spectrum  s (L x L, written, row-major [m][n]) = Re F G for a real kernel G[da][db] (L x L, read-only): forward
 *                        transform by the library's own passes, real part expanded from the half spectrum.  Uses the handle's
 *                        workspace (r, p): not while a solve is pending.  s must not alias G.  Asynchronous.
 *   fcg_force_apply      y = (I + K G) x = x + k o (G x); y must not alias k or x.  Asynchronous.
 *   fcg_force_solve      CG on eq. (2): right-hand side b_i = k_i * D formed in the residual pass (one multiply in the handle's dtype);
 *                        f in: initial guess (0 on broken bonds), out: forces; stop at the first iteration with
 *                        ||r||_2 <= tol ||b||_2; iters / rel_residual / status / scalars in double / determinism as fcg_solve.
 *                        k == 0 everywhere or D == 0 gives f = 0, 0 iterations.  One CUDA graph per solve.  Where reading
 *                        F1 holds for the call -- checked on the device first (one kernel over k and f, a 32-byte read-back):
 *                        all k_i in {0, kappa} and the start vector zero on the broken bonds -- the iteration is three
 *                        launches, with p.(I + K G)p = sum p^2 + kappa sum g |P|^2 as in fcg_solve (FCG_OPT_SPECTRAL_ALPHA);
 *                        otherwise four launches in the textbook order, for any k.  At L = 256 and 512 one cooperative launch
 *                        for the whole solve, textbook order (FCG_OPT_FUSED).  Blocks.
 *   fcg_force_break_step reading F2: the response is linear in D, so the bond that reaches its threshold first is
 *                        argmax over {k_i > 0} of f_i / t_i (one IEEE divide in double; ties -> lowest i; NaN skipped);
 *                        sets k_i = 0 AND f_i = 0 (a broken bond carries nothing).  ratio_host = the winning f/t: with f
 *                        computed at displacement D the bond breaks at D_c = D / ratio.  Blocks.
 *   fcg_force_fracture   nsteps times { fcg_force_solve warm-started from the current f; fcg_force_break_step } ("For each
 *                        step in the simulation, the displacement is set, and the resulting distribution of forces is
 *                        calculated ... bonds break").  index_host, iters_host, ratio_host (may be NULL): HOST
 *                        arrays of nsteps; stops early on a negative status; steps_done_host = completed steps.
 *                        At L = 256 and 512 the whole loop -- every solve and every break step -- is ONE cooperative launch
 *                        with k, f, t resident in shared memory (fcg_fused.cuh, FORCE variant); else one graph per solve
 *                        and one break kernel per step, driven from the host.  Blocks. */
/* The same state through the displacements (reading F7): eliminating f instead of u from (1a), (1b) gives
 * (K + G^-1) u = K D, the symmetric system of fcg_solve / fcg_pcg_solve with the spectrum 1 / g and the right-hand side K D; its
 * iteration count does not grow with L (24-34 against 60, 83, 144, .. of eq. (2) at L = 256, 512, 2048), so this is the fast
 * way to the forces.  The three element-wise maps of that route (all asynchronous, one IEEE operation per element and step):
 *   fcg_inverse_spectrum         s = 1 / g  (L x L, row-major [m][n]; may be in place): the spectrum of G^-1, for fcg_set_spectrum
 *   fcg_force_rhs                b = k * D  (the right-hand side K D; b must not alias k)
 *   fcg_force_from_displacement  f = -k (u - D), eq. (1a), evaluated as k * (D - u); f may alias u
 *
 *   fcg_force_fracture_displacement  the quasi-static loop of the force model on that route: nsteps times { b = K D;
 *                        (K + G^-1) u = b by fcg_solve, or fcg_pcg_solve when use_pcg != 0, warm-started from the current u;
 *                        f = -k (u - D); break argmax over {k_i > 0} of f_i / t_i (reading F2), k_i = 0 }.  u is the plate's
 *                        displacement and is not changed by a break.  Before the call: fcg_set_spectrum with 1 / g, and for
 *                        use_pcg fcg_set_preconditioner with the same spectrum and a kbar (fixed for the whole loop).  Results
 *                        as fcg_force_fracture (ratio = winning f/t: the bond breaks at D_c = D / ratio); the break sequence is
 *                        that of fcg_force_fracture wherever the top-2 gap exceeds the solver error.  At L = 256 and 512 ONE
 *                        cooperative launch for the whole loop (fcg_fused.cuh, FORCE = 2).  Blocks.
 *   fcg_force_fracture_displacement_begin / _end   the same loop in two halves, as fcg_fracture_begin / _end: _begin enqueues (and
 *                        returns at once where the loop is the cooperative kernel; elsewhere it runs the loop to its end), _end
 *                        blocks and fills the host arrays.  For ensembles of samples: one handle per sample, each on its own
 *                        stream, all in flight from one host thread.  k, u, t must stay valid and untouched in between. */
int fcg_force_fracture_displacement(fcg_handle h, void* k, double D, void* u, const void* t, int nsteps, double tol, int maxit,
                                    int use_pcg, long long* index_host, int* iters_host, double* ratio_host, int* steps_done_host);
int fcg_force_fracture_displacement_begin(fcg_handle h, void* k, double D, void* u, const void* t, int nsteps, double tol,
                                          int maxit, int use_pcg);
int fcg_force_fracture_displacement_end(fcg_handle h, long long* index_host, int* iters_host, double* ratio_host,
                                        int* steps_done_host);
int fcg_inverse_spectrum(fcg_handle h, const void* g, void* s);
int fcg_force_rhs(fcg_handle h, const void* k, double D, void* b);
int fcg_force_from_displacement(fcg_handle h, const void* k, double D, const void* u, void* f);
int fcg_green_function(fcg_handle h, double nu, double E, double a, void* G);
int fcg_kernel_spectrum(fcg_handle h, const void* G, void* s);
int fcg_force_apply(fcg_handle h, const void* k, const void* x, void* y);
int fcg_force_solve(fcg_handle h, const void* k, double D, void* f, double tol, int maxit,
                    int* iters_host, double* rel_residual_host);
int fcg_force_break_step(fcg_handle h, void* k, void* f, const void* t, long long* index_host, double* ratio_host);
int fcg_force_fracture(fcg_handle h, void* k, double D, void* f, const void* t, int nsteps, double tol, int maxit,
                       long long* index_host, int* iters_host, double* ratio_host, int* steps_done_host);

/* ---- Slab-decomposed conjugate gradient over several ranks (the paper's remark on the bus as the
 * bottleneck between devices) ----------------------------------------------------------------
 * The path shards by rows: rank g of G owns rows [g L/G, (g+1) L/G) of every vector (k, f, u and the library's r, p, q), i.e. the
 * row pairs [g L/2G, (g+1) L/2G).  The row passes are local.  The column pass needs whole columns, so the half spectrum is
 * transposed between the ranks before and after it: rank g ends up with the columns [g L/2G, (g+1) L/2G) (whole 128-byte lines of
 * T2: L/(2 NB G) column blocks of NB columns), and the two scalars of Listing 2 (p.q and r.r) are sums over the ranks.
 * The library provides the local passes and the scalar steps; the CALLER runs the two
 * collectives -- an all-to-all with equal chunks on the send / receive buffers and an all-reduce (sum) on a device buffer of two
 * doubles -- with whatever connects the ranks (torch.distributed over NCCL in paper_1305_3625_b200/slab.py; plain copies when
 * several logical ranks share one device).  One handle per rank (fcg_create on the rank's device, then fcg_slab_configure);
 * fcg_set_spectrum takes the full L x L spectrum on every rank.  Textbook order of Listing 2, one iteration =
 *     rows_fwd(cg) | all-to-all S->R | cols (on R, in place) | all-to-all R->S | rows_inv -> xch | all-reduce | scalar(1) |
 *     update_r -> xch | all-reduce | scalar(2) | poll
 * Every rank computes alpha, beta, the count and the stopping decision itself from the all-reduced sums: identical everywhere.
 *
 *   fcg_slab_shape_of   pure host arithmetic, no device needed: how the lattice splits over nranks (FCG_UNSUPPORTED unless nranks
 *                       divides L / (2 NB) and L / 2; NB = columns per 128-byte line: 4 for FCG_F64, 8 for FCG_F32; L >= 256)
 *   fcg_slab_configure  make this handle rank `rank` of `nranks` (this slice keeps the full-size workspace of fcg_create)
 *   fcg_slab_buffers    byte offsets into the handle's workspace of the send buffer S (T2 of the own rows, ordered by destination
 *                       rank: nranks chunks of chunk_bytes) and the receive buffer R (ordered by source rank), buffer_bytes each.
 *                       Forward exchange: all-to-all S -> R; backward: all-to-all R -> S.  (The workspace must be the caller's.)
 *   fcg_slab_setup      reset the scalar block: tol, maxit (before fcg_slab_rows_inv(residual = 1))
 *   fcg_slab_rows_fwd   cg = 0: row transforms of the own rows of xu (an input vector) into S;  cg = 1: u += alpha p (lagged one
 *                       pass), p = r + beta p, row transforms of p into S (xu = the own rows of u, updated in place)
 *   fcg_slab_cols       column pass on R in place: F^H (shat o F .) of the own columns.  R is read and written where the all-to-all
 *                       left it / will take it -- [source rank][local column block][local row pair][line] -- through a 5-D tensor map,
 *                       so nothing is repacked around the exchange.  Returns at once when the solve has finished.
 *   fcg_slab_rows_inv   inverse row transforms of S;  residual = 1: r = f - (k o u + C u), p := 0, xch = { r.r, f.f } of the own rows;
 *                       residual = 0: q = k o p + C p, xch[0] = p.q of the own rows.  xch: device, caller-owned (2 doubles
 *                       used here, 4 by the three-pass form below: allocate 4)
 *   fcg_slab_update_r   r -= alpha q on the own rows, xch[0] = their r.r
 *   fcg_slab_scalar     the scalar step on the ALL-REDUCED xch: what = 0 after the residual pass (rho, ||f||^2, early exit), 1 after
 *                       rows_inv (alpha, or breakdown), 2 after update_r (count, convergence / maxit, beta, rho)
 *   fcg_slab_finish     the last lagged u += alpha p on the own rows
 *   fcg_slab_poll       read the scalar block back (blocks): done flag, iteration count, relative residual, status
 * The same iteration with the SPECTRAL SEARCH LENGTH (DESIGN.md sections 12 and 18; xch: device, 4 doubles): p.Ap = sum k p^2 +
 * sum shat |P|^2 is known after the column pass, so the residual update rides in the last pass and the update_r pass disappears:
 *     rows_fwd(cg) | exchange | cols_energy -> xch | exchange, all-reduce | scalar(4) | rows_inv(2) -> xch | all-reduce | scalar(5)
 *   fcg_slab_kpp0       after rows_inv(residual = 1): xch[2] = sum k r^2 of the own rows (the first direction is p = r), so that the
 *                       one all-reduce of the set-up carries r.r, f.f and this; then fcg_slab_scalar(0) and fcg_slab_scalar(3)
 *   fcg_slab_cols_energy  fcg_slab_cols that also leaves xch[0] = this rank's share of sum shat |P|^2 (xch[1..3] = 0)
 *   fcg_slab_rows_inv(residual = 2)   r -= alpha (k o p + C p) on the own rows, q never stored (u, f unused);
 *                       xch = { r.r, sum k r^2, sum k r p } of the own rows (the new r)
 *   fcg_slab_scalar     what = 3: start of the recurrence for sum k p^2 (xch[2] of the set-up); 4: alpha = rho / (sum k p^2 + xch[0]),
 *                       or breakdown; 5: count, convergence / maxit, beta, rho from xch[0], and sum k p'^2 = xch[1] + 2 beta xch[2] +
 *                       beta^2 sum k p^2 for the next direction
 * All calls but fcg_slab_shape_of and fcg_slab_poll are asynchronous on the handle's stream. */
typedef struct {
    int nranks, rank;
    int columns_per_line;      /* NB */
    int column_blocks;         /* L / (2 NB): 128-byte-line blocks of NB columns */
    int column_blocks_local;   /* of which this rank owns L / (2 NB nranks) */
    int row_pairs_local;       /* L / (2 nranks) */
    int rows_local;            /* L / nranks: rows [rank * rows_local, ..) of every vector */
    int columns_local, column0;/* columns [column0, column0 + columns_local) of the half spectrum (column 0 = the packed n = 0, L/2 pair) */
    size_t line_bytes;         /* 128 */
    size_t chunk_bytes;        /* one (source rank, destination rank) piece of the exchange */
    size_t buffer_bytes;       /* nranks * chunk_bytes = N w / nranks */
} fcg_slab_shape;
int fcg_slab_shape_of(int L, fcg_dtype dt, int nranks, int rank, fcg_slab_shape* out);
int fcg_slab_configure(fcg_handle h, int nranks, int rank);
int fcg_slab_buffers(fcg_handle h, size_t* send_offset, size_t* recv_offset, size_t* bytes);
/* Peer mode: the exchange FUSED INTO THE PASSES over peer memory (NVLink / NVSwitch stores), no all-to-all at all.
 *   peer_send_host[g], peer_recv_host[g]   HOST arrays of nranks DEVICE addresses, valid on this handle's device, of rank g's S and
 *                       R buffers (the own ones included; 128-byte aligned): the other handles' buffers for logical ranks on one
 *                       device, peer-enabled or cudaIpcOpenMemHandle'd mappings for one process per GPU.
 * Afterwards fcg_slab_rows_fwd stores every 128-byte line of the row-transformed half spectrum straight into the exchange buffer
 * of the rank that owns its column block (R[my rank][..] there), and fcg_slab_cols scatters the row pairs of source rank s
 * straight into rank s's S (one TMA tensor map per peer), so the transfer overlaps the transforms line by line instead of
 * following them.  The caller replaces each all-to-all by a BARRIER between the ranks (all of them have finished the pass):
 * on one stream that is implicit, across processes any stream-ordered collective does it (slab.py uses the all-reduce).
 * NULL, NULL returns to the all-to-all mode. */
int fcg_slab_set_peers(fcg_handle h, void* const* peer_send_host, void* const* peer_recv_host);
/* The same for one process per GPU: fcg_slab_ipc_export fills FCG_SLAB_IPC_BYTES host bytes (the CUDA IPC handle of the allocation
 * that holds this rank's workspace, and the offsets of S and R in it); the caller gathers the blobs of all ranks in rank order
 * (nranks * FCG_SLAB_IPC_BYTES bytes) and hands them to fcg_slab_ipc_open on every rank, which maps the peers' buffers
 * (cudaIpcOpenMemHandle with lazy peer access, i.e. over NVLink between GPUs) and calls fcg_slab_set_peers.  The workspace must
 * come from cudaMalloc (torch's default allocator qualifies; expandable segments do not). */
#define FCG_SLAB_IPC_BYTES 80
int fcg_slab_ipc_export(fcg_handle h, void* blob_host);
int fcg_slab_ipc_open(fcg_handle h, const void* blobs_host);
int fcg_slab_setup(fcg_handle h, double tol, int maxit);
int fcg_slab_rows_fwd(fcg_handle h, int cg, void* xu);
int fcg_slab_cols(fcg_handle h);
int fcg_slab_cols_energy(fcg_handle h, void* xch);
int fcg_slab_kpp0(fcg_handle h, const void* k, void* xch);
int fcg_slab_rows_inv(fcg_handle h, int residual, const void* k, const void* u, const void* f, void* xch);
int fcg_slab_update_r(fcg_handle h, void* xch);
int fcg_slab_scalar(fcg_handle h, int what, const void* xch);
int fcg_slab_finish(fcg_handle h, void* u);
int fcg_slab_poll(fcg_handle h, int* done_host, int* iters_host, double* rel_residual_host, int* status_host);

/* ---- Break step that allocates NOTHING (no handle, no workspace) ---------------------------------------------------------------
 * For callers that cannot call cudaMalloc: code under CUDA-graph stream capture, tight serving loops, harnesses that forbid
 * allocation.  The same kernel and rule as fcg_break_step (configs[3], S5, S13: over {i : k_i > 0} the maximum of
 * (k_i * u_i) / t_i in double, ties -> lowest i, NaN skipped, k_i := 0 at the winner), but its scratch -- one partial (ratio,
 * index) per CTA and an arrival ticket -- lives in a static device array of FCG_BREAK_STATIC_SCRATCH_BYTES inside libfcg.so, which
 * every GPU that loads the library holds until the process exits.  The call enqueues one 4-byte memset (the ticket must start at
 * zero; the array otherwise keeps the last call's contents) and one kernel on `cuda_stream` of the CURRENT device and returns:
 * no cudaMalloc / cudaFree / allocating routine, no host synchronisation, no device-to-host copy.
 *   dt, n        element type and count of k, u, t;  1 <= n <= FCG_BREAK_STATIC_MAX_N (= 8192 * 8192, the largest lattice of
 *                this library), else FCG_UNSUPPORTED; the arrays need not be a square lattice
 *   k            device, in/out (k[index] := 0);  u, t  device, read-only;  all 16-byte aligned
 *   result_dev   device, 8-byte aligned, caller-owned: receives one fcg_break_result { index (-1: no candidate), ratio, status
 *                (FCG_OK or FCG_NO_CANDIDATE) } when the kernel has run
 *   cuda_stream  a cudaStream_t of the current device (NULL: default stream)
 * All calls on a device share the one array: calls whose kernels may OVERLAP on the GPU (different streams without an ordering
 * between them, concurrent graph branches) race on it and give wrong results -- keep them on one stream or order them.
 * Returns FCG_OK when enqueued; on error fcg_static_last_error() (per host thread) says why. */
#define FCG_BREAK_STATIC_MAX_N (8192LL * 8192LL)
#define FCG_BREAK_STATIC_SCRATCH_BYTES 19200
typedef struct { long long index; double ratio; int status; int pad_; } fcg_break_result;
int fcg_break_step_static(fcg_dtype dt, long long n, void* k, const void* u, const void* t, void* result_dev, void* cuda_stream);
const char* fcg_static_last_error(void);

/* Measurement aid: runs the set-up of fcg_solve and then `iters` iterations of the CG loop body as direct
 * launches with CUDA events between the four kernels (tol = 0: never stops early), and returns their mean
 * device times in milliseconds, ms_host[0..3] = { row pass forward (P1), column pass (P2), row pass inverse
 * (P3), residual update (P4) }; with the default three-launch iteration (FCG_OPT_SPECTRAL_ALPHA = 1) P3 includes the residual
 * update and ms_host[3] is the time between two adjacent events (~2.6 us).  Kernels run in loop order, so each sees the cache state its predecessor
 * leaves.  u is overwritten with an unfinished iterate.  Blocks until done.  Returns FCG_NOT_CONVERGED if the
 * loop flagged completion (times then include early exits and are not meaningful). */
int fcg_profile_iteration(fcg_handle h, const void* k, const void* f, void* u, int iters, double* ms_host);

/* The same for one iteration of fcg_pcg_solve (pipelined engine only, else FCG_UNSUPPORTED): ms_host[0..5] =
 * { P1 (u, p updates + row transforms), P2 (spectrum), P3 (q, p.q), r update + r.r + row transforms of r,
 *   P2 (preconditioner), P3 (z, r.z) }. */
int fcg_profile_pcg_iteration(fcg_handle h, const void* k, const void* f, void* u, int iters, double* ms_host);

/* Number of this library's kernel launches enqueued by the last fcg_solve / fcg_solve_host /
 * fcg_fracture call on this handle (graph kernel nodes counted once per execution). */
long long fcg_last_launch_count(fcg_handle h);

const char* fcg_last_error(fcg_handle h);
const char* fcg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FCG_H */
