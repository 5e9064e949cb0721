// fcg_passes.cuh -- the three transform passes of one operator application  q = k o p + C p
// (Listing 4), each fused with its neighbouring vector work of Listing 2
// (PAPER.md:88-100).  Data layout and byte counts: DESIGN.md sections 3-4.
//
//   row_fwd  (P1): [u += alpha p; p = r + beta p;]  T[n][a] = sum_b p[a,b] w^{n b},  n < L/2
//   col_conv (P2): T[n][.] <- F_col^H ( shat[n][.] o F_col T[n][.] )               (in place)
//   row_inv  (P3): c = F_row^H T;  q = k o p + c  [+ partial p.q]  (or residual / apply / plain)
//
// Two real rows are transformed by one complex FFT (z = x_even + i x_odd) and separated with
// X_even[n] = (Z[n] + conj Z[L-n])/2, X_odd[n] = (Z[n] - conj Z[L-n])/(2i).  Row n = 0 of T packs the
// two purely real columns n = 0 and n = L/2 as T[0][a] = X_a[0] + i X_a[L/2], so T is exactly
// L/2 x L complex.  T is stored transposed (n-major) so that the column pass streams contiguous
// columns; the transposition happens in the row passes through shared memory, with 2F*sizeof(complex)
// contiguous bytes per n.
//
// Every body is written against a Runner: run(f) executes f(tid) for each thread of the CTA followed
// by a CTA barrier.  On the device that is one call + __syncthreads(); the host harness
// (tests/emul) loops over tid instead, which lets the index algebra be checked without a GPU.
#pragma once
#include <type_traits>
#include "fcg_engine.cuh"

namespace fcg {

// Device-resident CG state (one per handle).  All scalars are double for both dtypes (reading S12).
struct Scalars {
    double rho, pq, alpha, beta, fn2, tol, relres;
    int it, maxit, done, status, zero_u, use_cond;
    unsigned int ticket[4];
    unsigned long long cond;       // cudaGraphConditionalHandle of the WHILE node (loop mode 0)
    int steps_done, pad_;          // fused quasi-static loop: completed break steps
    int pcg, pad2_;                // 1: preconditioned CG (rho = r.z, rr = r.r kept apart)
    double rr;                     // PCG: r.r of the current residual
    double kpp;                    // spectral search length: sum k p^2 from P1; P2 adds sum shat |P|^2
    unsigned int ticket2[2];       // [0] P1's k p^2 reduction, [1] P2's spectral-energy reduction
    unsigned int timeout, pad3_;   // raised by a pipelined pass whose mbarrier wait gave up (fcg_tma.cuh); sticky until fcg_destroy
};

enum { ROWF_PLAIN = 0, ROWF_CG = 1, ROWF_RUPD = 2 };   // RUPD (PCG): r -= alpha q, partial r.r, row transforms of r
enum { ROWI_PLAIN = 0, ROWI_CG = 1, ROWI_RESID = 2, ROWI_APPLY = 3, ROWI_PRECOND = 4, ROWI_CGF = 5 };   // PRECOND (PCG): z = M^-1 r, partial r.z (k = r)
enum { COL_CONV = 0, COL_FWD = 1, COL_INV = 2 };

template <typename T> struct RowFwdArgs {
    int mode;
    const T* x;            // PLAIN: input field
    T* u; T* p; const T* r;        // CG: vectors updated in place / read
    cx<T>* Tb;             // [L/2][L] transposed half spectrum
    const cx<T>* tw;       // per-stage twiddle tables (Plan::tw_off)
    Scalars* sc;
    int nsm;               // SMs of the device (persistent passes: tile assignment)
    int pdl;               // host side: launch with programmatic stream serialization
    int check_done;        // PLAIN inside the PCG loop: return at once when sc->done
    const T* q;            // RUPD: q = A p (read);  r is updated in place through rw
    T* rw;                 // RUPD: r (read / write)
    double* partial;       // RUPD: [gridDim.x] partial r.r
    int hints;             // L2 eviction-priority hints (FCG_OPT_L2_HINTS bit mask; pipelined passes only)
    unsigned int* tmo;     // pipelined passes: raised when an mbarrier wait gives up (fcg_tma.cuh); = &Scalars::timeout
    int ntile, astride;    // slab instantiation: row pairs of this rank, and row pairs per column block of ITS T2
    // slab, exchange fused into the pass (peer mode): the line of column block mb goes straight into the exchange buffer R of the rank
    // that owns the block, peerR[mb / mbl], at [my rank][mb % mbl][local row pair] -- a store over NVLink (or into the same device
    // for logical ranks).  npeer == 0: the lines stay in the own T2 (Tb) and an all-to-all moves them.
    int npeer, prank, mbl;
    cx<T>* peerR[16];
    int stagger_ns;        // start offset between the CTAs that share an SM (fcg_tma.cuh: stagger_wait); 0: none
};

template <typename T> struct ColArgs {
    int mode;
    cx<T>* Tb;             // in place
    const T* shat;         // [(L/2)+1][L], digit-reversed along m, pre-scaled by 1/L^2
    const cx<T>* tw;
    const Scalars* sc;
    int pdl;
    int hints;
    double* partial;       // ENERGY instantiation: [L/2] partial sums of shat |P|^2, one per column
    int nsm;               // persistent column pass: SMs of the device
    unsigned int* tmo;     // pipelined passes: raised when an mbarrier wait gives up
    int col0;              // slab instantiation: global number of this launch's first column (spectrum row, packed column 0)
    int nranks, al, boxa;  // slab: source ranks, row pairs per rank, row pairs per box of the 5-D map of the exchange buffer
    const void* peer_maps; // slab, peer mode: device array of nranks CUtensorMap, one per rank's T2 (rows side); the scatter of source
    int prank, mbl;        //   rank s's row pairs goes straight there, to column block prank * mbl + local block.  nullptr: back into R
    cx<T>* X;              // stand-alone transforms (col2_xpub_kernel): the public half spectrum X[m][n], L x (L/2+1)
    int stagger_ns;        // col2_kernel: start offset between the first-wave CTAs that share an SM (0: none)
};

template <typename T> struct RowInvArgs {
    int mode;
    const cx<T>* Tb;
    const cx<T>* tw;
    const T* k; const T* v; const T* f;   // CG: v = p;  RESID: v = u, f;  APPLY: v = x
    T* out; T* out2;                      // CG: q;  RESID: r, p(:=0);  APPLY: y;  PLAIN: x
    T scale;                              // PLAIN: 1/L^2
    double* partial;                      // [gridDim.x][2]
    Scalars* sc;
    int nsm;
    int pdl;
    int hints;
    const double* colsum;                 // CGF: the column pass's L/2 partial sums of shat |P|^2
    int form;                             // 0: A x = k o x + C x (BASELINE.json);  1: force formulation B x = x + k o (C x), the left side
                                          //    of eq. (2), PAPER.md:74 (CG, RESID, APPLY)
    T dval;                               // form 1, RESID: right-hand side b = k * dval (K D of eq. (2)); f is not read
    double kappa;                         // form 1, CGF (three launches, reading F1: k in {0, kappa}, vectors zero on broken bonds):
                                          //    p.(I + K G)p = sum p^2 + kappa sum g |P|^2
    unsigned int* tmo;                    // pipelined passes: raised when an mbarrier wait gives up
    int ntile;                            // slab instantiation: row pairs of this rank
    int stagger_ns;                       // start offset between the CTAs that share an SM; 0: none
    double* xch;                          // slab: the pass's grid-wide sums go HERE (device; 2 doubles, 4 in the fused form) and no scalar step follows:
                                          //       they are this rank's share, to be all-reduced first (fcg_slab_scalar)
};

template <int A, int B, typename F> FCG_HD void static_for_up(F&& f) {
    if constexpr (A <= B) { f(std::integral_constant<int, A>{}); static_for_up<A + 1, B>(f); }
}
template <int A, int B, typename F> FCG_HD void static_for_down(F&& f) {
    if constexpr (A >= B) { f(std::integral_constant<int, A>{}); static_for_down<A - 1, B>(f); }
}

// Region stride of one packed transform in shared memory (elements).  The +2 skew puts the F regions of a
// row-pass CTA on different banks when F lanes read the same position of F different transforms.
template <typename P> constexpr int region_stride() { return P::N + 2; }

// Host: fill the per-stage twiddle tables of plan P (layout: Plan::tw_off).  Every entry is evaluated in
// double from its own reduced angle index (no recurrences) and rounded once to T.
template <typename T, typename P>
inline void fill_twiddles(cx<T>* out) {
    for (int sv = 1; sv < P::S; ++sv) {
        const int R = P::radix(sv), M = P::mlen(sv), Q = M / R, off = P::tw_off(sv);
        for (int u = 1; u < R; ++u)
            for (int j = 0; j < Q; ++j) {
                const double ang = 2.0 * 3.14159265358979323846 * (double)((j * u) % M) / (double)M;
                cx<T> w; w.x = (T)cos(ang); w.y = (T)(-sin(ang));
                out[off + (u - 1) * Q + j] = w;
            }
    }
}

// shat[n][pos(m)] from the caller's s[m][n]: even part, 1/L^2, digit-reversed along m; row 0 and row L/2
// hold (s0 + sN)/2 and (s0 - sN)/2 for the packed n = 0 / n = L/2 column (col_body); within a row the entry of
// position e sits at Plan::shat_index(e).  idx = m*(L/2) + n.
// colpos = false: the row of column frequency n is n (classic passes);  colpos = true: it is the column's number in the
// position-ordered layout T2 of the pipelined passes, m = (e / RLAST)(RLAST/2) + e % RLAST with e = pos_of(n).
template <typename T, typename P>
FCG_HD void spectrum_prep_one(int idx, const T* __restrict__ s, T* __restrict__ shat, bool colpos = false) {
    constexpr int L = P::N;
    const T scale = (T)(1.0 / ((double)L * (double)L));
    const T h = (T)0.5;
    const int m = idx / (L / 2), n = idx % (L / 2);
    const int mm = (L - m) % L;
    const int e = P::shat_index(P::pos_of(m));
    if (n > 0) {
        const T ev = (s[(size_t)m * L + n] + s[(size_t)mm * L + (L - n)]) * h;
        const int en = P::pos_of(n);
        const int row = colpos ? (en / P::RLAST) * (P::RLAST / 2) + en % P::RLAST : n;
        shat[(size_t)row * L + e] = ev * scale;
    } else {
        const T s0 = (s[(size_t)m * L] + s[(size_t)mm * L]) * h * scale;
        const T sN = (s[(size_t)m * L + L / 2] + s[(size_t)mm * L + L / 2]) * h * scale;
        shat[e] = (s0 + sN) * h;
        shat[(size_t)(L / 2) * L + e] = (s0 - sN) * h;
    }
}

// --------------------------------------------------------------------------------------------- P1
template <typename T, typename P, int F, typename Runner>
FCG_HD void row_fwd_body(const RowFwdArgs<T>& A, int block, cx<T>* smem, Runner& run)
{
    constexpr int L = P::N, S = P::S, NT = P::NT;
    const int a0 = block * 2 * F;
    T alpha = (T)0, beta = (T)0;
    if (A.mode == ROWF_CG) { alpha = (T)A.sc->alpha; beta = (T)A.sc->beta; }

    // stage 1: global -> (vector update) -> butterfly -> shared
    run([&](int tid) {
        const int f = tid / NT, lt = tid % NT;
        SmemIO<T, P> io{smem + f * region_stride<P>()};
        const size_t row0 = (size_t)(a0 + 2 * f) * L, row1 = row0 + L;
        auto ld = [&](int e) -> cx<T> {
            if (A.mode == ROWF_CG) {
                T p0 = A.p[row0 + e], p1 = A.p[row1 + e];
                const T r0 = A.r[row0 + e], r1 = A.r[row1 + e];
                T u0 = A.u[row0 + e], u1 = A.u[row1 + e];
                u0 = u0 + alpha * p0; u1 = u1 + alpha * p1;       // new x, lagged one pass
                p0 = r0 + beta * p0;  p1 = r1 + beta * p1;        // new direction
                A.u[row0 + e] = u0; A.u[row1 + e] = u1;
                A.p[row0 + e] = p0; A.p[row1 + e] = p1;
                return mk<T>(p0, p1);
            }
            return mk<T>(A.x[row0 + e], A.x[row1 + e]);
        };
        run_stage<P, 1, -1, T>(lt, A.tw, ld, [&](int e, cx<T> v) { io.st(e, v); });
    });
    // stages 2..S in shared memory
    static_for_up<2, S>([&](auto s) {
        run([&](int tid) {
            const int f = tid / NT, lt = tid % NT;
            SmemIO<T, P> io{smem + f * region_stride<P>()};
            run_stage<P, decltype(s)::value, -1, T>(lt, A.tw, [&](int e) { return io.ld(e); },
                                                    [&](int e, cx<T> v) { io.st(e, v); });
        });
    });
    // separate the two rows of each packed transform and store transposed: lanes run over f first, so a
    // warp writes 2F consecutive complex numbers per n
    run([&](int tid) {
        constexpr int ITEMS = F * (L / 2), NTH = F * NT;
        const T h = (T)0.5;
#pragma unroll 4
        for (int item = tid; item < ITEMS; item += NTH) {
            const int f = item % F, n = item / F;
            SmemIO<T, P> io{smem + f * region_stride<P>()};
            cx<T> X0, X1;
            if (n == 0) {
                const cx<T> Z0 = io.ld(P::pos_of(0)), ZN = io.ld(P::pos_of(L / 2));
                X0 = mk<T>(Z0.x, ZN.x); X1 = mk<T>(Z0.y, ZN.y);
            } else {
                const cx<T> Za = io.ld(P::pos_of(n)), Zb = io.ld(P::pos_of(L - n));
                X0 = mk<T>((Za.x + Zb.x) * h, (Za.y - Zb.y) * h);
                X1 = mk<T>((Za.y + Zb.y) * h, (Zb.x - Za.x) * h);
            }
            cx<T>* dst = A.Tb + (size_t)n * L + a0 + 2 * f;
            dst[0] = X0; dst[1] = X1;
        }
    });
}

// --------------------------------------------------------------------------------------------- P2
// COLS columns per CTA, column n = block*COLS + c, region c of shared memory.
template <typename T, typename P, int COLS, typename Runner>
FCG_HD void col_body(const ColArgs<T>& A, int block, cx<T>* smem, Runner& run)
{
    constexpr int L = P::N, S = P::S, NT = P::NT;
    const int n0 = block * COLS;
    const bool special = (A.mode == COL_CONV) && (n0 == 0);    // this CTA holds the packed n=0 / n=L/2 column
    auto region = [&](int tid) { return SmemIO<T, P>{smem + (tid / NT) * region_stride<P>()}; };
    auto column = [&](int tid) { return A.Tb + (size_t)(n0 + tid / NT) * L; };

    auto fwd_stage = [&](auto s) {           // stage s forward: loads global iff s == 1, stores shared
        run([&](int tid) {
            auto io = region(tid); cx<T>* col = column(tid);
            constexpr int sv = decltype(s)::value;
            if constexpr (sv == 1)
                run_stage<P, 1, -1, T>(tid % NT, A.tw, [&](int e) { return col[e]; }, [&](int e, cx<T> v) { io.st(e, v); });
            else
                run_stage<P, sv, -1, T>(tid % NT, A.tw, [&](int e) { return io.ld(e); }, [&](int e, cx<T> v) { io.st(e, v); });
        });
    };
    auto inv_stage = [&](auto s) {           // stage s inverse: loads shared, stores global iff s == 1
        run([&](int tid) {
            auto io = region(tid); cx<T>* col = column(tid);
            constexpr int sv = decltype(s)::value;
            if constexpr (sv == 1)
                run_stage<P, 1, +1, T>(tid % NT, A.tw, [&](int e) { return io.ld(e); }, [&](int e, cx<T> v) { col[e] = v; });
            else
                run_stage<P, sv, +1, T>(tid % NT, A.tw, [&](int e) { return io.ld(e); }, [&](int e, cx<T> v) { io.st(e, v); });
        });
    };

    if (A.mode == COL_CONV && !special) {
        static_for_up<1, S - 1>(fwd_stage);
        run([&](int tid) {                   // last forward stage * shat * first inverse stage, in registers
            auto io = region(tid); cx<T>* col = column(tid);
            const T* sh = A.shat + (size_t)(n0 + tid / NT) * L;
            if constexpr (S == 1)
                run_middle<P, T>(tid % NT, [&](int e) { return col[e]; }, [&](int e, cx<T> v) { col[e] = v; },
                                 [&](int g, int u) { return sh[u * (L / P::RLAST) + g]; });
            else
                run_middle<P, T>(tid % NT, [&](int e) { return io.ld(e); }, [&](int e, cx<T> v) { io.st(e, v); },
                                 [&](int g, int u) { return sh[u * (L / P::RLAST) + g]; });
        });
        static_for_down<S - 1, 1>(inv_stage);
        return;
    }
    if (A.mode == COL_CONV) {                // special CTA: column 0 needs W[m] and W[-m] together
        static_for_up<1, S>(fwd_stage);
        run([&](int tid) {
            auto io = region(tid);
            const int c = tid / NT, lt = tid % NT;
            const T* sh = A.shat + (size_t)(n0 + c) * L;
            if (c == 0) {
                // packed column: W = Y0 + i YN.  W'[m] = sp[m] W[m] + sm[m] conj W[-m],
                // sp = (s0 + sN)/2 (row 0 of shat), sm = (s0 - sN)/2 (row L/2 of shat); pairs (m, L-m), m <= L/2
                const T* sm_ = A.shat + (size_t)(L / 2) * L;
                for (int m = lt; m <= L / 2; m += NT) {
                    const int e = P::pos_of(m), e2 = P::pos_of((L - m) % L);
                    const cx<T> Wa = io.ld(e), Wb = io.ld(e2);
                    cx<T> va, vb;
                    const int i1 = P::shat_index(e), i2 = P::shat_index(e2);
                    va.x = sh[i1] * Wa.x + sm_[i1] * Wb.x; va.y = sh[i1] * Wa.y - sm_[i1] * Wb.y;
                    vb.x = sh[i2] * Wb.x + sm_[i2] * Wa.x; vb.y = sh[i2] * Wb.y - sm_[i2] * Wa.y;
                    io.st(e, va);
                    if (e2 != e) io.st(e2, vb);
                }
            } else {
                for (int e = lt; e < L; e += NT) { cx<T> w = io.ld(e); const T sv = sh[P::shat_index(e)]; w.x *= sv; w.y *= sv; io.st(e, w); }
            }
        });
        static_for_down<S, 1>(inv_stage);
        return;
    }
    if (A.mode == COL_FWD) {                 // public transform: forward only, natural m order out (in place)
        static_for_up<1, S>(fwd_stage);
        run([&](int tid) {
            auto io = region(tid); cx<T>* col = column(tid);
            for (int m = tid % NT; m < L; m += NT) col[m] = io.ld(P::pos_of(m));
        });
        return;
    }
    // COL_INV: natural m order in, inverse only
    run([&](int tid) {
        auto io = region(tid); cx<T>* col = column(tid);
        for (int m = tid % NT; m < L; m += NT) io.st(P::pos_of(m), col[m]);
    });
    static_for_down<S, 1>(inv_stage);
}

// --------------------------------------------------------------------------------------------- P3
// acc[0], acc[1]: this thread's (device) or this CTA's (host harness) partial dot products.
template <typename T, typename P, int F, typename Runner>
FCG_HD void row_inv_body(const RowInvArgs<T>& A, int block, cx<T>* smem, Runner& run, double (&acc)[2])
{
    constexpr int L = P::N, S = P::S, NT = P::NT;
    const int a0 = block * 2 * F;
    // load T[n][a0 + 2f .. +1], rebuild the packed spectrum Z = X_even + i X_odd at its digit-reversed place
    run([&](int tid) {
        constexpr int ITEMS = F * (L / 2), NTH = F * NT;
#pragma unroll 4
        for (int item = tid; item < ITEMS; item += NTH) {
            const int f = item % F, n = item / F;
            SmemIO<T, P> io{smem + f * region_stride<P>()};
            const cx<T>* src = A.Tb + (size_t)n * L + a0 + 2 * f;
            const cx<T> X0 = src[0], X1 = src[1];
            if (n == 0) {
                io.st(P::pos_of(0), mk<T>(X0.x, X1.x));
                io.st(P::pos_of(L / 2), mk<T>(X0.y, X1.y));
            } else {
                io.st(P::pos_of(n), mk<T>(X0.x - X1.y, X0.y + X1.x));
                io.st(P::pos_of(L - n), mk<T>(X0.x + X1.y, X1.x - X0.y));
            }
        }
    });
    static_for_down<S, 2>([&](auto s) {
        run([&](int tid) {
            const int f = tid / NT, lt = tid % NT;
            SmemIO<T, P> io{smem + f * region_stride<P>()};
            run_stage<P, decltype(s)::value, +1, T>(lt, A.tw, [&](int e) { return io.ld(e); },
                                                    [&](int e, cx<T> v) { io.st(e, v); });
        });
    });
    // inverse stage 1 straight into the epilogue: natural order, re = even row, im = odd row
    run([&](int tid) {
        const int f = tid / NT, lt = tid % NT;
        SmemIO<T, P> io{smem + f * region_stride<P>()};
        const size_t row0 = (size_t)(a0 + 2 * f) * L, row1 = row0 + L;
        auto emit = [&](size_t i, T c) {
            if (A.mode == ROWI_PLAIN) { A.out[i] = c * A.scale; return; }
            if (A.mode == ROWI_PRECOND) {                          // z = M^-1 r, r.z  (PCG; k = r)
                A.out[i] = c; acc[0] += (double)A.k[i] * (double)c; return;
            }
            const T vi = A.v[i], ki = A.k[i];
            const T val = A.form ? vi + ki * c : ki * vi + c;      // k o x + C x, or x + k o (G x) (eq. (2))
            if (A.mode == ROWI_RESID) {
                const T fi = A.form ? ki * A.dval : A.f[i], ri = fi - val;   // r = f - A u;  form 1: f = K D
                A.out[i] = ri; A.out2[i] = (T)0;
                acc[0] += (double)ri * (double)ri; acc[1] += (double)fi * (double)fi;
            } else {
                A.out[i] = val;
                acc[0] += (double)vi * (double)val;                // search length p.Ap
            }
        };
        run_stage<P, 1, +1, T>(lt, A.tw, [&](int e) { return io.ld(e); },
                               [&](int e, cx<T> v) { emit(row0 + e, v.x); emit(row1 + e, v.y); });
    });
}

}  // namespace fcg
