// fcg_engine.cuh -- one transform stage as seen by one thread, with pluggable element load/store.
//
// A stage of plan P (fcg_math.cuh) consists of N/R independent radix-R butterflies.  A transform is
// worked on by P::NT = N/RMAX threads; thread `lt` owns butterflies g = lt + i*NT.  Consecutive
// threads own consecutive elements, so both the shared-memory accesses (after Swz) and the global
// accesses of the first/last stage are contiguous across a warp.
//
// ld(e) returns logical element e of the transform, st(e, v) stores it.  "Logical" means the plain
// in-place index; the caller maps it to swizzled shared memory or to global memory.
#pragma once
#include "fcg_math.cuh"

namespace fcg {

// tw = per-stage twiddle tables of the plan (Plan::tw_off, forward sign); the inverse uses the conjugate.
template <typename P, int s, int DIR, typename T, typename LD, typename ST>
FCG_HD void run_stage(int lt, const cx<T>* __restrict__ tw, LD ld, ST st)
{
    constexpr int R = P::radix(s);
    constexpr int M = P::mlen(s);          // sub-block length
    constexpr int Q = M / R;               // element stride inside a butterfly
    constexpr int NB = P::N / R;           // butterflies in this stage
    constexpr int PER = NB / P::NT;        // butterflies per thread
    constexpr int TWO = P::tw_off(s);      // w_M^{j u} = tw[TWO + (u-1) Q + j]
    static_assert(PER >= 1, "plan: NT too large for this radix");
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const int g = lt + i * P::NT;
        const int blk = g / Q, j = g % Q;
        const int base = blk * M + j;
        cx<T> a[R];
#pragma unroll
        for (int t = 0; t < R; ++t) a[t] = ld(base + t * Q);
        if (DIR < 0) {
            dftR<R, -1>(a);
            if (Q > 1) {
#pragma unroll
                for (int u = 1; u < R; ++u) a[u] = cmulw(a[u], tw[TWO + (u - 1) * Q + j]);
            }
        } else {
            if (Q > 1) {
#pragma unroll
                for (int u = 1; u < R; ++u) a[u] = cmulwc(a[u], tw[TWO + (u - 1) * Q + j]);
            }
            dftR<R, +1>(a);
        }
#pragma unroll
        for (int t = 0; t < R; ++t) st(base + t * Q, a[t]);
    }
}

template <typename P, int s> struct St {
    static constexpr int R = P::radix(s), M = P::mlen(s), Q = M / R, NB = P::N / R, PER = NB / P::NT, TWO = P::tw_off(s);
    static_assert(PER >= 1, "plan: NT too large for this radix");
};

// Which butterflies a thread owns.  Natural: g = lt + i NT (cyclic over the CTA's threads), which makes every stage depend on
// every thread of the previous one: a CTA barrier after each stage.  But after stage 1 a decimation-in-frequency transform
// falls apart into R1 independent sub-transforms of length N / R1 (and the adjoint inverse only joins them again in its last
// stage, stage 1), so the stages 2 .. S need no exchange between threads that own different sub-blocks.  GROUPED assignment:
// the NT threads form G groups of TPG consecutive threads (whole warps); group j owns the sub-blocks [j R1/G, (j+1) R1/G) in
// EVERY stage >= 2, i.e. the contiguous butterfly range [j PER TPG, (j+1) PER TPG) of each stage, dealt cyclically inside the
// group.  A warp instruction still covers 32 consecutive butterflies (same shared-memory bank behaviour), and between two
// stages >= 2 only the group has to synchronise: __syncwarp() where a group is one warp (every plan but L = 8192), a named
// barrier of TPG threads otherwise.  The groups of a CTA drift apart, so one group's shared-memory phase overlaps another's
// arithmetic -- with CTA barriers all warps alternate between the two in lock-step.
template <typename P> struct Grp {
    static constexpr int G_ = P::NT / 32 < P::R1 ? P::NT / 32 : P::R1;
    static constexpr int G = G_ < 1 ? 1 : G_;
    static constexpr int TPG = P::NT / G;
    static_assert(P::NT % G == 0 && P::R1 % G == 0, "groups must divide the threads and the stage-2 sub-blocks");
};
template <typename P, int s, bool GR> FCG_HD int bfly(int lt, int i) {
    if constexpr (!GR || s == 1) return lt + i * P::NT;
    else return (lt / Grp<P>::TPG) * (St<P, s>::PER * Grp<P>::TPG) + lt % Grp<P>::TPG + i * Grp<P>::TPG;
}
#ifdef __CUDACC__
// synchronise the threads that share sub-blocks with me (all of them call this): between two stages >= 2 of a GROUPED transform
template <typename P> __device__ __forceinline__ void group_sync(int lt) {
    if constexpr (Grp<P>::TPG == 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(2 + lt / Grp<P>::TPG), "n"(Grp<P>::TPG) : "memory");
}
#endif

// Last forward stage, a pointwise real multiply, and the first inverse stage, all in registers:
//   a <- DFT_R(a);  a[u] *= mul(e_u);  a <- DFT_R^H(a)
// (the last stage has Q = 1, so no twiddles are involved).  mul(g, u) returns the real factor for position g*R + u.
// ENERGY: *energy += sum of mul * |a|^2 over this thread's elements after the forward stage: the R products of one butterfly
// are summed in the working precision, the butterflies' sums in double.
template <typename P, typename T, bool ENERGY = false, bool GR = false, typename LD, typename ST, typename MUL>
FCG_HD void run_middle(int lt, LD ld, ST st, MUL mul, double* energy = nullptr)
{
    constexpr int R = P::RLAST;
    constexpr int NB = P::N / R;
    constexpr int PER = NB / P::NT;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const int g = bfly<P, P::S, GR>(lt, i);
        const int base = g * R;
        cx<T> a[R];
#pragma unroll
        for (int t = 0; t < R; ++t) a[t] = ld(base + t);
        dftR<R, -1>(a);
#ifdef FCG_ENERGY_WIDE
        double e = 0.0;
#else
        T e = (T)0;
#endif
#pragma unroll
        for (int u = 0; u < R; ++u) {
            const T sv = mul(g, u);
#ifdef FCG_ENERGY_WIDE
            if constexpr (ENERGY) e += (double)sv * ((double)a[u].x * (double)a[u].x + (double)a[u].y * (double)a[u].y);
#else
            if constexpr (ENERGY) e += sv * (a[u].x * a[u].x + a[u].y * a[u].y);
#endif
            a[u].x *= sv; a[u].y *= sv;
        }
        if constexpr (ENERGY) *energy += (double)e;
        dftR<R, +1>(a);
#pragma unroll
        for (int t = 0; t < R; ++t) st(base + t, a[t]);
    }
}

// ---- register-resident stages (used by the pipelined passes, fcg_async.cuh) ----------------------------
// The same stage split into load / math / store so that barriers, asynchronous-copy waits and fused epilogues
// can be placed between the steps.  Twiddles are not read from the [u][j] tables: each thread keeps the base
// twiddle w = w_M^j of each of its butterflies (one table entry, fetched once at kernel start) and forms the
// powers w^2 .. w^(R-1) by a product tree (apply_twiddles, error <= ~4 ulp), which costs no memory traffic.
// a[u] *= w^u (CONJ: conj(w)^u), u = 1 .. R-1.  Two ways to form the powers, chosen per kernel by measurement (it is a
// register-allocation matter: row_fwd2 at L=2048 fp64 runs 39 us with CHAIN and 44 us with the tree, row_inv2 36 vs 39):
//   tree : w^u = w^(u/2) w^(u - u/2), depth log2 R products (error <= ~4 ulp), all powers live at once;
//   CHAIN: w^2, w^3, w^4 by products, then four interleaved chains w^u = w^(u-4) w^4 (depth <= 5, <= ~6 ulp),
//          at most five powers live at a time.
template <int R, bool CONJ, bool CHAIN, typename C> FCG_HD void apply_twiddles(C (&a)[R], C w) {
    auto mul = [](C x, C t) { return CONJ ? cmulwc(x, t) : cmulw(x, t); };
    if constexpr (!CHAIN) {
        C pw[R];
        pw[0] = w;
        if constexpr (R > 1) pw[1] = w;
#pragma unroll
        for (int u = 2; u < R; ++u) pw[u] = cmulw(pw[u / 2], pw[u - u / 2]);
#pragma unroll
        for (int u = 1; u < R; ++u) a[u] = mul(a[u], pw[u]);
    } else {
        if constexpr (R > 1) a[1] = mul(a[1], w);
        if constexpr (R > 2) {
            const C w2 = cmulw(w, w);
            a[2] = mul(a[2], w2);
            if constexpr (R > 3) {
                const C w3 = cmulw(w2, w);
                a[3] = mul(a[3], w3);
                if constexpr (R > 4) {
                    const C w4 = cmulw(w2, w2);
                    C c0 = w4, c1 = w, c2 = w2, c3 = w3;          // c_k holds w^(4 j + k), advanced by w^4
                    a[4] = mul(a[4], c0);
#pragma unroll
                    for (int u = 5; u < R; ++u) {
                        C& c = (u % 4 == 0) ? c0 : (u % 4 == 1) ? c1 : (u % 4 == 2) ? c2 : c3;
                        c = cmulw(c, w4);
                        a[u] = mul(a[u], c);
                    }
                }
            }
        }
    }
}

// base twiddles of this thread's butterflies in stage s (u = 1 row of the stage's table)
template <typename P, int s, typename T, bool GR = false> FCG_HD void base_tw(int lt, const cx<T>* __restrict__ tw, cx<T>* w) {
    using I = St<P, s>;
    if constexpr (I::Q > 1) {
#pragma unroll
        for (int i = 0; i < I::PER; ++i) w[i] = tw[I::TWO + bfly<P, s, GR>(lt, i) % I::Q];
    }
}

template <typename P, int s, typename T, bool GR = false, typename LD>
FCG_HD void stage_ld(int lt, LD ld, cx<T> (&a)[St<P, s>::PER][St<P, s>::R]) {
    using I = St<P, s>;
#pragma unroll
    for (int i = 0; i < I::PER; ++i) {
        const int g = bfly<P, s, GR>(lt, i);
        const int base = (g / I::Q) * I::M + g % I::Q;
#pragma unroll
        for (int t = 0; t < I::R; ++t) a[i][t] = ld(base + t * I::Q);
    }
}
template <typename P, int s, typename T, bool GR = false, typename ST>
FCG_HD void stage_st(int lt, ST st, const cx<T> (&a)[St<P, s>::PER][St<P, s>::R]) {
    using I = St<P, s>;
#pragma unroll
    for (int i = 0; i < I::PER; ++i) {
        const int g = bfly<P, s, GR>(lt, i);
        const int base = (g / I::Q) * I::M + g % I::Q;
#pragma unroll
        for (int t = 0; t < I::R; ++t) st(base + t * I::Q, a[i][t]);
    }
}
// DIR < 0: a <- DFT_R(a), a[u] *= w^(u);   DIR > 0 (adjoint, run in reverse stage order): a[u] *= conj(w^u), a <- DFT_R^H(a)
template <typename P, int s, int DIR, typename T, bool CHAIN = false>
FCG_HD void stage_math(cx<T> (&a)[St<P, s>::PER][St<P, s>::R], const cx<T>* w) {
    using I = St<P, s>;
#pragma unroll
    for (int i = 0; i < I::PER; ++i) {
        if constexpr (DIR < 0) {
            dftR<I::R, -1>(a[i]);
            if constexpr (I::Q > 1) {
                apply_twiddles<I::R, false, CHAIN>(a[i], w[i]);
            }
        } else {
            if constexpr (I::Q > 1) {
                apply_twiddles<I::R, true, CHAIN>(a[i], w[i]);
            }
            dftR<I::R, +1>(a[i]);
        }
    }
}

// Compile-time loops over the middle stages (everything between the first and the last stage lives in
// shared memory and needs a barrier after each stage; `sync()` is __syncthreads on the device and a
// no-op in the host harness, which runs whole phases thread by thread instead).
template <typename T, typename P> struct SmemIO {
    using S = Swz<T, P::RLAST>;
    cx<T>* sm;
    FCG_HD cx<T> ld(int e) const { return sm[S::at(e)]; }
    FCG_HD void st(int e, cx<T> v) const { sm[S::at(e)] = v; }
};

}  // namespace fcg
