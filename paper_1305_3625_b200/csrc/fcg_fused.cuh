// fcg_fused.cuh -- a whole CG solve (Listing 2, around the operator of Listing 4, 141-151) as ONE
// cooperative kernel, for lattices small enough that launch latency, not bandwidth, sets the pace (L = 256, 512:
// BASELINE.json configs[3] is ~75 000 iterations of a 0.5 MiB problem).
//
//   * grid = G <= 256 co-resident CTAs (cudaLaunchCooperativeKernel); CTA c owns the row pairs c, c+G, .. and the columns
//     c, c+G, .. of T for the whole solve;
//   * its rows of k, f, u, r, p, q live in shared memory from the first iteration to the last; only T (the transposition
//     between the row and the column transforms) goes through global memory, i.e. through L2;
//   * preconditioned CG (A.mhat != nullptr): z = M^-1 r is one more operator-shaped round trip per iteration (rows of r ->
//     columns with the preconditioner's spectrum -> rows of z, r.z), three more grid barriers; z lives in q's slot;
//   * per iteration THREE grid barriers (an atomic counter in global memory): T complete -> columns done -> r.r known.  The
//     search length needs no barrier of its own: p.Ap = sum k p^2 (formed with the new direction, in shared memory) + sum shat |P|^2
//     (accumulated in the column phase), published before the "columns done" barrier and added up by
//     every CTA after it, so u and r are updated in the epilogue of the inverse row transforms and q is never stored.  Every CTA adds the G partial sums itself, in the same fixed order, so alpha, beta and the convergence
//     decision are bit-identical in all CTAs and no CTA ever waits for a broadcast;
//   * same stage arithmetic as the pipelined passes (fcg_engine.cuh: register twiddle powers, swizzled work buffer) and the
//     same column numbering / stored spectrum as them (AsyncShape, colpos layout), so fcg_set_spectrum is shared.
//
// Order of operations = the oracle's (u is updated as soon as alpha is known).  A spin that exceeds SPIN_CAP polls sets
// status FCG_CUDA_ERROR instead of hanging the device.
#pragma once
#include "fcg_async.cuh"

namespace fcg {

struct FusedArgs {
    const void* k; const void* f; void* u;     // caller vectors (device), N reals
    void* Tf;                                   // workspace: L/2 columns x L complex, column m contiguous
    const void* shat; const void* tw;
    double* partial;                            // 4 x G doubles
    unsigned int* counter;                      // grid barrier (set to counter_start by the host before the launch)
    unsigned int counter_start;                 // normally 0; FCG_OPT_BARRIER_START presets it (test of the wrap-around)
    Scalars* sc;                                // result: it, relres, status
    double tol; int maxit;
    // quasi-static loop (nsteps > 0): thresholds, k written back, per-step results, arg-max scratch (G entries each)
    int nsteps; const void* t; void* k_out; long long* out_index; int* out_iters; double* brk_r; long long* brk_i;
    const void* mhat;                           // preconditioned CG: stored spectrum of M^-1, or nullptr for plain CG
    // force formulation (I + K G) f = K D (eq. (2)): u holds the bond forces, f is not read
    // (b = k * D is formed in shared memory), out_ratio[step] = the winning f/t of the break step (may be nullptr)
    int form; double D; double* out_ratio;
    int two;                                    // form != 1: 1 = fewer grid barriers per iteration (TWO instantiations: 2 for CG, 4 for PCG)
};

template <typename T, typename P> struct FusedShape {
    static constexpr int L = P::N, NT = P::NT;
    static constexpr bool valid = AsyncShape<T, P>::valid && (L == 256 || L == 512) && NT % 32 == 0;
    static constexpr int G = L / 2 < 256 ? L / 2 : 256;          // CTAs (all co-resident: <= 2 per SM)
    static constexpr int TPC = (L / 2) / G;                      // row pairs (and columns) per CTA
    static constexpr size_t WBYTES = (size_t)L * 2 * sizeof(T);
    static constexpr size_t VBYTES = (size_t)2 * L * sizeof(T);  // one vector's two rows
    static constexpr size_t smem = WBYTES + (size_t)TPC * 7 * VBYTES + 128;     // k f u r p q t
    static constexpr size_t smem_two = smem;     // TWO = 1 keeps the own columns of the row-transformed direction in q's slot
    static constexpr size_t smem_two_pcg = smem + (size_t)TPC * VBYTES;          // TWO = 2 (PCG): q's slot holds z, an eighth slot the columns
    static_assert(WBYTES == VBYTES, "a column of T is as large as a vector's two rows");
};

#ifdef __CUDACC__

constexpr unsigned int SPIN_CAP = 1u << 26;

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ unsigned int ld_relaxed_u32(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// all CTAs of the (co-resident) grid; returns false if the spin cap was hit
__device__ __forceinline__ bool grid_barrier(unsigned int* counter, unsigned int& target, unsigned int G, int* ok_smem) {
    __syncthreads();
    if (threadIdx.x == 0) {
        // arrive with release, poll with acquire (gpu scope): the CTA's earlier writes -- ordered before this thread by the
        // bar.sync above -- are visible to every CTA that sees the count, without the two full membar.gpu of the classic form
        target += G;
        asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(counter), "r"(1u) : "memory");
        unsigned int spins = 0;
        // poll relaxed (no L1 invalidate per poll), with a short back-off so that G pollers do not crowd the arrivals out of
        // the counter's L2 slice; one acquire load once the count is there orders the other CTAs' writes before what follows
        // (wrap-safe: the counter is monotonic modulo 2^32 and never more than G ahead of any CTA's target, so the sign of the
        //  difference decides; a plain `counter < target` fails when target wraps to a small number after ~2^32 / G barriers,
        //  i.e. ~5.6 M CG iterations at L = 512 -- a run to failure gets there)
        while ((int)(ld_relaxed_u32(counter) - target) < 0 && ++spins < SPIN_CAP) { __nanosleep(32); }
        (void)ld_acquire_u32(counter);
        *ok_smem = spins < SPIN_CAP;
    }
    __syncthreads();
    return *ok_smem != 0;
}

// FORCE = 1: the paper's own system in the bond forces, in the textbook order of Listing 2 (q = (I + K G) p is formed and kept, p.q is a
// dot product, then u and r are updated: one more grid barrier per iteration than the spectral search length of the displacement
// form, which would need k o p = kappa p, i.e. reading F1, to hold exactly) -- the same arithmetic as the oracle for any k.
// FORCE = 2: the force model through the displacements (reading F7): the arithmetic of FORCE = 0 (spectral
// search length, optional preconditioner) on (K + G^-1) u = K D, with b = K D re-formed in shared memory at every step and the
// break rule of the force model, f_i / t_i with f_i = k_i (D - u_i) by eq. (1a); u is not touched by the break.
// TWO = true (plain CG only: FORCE = 0 or 2, no preconditioner): TWO grid barriers per iteration instead of three.  The row
// transforms are linear, so the row-transformed direction obeys the recurrence of Listing 2 itself: with p' = r' + beta p,
//     F_row p' = F_row r' + beta F_row p.
// Each CTA keeps its own columns of F_row p in shared memory (Pc) and transforms the RESIDUAL instead of the direction, which it
// can do as soon as it has formed its rows of r' -- before beta is known -- so that the barrier of the r.r sum is also the
// barrier that completes T:   .. -> rows_inverse: u, r' -> row transforms of r' -> [sum r.r | T complete] -> beta, p' (real
// space, for k o p and u), columns: Pc = T + beta Pc, column transforms, energy -> [sum p.Ap] -> alpha -> rows_inverse ..
// The recurrence starts afresh with every solve (p = 0), so its rounding does not accumulate over a quasi-static loop.
// TWO = 2: the same for preconditioned CG, FOUR barriers instead of six: r' is transformed where the operator's last phase forms it
// (the r.r barrier completes T for z = M^-1 r'), z where the preconditioner's last phase forms it (the r.z barrier completes T for
// the operator, whose column phase then forms F_row p' = F_row z + beta F_row p).  z keeps q's slot, the columns get an eighth one.
template <typename T, typename P, int FORCE = 0, int TWO = 0>
__global__ void __launch_bounds__(P::NT) cg_fused_kernel(const FusedArgs A)
{
    static_assert(!TWO || FORCE != 1, "the two-barrier iteration is for the displacement form");
    constexpr bool FQ = FORCE == 1, FD = FORCE == 2;
    using AS = AsyncShape<T, P>;
    using FS = FusedShape<T, P>;
    constexpr int L = P::N, S = P::S, NT = P::NT, R1 = AS::R1, Q1 = AS::Q1, PER1 = AS::PER1, PM = per_max<P>();
    constexpr int G = FS::G, TPC = FS::TPC;
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* const smem_raw = align128(smem_dyn);
    __shared__ double red[32];
    __shared__ double bcast;
    __shared__ int ok_smem;
    cx<T>* W = reinterpret_cast<cx<T>*>(smem_raw);
    T* const vecs = reinterpret_cast<T*>(smem_raw + FS::WBYTES);
    // TWO: the own columns of F_row p live in the slot of q (vector 5), which plain CG never stores: L complex = two real rows
    constexpr int NVEC = TWO == 2 ? 8 : 7, PCSLOT = TWO == 2 ? 7 : 5;
    auto PcOf = [&](int j) { return reinterpret_cast<cx<T>*>(vecs + ((size_t)(j * NVEC + PCSLOT) * 2) * L); };
    // vector v (0 k, 1 f, 2 u, 3 r, 4 p, 5 q, 6 t) of own tile j, row r (0/1)
    auto V = [&](int j, int v, int r) { return vecs + ((size_t)(j * NVEC + v) * 2 + r) * L; };
    SmemIO<T, P> io{W};
    const int lt = threadIdx.x, cta = (int)blockIdx.x;
    const T* gk = static_cast<const T*>(A.k); const T* gf = static_cast<const T*>(A.f); T* gu = static_cast<T*>(A.u);
    cx<T>* Tf = static_cast<cx<T>*>(A.Tf);
    const T* shat = static_cast<const T*>(A.shat);
    const cx<T>* tw = static_cast<const cx<T>*>(A.tw);
    unsigned int target = A.counter_start;
    int slot = 0;                                  // partial-sum slot, rotates over 4
    auto ld_sw = [&](int e) { return io.ld(e); };
    auto st_sw = [&](int e, cx<T> v) { io.st(e, v); };

    cx<T> wb[S + 1][PM];
    static_for_up<1, S - 1>([&](auto s) { base_tw<P, decltype(s)::value, T>(lt, tw, wb[decltype(s)::value]); });

    // sum of one double per thread over the CTA (fixed tree), result in every thread
    auto cta_sum = [&](double v) {
        double a[1] = {v};
        block_sum<1>(a, red);
        if (lt == 0) bcast = a[0];
        __syncthreads();
        const double r = bcast;
        __syncthreads();
        return r;
    };
    // this thread's share of G doubles, all loads in flight before the first add (same order of additions as a plain loop; the loop
    // form serialised G / NT L2 round trips per sum -- 10 % of the kernel's stall samples at L = 512, profiles/r1_ncu_fused_L512_f64.txt)
    auto sum_partials = [&](const double* ps) {
        constexpr int NP = (G + NT - 1) / NT;
        double t[NP];
#pragma unroll
        for (int c = 0; c < NP; ++c) t[c] = lt + c * NT < G ? __ldcg(ps + lt + c * NT) : 0.0;
        double v = 0.0;
#pragma unroll
        for (int c = 0; c < NP; ++c) v += t[c];
        return v;
    };
    // grid-wide sum: publish the CTA's partial, barrier, every CTA adds all G partials in the same order
    auto grid_sum = [&](double part, bool& ok) {
        const double mine = cta_sum(part);
        double* ps = A.partial + (size_t)slot * G;
        if (lt == 0) ps[cta] = mine;
        ok = grid_barrier(A.counter, target, G, &ok_smem);
        const double v = sum_partials(ps);
        slot = (slot + 1) & 3;
        return cta_sum(v);
    };

    // arg-max of (ratio, index) over the CTA, "larger ratio, then lower index" (better(), fcg_kernels.cuh); result in all threads
    __shared__ double am_r[32];
    __shared__ long long am_i[32];
    auto cta_argmax = [&](double& r, long long& i) {
        const int lane = lt & 31, w = lt >> 5;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double r2 = __shfl_down_sync(0xffffffffu, r, o);
            const long long i2 = __shfl_down_sync(0xffffffffu, i, o);
            if (better(r2, i2, r, i)) { r = r2; i = i2; }
        }
        if (lane == 0) { am_r[w] = r; am_i[w] = i; }
        __syncthreads();
        r = am_r[0]; i = am_i[0];
        for (int k2 = 1; k2 < NT / 32; ++k2)
            if (better(am_r[k2], am_i[k2], r, i)) { r = am_r[k2]; i = am_i[k2]; }
        __syncthreads();
    };

    // ---- the three phases of one operator application c = C x (x = vector `vx` of the own tiles); c is left in `out`
    // phase R1: row transforms of x -> columns of Tf
    auto rows_forward = [&](int vx) {
        for (int j = 0; j < TPC; ++j) {
            const int A2 = cta + j * G;
            const T* x0 = V(j, vx, 0); const T* x1 = V(j, vx, 1);
            {
                cx<T> a[PER1][R1];
                stage_ld<P, 1, T>(lt, [&](int e) { return mk<T>(x0[e], x1[e]); }, a);
                stage_math<P, 1, -1, T>(a, wb[1]);
                stage_st<P, 1, T>(lt, st_sw, a);
                __syncthreads();
            }
            static_for_up<2, S>([&](auto s) {
                constexpr int sv = decltype(s)::value;
                cx<T> a[St<P, sv>::PER][St<P, sv>::R];
                stage_ld<P, sv, T>(lt, ld_sw, a);
                stage_math<P, sv, -1, T>(a, wb[sv]);
                stage_st<P, sv, T>(lt, st_sw, a);
                __syncthreads();
            });
            const T h = (T)0.5;
            for (int m = lt; m < L / 2; m += NT) {
                const int e = AS::pos_of_col(m);
                const int n = P::freq_of(e);
                cx<T> X0, X1;
                if (n == 0) {
                    const cx<T> Z0 = io.ld(P::pos_of(0)), ZN = io.ld(P::pos_of(L / 2));
                    X0 = mk<T>(Z0.x, ZN.x); X1 = mk<T>(Z0.y, ZN.y);
                } else {
                    const cx<T> Za = io.ld(e), Zb = io.ld(P::pos_of(L - n));
                    X0 = mk<T>((Za.x + Zb.x) * h, (Za.y - Zb.y) * h);
                    X1 = mk<T>((Za.y + Zb.y) * h, (Zb.x - Za.x) * h);
                }
                store_pair<T>(Tf + (size_t)m * L + 2 * A2, X0, X1);
            }
            __syncthreads();
        }
    };
    // phase C: own columns, in place: forward, spectral multiply, inverse
    auto columns = [&](const T* spec, double* en, bool recur = false, T rb = (T)0) {      // en != nullptr: *en += this CTA's share of sum spec |P|^2
        for (int j = 0; j < TPC; ++j) {                     // recur (TWO): the column is T + rb * Pc, and becomes the new Pc
            const int m = cta + j * G;
            cx<T>* col = Tf + (size_t)m * L;
            if constexpr (TWO) {
                cx<T>* pc = PcOf(j);
                if (recur) {
                    for (int e = lt; e < L; e += NT) {
                        const cx<T> t = __ldcg(col + e), o = pc[e];
                        const cx<T> v = mk<T>(t.x + rb * o.x, t.y + rb * o.y);
                        pc[e] = v; W[e] = v;
                    }
                } else {
                    for (int e = lt; e < L; e += NT) W[e] = __ldcg(col + e);
                }
            } else {
                for (int e = lt; e < L; e += NT) W[e] = __ldcg(col + e);
            }
            __syncthreads();
            {
                cx<T> a[St<P, 1>::PER][St<P, 1>::R];
                stage_ld<P, 1, T>(lt, [&](int e) { return W[e]; }, a);
                __syncthreads();
                stage_math<P, 1, -1, T>(a, wb[1]);
                stage_st<P, 1, T>(lt, st_sw, a);
                __syncthreads();
            }
            auto fwd_stage = [&](auto s) {
                constexpr int sv = decltype(s)::value;
                cx<T> a[St<P, sv>::PER][St<P, sv>::R];
                stage_ld<P, sv, T>(lt, ld_sw, a);
                stage_math<P, sv, -1, T>(a, wb[sv]);
                stage_st<P, sv, T>(lt, st_sw, a);
                __syncthreads();
            };
            auto inv_stage = [&](auto s) {
                constexpr int sv = decltype(s)::value;
                cx<T> a[St<P, sv>::PER][St<P, sv>::R];
                stage_ld<P, sv, T>(lt, ld_sw, a);
                stage_math<P, sv, +1, T>(a, wb[sv]);
                stage_st<P, sv, T>(lt, st_sw, a);
                __syncthreads();
            };
            if (m != 0) {
                const T* sh = spec + (size_t)m * L;
                static_for_up<2, S - 1>(fwd_stage);
                if (en) {
                    double e2 = 0.0;
                    run_middle<P, T, true>(lt, ld_sw, st_sw, [&](int g, int u) { return sh[u * (L / P::RLAST) + g]; }, &e2);
                    *en += 2.0 * e2;                                 // column m stands for frequencies n and L - n
                } else {
                    run_middle<P, T>(lt, ld_sw, st_sw, [&](int g, int u) { return sh[u * (L / P::RLAST) + g]; });
                }
                __syncthreads();
                static_for_down<S - 1, 2>(inv_stage);
            } else {     // packed n = 0 / L/2 column (see col2_kernel)
                static_for_up<2, S>(fwd_stage);
                const T* sp_ = spec;
                const T* sm_ = spec + (size_t)(L / 2) * L;
                for (int mm = lt; mm <= L / 2; mm += NT) {
                    const int e = P::pos_of(mm), e2 = P::pos_of((L - mm) % L);
                    const cx<T> Wa = io.ld(e), Wb = io.ld(e2);
                    cx<T> va, vb;
                    const int i1 = P::shat_index(e), i2 = P::shat_index(e2);
                    va.x = sp_[i1] * Wa.x + sm_[i1] * Wb.x; va.y = sp_[i1] * Wa.y - sm_[i1] * Wb.y;
                    vb.x = sp_[i2] * Wb.x + sm_[i2] * Wa.x; vb.y = sp_[i2] * Wb.y - sm_[i2] * Wa.y;
                    if (en) {        // s0 |Y0|^2 + sN |YN|^2 at mm (and again at -mm), see col2_kernel
                        const double na = (double)Wa.x * (double)Wa.x + (double)Wa.y * (double)Wa.y;
                        const double nb = (double)Wb.x * (double)Wb.x + (double)Wb.y * (double)Wb.y;
                        const double re = (double)Wa.x * (double)Wb.x - (double)Wa.y * (double)Wb.y;
                        const double term = 0.5 * (double)sp_[i1] * (na + nb) + (double)sm_[i1] * re;
                        *en += e2 != e ? 2.0 * term : term;
                    }
                    io.st(e, va);
                    if (e2 != e) io.st(e2, vb);
                }
                __syncthreads();
                static_for_down<S, 2>(inv_stage);
            }
            {
                cx<T> a[St<P, 1>::PER][St<P, 1>::R];
                stage_ld<P, 1, T>(lt, ld_sw, a);
                stage_math<P, 1, +1, T>(a, wb[1]);
                __syncthreads();
                stage_st<P, 1, T>(lt, [&](int e, cx<T> v) { W[e] = v; }, a);
            }
            __syncthreads();
            for (int e = lt; e < L; e += NT) col[e] = W[e];
            __syncthreads();
        }
    };
    // phase R2: inverse row transforms; emit(j, e, c0, c1) receives c = (C x) at element e of rows 0/1 of own tile j
    auto rows_inverse = [&](auto emit) {
        for (int j = 0; j < TPC; ++j) {
            const int A2 = cta + j * G;
            // all of this thread's loads of T in flight before the first use (the plain loop, with its branch, serialised
            // L / (2 NT) L2 round trips per phase: the largest single stall site at L = 512, profiles/r1_ncu_fused_L512_f64.txt)
            constexpr int NM = (L / 2 + NT - 1) / NT;
            cx<T> xa[NM], xb[NM];
#pragma unroll
            for (int c = 0; c < NM; ++c) {
                const int m = lt + c * NT;
                if (m < L / 2) { const cx<T>* src = Tf + (size_t)m * L + 2 * A2; xa[c] = __ldcg(src); xb[c] = __ldcg(src + 1); }
            }
#pragma unroll
            for (int c = 0; c < NM; ++c) {
                const int m = lt + c * NT;
                if (m >= L / 2) break;
                const int e = AS::pos_of_col(m);
                const int n = P::freq_of(e);
                const cx<T> X0 = xa[c], X1 = xb[c];
                if (n == 0) {
                    io.st(P::pos_of(0), mk<T>(X0.x, X1.x));
                    io.st(P::pos_of(L / 2), mk<T>(X0.y, X1.y));
                } else {
                    io.st(e, mk<T>(X0.x - X1.y, X0.y + X1.x));
                    io.st(P::pos_of(L - n), mk<T>(X0.x + X1.y, X1.x - X0.y));
                }
            }
            __syncthreads();
            static_for_down<S, 2>([&](auto s) {
                constexpr int sv = decltype(s)::value;
                cx<T> a[St<P, sv>::PER][St<P, sv>::R];
                stage_ld<P, sv, T>(lt, ld_sw, a);
                stage_math<P, sv, +1, T>(a, wb[sv]);
                stage_st<P, sv, T>(lt, st_sw, a);
                __syncthreads();
            });
            cx<T> c[PER1][R1];
            stage_ld<P, 1, T>(lt, ld_sw, c);
            __syncthreads();
            stage_math<P, 1, +1, T>(c, wb[1]);
#pragma unroll
            for (int q = 0; q < PER1; ++q)
#pragma unroll
                for (int t = 0; t < R1; ++t) emit(j, lt + q * NT + t * Q1, c[q][t].x, c[q][t].y);
        }
    };

    // ---- load the CTA's rows once; they stay in shared memory for the whole solve (or the whole quasi-static loop)
    const bool frac = A.nsteps > 0;
    for (int j = 0; j < TPC; ++j) {
        const size_t row0 = (size_t)(2 * (cta + j * G)) * L;
        for (int e = lt; e < 2 * L; e += NT) {         // the two rows are adjacent in memory
            V(j, 0, 0)[e] = gk[row0 + e]; V(j, 2, 0)[e] = gu[row0 + e];
            if (FORCE == 0) V(j, 1, 0)[e] = gf[row0 + e];
            if (frac) V(j, 6, 0)[e] = static_cast<const T*>(A.t)[row0 + e];
        }
    }
    __syncthreads();
    // One solve is a small state machine, so that every phase of the operator-shaped round trip (rows -> columns -> rows) and the
    // grid-wide sum exist ONCE in the instruction stream (with several call sites the compiler stops inlining them: 64 registers,
    // a stack frame, and 17.7 instead of 12.4 us per iteration at L = 256):
    //   FN (once per launch: ||f||^2) -> RESID (r = f - A u, r.r) -> [Z (z = M^-1 r, r.z)] -> Q (p, A p, alpha, u, r, r.r) -> [Z] -> Q -> ..
    // Z only for preconditioned CG; z lives in the slot that used to hold q (q is consumed as it is formed).
    // FORCE: .. -> Q (p, q = p + k o G p, p.q) -> U (alpha, u, r, r.r) -> Q -> ..; ||b||^2 once per solve (b = K D changes with k).
    enum { PH_FN = 0, PH_RESID = 1, PH_Z = 2, PH_Q = 3, PH_U = 4 };
    bool ok = true, okb = true, have_fn = false;
    int it = 0, status = ST_OK, steps_done = 0;
    double rho = 0.0, fn2 = 0.0, rr = 0.0;         // rho = r.r (CG) or r.z (PCG); rr = r.r
    bool zero_u = false;
    const T* mhat = static_cast<const T*>(A.mhat);
    const bool pcg = mhat != nullptr;

    for (int step = 0; step < (frac ? A.nsteps : 1); ++step) {
        // ---- set up initial values: first direction from p = 0, beta = 0
        for (int j = 0; j < TPC; ++j) {
            T* pp = V(j, 4, 0);
            for (int e = lt; e < 2 * L; e += NT) pp[e] = (T)0;
            if constexpr (TWO) { cx<T>* pc = PcOf(j); for (int e = lt; e < L; e += NT) pc[e] = mk<T>((T)0, (T)0); }
        }
        if (FORCE != 0) {                                   // right-hand side b = K D (eq. (2)), one multiply in the working precision
            const T dv = (T)A.D;
            for (int j = 0; j < TPC; ++j) {
                const T* kk = V(j, 0, 0); T* bb = V(j, 1, 0);
                for (int e = lt; e < 2 * L; e += NT) bb[e] = kk[e] * dv;
            }
            __syncthreads();
        }
        it = 0; status = ST_OK; zero_u = false;
        double beta = 0.0;
        T al_u = (T)0;                                 // FORCE: the search length between phases Q and U
        int phase = (have_fn && FORCE == 0) ? PH_RESID : PH_FN;
        if constexpr (TWO) {
            // FN (||f||^2 where not known yet; row transforms of u) -> RESID (r = f - A u; row transforms of r) -> Q -> Q -> ..
            // (TWO = 2, PCG: .. RESID -> Z (z = M^-1 r, r.z; row transforms of z) -> Q (.. row transforms of r') -> Z -> Q -> ..)
            // every phase ends with the row transforms of the NEXT operand and the grid-wide sum whose barrier also completes T
            const bool need_fn = phase == PH_FN;
            phase = PH_FN;
            while (true) {
                double acc = 0.0, kpp = 0.0;
                bool bd = false;
                if (phase == PH_FN) {
                    if (need_fn)
                        for (int j = 0; j < TPC; ++j) {
                            const T* ff = V(j, 1, 0);
                            for (int e = lt; e < 2 * L; e += NT) acc += (double)ff[e] * (double)ff[e];
                        }
                } else {
                    if (phase == PH_Q) {                    // update calculation variables: new direction (98); sum k p^2 on the way
                        for (int j = 0; j < TPC; ++j) {
                            const T* dv = V(j, TWO == 2 ? 5 : 3, 0); T* pp = V(j, 4, 0); const T* kk = V(j, 0, 0);   // r, or z = M^-1 r
                            const T b = (T)beta;
                            for (int e = lt; e < 2 * L; e += NT) {
                                const T pn = dv[e] + b * pp[e];
                                pp[e] = pn;
                                kpp += (double)kk[e] * ((double)pn * (double)pn);
                            }
                        }
                        __syncthreads();
                    }
                    double en = 0.0;
                    columns(phase == PH_Z ? mhat : shat, phase == PH_Q ? &en : nullptr, phase == PH_Q, (T)beta);
                    double* ps = A.partial + (size_t)slot * G;
                    if (phase == PH_Q) {                    // this CTA's share of p.Ap = sum k p^2 + sum shat |P|^2
                        const double mine = cta_sum(kpp + en);
                        if (lt == 0) ps[cta] = mine;
                    }
                    ok = grid_barrier(A.counter, target, G, &ok_smem) && ok;
                    T al = (T)0;
                    if (phase == PH_Q) {                    // search length (94): every CTA adds the G shares in the same order
                        const double v = sum_partials(ps);
                        slot = (slot + 1) & 3;
                        const double pq = cta_sum(v);
                        if (!(pq > 0.0) || !isfinite(pq)) bd = true;
                        else al = (T)(rho / pq);
                    }
                    if (!bd) rows_inverse([&](int j, int e, T c0, T c1) {
                        const T* kk = V(j, 0, 0); T* uu = V(j, 2, 0); T* rv = V(j, 3, 0);
                        if (phase == PH_RESID) {                              // r = f - (k o u + C u)
                            const T* ff = V(j, 1, 0);
                            const T r0 = ff[e] - (kk[e] * uu[e] + c0), r1 = ff[L + e] - (kk[L + e] * uu[L + e] + c1);
                            rv[e] = r0; rv[L + e] = r1;
                            acc += (double)r0 * (double)r0; acc += (double)r1 * (double)r1;
                        } else if (TWO == 2 && phase == PH_Z) {               // z = M^-1 r, r.z
                            T* zz = V(j, 5, 0);
                            zz[e] = c0; zz[L + e] = c1;
                            acc += (double)rv[e] * (double)c0; acc += (double)rv[L + e] * (double)c1;
                        } else {                        // q = k o p + C p; new x (95), residue (96), residue length (97)
                            const T* pp = V(j, 4, 0);
                            const T p0 = pp[e], p1 = pp[L + e];
                            const T q0 = kk[e] * p0 + c0, q1 = kk[L + e] * p1 + c1;
                            uu[e] = uu[e] + al * p0; uu[L + e] = uu[L + e] + al * p1;
                            const T r0 = rv[e] - al * q0, r1 = rv[L + e] - al * q1;
                            rv[e] = r0; rv[L + e] = r1;
                            acc += (double)r0 * (double)r0; acc += (double)r1 * (double)r1;
                        }
                    });
                }
                if (bd) { status = ST_BREAKDOWN; break; }
                __syncthreads();                            // the epilogue's writes to r (u) are in place for every thread
                rows_forward(phase == PH_FN ? 2 : (TWO == 2 && phase == PH_Z) ? 5 : 3);   // u for the residual pass, z for the operator, else the residual just formed
                const double s0 = grid_sum(acc, okb); ok = ok && okb;
                if (!ok) { status = -3; break; }
                if (phase == PH_FN) { if (need_fn) { fn2 = s0; have_fn = true; } phase = PH_RESID; }
                else if (phase == PH_RESID) {
                    rr = s0; rho = rr;
                    if (fn2 == 0.0) { zero_u = true; rho = 0.0; rr = 0.0; break; }
                    if (sqrt(rr) <= A.tol * sqrt(fn2)) break;
                    if (A.maxit <= 0) { status = ST_NOT_CONVERGED; break; }
                    phase = TWO == 2 ? PH_Z : PH_Q;
                } else if (TWO == 2 && phase == PH_Z) {
                    if (!(s0 > 0.0) || !isfinite(s0)) { status = ST_BREAKDOWN; break; }
                    beta = it == 0 ? 0.0 : s0 / rho;
                    rho = s0; phase = PH_Q;
                } else {
                    rr = s0; ++it;
                    if (sqrt(rr) <= A.tol * sqrt(fn2)) { if (TWO != 2) rho = rr; break; }            // check convergence (99)
                    if (it >= A.maxit) { if (TWO != 2) rho = rr; status = ST_NOT_CONVERGED; break; }
                    if (TWO == 2) phase = PH_Z;
                    else { beta = rr / rho; rho = rr; }
                }
            }
        } else
        while (true) {
            double acc = 0.0, kpp = 0.0;
            bool bd = false;
            // ---- vector work of this phase on the CTA's own rows
            if (phase == PH_FN) {
                for (int j = 0; j < TPC; ++j) {
                    const T* ff = V(j, 1, 0);
                    for (int e = lt; e < 2 * L; e += NT) acc += (double)ff[e] * (double)ff[e];
                }
            } else if (phase == PH_Q) {                 // update calculation variables: new direction (98); sum k p^2 on the way
                for (int j = 0; j < TPC; ++j) {
                    const T* dv = V(j, pcg ? 5 : 3, 0); T* pp = V(j, 4, 0); const T* kk = V(j, 0, 0);     // r, or z = M^-1 r
                    const T b = (T)beta;
                    for (int e = lt; e < 2 * L; e += NT) {
                        const T pn = dv[e] + b * pp[e];
                        pp[e] = pn;
                        kpp += (double)kk[e] * ((double)pn * (double)pn);
                    }
                }
                __syncthreads();
            } else if (FQ && phase == PH_U) {        // new x (95), residue (96), residue length (97)
                for (int j = 0; j < TPC; ++j) {
                    T* uu = V(j, 2, 0); T* rv = V(j, 3, 0); const T* pp = V(j, 4, 0); const T* qq = V(j, 5, 0);
                    for (int e = lt; e < 2 * L; e += NT) {
                        uu[e] = uu[e] + al_u * pp[e];
                        const T rn = rv[e] - al_u * qq[e];
                        rv[e] = rn;
                        acc += (double)rn * (double)rn;
                    }
                }
            }
            // ---- operator-shaped round trip: C u (RESID), C p (Q: A * p) or M^-1 r (Z)
            if (phase != PH_FN && !(FQ && phase == PH_U)) {
                rows_forward(phase == PH_RESID ? 2 : (phase == PH_Q ? 4 : 3));
                ok = grid_barrier(A.counter, target, G, &ok_smem) && ok;
                double en = 0.0;
                columns(phase == PH_Z ? mhat : shat, (!FQ && phase == PH_Q) ? &en : nullptr);
                double* ps = A.partial + (size_t)slot * G;
                if (!FQ && phase == PH_Q) {                    // this CTA's share of p.Ap = sum k p^2 + sum shat |P|^2, published before the barrier
                    const double mine = cta_sum(kpp + en);
                    if (lt == 0) ps[cta] = mine;
                }
                ok = grid_barrier(A.counter, target, G, &ok_smem) && ok;
                T al = (T)0;
                if (!FQ && phase == PH_Q) {          // search length (94): every CTA adds the G shares in the same order
                    const double v = sum_partials(ps);
                    slot = (slot + 1) & 3;
                    const double pq = cta_sum(v);
                    if (!(pq > 0.0) || !isfinite(pq)) bd = true;
                    else al = (T)(rho / pq);
                }
                if (!bd) rows_inverse([&](int j, int e, T c0, T c1) {
                    if (phase == PH_RESID) {                                  // r = f - (k o u + C u);  FORCE: r = b - (u + k o G u)
                        const T* kk = V(j, 0, 0); const T* ff = V(j, 1, 0); const T* uu = V(j, 2, 0); T* rv = V(j, 3, 0);
                        const T r0 = ff[e] - (FQ ? uu[e] + kk[e] * c0 : kk[e] * uu[e] + c0),
                                r1 = ff[L + e] - (FQ ? uu[L + e] + kk[L + e] * c1 : kk[L + e] * uu[L + e] + c1);
                        rv[e] = r0; rv[L + e] = r1;
                        acc += (double)r0 * (double)r0; acc += (double)r1 * (double)r1;
                    } else if (FQ && phase == PH_Q) {                      // q = p + k o (G p) (eq. (2)), kept; p.q
                        const T* kk = V(j, 0, 0); const T* pp = V(j, 4, 0); T* qq = V(j, 5, 0);
                        const T p0 = pp[e], p1 = pp[L + e];
                        const T q0 = p0 + kk[e] * c0, q1 = p1 + kk[L + e] * c1;
                        qq[e] = q0; qq[L + e] = q1;
                        acc += (double)p0 * (double)q0; acc += (double)p1 * (double)q1;
                    } else if (phase == PH_Q) {         // q = k o p + C p; new x (95), residue (96), residue length (97)
                        const T* kk = V(j, 0, 0); const T* pp = V(j, 4, 0); T* uu = V(j, 2, 0); T* rv = V(j, 3, 0);
                        const T p0 = pp[e], p1 = pp[L + e];
                        const T q0 = kk[e] * p0 + c0, q1 = kk[L + e] * p1 + c1;
                        uu[e] = uu[e] + al * p0; uu[L + e] = uu[L + e] + al * p1;
                        const T r0 = rv[e] - al * q0, r1 = rv[L + e] - al * q1;
                        rv[e] = r0; rv[L + e] = r1;
                        acc += (double)r0 * (double)r0; acc += (double)r1 * (double)r1;
                    } else {                                                  // z = M^-1 r, r.z
                        const T* rv = V(j, 3, 0); T* zz = V(j, 5, 0);
                        zz[e] = c0; zz[L + e] = c1;
                        acc += (double)rv[e] * (double)c0; acc += (double)rv[L + e] * (double)c1;
                    }
                });
            }
            if (bd) { status = ST_BREAKDOWN; break; }
            const double s0 = grid_sum(acc, okb); ok = ok && okb;
            if (!ok) { status = -3; break; }
            // ---- scalar step, identical in every CTA
            if (phase == PH_FN) { fn2 = s0; have_fn = true; phase = PH_RESID; }
            else if (phase == PH_RESID) {
                rr = s0; rho = rr;
                if (fn2 == 0.0) { zero_u = true; rho = 0.0; rr = 0.0; break; }
                if (sqrt(rr) <= A.tol * sqrt(fn2)) break;
                if (A.maxit <= 0) { status = ST_NOT_CONVERGED; break; }
                phase = pcg ? PH_Z : PH_Q;
            } else if (phase == PH_Z) {
                if (!(s0 > 0.0) || !isfinite(s0)) { status = ST_BREAKDOWN; break; }
                beta = it == 0 ? 0.0 : s0 / rho;
                rho = s0; phase = PH_Q;
            } else if (FQ && phase == PH_Q) {        // search length (94): a dot product, as the oracle forms it
                if (!(s0 > 0.0) || !isfinite(s0)) { status = ST_BREAKDOWN; break; }
                al_u = (T)(rho / s0); phase = PH_U;
            } else {
                if (FQ) phase = PH_Q;
                rr = s0; ++it;
                if (sqrt(rr) <= A.tol * sqrt(fn2)) { if (!pcg) rho = rr; break; }                 // check convergence (99)
                if (it >= A.maxit) { if (!pcg) rho = rr; status = ST_NOT_CONVERGED; break; }
                if (pcg) phase = PH_Z;
                else { beta = rr / rho; rho = rr; }
            }
        }
        __syncthreads();
        if (zero_u)
            for (int j = 0; j < TPC; ++j) {
                T* uu = V(j, 2, 0);
                for (int e = lt; e < 2 * L; e += NT) uu[e] = (T)0;
            }
        if (!frac || status < 0) break;

        // ---- break step (rule of BASELINE.json configs[3]): arg-max over {k_i > 0} of (k_i u_i) / t_i, one IEEE
        //      multiply and one IEEE divide in double, ties -> lowest index, NaN skipped; the winner's k becomes 0
        __syncthreads();
        double br = 0.0; long long bi = -1;
        for (int j = 0; j < TPC; ++j) {
            const long long row0 = (long long)(2 * (cta + j * G)) * L;
            const T* kk = V(j, 0, 0); const T* uu = V(j, 2, 0); const T* tt = V(j, 6, 0);
            for (int e = lt; e < 2 * L; e += NT) {
                const T ki = kk[e];
                if (!(ki > (T)0)) continue;
                const double load = FQ ? (double)uu[e] : FD ? (double)(ki * ((T)A.D - uu[e])) : (double)ki * (double)uu[e];      // FORCE (reading F2): f_i / t_i
                const double rt = load / (double)tt[e];
                if (rt != rt) continue;
                if (better(rt, row0 + e, br, bi)) { br = rt; bi = row0 + e; }
            }
        }
        cta_argmax(br, bi);
        if (lt == 0) { A.brk_r[cta] = br; A.brk_i[cta] = bi; }
        ok = grid_barrier(A.counter, target, G, &ok_smem) && ok;
        br = 0.0; bi = -1;
        for (int i = lt; i < G; i += NT) {
            const double r2 = __ldcg(A.brk_r + i); const long long i2 = __ldcg(A.brk_i + i);
            if (better(r2, i2, br, bi)) { br = r2; bi = i2; }
        }
        cta_argmax(br, bi);
        if (!ok) { status = -3; break; }
        if (bi < 0) { status = -6; break; }                                   // FCG_NO_CANDIDATE
        {
            const int A2 = (int)(bi / (2 * L));
            if (A2 % G == cta && lt == 0) {
                V(A2 / G, 0, 0)[bi - (long long)A2 * 2 * L] = (T)0;
                if (FQ) V(A2 / G, 2, 0)[bi - (long long)A2 * 2 * L] = (T)0;        // a broken bond carries no force
            }
        }
        if (cta == 0 && lt == 0) {
            A.out_index[step] = bi; A.out_iters[step] = it;
            if (FORCE != 0 && A.out_ratio) A.out_ratio[step] = br;
        }
        steps_done = step + 1;
        status = ST_OK;
        __syncthreads();
        // the winners' slots are reused two barriers later at the earliest (the next step's set-up has three)
    }
    __syncthreads();
    for (int j = 0; j < TPC; ++j) {
        const size_t row0 = (size_t)(2 * (cta + j * G)) * L;
        const T* uu = V(j, 2, 0); const T* kk = V(j, 0, 0);
        for (int e = lt; e < 2 * L; e += NT) {
            gu[row0 + e] = uu[e];
            if (frac) static_cast<T*>(A.k_out)[row0 + e] = kk[e];
        }
    }
    if (cta == 0 && lt == 0) {
        Scalars* sc = A.sc;
        sc->it = it; sc->status = status; sc->done = 1; sc->rho = rho; sc->rr = rr; sc->fn2 = fn2; sc->steps_done = steps_done;
        sc->relres = fn2 > 0.0 ? sqrt(rr) / sqrt(fn2) : 0.0;
    }
}

#endif  // __CUDACC__

}  // namespace fcg
