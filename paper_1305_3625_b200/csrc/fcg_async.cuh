// fcg_async.cuh -- the three transform passes of one operator application (Listing 4) with their
// fused vector work (Listing 2), written for sm_100a's asynchronous copy engine:
//
//   * persistent CTAs, one transform (P::NT consumer threads) in flight per CTA, 2-4 CTAs resident per SM;
//   * every global read arrives through TMA (cp.async.bulk / cp.async.bulk.tensor) into shared memory and signals
//     an mbarrier: no register staging, no load latency on the instruction stream, depth bounded by shared memory;
//   * vectors that are read strip-wise (p, r, u in P1; k, p in P3) stream through rings of shared-memory slots beside
//     the transform's work buffer; producer warps keep the rings full ACROSS transforms, so the next transform's
//     inputs land while the current one is in its butterfly stages;
//   * T is kept in the line layout T2 (AsyncShape): the row passes move whole 128-byte lines, the
//     column pass gathers / scatters its column with 4-D TMA tensor copies and runs in place in shared memory;
//   * twiddles: one base twiddle per butterfly in registers + powers (fcg_engine.cuh), no table traffic.
//
// Every hand-over between the threads' own (generic-proxy) accesses to a shared-memory slot and a TMA (async-proxy)
// access to the same slot goes through an mbarrier: "full" barriers carry the copy's byte count, "empty" / "ready"
// barriers collect one arrival per warp.  A CTA barrier (bar.sync) is NOT used for that: it only orders the generic
// proxy.  A consumer releases a slot with fence.proxy.async + arrive (tma::mbar_warp_release): without the fence a
// still-queued ld.shared can be overtaken by the refill (measured, see fcg_tma.cuh).  bar.sync is used between
// butterfly stages only.
//
// Same mathematics (two rows per complex transform, packed n = 0 / L/2 column, digit-reversed spectrum) and modes as
// fcg_passes.cuh, which remains the path for small lattices (NT < 64), for the stand-alone transforms, and the
// host-replayable statement of the index algebra.  Byte counts per launch: DESIGN.md section 4.
#pragma once
#include <cuda.h>
#include "fcg_kernels.cuh"
#include "fcg_plans.cuh"
#include "fcg_tma.cuh"

namespace fcg {

template <typename T, typename P> struct AsyncShape {
    static constexpr int L = P::N, NT = P::NT, R1 = P::radix(1), Q1 = L / R1, PER1 = Q1 / NT;
    static constexpr bool valid = NT >= 64 && L >= 256;
    static constexpr size_t WBYTES = (size_t)L * 2 * sizeof(T);              // one complex transform (work buffer)
    static constexpr uint32_t PIECE = (uint32_t)(Q1 * sizeof(T));            // one stage-1 strip of one real row
    static constexpr int MAXSLOT = 16;

    // Layout of T for these passes: columns are numbered by their POSITION in the digit-reversed row
    // spectrum, m = 0 .. L/2-1 <-> position e(m) = (m / HR) RLAST + m % HR <-> frequency n = freq_of(e(m)) < L/2, and
    // NB consecutive columns x one row pair form one 128-byte line:  T2[m / NB][A][m % NB][r],  a = 2A + r.
    static constexpr int NB = 128 / (4 * (int)sizeof(T));
    static constexpr int HR = P::RLAST / 2;
    static constexpr int ABOX = L / 2 < 256 ? L / 2 : 256;                   // row pairs per box of the column tensor map
    static FCG_HD int pos_of_col(int m) { return (m / HR) * P::RLAST + m % HR; }
    static FCG_HD int col_of_pos(int e) { return (e / P::RLAST) * HR + e % P::RLAST; }
    static FCG_HD size_t t2_index(int m, int A) { return (((size_t)(m / NB) * (L / 2) + A) * NB + m % NB) * 2; }   // complex units, r = 0
    static FCG_HD size_t t2_index_s(int m, int A, int astride) { return (((size_t)(m / NB) * astride + A) * NB + m % NB) * 2; }   // a slab's T2

    // Shared memory.  The rings are sized for CRES resident CTAs per SM: 4 transforms in flight when a work buffer is
    // small, else 2 (1 when even that does not fit); whatever the work buffers leave goes to the rings, whose depth is
    // what hides the loaded DRAM latency.  2688 = static barriers + 1 KB per-CTA reserve + alignment slack.
    // Measured at the 64 KB work buffers (L = 4096 fp64, L = 8192 fp32): ONE resident CTA with rings of 160 KB beats two with
    // 47 KB each: P1 178 -> 145 us, 325 -> 277 us; the fused last pass 157 -> 128 us, 378 -> 290 us once its tile ring holds a whole
    // transform (with nobody else on the SM the wait for the tiles at the start of a transform is fully exposed otherwise).
    // At the 32 KB work buffers (L = 2048 fp64, L = 4096 fp32) one CTA loses in both passes (4-8 warps do not cover the stages).
    static constexpr int CRES = WBYTES <= 16384 ? 4 : (WBYTES < 65536 ? 2 : 1);                                   // P1
    static constexpr int CRES_I = WBYTES <= 16384 ? 4 : (WBYTES < 65536 ? 2 : 1);   // P3
    static constexpr size_t RING_BUDGET_F = ((size_t)FCG_MAX_SMEM / CRES - 2688 - WBYTES) / 128 * 128;
    static constexpr size_t RING_BUDGET = ((size_t)FCG_MAX_SMEM / CRES_I - 2688 - WBYTES) / 128 * 128;
    // P1: ring of NFS strips (p0 p1 r0 r1 u0 u1: 6 pieces each)
    static constexpr uint32_t FSLOTB = 6 * PIECE;
    static constexpr int NFS = RING_BUDGET_F / FSLOTB < 2 ? 2 : (RING_BUDGET_F / FSLOTB > MAXSLOT ? MAXSLOT : (int)(RING_BUDGET_F / FSLOTB));
    static constexpr size_t fwd_smem = WBYTES + (size_t)NFS * FSLOTB + 128;   // + 128: the kernels align the dynamic base themselves
    // P2: column + its spectrum row
    static constexpr size_t col_smem = WBYTES + (size_t)L * sizeof(T) + 128;
    // P3: NTS tiles of T2 (TSB bytes = TSUB columns x 2 rows each) and a ring of KRB bytes for strips of k, p (, f).
    // The strip ring gets at least two loop-mode strips (4 pieces each); the tiles get smaller if that is what it takes.
    static constexpr size_t TSB_MAX = WBYTES >= 16384 ? 8192 : WBYTES / 2;
    static constexpr size_t KMIN = 8 * (size_t)PIECE;
    static constexpr size_t TSB = RING_BUDGET >= KMIN + 2 * TSB_MAX ? TSB_MAX : TSB_MAX / 2;
    static constexpr int TSUB = (int)(TSB / (2 * 2 * sizeof(T)));            // columns per tile of T2
    static constexpr int NSUB = (L / 2) / TSUB;
    static constexpr int NTS_ = (int)((RING_BUDGET - KMIN) / TSB);
    static constexpr int NTS = NTS_ < 2 ? 2 : (NTS_ > NSUB ? NSUB : (NTS_ > MAXSLOT ? MAXSLOT : NTS_));
    static constexpr size_t KRB = RING_BUDGET - (size_t)NTS * TSB;
    static constexpr size_t inv_smem = WBYTES + (size_t)NTS * TSB + KRB + 128;
    static constexpr bool PRODUCER_WARPS = NT <= 256;                        // P3: dedicated TMA-issuing warps (else consumer warp 0 issues)
    static constexpr int thread_cap = sizeof(T) == 8 ? 640 : 1152;           // ~104-128 / ~56-64 registers per thread
    // P3 normally has TWO producer warps (tiles of T2 / strips of the vectors: each runs ahead across transforms on its own).  Where a
    // second one costs a resident CTA AND with that CTA every transform of the lattice is resident at once (L = 1024 fp64: 3 x 148 = 444
    // slots for 512 transforms with two, 4 x 148 = 592 with one), ONE producer warp issues tiles then strips of each transform in
    // consumption order: nothing runs ahead, but nothing has to -- each CTA has a single transform -- and the pass is one round instead
    // of two (measured 22.6 -> see DESIGN.md section 17).
    static constexpr int NSM_DESIGN = 148;
    static constexpr int slots_with(int extra) {
        const int by_smem = (int)((size_t)FCG_MAX_SMEM / ((size_t)FCG_MAX_SMEM / CRES_I + 1280 - 2688 + 1024 + 128));
        const int by_thr = thread_cap / (NT + extra) > 1 ? thread_cap / (NT + extra) : 1;
        return (by_smem < by_thr ? by_smem : by_thr) * NSM_DESIGN;
    }
    static constexpr int NPW = !PRODUCER_WARPS ? 0 : (slots_with(64) < L / 2 && slots_with(32) >= L / 2) ? 1 : 2;
    static constexpr int INV_THREADS = NT + 32 * NPW;

    // resident CTAs per SM to compile for: static_smem = the kernel's __shared__ barriers etc., extra = producer threads
    static constexpr int ctas(size_t smem, size_t static_smem, int extra) {
        const int by_smem = (int)((size_t)FCG_MAX_SMEM / (smem + static_smem + 1024));
        const int by_thr = thread_cap / (NT + extra) > 1 ? thread_cap / (NT + extra) : 1;
        return by_smem < 1 ? 1 : (by_smem < by_thr ? by_smem : by_thr);
    }
    static_assert(!valid || (KRB >= 6 * (size_t)PIECE && KRB >= KMIN), "strip ring too small");
    static_assert(!valid || (TSUB % NB == 0 && TSUB / NB <= 256 && (L / 2) % TSUB == 0 && NSUB >= 2 && NT % 32 == 0), "tile shape");
    static_assert(!valid || (fwd_smem <= (size_t)FCG_MAX_SMEM && inv_smem <= (size_t)FCG_MAX_SMEM && col_smem <= (size_t)FCG_MAX_SMEM), "shared memory");
};

#ifdef __CUDACC__

// TMA tensor tiles want a 128-byte aligned destination; the dynamic shared-memory base only promises 16
__device__ __forceinline__ unsigned char* align128(unsigned char* p) { return p + ((128u - (tma::smem_u32(p) & 127u)) & 127u); }

template <typename T> __device__ __forceinline__ void store_pair(cx<T>* dst, cx<T> a, cx<T> b);
template <> __device__ __forceinline__ void store_pair<double>(double2* dst, double2 a, double2 b) { dst[0] = a; dst[1] = b; }
template <> __device__ __forceinline__ void store_pair<float>(float2* dst, float2 a, float2 b) {
    *reinterpret_cast<float4*>(dst) = make_float4(a.x, a.y, b.x, b.y);
}

// the same with an L2 eviction-priority policy
__device__ __forceinline__ void store_pair_hint(double2* dst, double2 a, double2 b, uint64_t pol) { tma::st_hint(dst, a, pol); tma::st_hint(dst + 1, b, pol); }
__device__ __forceinline__ void store_pair_hint(float2* dst, float2 a, float2 b, uint64_t pol) {
    tma::st_hint(reinterpret_cast<float4*>(dst), make_float4(a.x, a.y, b.x, b.y), pol);
}

// CTA barrier among the first N threads only (the consumers of a warp-specialised kernel); barrier 0 stays __syncthreads
template <int N> __device__ __forceinline__ void bar_named() { asm volatile("bar.sync 1, %0;" ::"n"(N) : "memory"); }

// Grouped butterfly assignment in the stages >= 2 of the pipelined passes (fcg_engine.cuh, Grp), built with -DFCG_GROUPS.  Correct
// (parity green) but not faster: measured L = 2048 fp64 93.7 vs 94.2 us per iteration, and slower where it costs registers
// (L = 8192 fp32 826 vs 798 us, L = 4096 fp64 379 vs 369 us) -- the stage barriers are not what these kernels wait for.  Default:
// the cyclic assignment with a CTA barrier after every stage.
// Column gather by the LSU's asynchronous 16-byte copies (cp.async, SASS LDGSTS) instead of TMA tensor loads, the scatter staying
// on TMA: built with -DFCG_LSU_GATHER, measured, NOT the default.  Elimination runs (-DFCG_PROBE) show the column pass without
// its arithmetic at 0.7 ns per gathered / scattered cell whatever the cell's size (L = 2048 fp64: 32-byte cells, 18.0 of 27.1 us;
// L = 8192 fp32: 16-byte cells, 164 of 218 us), i.e. bound by the rate of small requests, not by HBM bytes.  Moving the gather's
// requests from the TMA engine to the load/store unit did not help -- L = 2048 fp64 28.4 vs 26.7 us, L = 8192 fp32 241 vs 220 us,
// parity green either way.  (A later timing probe with every column contiguous in T2 -- one bulk copy per column -- ran the pass
// only 1.5 us / 4 us faster: the number and size of the copy requests is not what limits it at all.  DESIGN.md section 17.)
#ifdef FCG_LSU_GATHER
constexpr bool LSU_GATHER = true;
#else
constexpr bool LSU_GATHER = false;
#endif
#ifdef FCG_GROUPS
constexpr bool GRP = true;
#else
constexpr bool GRP = false;
#endif
// Elimination runs (-DFCG_PROBE, measurement builds only; results are then wrong): bits of ColArgs/RowInvArgs/RowFwdArgs::hints
//   0x100 column pass without its stages   0x200 without its gather   0x400 without its scatter
//   0x800 last pass without its shared-memory stages   0x1000 first pass without them
#ifdef FCG_PROBE
#define FCG_PROBE_ON(bit) ((A.hints & (bit)) != 0)
#else
#define FCG_PROBE_ON(bit) false
#endif
// after a stage >= 2: only the threads that share my sub-blocks (GRP), else all NT consumers
template <typename P, int NT> __device__ __forceinline__ void stage_sync(int lt) {
    if constexpr (GRP) group_sync<P>(lt); else asm volatile("bar.sync 1, %0;" ::"n"(NT) : "memory");
}

template <typename P> constexpr int per_max() {
    int m = 1;
    for (int s = 1; s <= P::S; ++s) { const int per = (P::N / P::radix(s)) / P::NT; if (per > m) m = per; }
    return m;
}

// --------------------------------------------------------------------------------------------- P1
//   [u += alpha p;  p = r + beta p;]   columns of T2 at row pair a0/2 = row transforms of rows a0, a0+1 of p (or x)
// Persistent: grid = nsm x CTAS; the CTAs that share an SM (blockIdx % nsm, the usual placement) take the row pairs
// s, s+nsm, s+2nsm, .. in turn, so every SM gets floor or ceil of (L/2)/nsm transforms.
// Warp-specialised: NT consumer threads + one producer warp that only issues the strip copies, so the ring runs
// ahead across transforms (while one transform is in its butterfly stages the next one's strips are landing) and
// no consumer ever spends issue slots on address arithmetic for TMA.
// RUPD = true (a separate instantiation, so that the CG kernel's register allocation is untouched) is the PCG pass
//   r -= alpha q;  partial r.r -> last CTA: count, convergence;  columns of T2 = row transforms of the new r
// whose strips are r0 r1 q0 q1 (4 pieces) and which ends with the grid-wide reduction of cg_update_r_kernel.
template <typename T, typename P, int CTAS, int VAR = 0>
__global__ void __launch_bounds__(P::NT + 32, CTAS) row_fwd2_kernel(const RowFwdArgs<T> A)
{
    constexpr bool RUPD = VAR == 1;
    constexpr bool SLAB = VAR == 2;      // one rank's row slab: A.ntile row pairs, T2 of A.astride row pairs per column block
    using AS = AsyncShape<T, P>;
    constexpr int L = P::N, S = P::S, NT = P::NT, R1 = AS::R1, Q1 = AS::Q1, PER1 = AS::PER1, PM = per_max<P>();
    constexpr uint32_t PIECE = AS::PIECE;
    const int NTILE = SLAB ? A.ntile : L / 2, ASTR = SLAB ? A.astride : L / 2;
    constexpr int NSLOT = RUPD ? (AS::NFS * 6 / 4 > AS::MAXSLOT ? AS::MAXSLOT : AS::NFS * 6 / 4) : AS::NFS;
    constexpr uint32_t SLOTB = RUPD ? 4 * PIECE : AS::FSLOTB;
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* const smem_raw = align128(smem_dyn);
    unsigned char* const ring = smem_raw + AS::WBYTES;
    __shared__ __align__(8) uint64_t full[AS::MAXSLOT];
    __shared__ __align__(8) uint64_t empty[AS::MAXSLOT];
    cx<T>* W = reinterpret_cast<cx<T>*>(smem_raw);
    SmemIO<T, P> io{W};
    const int lt = threadIdx.x, lane = lt & 31, warp = lt >> 5;
    const bool cg = !RUPD && A.mode == ROWF_CG;
    const int nv = RUPD ? 4 : (cg ? 6 : 2);
    tma::grid_dep_launch();
    // Always true, but opaque to the compiler: guarding the global stores with it keeps them in basic blocks of their own
    // instead of interleaved with the shared-memory loads of the next strip.  Measured at L=2048 fp64: 39 vs 44 us.
    const bool st_on = A.mode >= 0;

    // my transforms: tile(i) = grp + nsm * (j + i * k)
    // (a grid that is not a whole multiple of the SM count is the one-transform-per-CTA launch: every transform resident at once)
    const int nsm = A.nsm < (int)gridDim.x ? A.nsm : (int)gridDim.x, grp = (int)blockIdx.x % nsm, jj = (int)blockIdx.x / nsm,
              kk = (int)gridDim.x / nsm;
    const bool whole = (int)gridDim.x % nsm == 0;
    auto tile_of = [&](int i) { return whole ? grp + nsm * (jj + i * kk) : (int)blockIdx.x + i * (int)gridDim.x; };
    int ntl = 0;
    while (tile_of(ntl) < NTILE) ++ntl;
    const int G = ntl * R1;                                       // strips this CTA will consume

    if (lt == 0) {
        for (int i = 0; i < NSLOT; ++i) { tma::mbar_init(&full[i], 1); tma::mbar_init(&empty[i], NT / 32); }
        tma::fence_mbar_init();
    }
    __syncthreads();
    tma::grid_dep_wait();                                         // everything above overlaps the previous kernel's tail
    if ((cg || RUPD || A.check_done) && A.sc->done) return;       // converged: nothing may change
    if (jj > 0 && A.stagger_ns > 0) {      // the later CTAs of an SM start a fraction of a transform time after the first (see stagger_wait)
        tma::stagger_wait((unsigned long long)jj * (unsigned long long)A.stagger_ns);
    }
    double acc[1] = {0.0};

    if (warp == NT / 32) {
        // ---- producer warp: strip g = (transform g / R1, strip g % R1) = elements [t Q1, (t+1) Q1) of
        //      p0 p1 r0 r1 u0 u1 (or x0 x1), one bulk copy per lane < nv, into slot g % NSLOT
        const T* base = RUPD ? (lane < 2 ? (const T*)A.rw : A.q) : cg ? (lane < 2 ? A.p : lane < 4 ? A.r : A.u) : A.x;
        base += (size_t)(lane & 1) * L;
        unsigned char* dst = ring + (size_t)lane * PIECE;
        int slot = 0;
        uint32_t phase = 0;
        // L2 hints (bit 0): u is not touched again before the next iteration's P1 -- its strips should not displace T2, q, r
        const uint64_t pol = (cg && lane >= 4 && (A.hints & 1)) ? tma::policy_evict_first() : tma::policy_evict_normal();
        for (int g = 0; g < G; ++g) {
            if (g >= NSLOT) tma::mbar_wait(&empty[slot], phase ^ 1u, A.tmo);          // the slot's previous strip has been read by every warp
            if (lane == 0) tma::mbar_expect_tx(&full[slot], nv * PIECE);
            __syncwarp();
            if (lane < nv)
                tma::bulk_g2s_hint(dst + (size_t)slot * SLOTB, base + (size_t)(2 * tile_of(g / R1)) * L + (size_t)(g % R1) * Q1, PIECE, &full[slot], pol);
            if (++slot == NSLOT) { slot = 0; phase ^= 1u; }
        }
        if constexpr (!RUPD) return;
    }

    // ---- consumers
    if (!RUPD || warp < NT / 32) {
    T alpha = (T)0, beta = (T)0;
    if (cg) { alpha = (T)A.sc->alpha; beta = (T)A.sc->beta; }
    if (RUPD) alpha = (T)A.sc->alpha;
    const uint64_t pol_u = (A.hints & 2) ? tma::policy_evict_first() : tma::policy_evict_normal();   // L2 hints (bit 1): the u stores
    const uint64_t pol_t2 = (A.hints & 64) ? tma::policy_evict_last() : tma::policy_evict_normal(); // (bit 6): T2 is read back by the next two passes
    cx<T> wb[S + 1][PM];
    static_for_up<1, S - 1>([&](auto s) { base_tw<P, decltype(s)::value, T, GRP>(lt, A.tw, wb[decltype(s)::value]); });

    int slot = 0;
    uint32_t phase = 0;
    for (int i = 0; i < ntl; ++i) {
        const int a0 = 2 * tile_of(i);
        const size_t row0 = (size_t)a0 * L;
        // phase A: strips stream through the ring; vector update on the fly; z = p_even + i p_odd
        cx<T> z[PER1][R1];
#pragma unroll
        for (int t = 0; t < R1; ++t) {
            tma::mbar_wait(&full[slot], phase, A.tmo);
            const T* sl = reinterpret_cast<const T*>(ring + (size_t)slot * SLOTB);
#pragma unroll
            for (int q = 0; q < PER1; ++q) {
                const int j = lt + q * NT;
                if constexpr (RUPD) {
                    T r0 = sl[j], r1 = sl[Q1 + j];
                    const T q0 = sl[2 * Q1 + j], q1 = sl[3 * Q1 + j];
                    r0 = r0 - alpha * q0; r1 = r1 - alpha * q1;       // residue
                    const size_t i0 = row0 + (size_t)t * Q1 + j;
                    if (st_on) { A.rw[i0] = r0; A.rw[i0 + L] = r1; }
                    acc[0] += (double)r0 * (double)r0; acc[0] += (double)r1 * (double)r1;   // residue length
                    z[q][t] = mk<T>(r0, r1);
                } else if (cg) {
                    T p0 = sl[j], p1 = sl[Q1 + j];
                    const T r0 = sl[2 * Q1 + j], r1 = sl[3 * Q1 + j];
                    T u0 = sl[4 * Q1 + j], u1 = sl[5 * Q1 + j];
                    u0 = u0 + alpha * p0; u1 = u1 + alpha * p1;       // new x, lagged one pass
                    p0 = r0 + beta * p0;  p1 = r1 + beta * p1;        // new direction
                    const size_t i0 = row0 + (size_t)t * Q1 + j;
                    if (st_on) { tma::st_hint(A.u + i0, u0, pol_u); tma::st_hint(A.u + i0 + L, u1, pol_u); A.p[i0] = p0; A.p[i0 + L] = p1; }
                    z[q][t] = mk<T>(p0, p1);
                } else {
                    z[q][t] = mk<T>(sl[j], sl[Q1 + j]);
                }
            }
            if (i * R1 + t + NSLOT < G) {                               // this warp has read the slot
                if (cg || RUPD) tma::mbar_warp_release_consumed(&empty[slot]);  // (values already used by the update above)
                else tma::mbar_warp_release(&empty[slot]);
            }
            if (++slot == NSLOT) { slot = 0; phase ^= 1u; }
        }
        bar_named<NT>();                                          // the previous transform's separation has left W
        stage_math<P, 1, -1, T, true>(z, wb[1]);
        stage_st<P, 1, T>(lt, [&](int e, cx<T> v) { io.st(e, v); }, z);
        bar_named<NT>();
        if (!FCG_PROBE_ON(0x1000))
        static_for_up<2, S>([&](auto s) {
            constexpr int sv = decltype(s)::value;
            cx<T> a[St<P, sv>::PER][St<P, sv>::R];
            stage_ld<P, sv, T, GRP>(lt, [&](int e) { return io.ld(e); }, a);
            stage_math<P, sv, -1, T, true>(a, wb[sv]);
            stage_st<P, sv, T, GRP>(lt, [&](int e, cx<T> v) { io.st(e, v); }, a);
            if constexpr (sv == S) bar_named<NT>();           // the separation below reads Z[n] and Z[L - n]: everybody's
            else stage_sync<P, NT>(lt);
        });
        // Separate the two rows and store them as column m of T2 (X_even[n], X_odd[n] side by side).  Consecutive
        // threads take consecutive POSITIONS e of the digit-reversed spectrum (n = freq_of(e), n < L/2 <=> the last
        // digit e % RLAST is in its lower half), so the reads of Z[n] and of its mirror Z[L-n] are contiguous runs.
        const T h = (T)0.5;
#pragma unroll 4
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
            if constexpr (SLAB) {
                cx<T>* dst;
                if (A.npeer) {         // straight into the owner's exchange buffer: R[my rank][local block][row pair][column][2]
                    const int mb = m / AS::NB;
                    dst = A.peerR[mb / A.mbl] + ((((size_t)A.prank * A.mbl + mb % A.mbl) * ASTR + (a0 >> 1)) * AS::NB + m % AS::NB) * 2;
                } else {
                    dst = A.Tb + AS::t2_index_s(m, a0 >> 1, ASTR);
                }
                if (st_on) store_pair_hint(dst, X0, X1, pol_t2);
            } else {
                if (st_on) store_pair_hint(A.Tb + AS::t2_index(m, a0 >> 1), X0, X1, pol_t2);
            }
        }
    }
    }
    if constexpr (RUPD) {        // all warps (the producer contributes zero): r.r, count, convergence
        __shared__ double red[32];
        double tot[1];
        if (!grid_sum_last<1>(acc, A.partial, &A.sc->ticket[1], red, tot)) return;
        if (threadIdx.x == 0) cg_after_rr(A.sc, tot[0]);
    }
}

// --------------------------------------------------------------------------------------------- P2
//   column m of T2, in place:  T2[m][.] <- F^H ( shat[m][.] o F T2[m][.] )
// ENERGY = true (a separate instantiation) also accumulates the spectral half of the search length,
//   p.Cp = sum over the full spectrum of shat |P|^2 = 2 x (columns 0 < n < L/2) + (columns n = 0, L/2)      (Parseval),
// in the registers of the spectral multiply, and leaves one partial sum per column; row_inv2_kernel<.., 2> adds them up.
// SLAB = true (a separate instantiation): the launch covers the columns one rank owns; blockIdx.x numbers them locally (tensor-map
// coordinates), A.col0 + blockIdx.x is the global column (spectrum row, packed column 0).
template <typename T, typename P, int CTAS, bool ENERGY = false, bool SLAB = false>
__global__ void __launch_bounds__(P::NT, CTAS) col2_kernel(const ColArgs<T> A, const __grid_constant__ CUtensorMap tmap)
{
    using AS = AsyncShape<T, P>;
    constexpr int L = P::N, S = P::S, NT = P::NT, PM = per_max<P>();
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* const smem_raw = align128(smem_dyn);
    __shared__ __align__(8) uint64_t bar, ready;
    cx<T>* W = reinterpret_cast<cx<T>*>(smem_raw);
    T* sh = reinterpret_cast<T*>(smem_raw + AS::WBYTES);
    SmemIO<T, P> io{W};
    // column m of T2 (frequency freq_of(pos_of_col(m)); m = 0 is the packed n = 0 / L/2 column): 2 complex per row pair,
    // gathered by TMA into natural row order a = 2A + r, and scattered back the same way at the end
    const int lt = threadIdx.x, nl = (int)blockIdx.x, n = SLAB ? nl + A.col0 : nl;      // local (T2 of this launch) and global column
    constexpr int ABOX = AS::ABOX;
    constexpr uint32_t BOXB = (uint32_t)(ABOX * 2 * sizeof(cx<T>));
    if (A.pdl != 2) tma::grid_dep_launch();                 // pdl == 2: triggered after this kernel's own wait (below), see row_inv2_kernel
    constexpr bool LG = LSU_GATHER && !SLAB;                      // (the slab instantiation keeps the TMA gather: its T2 has another extent)
    if (lt == 0) {
        tma::prefetch_tmap(&tmap);
        tma::mbar_init(&bar, LG ? NT + 1 : 1);
        tma::mbar_init(&ready, NT / 32);
        tma::fence_mbar_init();
    }
    cx<T> wb[S + 1][PM];
    static_for_up<1, S - 1>([&](auto s) { base_tw<P, decltype(s)::value, T, GRP>(lt, A.tw, wb[decltype(s)::value]); });
    __syncthreads();                                              // the barriers exist before anybody arrives on them
    tma::grid_dep_wait();                                         // everything above overlaps the previous kernel's tail
    if (A.pdl == 2) tma::grid_dep_launch();
    // The CTAs that share an SM in the FIRST wave start a fraction of a column time apart (later waves inherit the offsets), so that one's
    // gather overlaps another's arithmetic instead of all of them moving through the same phase together.  Measured at L = 2048 fp64
    // (3 CTAs per SM): 1.5 us apart 93.2 -> 91.7 us per iteration, 0.8 us 91.9, 2 us 92.1, 3 us no gain.
    if (A.sc && A.sc->done) return;                               // after the stop: before any copy is issued (a no-op launch costs its launch only)
    if (A.stagger_ns > 0 && blockIdx.x >= (unsigned)A.nsm && blockIdx.x < (unsigned)(CTAS * A.nsm)) {
        tma::stagger_wait((unsigned long long)(blockIdx.x / (unsigned)A.nsm) * (unsigned long long)A.stagger_ns);
    }
    if constexpr (LG) {
        // column nl: cell (row pair a2) = 2 complex at T2[nl / NB][a2][nl % NB], CB bytes, to natural order in shared memory
        constexpr int CB = (int)(2 * sizeof(cx<T>)), PIECES = CB / 16;
        const unsigned char* src = reinterpret_cast<const unsigned char*>(A.Tb + AS::t2_index(nl, 0));
        constexpr size_t ASTRIDE = (size_t)AS::NB * CB;           // bytes between consecutive row pairs of one column
#pragma unroll 8
        for (int i = lt; i < (L / 2) * PIECES; i += NT)
            tma::cp_async16(smem_raw + (size_t)i * 16, src + (size_t)(i / PIECES) * ASTRIDE + (size_t)(i % PIECES) * 16);
        tma::cp_async_arrive(&bar);
    }
    if (lt == 0 && !FCG_PROBE_ON(0x200)) {
        tma::mbar_expect_tx(&bar, (uint32_t)((LG ? 0 : AS::WBYTES) + (n ? L * sizeof(T) : 0)));
        if constexpr (SLAB) {
            // straight from the exchange buffer R[source rank][local column block][local row pair][column][2 complex] (5-D map): row pair
            // s al + a of the column lands at its natural place, so nothing has to be repacked after the all-to-all
            for (int s2 = 0; s2 < A.nranks; ++s2)
                for (int a = 0; a < A.al; a += A.boxa)
                    tma::tensor_g2s_5d(smem_raw + (size_t)(s2 * A.al + a) * (2 * sizeof(cx<T>)), &tmap, 0, nl % AS::NB, a, nl / AS::NB, s2, &bar);
        } else if constexpr (!LG) {
#pragma unroll
        for (int b = 0; b < (L / 2) / ABOX; ++b)
            tma::tensor_g2s_4d(smem_raw + (size_t)b * BOXB, &tmap, 0, nl % AS::NB, b * ABOX, nl / AS::NB, &bar);
        }
        if (n) tma::bulk_g2s_hint(sh, A.shat + (size_t)n * L, (uint32_t)(L * sizeof(T)), &bar,
                                  (A.hints & 4) ? tma::policy_evict_first() : tma::policy_evict_normal());   // read once per iteration
    }
    if (!FCG_PROBE_ON(0x200)) tma::mbar_wait(&bar, 0, A.tmo);
    double energy = 0.0;

    auto ld_sw = [&](int e) { return io.ld(e); };
    auto st_sw = [&](int e, cx<T> v) { io.st(e, v); };
    // stages >= 2: grouped assignment, only the group synchronises (fcg_engine.cuh); a CTA barrier where all sub-blocks meet --
    // before the packed column's pair loop (after forward stage S) and before inverse stage 1 (after inverse stage 2)
    auto fwd_smem_stage = [&](auto s) {
        constexpr int sv = decltype(s)::value;
        cx<T> a[St<P, sv>::PER][St<P, sv>::R];
        stage_ld<P, sv, T, GRP>(lt, ld_sw, a);
        stage_math<P, sv, -1, T>(a, wb[sv]);
        stage_st<P, sv, T, GRP>(lt, st_sw, a);
        if constexpr (sv == S) __syncthreads(); else stage_sync<P, NT>(lt);
    };
    auto inv_smem_stage = [&](auto s) {
        constexpr int sv = decltype(s)::value;
        cx<T> a[St<P, sv>::PER][St<P, sv>::R];
        stage_ld<P, sv, T, GRP>(lt, ld_sw, a);
        stage_math<P, sv, +1, T>(a, wb[sv]);
        stage_st<P, sv, T, GRP>(lt, st_sw, a);
        if constexpr (sv == 2) __syncthreads(); else stage_sync<P, NT>(lt);
    };
    if (!FCG_PROBE_ON(0x100)) {
    {   // forward stage 1: the column arrived in natural (linear) order; it leaves the stage swizzled
        cx<T> a[St<P, 1>::PER][St<P, 1>::R];
        stage_ld<P, 1, T>(lt, [&](int e) { return W[e]; }, a);
        __syncthreads();
        stage_math<P, 1, -1, T>(a, wb[1]);
        stage_st<P, 1, T>(lt, st_sw, a);
        __syncthreads();
    }
    if (n != 0) {
        static_for_up<2, S - 1>(fwd_smem_stage);
        // last forward stage * shat * first inverse stage, in registers
        if constexpr (ENERGY) {
            run_middle<P, T, true, GRP>(lt, ld_sw, st_sw, [&](int g, int u) { return sh[u * (L / P::RLAST) + g]; }, &energy);
            energy *= 2.0;                                       // column n stands for n and L - n
        } else {
            run_middle<P, T, false, GRP>(lt, ld_sw, st_sw, [&](int g, int u) { return sh[u * (L / P::RLAST) + g]; });
        }
        if constexpr (S - 1 >= 2) stage_sync<P, NT>(lt); else __syncthreads();
        static_for_down<S - 1, 2>(inv_smem_stage);
    } else {
        // packed column: W = Y0 + i YN.  W'[m] = sp[m] W[m] + sm[m] conj W[-m], sp = (s0+sN)/2 (row 0 of shat),
        // sm = (s0-sN)/2 (row L/2 of shat); pairs (m, L-m), m <= L/2
        static_for_up<2, S>(fwd_smem_stage);
        const T* sp_ = A.shat;
        const T* sm_ = A.shat + (size_t)(L / 2) * L;
        for (int m = lt; m <= L / 2; m += NT) {
            const int e = P::pos_of(m), e2 = P::pos_of((L - m) % L);
            const cx<T> Wa = io.ld(e), Wb = io.ld(e2);
            cx<T> va, vb;
            const int i1 = P::shat_index(e), i2 = P::shat_index(e2);
            va.x = sp_[i1] * Wa.x + sm_[i1] * Wb.x; va.y = sp_[i1] * Wa.y - sm_[i1] * Wb.y;
            vb.x = sp_[i2] * Wb.x + sm_[i2] * Wa.x; vb.y = sp_[i2] * Wb.y - sm_[i2] * Wa.y;
            if constexpr (ENERGY) {
                // s0 |Y0|^2 + sN |YN|^2 at m (and the same again at -m) = sp/2 (|Wa|^2 + |Wb|^2) + sm Re(Wa Wb)
                const double na = (double)Wa.x * (double)Wa.x + (double)Wa.y * (double)Wa.y;
                const double nb = (double)Wb.x * (double)Wb.x + (double)Wb.y * (double)Wb.y;
                const double re = (double)Wa.x * (double)Wb.x - (double)Wa.y * (double)Wb.y;
                const double term = 0.5 * (double)sp_[i1] * (na + nb) + (double)sm_[i1] * re;
                energy += e2 != e ? 2.0 * term : term;
            }
            io.st(e, va);
            if (e2 != e) io.st(e2, vb);
        }
        __syncthreads();
        static_for_down<S, 2>(inv_smem_stage);
    }
    {   // inverse stage 1: swizzled in, natural order out, ready for the bulk store
        cx<T> a[St<P, 1>::PER][St<P, 1>::R];
        stage_ld<P, 1, T>(lt, ld_sw, a);
        stage_math<P, 1, +1, T>(a, wb[1]);
        __syncthreads();
        stage_st<P, 1, T>(lt, [&](int e, cx<T> v) { W[e] = v; }, a);
    }
    }
    tma::fence_proxy_async();                 // my writes -> visible to the async proxy
    tma::mbar_warp_arrive(&ready);
    if (lt == 0) {
        tma::mbar_wait(&ready, 0, A.tmo);            // every warp's part of the column is in place
        if constexpr (SLAB) {
            const CUtensorMap* pm = static_cast<const CUtensorMap*>(A.peer_maps);
            for (int s2 = 0; s2 < A.nranks; ++s2)
                for (int a = 0; a < A.al; a += A.boxa) {
                    const void* src = smem_raw + (size_t)(s2 * A.al + a) * (2 * sizeof(cx<T>));
                    if (pm) tma::tensor_s2g_4d(pm + s2, 0, nl % AS::NB, a, A.prank * A.mbl + nl / AS::NB, src);   // rank s2's T2, over NVLink
                    else tma::tensor_s2g_5d(&tmap, 0, nl % AS::NB, a, nl / AS::NB, s2, src);
                }
        } else if (!FCG_PROBE_ON(0x400)) {
#pragma unroll
        for (int b = 0; b < (L / 2) / ABOX; ++b)
            tma::tensor_s2g_4d(&tmap, 0, nl % AS::NB, b * ABOX, nl / AS::NB, smem_raw + (size_t)b * BOXB);
        }
        tma::bulk_commit();
    }
    if constexpr (ENERGY) {      // this column's share of sum shat |P|^2, while the scatter drains; the next pass adds the L/2 shares
        __shared__ double red[32];
        double ev[1] = {energy};
        block_sum<1>(ev, red);
        if (lt == 0) A.partial[nl] = ev[0];       // (slab: one per column of THIS rank; fcg_slab_cols_energy sums them)
    }
    if (lt == 0) tma::bulk_wait_read0();          // shared memory must outlive the store's read
}

// --------------------------------------------------------------------------------------------- P2, persistent
// The same column pass with the gather of the NEXT column in flight while the current one is being transformed: grid = SMs x
// CTAS persistent CTAs, two column buffers (column + spectrum row) per CTA, NT consumer threads + one producer warp whose lane 0
// owns every asynchronous copy:   G(0) G(1) | ready(0) -> S(0) -> read of S(0) done -> G(2) | ready(1) -> S(1) -> G(3) | ..
// (G = TMA gather of a column into its buffer, S = TMA scatter back).  col2_kernel leaves that overlap to the 3-6 CTAs that
// share an SM and loses the gather latency (~2 us of ~8 us per column at L = 2048 fp64) whenever they fall into step.
// Used where two buffers fit at least twice per SM (ColPShape::valid); otherwise col2_kernel.
template <typename T, typename P> struct ColPShape {
    using AS = AsyncShape<T, P>;
    static constexpr size_t BUF = AS::WBYTES + (size_t)P::N * sizeof(T);
    static constexpr size_t smem = 2 * BUF + 128;
    static constexpr int by_smem = (int)((size_t)FCG_MAX_SMEM / (smem + 1024 + 512));
    static constexpr int by_thr = AS::thread_cap / (P::NT + 32);
    static constexpr int CTAS = by_smem < by_thr ? by_smem : by_thr;
    static constexpr bool valid = AS::valid && CTAS >= 1;
};

template <typename T, typename P, int CTAS, bool ENERGY = false>
__global__ void __launch_bounds__(P::NT + 32, CTAS) col2p_kernel(const ColArgs<T> A, const __grid_constant__ CUtensorMap tmap)
{
    using AS = AsyncShape<T, P>;
    using CP = ColPShape<T, P>;
    constexpr int L = P::N, S = P::S, NT = P::NT, PM = per_max<P>();
    constexpr int ABOX = AS::ABOX;
    constexpr uint32_t BOXB = (uint32_t)(ABOX * 2 * sizeof(cx<T>));
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* const smem_raw = align128(smem_dyn);
    __shared__ __align__(8) uint64_t full[2], ready[2];
    __shared__ double red[32];
    const int lt = threadIdx.x, lane = lt & 31, warp = lt >> 5;
    int cnt = 0;
    while ((int)blockIdx.x + cnt * (int)gridDim.x < L / 2) ++cnt;
    auto col_of = [&](int i) { return (int)blockIdx.x + i * (int)gridDim.x; };
    if (A.pdl != 2) tma::grid_dep_launch();                 // pdl == 2: triggered after this kernel's own wait (below), see row_inv2_kernel
    if (lt == 0) {
        tma::prefetch_tmap(&tmap);
        for (int b = 0; b < 2; ++b) { tma::mbar_init(&full[b], LSU_GATHER ? 33 : 1); tma::mbar_init(&ready[b], NT / 32); }
        tma::fence_mbar_init();
    }
    __syncthreads();
    tma::grid_dep_wait();
    if (A.pdl == 2) tma::grid_dep_launch();
    if (A.sc && A.sc->done) return;                              // before any copy is issued

    if (warp == NT / 32) {
        // producer warp.  Lane 0 owns the TMA copies (spectrum row in, scatter out); with LSU_GATHER all 32 lanes gather the column
        // itself with 16-byte asynchronous copies (one arrival each on full[b] when theirs have landed) -- see LSU_GATHER above.
        const uint64_t pol = (A.hints & 4) ? tma::policy_evict_first() : tma::policy_evict_normal();   // spectrum rows: read once per iteration
        auto gather = [&](int i) {
            const int n = col_of(i), b = i & 1;
            unsigned char* Wb = smem_raw + (size_t)b * CP::BUF;
            if (FCG_PROBE_ON(0x200)) { if (LSU_GATHER || lane == 0) tma::mbar_arrive(&full[b]); if (LSU_GATHER && lane == 0) tma::mbar_arrive(&full[b]); return; }
            if constexpr (LSU_GATHER) {
                constexpr int CB = (int)(2 * sizeof(cx<T>)), PIECES = CB / 16;
                const unsigned char* src = reinterpret_cast<const unsigned char*>(A.Tb + AS::t2_index(n, 0));
                constexpr size_t ASTRIDE = (size_t)AS::NB * CB;
#pragma unroll 8
                for (int c = lane; c < (L / 2) * PIECES; c += 32)
                    tma::cp_async16(Wb + (size_t)c * 16, src + (size_t)(c / PIECES) * ASTRIDE + (size_t)(c % PIECES) * 16);
                tma::cp_async_arrive(&full[b]);
            }
            if (lane == 0) {
                tma::mbar_expect_tx(&full[b], (uint32_t)((LSU_GATHER ? 0 : AS::WBYTES) + (n ? L * sizeof(T) : 0)));
                if constexpr (!LSU_GATHER) {
#pragma unroll
                    for (int q = 0; q < (L / 2) / ABOX; ++q)
                        tma::tensor_g2s_4d(Wb + (size_t)q * BOXB, &tmap, 0, n % AS::NB, q * ABOX, n / AS::NB, &full[b]);
                }
                if (n) tma::bulk_g2s_hint(Wb + AS::WBYTES, A.shat + (size_t)n * L, (uint32_t)(L * sizeof(T)), &full[b], pol);
            }
        };
        if (!LSU_GATHER && lane != 0) return;
        if (cnt > 0) gather(0);
        if (cnt > 1) gather(1);
        for (int i = 0; i < cnt; ++i) {
            const int n = col_of(i), b = i & 1;
            unsigned char* Wb = smem_raw + (size_t)b * CP::BUF;
            tma::mbar_wait(&ready[b], (uint32_t)((i >> 1) & 1), A.tmo);          // every consumer warp's part of column i is in place
            if (lane == 0) {
                if (!FCG_PROBE_ON(0x400)) {
#pragma unroll
                for (int q = 0; q < (L / 2) / ABOX; ++q)
                    tma::tensor_s2g_4d(&tmap, 0, n % AS::NB, q * ABOX, n / AS::NB, Wb + (size_t)q * BOXB);
                }
                tma::bulk_commit();
                tma::bulk_wait_read0();                                        // the buffer may be refilled (or the CTA may exit)
            }
            if constexpr (LSU_GATHER) __syncwarp();                            // .. by every lane
            if (i + 2 < cnt) gather(i + 2);
        }
        return;
    }

    // ---- consumers
    cx<T> wb[S + 1][PM];
    static_for_up<1, S - 1>([&](auto s) { base_tw<P, decltype(s)::value, T, GRP>(lt, A.tw, wb[decltype(s)::value]); });
    for (int i = 0; i < cnt; ++i) {
        const int n = col_of(i), b = i & 1;
        cx<T>* W = reinterpret_cast<cx<T>*>(smem_raw + (size_t)b * CP::BUF);
        const T* sh = reinterpret_cast<const T*>(smem_raw + (size_t)b * CP::BUF + AS::WBYTES);
        SmemIO<T, P> io{W};
        double energy = 0.0;
        tma::mbar_wait(&full[b], (uint32_t)((i >> 1) & 1), A.tmo);
        auto ld_sw = [&](int e) { return io.ld(e); };
        auto st_sw = [&](int e, cx<T> v) { io.st(e, v); };
        auto fwd_smem_stage = [&](auto s) {              // (grouped stages and their barriers: see col2_kernel)
            constexpr int sv = decltype(s)::value;
            cx<T> a[St<P, sv>::PER][St<P, sv>::R];
            stage_ld<P, sv, T, GRP>(lt, ld_sw, a);
            stage_math<P, sv, -1, T>(a, wb[sv]);
            stage_st<P, sv, T, GRP>(lt, st_sw, a);
            if constexpr (sv == S) bar_named<NT>(); else stage_sync<P, NT>(lt);
        };
        auto inv_smem_stage = [&](auto s) {
            constexpr int sv = decltype(s)::value;
            cx<T> a[St<P, sv>::PER][St<P, sv>::R];
            stage_ld<P, sv, T, GRP>(lt, ld_sw, a);
            stage_math<P, sv, +1, T>(a, wb[sv]);
            stage_st<P, sv, T, GRP>(lt, st_sw, a);
            if constexpr (sv == 2) bar_named<NT>(); else stage_sync<P, NT>(lt);
        };
        if (!FCG_PROBE_ON(0x100)) {
        {   // forward stage 1: the column arrived in natural (linear) order; it leaves the stage swizzled
            cx<T> a[St<P, 1>::PER][St<P, 1>::R];
            stage_ld<P, 1, T>(lt, [&](int e) { return W[e]; }, a);
            bar_named<NT>();
            stage_math<P, 1, -1, T>(a, wb[1]);
            stage_st<P, 1, T>(lt, st_sw, a);
            bar_named<NT>();
        }
        if (n != 0) {
            static_for_up<2, S - 1>(fwd_smem_stage);
            if constexpr (ENERGY) {
                run_middle<P, T, true, GRP>(lt, ld_sw, st_sw, [&](int g, int u) { return sh[u * (L / P::RLAST) + g]; }, &energy);
                energy *= 2.0;
            } else {
                run_middle<P, T, false, GRP>(lt, ld_sw, st_sw, [&](int g, int u) { return sh[u * (L / P::RLAST) + g]; });
            }
            if constexpr (S - 1 >= 2) stage_sync<P, NT>(lt); else bar_named<NT>();
            static_for_down<S - 1, 2>(inv_smem_stage);
        } else {         // packed n = 0 / L/2 column, see col2_kernel
            static_for_up<2, S>(fwd_smem_stage);
            const T* sp_ = A.shat;
            const T* sm_ = A.shat + (size_t)(L / 2) * L;
            for (int m = lt; m <= L / 2; m += NT) {
                const int e = P::pos_of(m), e2 = P::pos_of((L - m) % L);
                const cx<T> Wa = io.ld(e), Wb = io.ld(e2);
                cx<T> va, vb;
                const int i1 = P::shat_index(e), i2 = P::shat_index(e2);
                va.x = sp_[i1] * Wa.x + sm_[i1] * Wb.x; va.y = sp_[i1] * Wa.y - sm_[i1] * Wb.y;
                vb.x = sp_[i2] * Wb.x + sm_[i2] * Wa.x; vb.y = sp_[i2] * Wb.y - sm_[i2] * Wa.y;
                if constexpr (ENERGY) {
                    const double na = (double)Wa.x * (double)Wa.x + (double)Wa.y * (double)Wa.y;
                    const double nb = (double)Wb.x * (double)Wb.x + (double)Wb.y * (double)Wb.y;
                    const double re = (double)Wa.x * (double)Wb.x - (double)Wa.y * (double)Wb.y;
                    const double term = 0.5 * (double)sp_[i1] * (na + nb) + (double)sm_[i1] * re;
                    energy += e2 != e ? 2.0 * term : term;
                }
                io.st(e, va);
                if (e2 != e) io.st(e2, vb);
            }
            bar_named<NT>();
            static_for_down<S, 2>(inv_smem_stage);
        }
        {   // inverse stage 1: swizzled in, natural order out, ready for the scatter
            cx<T> a[St<P, 1>::PER][St<P, 1>::R];
            stage_ld<P, 1, T>(lt, ld_sw, a);
            stage_math<P, 1, +1, T>(a, wb[1]);
            bar_named<NT>();
            stage_st<P, 1, T>(lt, [&](int e, cx<T> v) { W[e] = v; }, a);
        }
        }
        tma::fence_proxy_async();                 // my writes -> visible to the async proxy
        tma::mbar_warp_arrive(&ready[b]);
        if constexpr (ENERGY) {                   // this column's share of sum shat |P|^2 (consumers only; fixed order)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) energy += __shfl_down_sync(0xffffffffu, energy, o);
            if (lane == 0) red[warp] = energy;
            bar_named<NT>();
            if (lt == 0) {
                double e = 0.0;
                for (int w2 = 0; w2 < NT / 32; ++w2) e += red[w2];
                A.partial[n] = e;
            }
        }
    }
}

// --------------------------------------------------------------------------------------------- stand-alone transforms
// Column pass of fcg_fft_fwd / fcg_fft_inv on the T2 layout: forward only (DIR < 0, natural row-frequency order out) or
// inverse only (DIR > 0, natural order in).  Same gather / in-place / scatter plumbing as col2_kernel; kept as a kernel
// of its own so that the loop kernel's register allocation is not disturbed.
template <typename T, typename P, int CTAS, int DIR>
__global__ void __launch_bounds__(P::NT, CTAS) col2_xform_kernel(const ColArgs<T> A, const __grid_constant__ CUtensorMap tmap)
{
    using AS = AsyncShape<T, P>;
    constexpr int L = P::N, S = P::S, NT = P::NT, PM = per_max<P>(), EPT = L / NT;
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* const smem_raw = align128(smem_dyn);
    __shared__ __align__(8) uint64_t bar, ready;
    cx<T>* W = reinterpret_cast<cx<T>*>(smem_raw);
    SmemIO<T, P> io{W};
    const int lt = threadIdx.x, n = (int)blockIdx.x;
    constexpr int ABOX = AS::ABOX;
    constexpr uint32_t BOXB = (uint32_t)(ABOX * 2 * sizeof(cx<T>));
    if (lt == 0) {
        tma::prefetch_tmap(&tmap);
        tma::mbar_init(&bar, 1);
        tma::mbar_init(&ready, NT / 32);
        tma::fence_mbar_init();
        tma::mbar_expect_tx(&bar, (uint32_t)AS::WBYTES);
#pragma unroll
        for (int b = 0; b < (L / 2) / ABOX; ++b)
            tma::tensor_g2s_4d(smem_raw + (size_t)b * BOXB, &tmap, 0, n % AS::NB, b * ABOX, n / AS::NB, &bar);
    }
    __syncthreads();
    cx<T> wb[S + 1][PM];
    static_for_up<1, S - 1>([&](auto s) { base_tw<P, decltype(s)::value, T>(lt, A.tw, wb[decltype(s)::value]); });
    tma::mbar_wait(&bar, 0, A.tmo);
    auto ld_sw = [&](int e) { return io.ld(e); };
    auto st_sw = [&](int e, cx<T> v) { io.st(e, v); };
    if constexpr (DIR < 0) {
        {   // stage 1: linear in, swizzled out
            cx<T> a[St<P, 1>::PER][St<P, 1>::R];
            stage_ld<P, 1, T>(lt, [&](int e) { return W[e]; }, a);
            __syncthreads();
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
        cx<T> v[EPT];                       // digit-reversed -> natural order, through registers
#pragma unroll
        for (int i = 0; i < EPT; ++i) v[i] = io.ld(P::pos_of(lt + i * NT));
        __syncthreads();
#pragma unroll
        for (int i = 0; i < EPT; ++i) W[lt + i * NT] = v[i];
    } else {
        cx<T> v[EPT];                       // natural order -> digit-reversed positions
#pragma unroll
        for (int i = 0; i < EPT; ++i) v[i] = W[lt + i * NT];
        __syncthreads();
#pragma unroll
        for (int i = 0; i < EPT; ++i) io.st(P::pos_of(lt + i * NT), v[i]);
        __syncthreads();
        static_for_down<S, 2>([&](auto s) {
            constexpr int sv = decltype(s)::value;
            cx<T> a[St<P, sv>::PER][St<P, sv>::R];
            stage_ld<P, sv, T>(lt, ld_sw, a);
            stage_math<P, sv, +1, T>(a, wb[sv]);
            stage_st<P, sv, T>(lt, st_sw, a);
            __syncthreads();
        });
        cx<T> a[St<P, 1>::PER][St<P, 1>::R];
        stage_ld<P, 1, T>(lt, ld_sw, a);
        stage_math<P, 1, +1, T>(a, wb[1]);
        __syncthreads();
        stage_st<P, 1, T>(lt, [&](int e, cx<T> x) { W[e] = x; }, a);
    }
    tma::fence_proxy_async();
    tma::mbar_warp_arrive(&ready);
    if (lt == 0) {
        tma::mbar_wait(&ready, 0, A.tmo);
#pragma unroll
        for (int b = 0; b < (L / 2) / ABOX; ++b)
            tma::tensor_s2g_4d(&tmap, 0, n % AS::NB, b * ABOX, n / AS::NB, smem_raw + (size_t)b * BOXB);
        tma::bulk_commit();
        tma::bulk_wait_read0();
    }
}

// Column pass of fcg_fft_fwd / fcg_fft_inv that reads / writes the PUBLIC half spectrum X[m][n] (L x (L/2+1), n fastest) itself, so
// that a stand-alone transform is two launches (row pass + this) instead of three (+ t2_export / t2_import, 2 N w of pure layout
// traffic).  Column c of T2 is frequency n = freq_of(pos_of_col(c)); its L outputs are the strided column X[.][n]:
//   * FCG_F64: one complex is 16 bytes and a row of X is 16 (L/2+1) bytes, so the column is a legal TMA tensor tile (xmap: 3-D,
//     box = 1 complex x 1 column x XBOX rows) -- stored from / loaded into the natural-order column in shared memory;
//   * FCG_F32: 8-byte elements at a stride that is not a multiple of 16 bytes cannot be a tensor map: plain 8-byte accesses
//     straight from / to the registers that hold the natural-order column (neighbouring columns run on neighbouring SMs at the
//     same time, so L2 merges the pieces of a sector);
//   * column 0 is the packed pair n = 0, L/2 (W = Y0 + i YN): unpacked / packed with its mirror element, plain accesses.
template <typename T, typename P, int CTAS, int DIR>
__global__ void __launch_bounds__(P::NT, CTAS) col2_xpub_kernel(const ColArgs<T> A, const __grid_constant__ CUtensorMap tmap,
                                                                const __grid_constant__ CUtensorMap xmap)
{
    using AS = AsyncShape<T, P>;
    constexpr int L = P::N, S = P::S, NT = P::NT, PM = per_max<P>(), EPT = L / NT, XW = L / 2 + 1;
    constexpr bool XTMA = sizeof(T) == 8;
    constexpr int XBOX = L < 256 ? L : 256;
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* const smem_raw = align128(smem_dyn);
    __shared__ __align__(8) uint64_t bar, ready;
    cx<T>* W = reinterpret_cast<cx<T>*>(smem_raw);
    SmemIO<T, P> io{W};
    const int lt = threadIdx.x, c = (int)blockIdx.x;
    const int n = P::freq_of(AS::pos_of_col(c));                  // 0 for the packed column
    constexpr int ABOX = AS::ABOX;
    constexpr uint32_t BOXB = (uint32_t)(ABOX * 2 * sizeof(cx<T>));
    constexpr uint32_t XBOXB = (uint32_t)(XBOX * sizeof(cx<T>));
    cx<T>* const X = A.X;
    if (lt == 0) {
        tma::prefetch_tmap(&tmap);
        if (XTMA) tma::prefetch_tmap(&xmap);
        tma::mbar_init(&bar, 1);
        tma::mbar_init(&ready, NT / 32);
        tma::fence_mbar_init();
        if (DIR < 0) {
            tma::mbar_expect_tx(&bar, (uint32_t)AS::WBYTES);
#pragma unroll
            for (int b = 0; b < (L / 2) / ABOX; ++b)
                tma::tensor_g2s_4d(smem_raw + (size_t)b * BOXB, &tmap, 0, c % AS::NB, b * ABOX, c / AS::NB, &bar);
        } else if (XTMA && c != 0) {
            tma::mbar_expect_tx(&bar, (uint32_t)AS::WBYTES);
#pragma unroll
            for (int b = 0; b < L / XBOX; ++b)
                tma::tensor_g2s_3d(smem_raw + (size_t)b * XBOXB, &xmap, 0, n, b * XBOX, &bar);
        }
    }
    __syncthreads();
    cx<T> wb[S + 1][PM];
    static_for_up<1, S - 1>([&](auto s) { base_tw<P, decltype(s)::value, T>(lt, A.tw, wb[decltype(s)::value]); });
    auto ld_sw = [&](int e) { return io.ld(e); };
    auto st_sw = [&](int e, cx<T> v) { io.st(e, v); };
    const T h = (T)0.5;
    if constexpr (DIR < 0) {
        tma::mbar_wait(&bar, 0, A.tmo);
        {   // stage 1: linear in, swizzled out
            cx<T> a[St<P, 1>::PER][St<P, 1>::R];
            stage_ld<P, 1, T>(lt, [&](int e) { return W[e]; }, a);
            __syncthreads();
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
        cx<T> v[EPT];                       // digit-reversed -> natural order m = lt + i NT, in registers
#pragma unroll
        for (int i = 0; i < EPT; ++i) v[i] = io.ld(P::pos_of(lt + i * NT));
        if (c == 0) {                       // packed pair: X[m][0] and X[m][L/2] from Z[m] and its mirror Z[L - m]
#pragma unroll
            for (int i = 0; i < EPT; ++i) {
                const int m = lt + i * NT;
                const cx<T> a = v[i], b = io.ld(P::pos_of((L - m) % L));
                X[(size_t)m * XW] = mk<T>((a.x + b.x) * h, (a.y - b.y) * h);
                X[(size_t)m * XW + L / 2] = mk<T>((a.y + b.y) * h, (b.x - a.x) * h);
            }
            return;
        }
        if constexpr (!XTMA) {
#pragma unroll
            for (int i = 0; i < EPT; ++i) X[(size_t)(lt + i * NT) * XW + n] = v[i];
            return;
        } else {
            __syncthreads();
#pragma unroll
            for (int i = 0; i < EPT; ++i) W[lt + i * NT] = v[i];
            tma::fence_proxy_async();
            tma::mbar_warp_arrive(&ready);
            if (lt == 0) {
                tma::mbar_wait(&ready, 0, A.tmo);
#pragma unroll
                for (int b = 0; b < L / XBOX; ++b)
                    tma::tensor_s2g_3d(&xmap, 0, n, b * XBOX, smem_raw + (size_t)b * XBOXB);
                tma::bulk_commit();
                tma::bulk_wait_read0();
            }
        }
    } else {
        cx<T> v[EPT];                       // natural order in -> digit-reversed positions
        if (c == 0) {
#pragma unroll
            for (int i = 0; i < EPT; ++i) {
                const int m = lt + i * NT;
                const cx<T> x0 = X[(size_t)m * XW], xN = X[(size_t)m * XW + L / 2];
                v[i] = mk<T>(x0.x - xN.y, x0.y + xN.x);
            }
        } else if constexpr (!XTMA) {
#pragma unroll
            for (int i = 0; i < EPT; ++i) v[i] = X[(size_t)(lt + i * NT) * XW + n];
        } else {
            tma::mbar_wait(&bar, 0, A.tmo);
#pragma unroll
            for (int i = 0; i < EPT; ++i) v[i] = W[lt + i * NT];
            __syncthreads();
        }
#pragma unroll
        for (int i = 0; i < EPT; ++i) io.st(P::pos_of(lt + i * NT), v[i]);
        __syncthreads();
        static_for_down<S, 2>([&](auto s) {
            constexpr int sv = decltype(s)::value;
            cx<T> a[St<P, sv>::PER][St<P, sv>::R];
            stage_ld<P, sv, T>(lt, ld_sw, a);
            stage_math<P, sv, +1, T>(a, wb[sv]);
            stage_st<P, sv, T>(lt, st_sw, a);
            __syncthreads();
        });
        cx<T> a[St<P, 1>::PER][St<P, 1>::R];
        stage_ld<P, 1, T>(lt, ld_sw, a);
        stage_math<P, 1, +1, T>(a, wb[1]);
        __syncthreads();
        stage_st<P, 1, T>(lt, [&](int e, cx<T> x) { W[e] = x; }, a);
        tma::fence_proxy_async();
        tma::mbar_warp_arrive(&ready);
        if (lt == 0) {
            tma::mbar_wait(&ready, 0, A.tmo);
#pragma unroll
            for (int b = 0; b < (L / 2) / ABOX; ++b)
                tma::tensor_s2g_4d(&tmap, 0, c % AS::NB, b * ABOX, c / AS::NB, smem_raw + (size_t)b * BOXB);
            tma::bulk_commit();
            tma::bulk_wait_read0();
        }
    }
}

// T2 (columns in position order, row frequencies m in natural order after col2_xform<-1>) -> public half spectrum
// X[m][n], n = 0 .. L/2.  One CTA per row pair (m = 2A, 2A+1): its L complex numbers are whole 128-byte lines of T2; they are
// permuted to frequency order through shared memory and leave as two contiguous rows.  The packed column 0 (W = Y0 + i YN)
// is unpacked with its mirror row L - m, read straight from T2.
template <typename T, typename P>
__global__ void __launch_bounds__(256) t2_export_kernel(const cx<T>* __restrict__ T2, cx<T>* __restrict__ X)
{
    using AS = AsyncShape<T, P>;
    constexpr int L = P::N, XW = L / 2 + 1, SK = L / P::radix(1);     // consecutive frequencies sit SK tile entries apart: skew them
    auto sk = [](int i) { return i + i / SK; };
    extern __shared__ unsigned char smem_dyn[];
    cx<T>* tile = reinterpret_cast<cx<T>*>(smem_dyn);                 // [m][r]
    const int A2 = (int)blockIdx.x, tid = threadIdx.x;
    for (int i = tid; i < L; i += 256) {                               // i = 2 m + r; 2 NB consecutive i are one line
        const int m = i >> 1;
        tile[sk(i)] = T2[AS::t2_index(m, A2) + (i & 1)];
    }
    __syncthreads();
    const T h = (T)0.5;
    for (int i = tid; i < 2 * XW; i += 256) {
        const int r = i / XW, nn = i % XW, mrow = 2 * A2 + r;
        cx<T> out;
        if (nn == 0 || nn == L / 2) {
            const int mm = (L - mrow) % L;
            const cx<T> a = tile[sk(r)], b = T2[AS::t2_index(0, mm >> 1) + (mm & 1)];
            out = nn == 0 ? mk<T>((a.x + b.x) * h, (a.y - b.y) * h) : mk<T>((a.y + b.y) * h, (b.x - a.x) * h);
        } else {
            out = tile[sk(2 * AS::col_of_pos(P::pos_of(nn)) + r)];
        }
        X[(size_t)mrow * XW + nn] = out;
    }
}

// public half spectrum -> T2 (the inverse of t2_export_kernel)
template <typename T, typename P>
__global__ void __launch_bounds__(256) t2_import_kernel(const cx<T>* __restrict__ X, cx<T>* __restrict__ T2)
{
    using AS = AsyncShape<T, P>;
    constexpr int L = P::N, XW = L / 2 + 1, SK = L / P::radix(1);
    auto sk = [](int i) { return i + i / SK; };
    extern __shared__ unsigned char smem_dyn[];
    cx<T>* tile = reinterpret_cast<cx<T>*>(smem_dyn);                 // [m][r]
    const int A2 = (int)blockIdx.x, tid = threadIdx.x;
    for (int i = tid; i < 2 * XW; i += 256) {
        const int r = i / XW, nn = i % XW, mrow = 2 * A2 + r;
        if (nn == L / 2) continue;
        const cx<T> v = X[(size_t)mrow * XW + nn];
        if (nn == 0) {
            const cx<T> xN = X[(size_t)mrow * XW + L / 2];
            tile[sk(r)] = mk<T>(v.x - xN.y, v.y + xN.x);
        } else {
            tile[sk(2 * AS::col_of_pos(P::pos_of(nn)) + r)] = v;
        }
    }
    __syncthreads();
    for (int i = tid; i < L; i += 256) T2[AS::t2_index(i >> 1, A2) + (i & 1)] = tile[sk(i)];
}

// --------------------------------------------------------------------------------------------- P3
//   c = F_row^H T (rows a0, a0+1);  q = k o p + c  [+ partial p.q]   (or residual / apply / plain)
// Persistent and warp-specialised like P1.  The producer warp feeds two rings in consumption order: tiles of T2
// (TSUB columns x 2 rows as whole 128-byte lines, TMA tensor loads) for the rebuild of the packed spectrum, and strips
// of k, p (, f) for the epilogue; both run ahead across transforms as far as shared memory allows.
// PRE = true (a separate instantiation) is the preconditioner pass of PCG: z = c, partial r.z, strips r0 r1 (k = r).
// VAR = 2 (CGF) is the last pass of the spectral-search-length path.  p.Ap = sum k p^2 + sum shat |P|^2
// (Parseval) is known before the pass starts: the first term is carried by a scalar recurrence (below), the second is the sum
// of the column pass's L/2 partial sums, which every CTA adds up itself in the same fixed order (bit-identical alpha in all
// CTAs, no broadcast).  So q = k o p + c is consumed on the spot -- r -= alpha q, r.r -> count, convergence, beta -- and never
// stored: strips k0 k1 p0 p1 r0 r1, output r in place.  The pass also accumulates t = sum k r'^2 and v = sum k r' p for
//     sum k p'^2 = t + 2 beta v + beta^2 sum k p^2        (p' = r' + beta p, the next direction).
// VAR = 3 is the same pass for the force formulation under reading F1: q = p + k o G p, and because every
// CG vector is zero on the broken bonds and k = kappa on the others, p.q = sum p^2 + kappa sum g |P|^2 -- the recurrence runs with
// unit weights (t = sum r'^2, v = sum r' p) and the column pass's energy is scaled by kappa.
template <typename T, typename P, int CTAS, int VAR = 0>
__global__ void __launch_bounds__(AsyncShape<T, P>::INV_THREADS, CTAS) row_inv2_kernel(const RowInvArgs<T> A, const __grid_constant__ CUtensorMap tmap)
{
    using AS = AsyncShape<T, P>;
    constexpr int L = P::N, S = P::S, NT = P::NT, R1 = AS::R1, Q1 = AS::Q1, PER1 = AS::PER1, PM = per_max<P>();
    constexpr bool PRE = VAR == 1, CGF = VAR == 2 || VAR == 3 || VAR == 5, FCGF = VAR == 3;
    constexpr bool SLAB = VAR == 4 || VAR == 5;      // one rank's row slab: A.ntile row pairs; sums go to A.xch, no scalar step
    constexpr bool SCGF = VAR == 5;      // slab + fused residual update: alpha comes from the scalar block (fcg_slab_scalar(4) after the all-reduce
                                         // of the ranks' spectral sums), the three sums of the own rows go to A.xch
    constexpr int TSUB = AS::TSUB, NSUB = AS::NSUB;
    constexpr uint32_t TBYTES = (uint32_t)AS::TSB;
    // CGF moves three vectors of strips per transform against one of tiles: the tile ring is kept short (TCAP) and the strips
    // get the rest; where whole stage-1 strips would leave too few slots they are NT elements long (SPT of them per stage-1 strip)
    // (whole stage-1 strips where three slots of those fit beside two tiles: 512-byte pieces cost more than they bring)
    constexpr bool FINE = CGF && (AS::RING_BUDGET - 2 * AS::TSB) / (6 * (size_t)AS::PIECE) < 3;
    constexpr int SPT = FINE ? PER1 : 1, QV = FINE ? NT : Q1;
    constexpr uint32_t PIECE = (uint32_t)(QV * sizeof(T));
    constexpr int NTSF_ = (int)((AS::RING_BUDGET - 12 * (size_t)PIECE) / AS::TSB);
    constexpr int TCAP = (int)(20480 / AS::TSB) < 2 ? 2 : (int)(20480 / AS::TSB);     // ~20 KB of tiles in flight (measured: 2 x 8 KB at L = 2048 fp64, 5 x 4 KB at L = 8192 fp32)
    constexpr int TCAP1 = AS::CRES_I == 1 ? NSUB : TCAP;   // one resident CTA: nobody else covers the rebuild's wait, keep a whole transform of tiles
    constexpr int TCAP2 = TCAP1 > NSUB ? NSUB : (TCAP1 > AS::MAXSLOT ? AS::MAXSLOT : TCAP1);
    constexpr int NTS = CGF ? (NTSF_ < 2 ? 2 : (NTSF_ > TCAP2 ? TCAP2 : NTSF_)) : AS::NTS;
    constexpr size_t KRB = CGF ? AS::RING_BUDGET - (size_t)NTS * AS::TSB : AS::KRB;
    static_assert(NTS <= AS::MAXSLOT && KRB >= 6 * (size_t)PIECE, "P3 rings");
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* const smem_raw = align128(smem_dyn);
    __shared__ __align__(8) uint64_t tfull[AS::MAXSLOT], tempty[AS::MAXSLOT];
    __shared__ __align__(8) uint64_t kfull[AS::MAXSLOT], kempty[AS::MAXSLOT];
    __shared__ double red[3 * 32];                // (one array for all variants: a second one costs the fourth CTA per SM at L = 2048 fp32)
    cx<T>* W = reinterpret_cast<cx<T>*>(smem_raw);
    unsigned char* const tring = smem_raw + AS::WBYTES;
    unsigned char* const kring = tring + (size_t)NTS * AS::TSB;
    SmemIO<T, P> io{W};
    const int lt = threadIdx.x, lane = lt & 31, warp = lt >> 5;
    const int mode = PRE ? (int)ROWI_PRECOND : CGF ? (int)ROWI_CGF : A.mode;
    const bool force = FCGF || (!PRE && !CGF && A.form != 0);
    tma::grid_dep_launch();
    const bool st_on = A.mode >= 0;                               // always true, opaque to the compiler (as in row_fwd2_kernel)
    const int nv = PRE ? 2 : CGF ? 6 : (mode == ROWI_PLAIN ? 0 : (mode == ROWI_RESID ? 6 : 4));
    int nks = nv ? (int)(KRB / (nv * PIECE)) : 1;
    nks = nks > AS::MAXSLOT ? AS::MAXSLOT : nks;
    const uint32_t kslotb = nv * PIECE;

    const int nsm = A.nsm < (int)gridDim.x ? A.nsm : (int)gridDim.x, grp = (int)blockIdx.x % nsm, jj = (int)blockIdx.x / nsm,
              kk = (int)gridDim.x / nsm;
    const bool whole = (int)gridDim.x % nsm == 0;        // else: one transform per CTA, every transform resident at once
    auto tile_of = [&](int i) { return whole ? grp + nsm * (jj + i * kk) : (int)blockIdx.x + i * (int)gridDim.x; };
    int ntl = 0;
    while (tile_of(ntl) < (SLAB ? A.ntile : L / 2)) ++ntl;

    if (lt == 0) {
        tma::prefetch_tmap(&tmap);
        for (int i = 0; i < NTS; ++i) { tma::mbar_init(&tfull[i], 1); tma::mbar_init(&tempty[i], NT / 32); }
        for (int i = 0; i < AS::MAXSLOT; ++i) { tma::mbar_init(&kfull[i], 1); tma::mbar_init(&kempty[i], NT / 32); }
        tma::fence_mbar_init();
    }
    __syncthreads();

    double acc[2] = {0.0, 0.0};
    double acc3[3] = {0.0, 0.0, 0.0};            // CGF: r'.r', sum k r'^2, sum k r' p
    double alpha_d = 0.0, pq_d = 0.0;
    T alpha = (T)0;
    // Producer state: next tile of T2 / next strip to issue, in consumption order.  With PW (small transforms) two extra
    // warps run these loops; otherwise (NT >= 512, where two more warps would cost 8 registers per thread) consumer warp 0
    // issues the successor of every slot it has just seen released.
    constexpr bool PW = AS::PRODUCER_WARPS;
    int p_ts = 0, p_tn = 0, p_ks = 0, p_kn = 0;
    uint32_t p_tph = 0, p_kph = 0;
    const int GT = ntl * NSUB, GK = nv ? ntl * R1 * SPT : 0;
    const T* kbase = nullptr;
    if (nv) kbase = (lane < 2 ? A.k : lane < 4 ? A.v : A.f) + (size_t)(lane & 1) * L;
    // L2 hints: T2 is dead once this pass has read it (bit 3); k comes back only in the next iteration (bit 4)
    const uint64_t pol_t = (A.hints & 8) ? tma::policy_evict_first() : tma::policy_evict_normal();
    const uint64_t pol_r = (A.hints & 128) ? tma::policy_evict_last() : tma::policy_evict_normal();   // (bit 7) the new r is read back by the next P1
    const uint64_t pol_k = (lane < 2 && !PRE && (A.hints & 16)) ? tma::policy_evict_first() : tma::policy_evict_normal();
    auto issue_next_T = [&]() {          // whole warp; tile p_tn = (transform p_tn / NSUB, part p_tn % NSUB): TSUB / NB whole lines
        if (p_tn >= NTS) tma::mbar_wait(&tempty[p_ts], p_tph ^ 1u, A.tmo);
        if (lane == 0) {
            tma::mbar_expect_tx(&tfull[p_ts], TBYTES);
            tma::tensor_g2s_3d_hint(tring + (size_t)p_ts * TBYTES, &tmap, 0, tile_of(p_tn / NSUB), (p_tn % NSUB) * (TSUB / AS::NB), &tfull[p_ts], pol_t);
        }
        ++p_tn;
        if (++p_ts == NTS) { p_ts = 0; p_tph ^= 1u; }
    };
    auto issue_next_K = [&]() {          // whole warp; strip p_kn % (R1 SPT) of k0 k1 v0 v1 (f0 f1) of transform p_kn / (R1 SPT), one bulk copy per lane < nv
        if (p_kn >= nks) tma::mbar_wait(&kempty[p_ks], p_kph ^ 1u, A.tmo);
        if (lane == 0) tma::mbar_expect_tx(&kfull[p_ks], kslotb);
        __syncwarp();
        if (lane < nv)
            tma::bulk_g2s_hint(kring + (size_t)p_ks * kslotb + (size_t)lane * PIECE,
                               kbase + (size_t)(2 * tile_of(p_kn / (R1 * SPT))) * L + (size_t)((p_kn % (R1 * SPT)) / SPT) * Q1 + (size_t)(p_kn % SPT) * QV,
                               PIECE, &kfull[p_ks], pol_k);
        ++p_kn;
        if (++p_ks == nks) { p_ks = 0; p_kph ^= 1u; }
    };
    // pdl == 2 (programmatic dependent launch with the column pass triggering after ITS wait, so that this section never runs before the
    // previous iteration has completed): the strips k, p, r depend on nothing the column pass writes -- the strip producer fills its
    // ring during the column pass's tail.
    constexpr bool EARLY = CGF && !SLAB && PW && AS::NPW == 2;
    if constexpr (EARLY) {
        if (A.pdl == 2 && warp == NT / 32 + 1 && !*reinterpret_cast<const volatile int*>(&A.sc->done))
            while (p_kn < GK && p_kn < nks) issue_next_K();
    }
    tma::grid_dep_wait();                                         // everything above overlaps the previous kernel's tail
    if ((mode == ROWI_CG || PRE || CGF) && A.sc->done) return;
    if (jj > 0 && A.stagger_ns > 0) {      // the later CTAs of an SM start a fraction of a transform time after the first (see stagger_wait)
        tma::stagger_wait((unsigned long long)jj * (unsigned long long)A.stagger_ns);
    }
    if constexpr (SCGF) {
        pq_d = A.sc->pq; alpha_d = A.sc->alpha; alpha = (T)alpha_d;      // (a breakdown has set sc->done: the pass returned above)
    } else if constexpr (CGF) {
        // search length from the column pass's partial sums, by ALL threads before the roles split (a breakdown must
        // stop producers and consumers alike); same order in every CTA, so alpha is bit-identical everywhere
        double e = 0.0;
        for (int i = lt; i < L / 2; i += (int)blockDim.x) e += __ldcg(A.colsum + i);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
        if (lane == 0) red[warp] = e;
        __syncthreads();
        e = 0.0;
        for (int w2 = 0; w2 < (int)(blockDim.x >> 5); ++w2) e += red[w2];
        __syncthreads();
        pq_d = A.sc->kpp + (FCGF ? A.kappa * e : e);
        if (!(pq_d > 0.0) || !isfinite(pq_d)) {                   // breakdown: nothing may change; CTA 0 reports it
            if (blockIdx.x == 0 && lt == 0) { A.sc->pq = pq_d; A.sc->status = ST_BREAKDOWN; A.sc->done = 1; A.sc->alpha = 0.0; set_cond(A.sc, false); }
            if constexpr (EARLY) {                                // strips issued before the wait must have landed before the CTA leaves
                if (warp == NT / 32 + 1) for (int s2 = 0; s2 < p_kn; ++s2) tma::mbar_wait(&kfull[s2], 0u, A.tmo);
            }
            return;
        }
        alpha_d = A.sc->rho / pq_d;
        alpha = (T)alpha_d;
    }
    if (PW && AS::NPW == 1 && warp == NT / 32) {       // one producer warp: tiles, then strips, of each transform in consumption order
        for (int i = 0; i < ntl; ++i) {
            for (int c = 0; c < NSUB; ++c) issue_next_T();
            if (nv) for (int c = 0; c < R1 * SPT; ++c) issue_next_K();
        }
    } else if (PW && AS::NPW == 2 && warp == NT / 32) {
        while (p_tn < GT) issue_next_T();
    } else if (PW && AS::NPW == 2 && warp == NT / 32 + 1) {
        while (p_kn < GK) issue_next_K();
    } else if (warp < NT / 32) {
        if (!PW && warp == 0) {
            while (p_tn < GT && p_tn < NTS) issue_next_T();
            while (p_kn < GK && p_kn < nks) issue_next_K();
        }
        // ---- consumers
        cx<T> wb[S + 1][PM];
        static_for_up<1, S - 1>([&](auto s) { base_tw<P, decltype(s)::value, T, GRP>(lt, A.tw, wb[decltype(s)::value]); });
        int ts = 0, ks = 0;
        uint32_t tph = 0, kph = 0;
        for (int i = 0; i < ntl; ++i) {
            const int a0 = 2 * tile_of(i);
            const size_t row0 = (size_t)a0 * L;
            // rebuild the packed spectrum Z = X_even + i X_odd at its digit-reversed place, tile by tile
            for (int sub = 0; sub < NSUB; ++sub) {
                tma::mbar_wait(&tfull[ts], tph, A.tmo);
                const cx<T>* Ts = reinterpret_cast<const cx<T>*>(tring + (size_t)ts * TBYTES);
#pragma unroll 4
                for (int ml = lt; ml < TSUB; ml += NT) {
                    const int e = AS::pos_of_col(sub * TSUB + ml);
                    const int n = P::freq_of(e);
                    const cx<T> X0 = Ts[2 * ml], X1 = Ts[2 * ml + 1];
                    if (n == 0) {
                        io.st(P::pos_of(0), mk<T>(X0.x, X1.x));
                        io.st(P::pos_of(L / 2), mk<T>(X0.y, X1.y));
                    } else {
                        io.st(e, mk<T>(X0.x - X1.y, X0.y + X1.x));
                        io.st(P::pos_of(L - n), mk<T>(X0.x + X1.y, X1.x - X0.y));
                    }
                }
                tma::mbar_warp_release_consumed(&tempty[ts]);         // this warp has read the tile (and used every value)
                if (!PW && warp == 0 && p_tn < GT) issue_next_T();
                if (++ts == NTS) { ts = 0; tph ^= 1u; }
            }
            bar_named<NT>();                                          // Z complete in W
            if (!FCG_PROBE_ON(0x800))
            static_for_down<S, 2>([&](auto s) {
                constexpr int sv = decltype(s)::value;
                cx<T> a[St<P, sv>::PER][St<P, sv>::R];
                stage_ld<P, sv, T, GRP>(lt, [&](int e) { return io.ld(e); }, a);
                stage_math<P, sv, +1, T>(a, wb[sv]);
                stage_st<P, sv, T, GRP>(lt, [&](int e, cx<T> v) { io.st(e, v); }, a);
                if constexpr (sv == 2) bar_named<NT>();           // stage 1 joins the sub-blocks: everybody's
                else stage_sync<P, NT>(lt);
            });
            // inverse stage 1 straight into the epilogue: natural order, re = even row, im = odd row
            cx<T> c[PER1][R1];
            stage_ld<P, 1, T>(lt, [&](int e) { return io.ld(e); }, c);
            bar_named<NT>();                                          // W may now be rebuilt for the next transform
            stage_math<P, 1, +1, T>(c, wb[1]);
            double f_rr = 0.0, f_t = 0.0, f_v = 0.0;                 // CGF: products and sums in double for both dtypes (reading S12)
#pragma unroll
            for (int t = 0; t < R1; ++t) {
#pragma unroll
              for (int qq = 0; qq < SPT; ++qq) {
                const T* sl = nullptr;
                if (nv) {
                    tma::mbar_wait(&kfull[ks], kph, A.tmo);
                    sl = reinterpret_cast<const T*>(kring + (size_t)ks * kslotb);
                }
#pragma unroll
                for (int q = FINE ? qq : 0; q < (FINE ? qq + 1 : PER1); ++q) {
                    const int j = FINE ? lt : lt + q * NT;              // element within the piece
                    const size_t i0 = row0 + (size_t)t * Q1 + lt + q * NT;
                    const T c0 = c[q][t].x, c1 = c[q][t].y;
                    if (mode == ROWI_PLAIN) { A.out[i0] = c0 * A.scale; A.out[i0 + L] = c1 * A.scale; continue; }
                    if constexpr (PRE) {                                                   // z = M^-1 r, r.z
                        if (st_on) { A.out[i0] = c0; A.out[i0 + L] = c1; }
                        acc[0] += (double)sl[j] * (double)c0; acc[0] += (double)sl[QV + j] * (double)c1;
                        continue;
                    }
                    const T v0 = sl[2 * QV + j], v1 = sl[3 * QV + j];
                    const T val0 = force ? v0 + sl[j] * c0 : sl[j] * v0 + c0,            // k o x + C x, or the force
                            val1 = force ? v1 + sl[QV + j] * c1 : sl[QV + j] * v1 + c1;  // formulation x + k o (G x) (eq. (2))
                    if constexpr (CGF) {
                        const T r0 = sl[4 * QV + j] - alpha * val0, r1 = sl[5 * QV + j] - alpha * val1;   // residue
                        if (st_on) { tma::st_hint(A.out + i0, r0, pol_r); tma::st_hint(A.out + i0 + L, r1, pol_r); }
                        const double r0d = (double)r0, r1d = (double)r1;
                        f_rr += r0d * r0d; f_rr += r1d * r1d;                                               // residue length (97)
                        const double kr0 = FCGF ? r0d : (double)sl[j] * r0d, kr1 = FCGF ? r1d : (double)sl[QV + j] * r1d;
                        f_t += kr0 * r0d; f_t += kr1 * r1d;
                        f_v += kr0 * (double)v0; f_v += kr1 * (double)v1;
                        continue;
                    }
                    if (mode == ROWI_RESID) {
                        const T f0 = force ? sl[j] * A.dval : sl[4 * QV + j], f1 = force ? sl[QV + j] * A.dval : sl[5 * QV + j];   // form 1: f = K D
                        const T r0 = f0 - val0, r1 = f1 - val1;                           // r = f - A u
                        A.out[i0] = r0; A.out[i0 + L] = r1; A.out2[i0] = (T)0; A.out2[i0 + L] = (T)0;
                        acc[0] += (double)r0 * (double)r0; acc[0] += (double)r1 * (double)r1;
                        acc[1] += (double)f0 * (double)f0; acc[1] += (double)f1 * (double)f1;
                    } else {
                        if (st_on) { A.out[i0] = val0; A.out[i0 + L] = val1; }
                        acc[0] += (double)v0 * (double)val0; acc[0] += (double)v1 * (double)val1;   // search length p.Ap
                    }
                }
                if (nv) {
                    tma::mbar_warp_release_consumed(&kempty[ks]);
                    if (!PW && warp == 0 && p_kn < GK) issue_next_K();
                    if (++ks == nks) { ks = 0; kph ^= 1u; }
                }
              }
            }
            if constexpr (CGF) { acc3[0] += f_rr; acc3[1] += f_t; acc3[2] += f_v; }
        }
    }
    if constexpr (CGF) {         // all warps (the producers contribute zeros)
        double tot[3];
        if (!grid_sum_last<3>(acc3, A.partial, &A.sc->ticket[0], red, tot)) return;
        if constexpr (SCGF) {
            if (threadIdx.x == 0) { A.xch[0] = tot[0]; A.xch[1] = tot[1]; A.xch[2] = tot[2]; A.xch[3] = 0.0; }
            return;
        }
        if (threadIdx.x == 0) {
            Scalars* sc = A.sc;
            sc->alpha = alpha_d; sc->pq = pq_d;
            const double kpp = sc->kpp;
            cg_after_rr(sc, tot[0]);                                                  // count, convergence, beta, rho
            if (!sc->done) sc->kpp = tot[1] + 2.0 * sc->beta * tot[2] + sc->beta * sc->beta * kpp;
        }
        return;
    }
    row_inv_reduce_finalize<T>(A, acc, red);      // all warps (the producer contributes zeros)
}

#endif  // __CUDACC__

}  // namespace fcg
