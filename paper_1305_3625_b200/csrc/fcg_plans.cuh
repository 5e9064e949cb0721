// fcg_plans.cuh -- radix plans and launch shapes per (dtype, L), and the type-erased launcher table
// each per-L translation unit (fcg_inst.cu) exports to fcg.cu.
#pragma once
#include <cuda_runtime.h>
#include "fcg_math.cuh"

namespace fcg {

// Radix choice: as few stages as possible (each stage is one shared-memory round trip), radix <= 16
// (64 fp64 registers of data per thread), and the last radix >= the number of complex elements per
// 128 B where possible so that the stride-1 runs of the earlier stages cover whole bank groups
// (8 for fp64, 16 for fp32).
template <typename T, int L> struct PlanFor;
#define FCG_PLAN(TYPE, L, R1, R2, R3, R4) \
    template <> struct PlanFor<TYPE, L> { using type = Plan<L, R1, R2, R3, R4>; };
FCG_PLAN(double, 16, 4, 4, 1, 1)      FCG_PLAN(float, 16, 4, 4, 1, 1)
FCG_PLAN(double, 32, 4, 8, 1, 1)      FCG_PLAN(float, 32, 4, 8, 1, 1)
FCG_PLAN(double, 64, 8, 8, 1, 1)      FCG_PLAN(float, 64, 4, 16, 1, 1)
FCG_PLAN(double, 128, 16, 8, 1, 1)    FCG_PLAN(float, 128, 8, 16, 1, 1)
FCG_PLAN(double, 256, 4, 4, 4, 4)     FCG_PLAN(float, 256, 4, 4, 4, 4)
FCG_PLAN(double, 512, 8, 8, 8, 1)     FCG_PLAN(float, 512, 4, 8, 16, 1)
// L = 1024 and 2048 in fp64: measured in round 2 (interleaved runs on one box, us per CG iteration): 1024: (8,8,4,4) 42.5, (16,8,8) 47.5,
// (8,16,8) 41.0, (16,16,4) 48.3, (4,4,8,8) 40.2;  2048: (16,16,8) 94.5, (8,8,4,8) 100.2, (4,8,8,8) 103.1, (16,8,16) 95.9, (8,16,16) 93.1 --
// a last radix that spans a whole 128-byte line (8 in fp64) or two helps the last pass; 256 threads per transform lose in the column pass.
#ifndef FCG_P1024D_R1        // (-DFCG_P1024D_R1=.. -DFCG_P1024D_R2=.. ..; the same for 2048: plan experiments)
#define FCG_P1024D_R1 4
#define FCG_P1024D_R2 4
#define FCG_P1024D_R3 8
#define FCG_P1024D_R4 8
#endif
#ifndef FCG_P2048D_R1
#define FCG_P2048D_R1 8
#define FCG_P2048D_R2 16
#define FCG_P2048D_R3 16
#define FCG_P2048D_R4 1
#endif
FCG_PLAN(double, 1024, FCG_P1024D_R1, FCG_P1024D_R2, FCG_P1024D_R3, FCG_P1024D_R4)   FCG_PLAN(float, 1024, 8, 8, 16, 1)
FCG_PLAN(double, 2048, FCG_P2048D_R1, FCG_P2048D_R2, FCG_P2048D_R3, FCG_P2048D_R4)  FCG_PLAN(float, 2048, 8, 16, 16, 1)
FCG_PLAN(double, 4096, 16, 16, 16, 1) FCG_PLAN(float, 4096, 16, 16, 16, 1)
FCG_PLAN(double, 8192, 16, 8, 8, 8)   FCG_PLAN(float, 8192, 8, 8, 8, 16)
#undef FCG_PLAN

constexpr int FCG_MAX_SMEM = 227 * 1024;
constexpr int FCG_NROWVAR = 4;

// Row-pass variants: F packed transforms (2F rows) per CTA, F = Fmin * 2^v.  A variant is valid when the
// CTA fits (threads <= 1024, shared memory <= 227 KB) and does not exceed the lattice.
template <typename T, typename P> struct RowShape {
    static constexpr int FMIN = (32 / P::NT) > 1 ? (32 / P::NT) : 1;
    static constexpr int F(int v) { return FMIN << v; }
    static constexpr size_t smem(int v) { return (size_t)F(v) * (P::N + 2) * 2 * sizeof(T); }
    static constexpr bool valid(int v) {
        return 2 * F(v) <= P::N && F(v) * P::NT <= 1024 && smem(v) <= (size_t)FCG_MAX_SMEM;
    }
};
// Column pass: COLS columns per CTA so that a CTA has at least 64 threads (one column once NT >= 64).
template <typename T, typename P> struct ColShape {
    static constexpr int COLS0 = (64 / P::NT) > 1 ? (64 / P::NT) : 1;
    static constexpr int COLS = COLS0 > P::N / 2 ? P::N / 2 : COLS0;
    static constexpr size_t smem = (size_t)COLS * (P::N + 2) * 2 * sizeof(T);
    static_assert(smem <= (size_t)FCG_MAX_SMEM, "column does not fit in shared memory");
};

// What fcg.cu sees of one (L, dtype): plain function pointers, arguments type-erased
// (RowFwdArgs<T>*, ColArgs<T>*, RowInvArgs<T>* of the matching T).
struct PassTable {
    int L, dtype;
    int row_valid[FCG_NROWVAR], row_F[FCG_NROWVAR], row_threads[FCG_NROWVAR];
    size_t row_smem[FCG_NROWVAR];
    int cols, col_threads; size_t col_smem;
    int tw_total;                                  // entries of the per-stage twiddle tables (Plan::TW_TOTAL)
    void (*fill_twiddles)(void* host_buf);         // host_buf: tw_total complex numbers of the table's dtype
    cudaError_t (*init)();
    cudaError_t (*row_fwd)(int var, const void* args, cudaStream_t st);
    cudaError_t (*col)(const void* args, cudaStream_t st);
    cudaError_t (*row_inv)(int var, const void* args, cudaStream_t st);
    cudaError_t (*spectrum_prep)(const void* s, void* shat, int colpos, cudaStream_t st);
    // pipelined (TMA) passes of fcg_async.cuh; v2 == 0 when the size is too small for them
    int v2, v2_nb, v2_abox, v2_tsub, v2_threads, v2_ctas[3];   // nb: columns per 128-byte line of T2; abox: row pairs per column box;
                                                   // tsub: columns per row-pass tile; ctas: resident CTAs/SM asked for (fwd, col, inv)
    size_t v2_smem[3];
    cudaError_t (*row_fwd2)(const void* args, cudaStream_t st);
    cudaError_t (*col2)(const void* args, const void* tensor_map, cudaStream_t st);
    cudaError_t (*row_inv2)(const void* args, const void* tensor_map, cudaStream_t st);
    // spectral search length: P2 with the spectral energy, P3 with alpha and the residual update fused
    // (q never stored); sl_ok == 0 when the size has no such instantiation
    int sl_ok;
    cudaError_t (*col2_energy)(const void* args, const void* tensor_map, cudaStream_t st);
    cudaError_t (*row_inv2_cgf)(const void* args, const void* tensor_map, cudaStream_t st);
    cudaError_t (*row_inv2_cgf_force)(const void* args, const void* tensor_map, cudaStream_t st);   // force formulation under reading F1
    // persistent, double-buffered column pass (col2p_kernel); colp_ok == 0 where two column buffers do not fit twice per SM
    int colp_ok, colp_ctas;
    cudaError_t (*col2p)(const void* args, const void* tensor_map, int energy, cudaStream_t st);
    cudaError_t (*row_fwd2_rupd)(const void* args, cudaStream_t st);                                // PCG: r update + r.r + row transforms of r
    cudaError_t (*row_inv2_pre)(const void* args, const void* tensor_map, cudaStream_t st);        // PCG: z = M^-1 r, r.z
    cudaError_t (*col2_xform)(const void* args, const void* tensor_map, int inverse, cudaStream_t st);   // stand-alone transforms
    cudaError_t (*col2_xpub)(const void* args, const void* tensor_map, const void* x_map, int inverse, cudaStream_t st);   // .. straight to / from X[m][n]
    cudaError_t (*t2_export)(const void* T2, void* X, cudaStream_t st);
    cudaError_t (*t2_import)(const void* X, void* T2, cudaStream_t st);
    // slab-decomposed CG: the three passes on one rank's share -- row pairs [0, ntile) of its own vectors,
    // `ncols` columns starting at global column col0
    cudaError_t (*row_fwd2_slab)(const void* args, cudaStream_t st);
    cudaError_t (*col2_slab)(const void* args, const void* tensor_map, int ncols, cudaStream_t st);
    cudaError_t (*row_inv2_slab)(const void* args, const void* tensor_map, cudaStream_t st);
    // the same with the spectral search length: column pass with its share of sum shat |P|^2, last pass with the residual update fused in
    cudaError_t (*col2_slab_e)(const void* args, const void* tensor_map, int ncols, cudaStream_t st);
    cudaError_t (*row_inv2_slab_f)(const void* args, const void* tensor_map, cudaStream_t st);
    // whole solve as one cooperative kernel (fcg_fused.cuh); fused == 0 when the size has none
    int fused, fused_grid;
    cudaError_t (*fused_solve)(const void* fused_args, cudaStream_t st);
};

#define FCG_DECL_TABLE(L) const PassTable* fcg_pass_table_##L(int dtype);
FCG_DECL_TABLE(16) FCG_DECL_TABLE(32) FCG_DECL_TABLE(64) FCG_DECL_TABLE(128) FCG_DECL_TABLE(256)
FCG_DECL_TABLE(512) FCG_DECL_TABLE(1024) FCG_DECL_TABLE(2048) FCG_DECL_TABLE(4096) FCG_DECL_TABLE(8192)
#undef FCG_DECL_TABLE

}  // namespace fcg
