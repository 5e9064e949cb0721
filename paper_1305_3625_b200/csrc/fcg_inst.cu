// fcg_inst.cu -- instantiates the transform passes for one lattice size.  Compiled once per supported L
// with -DFCG_INST_L=<L> (paper_1305_3625_b200/build.py) so the sizes build in parallel.
#include <cmath>
#include "fcg_plans.cuh"
#include "fcg_async.cuh"
#include "fcg_fused.cuh"

#ifndef FCG_INST_L
#error "compile with -DFCG_INST_L=<L>"
#endif

namespace fcg {
namespace {

template <typename T> struct Inst {
    using P = typename PlanFor<T, FCG_INST_L>::type;
    using RS = RowShape<T, P>;
    using CS = ColShape<T, P>;
    using AS = AsyncShape<T, P>;
    static constexpr int L = FCG_INST_L;
    static constexpr bool V2 = AS::valid;
    static constexpr int C_FWD = AS::ctas(AS::fwd_smem, 320, 32), C_COL = AS::ctas(AS::col_smem, 64, 64),
                         C_INV = AS::ctas(AS::inv_smem, 1280, AS::INV_THREADS - P::NT);

    // opt in to > 48 KB of dynamic shared memory and ask for the largest shared-memory carveout, so that as
    // many CTAs as the register file allows are resident
    template <typename K> static cudaError_t prep(K kernel, size_t smem) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        return cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    }
    template <int V> static cudaError_t init_row() {
        if constexpr (RS::valid(V)) {
            cudaError_t e = prep(row_fwd_kernel<T, P, RS::F(V)>, RS::smem(V));
            if (e != cudaSuccess) return e;
            return prep(row_inv_kernel<T, P, RS::F(V)>, RS::smem(V));
        }
        return cudaSuccess;
    }
    static cudaError_t init() {
        cudaError_t e;
        if ((e = init_row<0>()) != cudaSuccess) return e;
        if ((e = init_row<1>()) != cudaSuccess) return e;
        if ((e = init_row<2>()) != cudaSuccess) return e;
        if ((e = init_row<3>()) != cudaSuccess) return e;
        if constexpr (V2) {
            if ((e = prep(row_fwd2_kernel<T, P, C_FWD>, AS::fwd_smem)) != cudaSuccess) return e;
            if ((e = prep(col2_kernel<T, P, C_COL>, AS::col_smem)) != cudaSuccess) return e;
            if ((e = prep(row_inv2_kernel<T, P, C_INV>, AS::inv_smem)) != cudaSuccess) return e;
            if ((e = prep(row_fwd2_kernel<T, P, C_FWD, 1>, AS::fwd_smem)) != cudaSuccess) return e;
            if ((e = prep(row_inv2_kernel<T, P, C_INV, 1>, AS::inv_smem)) != cudaSuccess) return e;
            if ((e = prep(col2_kernel<T, P, C_COL, true>, AS::col_smem)) != cudaSuccess) return e;
            if constexpr (COLP) {
                if ((e = prep(col2p_kernel<T, P, CPS::CTAS, true>, CPS::smem)) != cudaSuccess) return e;
                if ((e = prep(col2p_kernel<T, P, CPS::CTAS, false>, CPS::smem)) != cudaSuccess) return e;
            }
            if ((e = prep(row_inv2_kernel<T, P, C_INV, 2>, AS::inv_smem)) != cudaSuccess) return e;
            if ((e = prep(row_inv2_kernel<T, P, C_INV, 3>, AS::inv_smem)) != cudaSuccess) return e;
            if ((e = prep(row_fwd2_kernel<T, P, C_FWD, 2>, AS::fwd_smem)) != cudaSuccess) return e;
            if ((e = prep(col2_kernel<T, P, C_COL, false, true>, AS::col_smem)) != cudaSuccess) return e;
            if ((e = prep(row_inv2_kernel<T, P, C_INV, 4>, AS::inv_smem)) != cudaSuccess) return e;
            if ((e = prep(col2_kernel<T, P, C_COL, true, true>, AS::col_smem)) != cudaSuccess) return e;
            if ((e = prep(row_inv2_kernel<T, P, C_INV, 5>, AS::inv_smem)) != cudaSuccess) return e;
            if ((e = prep(col2_xform_kernel<T, P, C_COL, -1>, AS::WBYTES + 128)) != cudaSuccess) return e;
            if ((e = prep(col2_xform_kernel<T, P, C_COL, +1>, AS::WBYTES + 128)) != cudaSuccess) return e;
            if ((e = prep(col2_xpub_kernel<T, P, C_COL, -1>, AS::WBYTES + 128)) != cudaSuccess) return e;
            if ((e = prep(col2_xpub_kernel<T, P, C_COL, +1>, AS::WBYTES + 128)) != cudaSuccess) return e;
            if ((e = prep(t2_export_kernel<T, P>, AS::WBYTES + 1024)) != cudaSuccess) return e;
            if ((e = prep(t2_import_kernel<T, P>, AS::WBYTES + 1024)) != cudaSuccess) return e;
        }
        if constexpr (FS::valid) {
            if ((e = prep(cg_fused_kernel<T, P>, FS::smem)) != cudaSuccess) return e;
            if ((e = prep(cg_fused_kernel<T, P, 1>, FS::smem)) != cudaSuccess) return e;
            if ((e = prep(cg_fused_kernel<T, P, 2>, FS::smem)) != cudaSuccess) return e;
            if ((e = prep(cg_fused_kernel<T, P, 0, 1>, FS::smem_two)) != cudaSuccess) return e;
            if ((e = prep(cg_fused_kernel<T, P, 2, 1>, FS::smem_two)) != cudaSuccess) return e;
            if ((e = prep(cg_fused_kernel<T, P, 0, 2>, FS::smem_two_pcg)) != cudaSuccess) return e;
            if ((e = prep(cg_fused_kernel<T, P, 2, 2>, FS::smem_two_pcg)) != cudaSuccess) return e;
        }
        return prep(col_kernel<T, P, CS::COLS>, CS::smem);
    }
    // launch, optionally with programmatic stream serialization (the kernels call griddepcontrol.wait before their first
    // dependent access, so the next kernel's prologue overlaps this one's tail)
    template <typename K, typename... Args>
    static cudaError_t launch(K kernel, int grid, int block, size_t smem, cudaStream_t st, int pdl, Args... args) {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = pdl ? 1u : 0u;
        return cudaLaunchKernelEx(&cfg, kernel, args...);
    }
    // persistent grid: CTAS CTAs on each of nsm SMs, but never more CTAs than transforms (whole multiples of nsm)
    static int pgrid(int nsm, int ctas) {
        if (nsm * ctas >= L / 2 && nsm < L / 2) return L / 2;      // every transform resident at once: one CTA each, a single round
        int k = ctas;
        while (k > 1 && nsm * k > L / 2) --k;
        return nsm * k > L / 2 ? L / 2 : nsm * k;
    }
    static int pgrid_n(int nsm, int ctas, int ntile) {       // the same for a slab of ntile row pairs
        int k = ctas;
        while (k > 1 && nsm * k > ntile) --k;
        return nsm * k > ntile ? ntile : nsm * k;
    }
    static cudaError_t row_fwd2_slab(const void* args, cudaStream_t st) {
        if constexpr (V2) {
            const RowFwdArgs<T>& A = *static_cast<const RowFwdArgs<T>*>(args);
            return launch(row_fwd2_kernel<T, P, C_FWD, 2>, pgrid_n(A.nsm, C_FWD, A.ntile), P::NT + 32, AS::fwd_smem, st, 0, A);
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t col2_slab(const void* args, const void* tensor_map, int ncols, cudaStream_t st) {
        if constexpr (V2) {
            const ColArgs<T>& A = *static_cast<const ColArgs<T>*>(args);
            return launch(col2_kernel<T, P, C_COL, false, true>, ncols, P::NT, AS::col_smem, st, 0, A, *static_cast<const CUtensorMap*>(tensor_map));
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t col2_slab_e(const void* args, const void* tensor_map, int ncols, cudaStream_t st) {
        if constexpr (V2) {
            const ColArgs<T>& A = *static_cast<const ColArgs<T>*>(args);
            return launch(col2_kernel<T, P, C_COL, true, true>, ncols, P::NT, AS::col_smem, st, 0, A, *static_cast<const CUtensorMap*>(tensor_map));
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t row_inv2_slab_f(const void* args, const void* tensor_map, cudaStream_t st) {
        if constexpr (V2) {
            const RowInvArgs<T>& A = *static_cast<const RowInvArgs<T>*>(args);
            return launch(row_inv2_kernel<T, P, C_INV, 5>, pgrid_n(A.nsm, C_INV, A.ntile), AS::INV_THREADS, AS::inv_smem, st, 0, A,
                          *static_cast<const CUtensorMap*>(tensor_map));
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t row_inv2_slab(const void* args, const void* tensor_map, cudaStream_t st) {
        if constexpr (V2) {
            const RowInvArgs<T>& A = *static_cast<const RowInvArgs<T>*>(args);
            return launch(row_inv2_kernel<T, P, C_INV, 4>, pgrid_n(A.nsm, C_INV, A.ntile), AS::INV_THREADS, AS::inv_smem, st, 0, A,
                          *static_cast<const CUtensorMap*>(tensor_map));
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t row_fwd2(const void* args, cudaStream_t st) {
        if constexpr (V2) {
            const RowFwdArgs<T>& A = *static_cast<const RowFwdArgs<T>*>(args);
            return launch(row_fwd2_kernel<T, P, C_FWD>, pgrid(A.nsm, C_FWD), P::NT + 32, AS::fwd_smem, st, A.pdl == 1, A);
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t row_fwd2_rupd(const void* args, cudaStream_t st) {
        if constexpr (V2) {
            const RowFwdArgs<T>& A = *static_cast<const RowFwdArgs<T>*>(args);
            return launch(row_fwd2_kernel<T, P, C_FWD, 1>, pgrid(A.nsm, C_FWD), P::NT + 32, AS::fwd_smem, st, A.pdl == 1, A);
        }
        return cudaErrorInvalidValue;
    }
    static constexpr bool SL = V2;
    using CPS = ColPShape<T, P>;
    static constexpr bool COLP = V2 && CPS::valid;
    static cudaError_t col2p(const void* args, const void* tensor_map, int energy, cudaStream_t st) {
        if constexpr (COLP) {
            const ColArgs<T>& A = *static_cast<const ColArgs<T>*>(args);
            int grid = A.nsm * CPS::CTAS;
            if (grid > L / 2) grid = L / 2;
            const CUtensorMap& tm = *static_cast<const CUtensorMap*>(tensor_map);
            if (energy) return launch(col2p_kernel<T, P, CPS::CTAS, true>, grid, P::NT + 32, CPS::smem, st, A.pdl == 1, A, tm);
            return launch(col2p_kernel<T, P, CPS::CTAS, false>, grid, P::NT + 32, CPS::smem, st, A.pdl == 1, A, tm);
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t col2_energy(const void* args, const void* tensor_map, cudaStream_t st) {
        if constexpr (SL) {
            const ColArgs<T>& A = *static_cast<const ColArgs<T>*>(args);
            return launch(col2_kernel<T, P, C_COL, true>, L / 2, P::NT, AS::col_smem, st, A.pdl == 1, A, *static_cast<const CUtensorMap*>(tensor_map));
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t row_inv2_cgf(const void* args, const void* tensor_map, cudaStream_t st) {
        if constexpr (SL) {
            const RowInvArgs<T>& A = *static_cast<const RowInvArgs<T>*>(args);
            return launch(row_inv2_kernel<T, P, C_INV, 2>, pgrid(A.nsm, C_INV), AS::INV_THREADS, AS::inv_smem, st, A.pdl, A,
                          *static_cast<const CUtensorMap*>(tensor_map));
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t row_inv2_cgf_force(const void* args, const void* tensor_map, cudaStream_t st) {
        if constexpr (SL) {
            const RowInvArgs<T>& A = *static_cast<const RowInvArgs<T>*>(args);
            return launch(row_inv2_kernel<T, P, C_INV, 3>, pgrid(A.nsm, C_INV), AS::INV_THREADS, AS::inv_smem, st, A.pdl, A,
                          *static_cast<const CUtensorMap*>(tensor_map));
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t row_inv2_pre(const void* args, const void* tensor_map, cudaStream_t st) {
        if constexpr (V2) {
            const RowInvArgs<T>& A = *static_cast<const RowInvArgs<T>*>(args);
            return launch(row_inv2_kernel<T, P, C_INV, 1>, pgrid(A.nsm, C_INV), AS::INV_THREADS, AS::inv_smem, st, A.pdl, A,
                          *static_cast<const CUtensorMap*>(tensor_map));
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t col2(const void* args, const void* tensor_map, cudaStream_t st) {
        if constexpr (V2) {
            const ColArgs<T>& A = *static_cast<const ColArgs<T>*>(args);
            return launch(col2_kernel<T, P, C_COL>, L / 2, P::NT, AS::col_smem, st, A.pdl == 1, A, *static_cast<const CUtensorMap*>(tensor_map));
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t col2_xform(const void* args, const void* tensor_map, int inverse, cudaStream_t st) {
        if constexpr (V2) {
            const ColArgs<T>& A = *static_cast<const ColArgs<T>*>(args);
            const CUtensorMap& tm = *static_cast<const CUtensorMap*>(tensor_map);
            if (inverse) col2_xform_kernel<T, P, C_COL, +1><<<L / 2, P::NT, AS::WBYTES + 128, st>>>(A, tm);
            else col2_xform_kernel<T, P, C_COL, -1><<<L / 2, P::NT, AS::WBYTES + 128, st>>>(A, tm);
            return cudaGetLastError();
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t col2_xpub(const void* args, const void* tensor_map, const void* x_map, int inverse, cudaStream_t st) {
        if constexpr (V2) {
            const ColArgs<T>& A = *static_cast<const ColArgs<T>*>(args);
            const CUtensorMap& tm = *static_cast<const CUtensorMap*>(tensor_map);
            const CUtensorMap& xm = *static_cast<const CUtensorMap*>(x_map);
            if (inverse) col2_xpub_kernel<T, P, C_COL, +1><<<L / 2, P::NT, AS::WBYTES + 128, st>>>(A, tm, xm);
            else col2_xpub_kernel<T, P, C_COL, -1><<<L / 2, P::NT, AS::WBYTES + 128, st>>>(A, tm, xm);
            return cudaGetLastError();
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t t2_export(const void* T2, void* X, cudaStream_t st) {
        if constexpr (V2) {
            t2_export_kernel<T, P><<<L / 2, 256, AS::WBYTES + 1024, st>>>(static_cast<const cx<T>*>(T2), static_cast<cx<T>*>(X));
            return cudaGetLastError();
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t t2_import(const void* X, void* T2, cudaStream_t st) {
        if constexpr (V2) {
            t2_import_kernel<T, P><<<L / 2, 256, AS::WBYTES + 1024, st>>>(static_cast<const cx<T>*>(X), static_cast<cx<T>*>(T2));
            return cudaGetLastError();
        }
        return cudaErrorInvalidValue;
    }
    using FS = FusedShape<T, P>;
    static cudaError_t fused_solve(const void* fused_args, cudaStream_t st) {
        if constexpr (FS::valid) {
            FusedArgs A = *static_cast<const FusedArgs*>(fused_args);
            void* params[] = {&A};
            const int two = (A.two && A.form != 1) ? (A.mhat ? 2 : 1) : 0;        // fewer grid barriers per iteration (CG: 2, PCG: 4)
            const void* fn;
            if (A.form == 1) fn = (const void*)cg_fused_kernel<T, P, 1>;
            else if (A.form == 2) fn = two == 2 ? (const void*)cg_fused_kernel<T, P, 2, 2> : two == 1 ? (const void*)cg_fused_kernel<T, P, 2, 1> : (const void*)cg_fused_kernel<T, P, 2>;
            else fn = two == 2 ? (const void*)cg_fused_kernel<T, P, 0, 2> : two == 1 ? (const void*)cg_fused_kernel<T, P, 0, 1> : (const void*)cg_fused_kernel<T, P>;
            const size_t smem = two == 2 ? FS::smem_two_pcg : two == 1 ? FS::smem_two : FS::smem;
            return cudaLaunchCooperativeKernel(fn, dim3(FS::G), dim3(P::NT), params, smem, st);
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t row_inv2(const void* args, const void* tensor_map, cudaStream_t st) {
        if constexpr (V2) {
            const RowInvArgs<T>& A = *static_cast<const RowInvArgs<T>*>(args);
            return launch(row_inv2_kernel<T, P, C_INV>, pgrid(A.nsm, C_INV), AS::INV_THREADS, AS::inv_smem, st, A.pdl, A,
                          *static_cast<const CUtensorMap*>(tensor_map));
        }
        return cudaErrorInvalidValue;
    }

    template <int V> static cudaError_t row_fwd_v(const RowFwdArgs<T>& A, cudaStream_t st) {
        if constexpr (RS::valid(V)) {
            row_fwd_kernel<T, P, RS::F(V)><<<L / (2 * RS::F(V)), RS::F(V) * P::NT, RS::smem(V), st>>>(A);
            return cudaGetLastError();
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t row_fwd(int var, const void* args, cudaStream_t st) {
        const RowFwdArgs<T>& A = *static_cast<const RowFwdArgs<T>*>(args);
        switch (var) {
            case 0: return row_fwd_v<0>(A, st);
            case 1: return row_fwd_v<1>(A, st);
            case 2: return row_fwd_v<2>(A, st);
            case 3: return row_fwd_v<3>(A, st);
        }
        return cudaErrorInvalidValue;
    }
    template <int V> static cudaError_t row_inv_v(const RowInvArgs<T>& A, cudaStream_t st) {
        if constexpr (RS::valid(V)) {
            row_inv_kernel<T, P, RS::F(V)><<<L / (2 * RS::F(V)), RS::F(V) * P::NT, RS::smem(V), st>>>(A);
            return cudaGetLastError();
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t row_inv(int var, const void* args, cudaStream_t st) {
        const RowInvArgs<T>& A = *static_cast<const RowInvArgs<T>*>(args);
        switch (var) {
            case 0: return row_inv_v<0>(A, st);
            case 1: return row_inv_v<1>(A, st);
            case 2: return row_inv_v<2>(A, st);
            case 3: return row_inv_v<3>(A, st);
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t col(const void* args, cudaStream_t st) {
        const ColArgs<T>& A = *static_cast<const ColArgs<T>*>(args);
        col_kernel<T, P, CS::COLS><<<(L / 2) / CS::COLS, CS::COLS * P::NT, CS::smem, st>>>(A);
        return cudaGetLastError();
    }
    static cudaError_t spectrum_prep(const void* s, void* shat, int colpos, cudaStream_t st) {
        spectrum_prep_kernel<T, P><<<148 * 2, 256, 0, st>>>(static_cast<const T*>(s), static_cast<T*>(shat), colpos != 0);
        return cudaGetLastError();
    }
    static PassTable make(int dtype) {
        PassTable t{};
        t.L = L; t.dtype = dtype;
        for (int v = 0; v < FCG_NROWVAR; ++v) {
            t.row_valid[v] = RS::valid(v); t.row_F[v] = RS::F(v);
            t.row_threads[v] = RS::F(v) * P::NT; t.row_smem[v] = RS::smem(v);
        }
        t.cols = CS::COLS; t.col_threads = CS::COLS * P::NT; t.col_smem = CS::smem;
        t.tw_total = P::TW_TOTAL;
        t.fill_twiddles = [](void* buf) { fill_twiddles<T, P>(static_cast<cx<T>*>(buf)); };
        t.v2 = V2 ? 1 : 0; t.v2_nb = AS::NB; t.v2_abox = AS::ABOX; t.v2_tsub = AS::TSUB; t.v2_threads = P::NT;
        t.v2_ctas[0] = C_FWD; t.v2_ctas[1] = C_COL; t.v2_ctas[2] = C_INV;
        t.v2_smem[0] = AS::fwd_smem; t.v2_smem[1] = AS::col_smem; t.v2_smem[2] = AS::inv_smem;
        t.row_fwd2 = &row_fwd2; t.col2 = &col2; t.row_inv2 = &row_inv2; t.row_fwd2_rupd = &row_fwd2_rupd; t.row_inv2_pre = &row_inv2_pre;
        t.colp_ok = COLP ? 1 : 0; t.colp_ctas = COLP ? CPS::CTAS : 0; t.col2p = &col2p;
        t.sl_ok = SL ? 1 : 0; t.col2_energy = &col2_energy; t.row_inv2_cgf = &row_inv2_cgf; t.row_inv2_cgf_force = &row_inv2_cgf_force;
        t.row_fwd2_slab = &row_fwd2_slab; t.col2_slab = &col2_slab; t.row_inv2_slab = &row_inv2_slab;
        t.col2_slab_e = &col2_slab_e; t.row_inv2_slab_f = &row_inv2_slab_f;
        t.col2_xform = &col2_xform; t.col2_xpub = &col2_xpub; t.t2_export = &t2_export; t.t2_import = &t2_import;
        t.fused = FS::valid ? 1 : 0; t.fused_grid = FS::G; t.fused_solve = &fused_solve;
        t.init = &init; t.row_fwd = &row_fwd; t.col = &col; t.row_inv = &row_inv; t.spectrum_prep = &spectrum_prep;
        return t;
    }
};

}  // namespace

#define FCG_CAT2(a, b) a##b
#define FCG_CAT(a, b) FCG_CAT2(a, b)
const PassTable* FCG_CAT(fcg_pass_table_, FCG_INST_L)(int dtype) {
    static const PassTable t32 = Inst<float>::make(0);
    static const PassTable t64 = Inst<double>::make(1);
    return dtype == 0 ? &t32 : &t64;
}

}  // namespace fcg
