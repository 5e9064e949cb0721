// fcg.cu -- the C ABI of include/fcg.h: handle, workspace, launch sequences, CUDA-graph construction.
// Kernels live in fcg_kernels.cuh / fcg_passes.cuh; the transform passes are instantiated per lattice
// size in fcg_inst.cu.  No cuFFT, no cuBLAS, no host arithmetic on the data path.
#define FCG_MAIN_TU
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include <cuda.h>

#include "../../include/fcg.h"
#include "fcg_kernels.cuh"
#include "fcg_plans.cuh"
#include "fcg_fused.cuh"

using namespace fcg;

namespace {

constexpr int VEC_BLOCKS_MAX = 148 * 8;   // 8 CTAs of 256 threads per SM
constexpr size_t ALIGN = 256;
size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

const PassTable* get_table(int L, int dtype) {
    switch (L) {
        case 16: return fcg_pass_table_16(dtype);
        case 32: return fcg_pass_table_32(dtype);
        case 64: return fcg_pass_table_64(dtype);
        case 128: return fcg_pass_table_128(dtype);
        case 256: return fcg_pass_table_256(dtype);
        case 512: return fcg_pass_table_512(dtype);
        case 1024: return fcg_pass_table_1024(dtype);
        case 2048: return fcg_pass_table_2048(dtype);
        case 4096: return fcg_pass_table_4096(dtype);
        case 8192: return fcg_pass_table_8192(dtype);
    }
    return nullptr;
}

struct Layout {            // byte offsets into the workspace
    size_t Tb, shat, mhat, r, p, q, z, tw, partial_row, partial_col, partial_vec, brk_r, brk_i, scalars, brk_out, brk_ticket, uni, total;
};
Layout make_layout(int L, size_t w) {
    const size_t N = (size_t)L * L;
    Layout o{}; size_t off = 0;
    auto take = [&](size_t bytes) { size_t at = off; off = align_up(off + bytes); return at; };
    o.Tb = take(N * w);                                   // (L/2) x L complex
    o.shat = take(((size_t)L / 2 + 1) * L * w);
    o.mhat = take(((size_t)L / 2 + 1) * L * w);           // PCG: eigenvalues of M^-1, same layout as shat
    o.r = take(N * w); o.p = take(N * w); o.q = take(N * w);
    o.z = take(N * w);                                    // PCG: z = M^-1 r
    o.tw = take((size_t)L * 2 * w);
    o.partial_row = take((size_t)L * 2 * sizeof(double));
    o.partial_col = take((size_t)L / 2 * sizeof(double));      // spectral search length: one partial sum per column
    o.partial_vec = take(VEC_BLOCKS_MAX * sizeof(double));
    o.brk_r = take(VEC_BLOCKS_MAX * sizeof(double));
    o.brk_i = take(VEC_BLOCKS_MAX * sizeof(long long));
    o.scalars = take(sizeof(Scalars));
    o.brk_out = take(sizeof(BreakResult));
    o.brk_ticket = take(2 * sizeof(unsigned int));        // arrival ticket + key of the screen's running maximum (break_argmax_kernel)
    o.uni = take(4 * sizeof(unsigned long long));         // force_uniform_kernel's result (reading F1 check)
    o.total = off;
    return o;
}

struct GraphEntry {
    const void *k, *f; void* u; double tol; int maxit, var, unroll, pdl, pcg, force; double D, kappa;   // pcg: bit 0 = preconditioned, the rest = launch options (key)
    cudaGraph_t graph; cudaGraphExec_t exec; unsigned long long stamp;
};

}  // namespace

struct AsyncSolve { int enqueued; long long unroll, outside, per_iteration; };

struct fcg_handle_s {
    int L = 0, dtype = 0; size_t w = 0, N = 0;
    const PassTable* tab = nullptr;
    cudaStream_t stream = nullptr, cap_stream = nullptr;
    char* ws = nullptr; bool own_ws = false;
    Layout lay{};
    bool have_spectrum = false, have_precond = false;
    int loop_mode = 0, chunk = 16, row_var_opt = -1, engine_opt = 0, nsm = 148, unroll_opt = -1, pdl_opt = -1, fused_opt = 1, hints = 63, sl_opt = 1, colp_opt = -1;
    alignas(64) CUtensorMap tmap_row;   // T2 as [L/(2 NB)][L/2][128 B]: box = v2_tsub/NB lines of one row pair (row_inv2 tiles)
    alignas(64) CUtensorMap tmap_col;   // T2 as [L/(2 NB)][L/2][NB][2 complex]: box = one column x v2_abox row pairs (col2 gather / scatter)
    bool have_tmap = false;
    int spectrum_colpos = 0;            // layout the stored spectrum was prepared for (1: T2 column order)
    bool v2() const { return engine_opt == 0 && tab->v2 && have_tmap; }
    // persistent column pass: measured faster for fp32 (L = 2048: 23.2 -> 20.6 us, L = 4096: 59.1 -> 53.1) and for fp64 up to
    // L = 1024; slower at L = 2048 fp64 (two CTAs of 4 warps per SM instead of three: 26.5 -> 31.0 us), hence the automatic rule
    bool colp() const { return tab->colp_ok && (colp_opt < 0 ? (dtype == FCG_F32 || L <= 1024) : colp_opt != 0); }
    // programmatic dependent launch of the loop kernels (FCG_OPT_PDL).  Measured per CG iteration, interleaved runs on one B200:
    // mode 1 (every kernel may start under its predecessor's tail) L = 1024 fp64 37.9 -> 36.2 us, but 2048 fp64 89.1 -> 96.1, 2048 fp32
    // 57.4 -> 60.2, 4096 fp32 201 -> 218, 8192 fp32 807 -> 839, 1024 fp32 30.4 -> 32.0; mode 2 (only the fused last pass starts early and
    // fills its strip ring during the column pass's tail) 1024 fp32 30.4 -> 29.9, 1024 fp64 36.7, 2048 fp64 89.4, 4096 fp64 387 -> 385,
    // others within noise.  Hence the automatic rule: L = 1024 only.
    // CG iterations per evaluation of the graph's WHILE condition (FCG_OPT_UNROLL; -1 = automatic).  Iterations after the stop are no-op
    // launches (each kernel returns before it issues anything), an evaluation costs a node boundary.  Measured, whole solves to the
    // configs' tolerances, us per iteration with 4 / 8 / 16 / 32: L = 2048 fp64 (100 iterations) 87.3 / 85.2 / 87.1 / 86.0, L = 1024 fp64 (77)
    // 35.6 / 34.5 / 34.8 / 34.7; L = 2048 fp32 (33) 57.5 / 58.5 / 58.5 / 61.6, PCG at L = 2048 fp64 (10) 166 / 170 / 169 / 186, L = 4096 and
    // 8192: within noise.  Hence 8 for un-preconditioned fp64 solves at L = 1024 and 2048, 4 otherwise.
    int unroll(bool pcg) const { return unroll_opt > 0 ? unroll_opt : (!pcg && dtype == FCG_F64 && (L == 1024 || L == 2048) ? 8 : 4); }
    int pdl() const { return pdl_opt >= 0 ? pdl_opt : (L == 1024 && v2() ? (dtype == FCG_F64 ? 1 : 2) : 0); }
    // start offsets in ns between the CTAs that share an SM, per pass (P1, P2, P3): -1 = the measured default for this size (stagger())
    int stag_opt[3] = {-1, -1, -1};
    int stagger(int pass) const {
        if (stag_opt[pass] >= 0) return stag_opt[pass];
        // measured (us per CG iteration, interleaved runs on one B200): L = 2048 fp64 91.8 -> 89.0 with the last pass 2 us apart (after 93.2 ->
        // 91.8 from the column pass), nothing from the first pass; L = 2048 fp32 and L = 4096 lose or stay; L = 1024 gained (40.5 -> 38.9) only
        // until its row passes got one CTA per transform (fcg_inst.cu pgrid: 37.9 with or without offsets)
        if (dtype == FCG_F64 && L == 2048) return pass == 0 ? 0 : pass == 1 ? 1500 : 2000;
        return 0;
    }
    bool sl() const { return sl_opt && v2() && tab->sl_ok; }     // spectral search length: 3 launches per CG iteration
    bool fused() const { return fused_opt && tab->fused && v2() && loop_mode == 0; }   // whole solve in one cooperative kernel
    Scalars* h_sc = nullptr;            // pinned
    BreakResult* h_brk = nullptr;       // pinned
    unsigned long long* h_uni = nullptr; // pinned: result of the reading-F1 check of fcg_force_solve
    void *hk = nullptr, *hf = nullptr, *hu = nullptr;   // device staging of fcg_solve_host
    // fcg_solve_host_submit / _wait: two staging sets, a stream for the inputs and one for the results, so that the copies of the
    // neighbouring solves run under the current one
    void* pset[2][3] = {};
    cudaStream_t pin_stream = nullptr, pout_stream = nullptr;
    cudaEvent_t pev_in[2] = {}, pev_solved[2] = {}, pev_out[2] = {};
    Scalars* pres = nullptr;             // pinned: the scalar block of each outstanding solve
    int phead = 0, pcount = 0, pstatus[2] = {}, penq[2] = {};
    long long punroll[2] = {}, poutside[2] = {}, pper[2] = {};
    long long* frac_idx = nullptr; int* frac_it = nullptr; double* frac_ratio = nullptr; int frac_cap = 0;   // device results of the fused quasi-static loop
    int pend_nsteps = -1, pend_done = 0, pend_status = 0; bool pend_async = false;   // fcg_fracture_begin / _end
    std::vector<long long> pend_idx; std::vector<int> pend_it; std::vector<double> pend_ratio;
    int pend_kind = 0;                  // 0: fcg_fracture_begin, 1: fcg_force_fracture_displacement_begin
    std::vector<GraphEntry> graphs; unsigned long long stamp = 0;
    long long launches = 0;
    std::string err;
    // slab-decomposed CG: this handle is rank `slab_rank` of `slab_G`
    int slab_G = 0, slab_rank = 0, slab_Al = 0, slab_MBl = 0, slab_boxa = 0;     // row pairs and column blocks this rank owns; row pairs per column box
    size_t slab_S = 0, slab_R = 0, slab_bytes = 0;                 // workspace offsets of T2 (rows side) and of the exchange buffer (= the columns side)
    void* slab_ipc_base[16] = {};        // peer mode across processes: the peers' workspaces as opened by fcg_slab_ipc_open (closed in fcg_destroy)
    void* slab_peerR[16] = {};           // peer mode (fcg_slab_set_peers): every rank's exchange buffer R ..
    CUtensorMap* slab_peer_maps = nullptr;   // .. and a device array of tensor maps of every rank's T2 (rows side, S); nullptr: exchange by all-to-all
    alignas(64) CUtensorMap tmap_row_s;  // S as [L/(2 NB)][Al][128 B]
    alignas(64) CUtensorMap tmap_col_s;  // R as [source rank][MBl][Al][NB][2 complex] (5-D)
    alignas(64) CUtensorMap tmap_x;      // FCG_F64: the caller's half spectrum X[m][n] as a tensor of columns (fft_impl; re-encoded when X moves)
    const void* tmap_x_ptr = nullptr;
    int fft_pub = -1;                   // FCG_OPT_FFT_DIRECT (-1: automatic)
    // Automatic rule, from measurements on one B200.  Writing X column by column leaves every 32-byte sector
    // of X to be completed by the neighbouring column's CTA: fine while X stays in L2 until then (L = 2048 fp64: 67.8 -> 55.5 us),
    // a read-modify-write storm once it does not (L = 4096 fp64 forward 254 -> 321 us, L = 8192 fp32 509 -> 1508 us).  Reading X
    // column by column has no such cliff for 16-byte elements (L = 4096 fp64 inverse 241 -> 199 us) but 8-byte elements waste
    // three quarters of every sector (L = 8192 fp32 inverse 609 -> 1273 us).
    bool fft_direct(bool inverse) const {
        if (fft_pub >= 0) return fft_pub != 0;
        const bool small = N * w <= ((size_t)64 << 20);
        return inverse ? (dtype == FCG_F64 || small) : small;
    }
    int device = 0;                     // the device the handle was created on; every entry point runs with it current
    unsigned int barrier_start = 0;     // FCG_OPT_BARRIER_START: initial value of the cooperative kernel's barrier counter
    int fused_two = 1;                  // FCG_OPT_FUSED_TWO: plain CG in the one-launch kernel with two grid barriers per iteration

    template <typename U> U* at(size_t off) const { return reinterpret_cast<U*>(ws + off); }
    Scalars* sc() const { return at<Scalars>(lay.scalars); }
    int vec_blocks() const {
        size_t nvec = N / (dtype == FCG_F64 ? 2 : 4);
        size_t b = (nvec + 255) / 256;
        return (int)(b < (size_t)VEC_BLOCKS_MAX ? b : (size_t)VEC_BLOCKS_MAX);
    }
    // Grid of cg_update_r_kernel: every thread makes the same whole number of unrolled trips (4 vectors of 16 bytes each), so
    // that no thread is left with a tail of serially dependent single loads: at L = 2048 fp64 1184 CTAs meant one unrolled
    // trip + up to three dependent ones, 1024 CTAs are exactly two unrolled trips
    int update_blocks() const {
        const size_t nvec = N / (dtype == FCG_F64 ? 2 : 4), per = 256 * 4;
        size_t b = (nvec + per - 1) / per;
        if (b > (size_t)VEC_BLOCKS_MAX) {
            const size_t trips = (nvec + (size_t)VEC_BLOCKS_MAX * per - 1) / ((size_t)VEC_BLOCKS_MAX * per);
            b = (nvec + per * trips - 1) / (per * trips);
        }
        return (int)(b < 1 ? 1 : b);
    }
    int row_var() const {
        if (row_var_opt >= 0 && row_var_opt < FCG_NROWVAR && tab->row_valid[row_var_opt]) return row_var_opt;
        int best = 0;
        for (int v = 0; v < FCG_NROWVAR; ++v)
            if (tab->row_valid[v] && tab->row_smem[v] <= 72 * 1024 && L / (2 * tab->row_F[v]) >= 256) best = v;
        return best;
    }
};

namespace {

#define FCG_CK(h, expr)                                                                          \
    do {                                                                                         \
        cudaError_t e_ = (expr);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            (h)->err = std::string(#expr) + ": " + cudaGetErrorString(e_);                       \
            return FCG_CUDA_ERROR;                                                               \
        }                                                                                        \
    } while (0)

int fail(fcg_handle h, int code, const char* msg) { if (h) h->err = msg; return code; }

// Every entry point runs with the handle's device current and restores the caller's on return (a caller that switched devices
// between fcg_create and a later call -- common with torch and several GPUs -- would otherwise launch on the wrong device).
struct DeviceGuard {
    int prev = -1; bool ok = true, switched = false;
    explicit DeviceGuard(int want) {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; cudaGetLastError(); return; }
        if (prev != want) { ok = cudaSetDevice(want) == cudaSuccess; switched = ok; if (!ok) cudaGetLastError(); }
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
#define FCG_ENTER(h)                                                                                                   \
    DeviceGuard dev_guard_((h)->device);                                                                               \
    if (!dev_guard_.ok) return fail((h), FCG_CUDA_ERROR, "cannot make the handle's device current");                   \
    if ((h)->pend_async) return fail((h), FCG_INVALID_ARG, "a quasi-static loop is pending on this handle: call its _end first");  \
    if ((h)->tab->v2 && (h)->engine_opt == 0 && !(h)->have_tmap)                                                       \
        return fail((h), FCG_UNSUPPORTED, "cuTensorMapEncodeTiled unavailable: the pipelined passes cannot run; FCG_OPT_ENGINE = 1 selects the classic passes")
#define FCG_ENTER_OPT(h)                                                                                               \
    DeviceGuard dev_guard_((h)->device);                                                                               \
    if (!dev_guard_.ok) return fail((h), FCG_CUDA_ERROR, "cannot make the handle's device current");                   \
    if ((h)->pend_async) return fail((h), FCG_INVALID_ARG, "a quasi-static loop is pending on this handle: call its _end first")
#define FCG_ENTER_END(h)                                                                                               \
    DeviceGuard dev_guard_((h)->device);                                                                               \
    if (!dev_guard_.ok) return fail((h), FCG_CUDA_ERROR, "cannot make the handle's device current")

bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

// CUDA events that are destroyed on every path out of the profiling calls
struct EventList {
    std::vector<cudaEvent_t> ev;
    ~EventList() { for (auto e : ev) if (e) cudaEventDestroy(e); }
    cudaError_t create(size_t n) {
        ev.assign(n, nullptr);
        for (auto& e : ev) { cudaError_t r = cudaEventCreate(&e); if (r != cudaSuccess) return r; }
        return cudaSuccess;
    }
    cudaEvent_t* operator+(size_t i) { return ev.data() + i; }
    cudaEvent_t operator[](size_t i) const { return ev[i]; }
};

// one cooperative launch of fcg_fused.cuh: scalar block zeroed, barrier counter preset, kernel enqueued
cudaError_t fused_launch(fcg_handle h, FusedArgs& A) {
    cudaError_t e = cudaMemsetAsync(h->sc(), 0, sizeof(Scalars), h->stream);
    if (e != cudaSuccess) return e;
    A.counter_start = h->barrier_start;
    A.two = h->fused_two;
    if (h->barrier_start != 0u &&
        (e = cudaMemcpyAsync(A.counter, &h->barrier_start, sizeof(unsigned int), cudaMemcpyHostToDevice, h->stream)) != cudaSuccess) return e;
    return h->tab->fused_solve(&A, h->stream);
}

// ---- launch sequences (typed) ---------------------------------------------------------------
template <typename T> struct Seq {
    fcg_handle h; cudaStream_t st; bool classic = false;      // classic: force the synchronous passes (stand-alone transforms)
    bool pcg = false;                                         // preconditioned CG: directions from z = M^-1 r
    bool force = false; double D = 0.0;                       // force formulation (I + K G) f = K D (eq. (2))
    double kappa = 0.0;                                       // force: > 0 when reading F1 was verified for this call (k in {0, kappa}): three launches
    bool v2() const { return h->v2() && !classic; }
    const T* mhat() const { return h->at<T>(h->lay.mhat); }
    T* z() const { return h->at<T>(h->lay.z); }
    cx<T>* Tb() const { return h->at<cx<T>>(h->lay.Tb); }
    const cx<T>* tw() const { return h->at<cx<T>>(h->lay.tw); }
    const T* shat() const { return h->at<T>(h->lay.shat); }
    T* r() const { return h->at<T>(h->lay.r); }
    T* p() const { return h->at<T>(h->lay.p); }
    T* q() const { return h->at<T>(h->lay.q); }

    cudaError_t row_fwd(int mode, const T* x, T* u, int check_done = 0) const {
        RowFwdArgs<T> A{}; A.mode = mode; A.x = x; A.u = u; A.p = p(); A.r = pcg ? z() : r(); A.check_done = check_done; A.stagger_ns = mode == ROWF_CG ? h->stagger(0) : 0; A.hints = h->hints; A.Tb = Tb(); A.tw = tw(); A.sc = h->sc(); A.nsm = h->nsm; A.pdl = h->pdl(); A.tmo = &h->sc()->timeout;
        ++h->launches;
        return v2() ? h->tab->row_fwd2(&A, st) : h->tab->row_fwd(h->row_var(), &A, st);
    }
    cudaError_t col(int mode, bool cg, bool precond = false) const {
        ColArgs<T> A{}; A.mode = mode; A.Tb = Tb(); A.shat = precond ? mhat() : shat(); A.hints = h->hints; A.tw = tw(); A.sc = cg ? h->sc() : nullptr; A.pdl = h->pdl(); A.tmo = &h->sc()->timeout;
        A.nsm = h->nsm; A.stagger_ns = cg ? h->stagger(1) : 0;
        ++h->launches;
        if (v2() && mode == COL_CONV && h->colp()) return h->tab->col2p(&A, &h->tmap_col, 0, st);
        return (v2() && mode == COL_CONV) ? h->tab->col2(&A, &h->tmap_col, st) : h->tab->col(&A, st);
    }
    cudaError_t row_inv(int mode, const T* k, const T* v, const T* f, T* out, T* out2) const {
        RowInvArgs<T> A{}; A.mode = mode; A.Tb = Tb(); A.tw = tw(); A.k = k; A.v = v; A.f = f; A.out = out; A.out2 = out2;
        A.scale = (T)(1.0 / ((double)h->L * (double)h->L)); A.hints = h->hints; A.form = force ? 1 : 0; A.dval = (T)D;
        A.partial = h->at<double>(h->lay.partial_row); A.sc = h->sc(); A.nsm = h->nsm; A.pdl = h->pdl(); A.tmo = &h->sc()->timeout;
        A.stagger_ns = mode == ROWI_CG ? h->stagger(2) : 0;
        ++h->launches;
        return v2() ? h->tab->row_inv2(&A, &h->tmap_row, st) : h->tab->row_inv(h->row_var(), &A, st);
    }
    // set up initial values: r = f - A u, p = 0 (first direction p = r + 0*p), rho, ||f||^2
    // PCG: then z = M^-1 r, rho = r.z (first direction p = z + 0*p)
    cudaError_t init(const T* k, const T* f, T* u, double tol, int maxit, bool use_cond, unsigned long long cond) const {
        SetupArgs sa{tol, maxit, use_cond ? 1 : 0, cond, pcg ? 1 : 0};
        cg_setup_kernel<<<1, 32, 0, st>>>(h->sc(), sa); ++h->launches;
        cudaError_t e;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        if ((e = row_fwd(ROWF_PLAIN, u, nullptr)) != cudaSuccess) return e;
        if ((e = col(COL_CONV, false)) != cudaSuccess) return e;
        if ((e = row_inv(ROWI_RESID, k, u, force ? k : f, r(), p())) != cudaSuccess) return e;   // (force: b = K D is formed in the pass)
        if (sl()) {      // start value of the sum k p^2 recurrence: the first direction is p = r  (force: sum p^2)
            cg_kpp0_kernel<T><<<h->vec_blocks(), 256, 0, st>>>(force ? (const T*)nullptr : k, (const T*)r(), h->N / Vec<T>::W, h->at<double>(h->lay.partial_vec), h->sc());
            ++h->launches;
            return cudaGetLastError();
        }
        if (!pcg) return e;
        if ((e = row_fwd(ROWF_PLAIN, r(), nullptr, 1)) != cudaSuccess) return e;
        return it_precond();
    }
    // PCG: column pass with the preconditioner's spectrum, then z = inverse row transforms, r.z -> rho', beta
    cudaError_t it_col_m() const { return col(COL_CONV, true, true); }
    cudaError_t it_row_pre() const {
        RowInvArgs<T> A{}; A.mode = ROWI_PRECOND; A.Tb = Tb(); A.tw = tw(); A.k = r(); A.out = z(); A.hints = h->hints; A.stagger_ns = h->stagger(2);
        A.partial = h->at<double>(h->lay.partial_row); A.sc = h->sc(); A.nsm = h->nsm; A.pdl = h->pdl(); A.tmo = &h->sc()->timeout;
        ++h->launches;
        return v2() ? h->tab->row_inv2_pre(&A, &h->tmap_row, st) : h->tab->row_inv(h->row_var(), &A, st);
    }
    cudaError_t it_precond() const {
        cudaError_t e = it_col_m();
        return e != cudaSuccess ? e : it_row_pre();
    }
    // PCG: r -= alpha q, r.r, count, convergence, and the row transforms of the new r -- one pass with the pipelined
    // engine, the vector kernel followed by a plain row pass with the classic one
    cudaError_t it_rupd() const {
        if (!v2()) {
            cudaError_t e = it_update_r();
            return e != cudaSuccess ? e : row_fwd(ROWF_PLAIN, r(), nullptr, 1);
        }
        RowFwdArgs<T> A{}; A.mode = ROWF_RUPD; A.stagger_ns = h->stagger(0); A.hints = h->hints; A.rw = r(); A.q = q(); A.Tb = Tb(); A.tw = tw(); A.sc = h->sc(); A.nsm = h->nsm; A.pdl = h->pdl(); A.tmo = &h->sc()->timeout;
        A.partial = h->at<double>(h->lay.partial_vec);
        ++h->launches;
        return h->tab->row_fwd2_rupd(&A, st);
    }
    int launches_per_iteration() const { return pcg ? (v2() ? 6 : 7) : (sl() ? 3 : 4); }
    int launches_outside_loop() const { return pcg ? 8 : (sl() ? 6 : 5); }
    // one pass of Listing 2, as four launches
    cudaError_t it_row_fwd(T* u) const { return row_fwd(ROWF_CG, nullptr, u); }                    // new x (lagged), new p, row transform
    cudaError_t it_col() const { return col(COL_CONV, true); }                                     // column transform * spectrum * inverse
    cudaError_t it_row_inv(const T* k) const { return row_inv(ROWI_CG, k, p(), nullptr, q(), nullptr); }   // q = A p, p.q, alpha
    cudaError_t it_update_r() const {                                                              // r, r.r, beta, convergence
        const size_t nvec = h->N / Vec<T>::W;
        ++h->launches;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)h->update_blocks()); cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = 0; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = h->pdl() == 1 ? 1u : 0u;
        return cudaLaunchKernelEx(&cfg, cg_update_r_kernel<T>, r(), (const T*)q(), nvec, h->at<double>(h->lay.partial_vec), h->sc(), h->hints, (double*)nullptr);
    }
    // spectral search length: alpha is known after the column pass, so the residual update rides in P3
    cudaError_t it_col_e() const {
        ColArgs<T> A{}; A.mode = COL_CONV; A.Tb = Tb(); A.shat = shat(); A.hints = h->hints; A.tw = tw(); A.sc = h->sc(); A.pdl = h->pdl(); A.tmo = &h->sc()->timeout;
        A.partial = h->at<double>(h->lay.partial_col); A.nsm = h->nsm; A.stagger_ns = h->stagger(1);
        ++h->launches;
        if (h->colp()) return h->tab->col2p(&A, &h->tmap_col, 1, st);
        return h->tab->col2_energy(&A, &h->tmap_col, st);
    }
    cudaError_t it_row_inv_f(const T* k) const {
        RowInvArgs<T> A{}; A.mode = ROWI_CGF; A.Tb = Tb(); A.tw = tw(); A.k = k; A.v = p(); A.f = r(); A.out = r(); A.hints = h->hints; A.stagger_ns = h->stagger(2);
        A.partial = h->at<double>(h->lay.partial_row); A.colsum = h->at<double>(h->lay.partial_col);
        A.sc = h->sc(); A.nsm = h->nsm; A.pdl = h->pdl(); A.tmo = &h->sc()->timeout;
        ++h->launches;
        if (force) { A.form = 1; A.kappa = kappa; return h->tab->row_inv2_cgf_force(&A, &h->tmap_row, st); }
        return h->tab->row_inv2_cgf(&A, &h->tmap_row, st);
    }
    bool sl() const { return !pcg && !classic && h->sl() && (!force || kappa > 0.0); }
    cudaError_t iteration(const T* k, T* u) const {
        cudaError_t e;
        if (sl()) {
            if ((e = it_row_fwd(u)) != cudaSuccess) return e;
            if ((e = it_col_e()) != cudaSuccess) return e;
            return it_row_inv_f(k);
        }
        if ((e = it_row_fwd(u)) != cudaSuccess) return e;
        if ((e = it_col()) != cudaSuccess) return e;
        if ((e = it_row_inv(k)) != cudaSuccess) return e;
        if (!pcg) return it_update_r();
        if ((e = it_rupd()) != cudaSuccess) return e;
        return it_precond();
    }
    cudaError_t finish(T* u) const {
        const size_t nvec = h->N / Vec<T>::W;
        cg_finish_kernel<T><<<h->vec_blocks(), 256, 0, st>>>(u, p(), nvec, h->sc()); ++h->launches;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        return cudaMemcpyAsync(h->h_sc, h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, st);
    }
};

void drop_graph(GraphEntry& g) {
    if (g.exec) cudaGraphExecDestroy(g.exec);
    if (g.graph) cudaGraphDestroy(g.graph);
    g.exec = nullptr; g.graph = nullptr;
}

// Whole solve as one graph:  init  ->  WHILE(cond){ iteration }  ->  finish + D2H of the scalars.
// cond is written on the device by the residual / r-update kernels (cudaGraphSetConditional).
template <typename T>
cudaError_t build_graph(fcg_handle h, GraphEntry& ge) {
    cudaError_t e;
    cudaStream_t cs = h->cap_stream;
    Seq<T> s{h, cs}; s.pcg = (ge.pcg & 1) != 0; s.force = ge.force != 0; s.D = ge.D; s.kappa = ge.kappa;
    const long long saved = h->launches;
    ge.graph = nullptr; ge.exec = nullptr;
    if ((e = cudaGraphCreate(&ge.graph, 0)) != cudaSuccess) return e;
    cudaGraphConditionalHandle cond;
    if ((e = cudaGraphConditionalHandleCreate(&cond, ge.graph, 0, cudaGraphCondAssignDefault)) != cudaSuccess) return e;

    if ((e = cudaStreamBeginCaptureToGraph(cs, ge.graph, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed)) != cudaSuccess) return e;
    e = s.init((const T*)ge.k, (const T*)ge.f, (T*)ge.u, ge.tol, ge.maxit, true, (unsigned long long)cond);
    cudaStreamCaptureStatus cst; const cudaGraphNode_t* deps = nullptr; size_t ndeps = 0;
    cudaError_t e2 = cudaStreamGetCaptureInfo(cs, &cst, nullptr, nullptr, &deps, &ndeps);
    std::vector<cudaGraphNode_t> dep(deps, deps + (e2 == cudaSuccess ? ndeps : 0));
    cudaGraph_t tmp;
    cudaError_t e3 = cudaStreamEndCapture(cs, &tmp);
    if (e != cudaSuccess) return e;
    if (e2 != cudaSuccess) return e2;
    if (e3 != cudaSuccess) return e3;

    cudaGraphNodeParams np{};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = cond;
    np.conditional.type = cudaGraphCondTypeWhile;
    np.conditional.size = 1;
    cudaGraphNode_t wnode;
    if ((e = cudaGraphAddNode(&wnode, ge.graph, dep.data(), dep.size(), &np)) != cudaSuccess) return e;
    cudaGraph_t body = np.conditional.phGraph_out[0];

    if ((e = cudaStreamBeginCaptureToGraph(cs, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed)) != cudaSuccess) return e;
    // `unroll` iterations per evaluation of the WHILE condition (each evaluation costs ~6 us on B200); once the device flag
    // is set the remaining kernels of the body return at once without touching anything
    for (int r = 0; r < ge.unroll && e == cudaSuccess; ++r) e = s.iteration((const T*)ge.k, (T*)ge.u);
    e3 = cudaStreamEndCapture(cs, &tmp);
    if (e != cudaSuccess) return e;
    if (e3 != cudaSuccess) return e3;

    if ((e = cudaStreamBeginCaptureToGraph(cs, ge.graph, &wnode, nullptr, 1, cudaStreamCaptureModeRelaxed)) != cudaSuccess) return e;
    e = s.finish((T*)ge.u);
    e3 = cudaStreamEndCapture(cs, &tmp);
    if (e != cudaSuccess) return e;
    if (e3 != cudaSuccess) return e3;

    h->launches = saved;
    return cudaGraphInstantiate(&ge.exec, ge.graph, 0);
}

template <typename T>
int solve_impl(fcg_handle h, const void* k, const void* f, void* u, double tol, int maxit, int* iters, double* relres, bool pcg = false,
               bool force = false, double D = 0.0, AsyncSolve* async = nullptr) {
    // async (fcg_solve_host_submit): where the solve is one graph launch, enqueue it and return without waiting; *async then says how
    // to count its launches once the scalar block has been read back.  Every other path runs to completion as usual (async->enqueued = 0).
    if (async) async->enqueued = 0;
    h->launches = 0;
    if (h->fused() && !(force && pcg)) {
        // small lattices: the whole solve is one cooperative kernel with the vectors resident in shared memory (fcg_fused.cuh)
        FusedArgs A{};
        A.mhat = pcg ? h->ws + h->lay.mhat : nullptr;
        A.form = force ? 1 : 0; A.D = D;
        A.k = k; A.f = f; A.u = u; A.Tf = h->ws + h->lay.Tb; A.shat = h->ws + h->lay.shat; A.tw = h->ws + h->lay.tw;
        A.partial = h->at<double>(h->lay.partial_row); A.counter = &h->sc()->ticket[3]; A.sc = h->sc(); A.tol = tol; A.maxit = maxit;
        cudaError_t e = fused_launch(h, A);
        if (e == cudaSuccess) {
            FCG_CK(h, cudaMemcpyAsync(h->h_sc, h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
            FCG_CK(h, cudaStreamSynchronize(h->stream));
            h->launches = 1;
            if (iters) *iters = h->h_sc->it;
            if (relres) *relres = h->h_sc->relres;
            if (h->h_sc->status == FCG_CUDA_ERROR) h->err = "fused solve: grid barrier timed out";
            return h->h_sc->status;
        }
        cudaGetLastError();
        h->err = std::string("cooperative launch failed (") + cudaGetErrorString(e) + "); using the graph path";
        h->fused_opt = 0;
    }
    // force formulation: the three-launch iteration needs reading F1 (k in {0, kappa}, start vector zero on broken bonds); one small
    // kernel and a 32-byte read-back decide it per call (~30 us against milliseconds of solve); otherwise four launches, any k
    double kappa = 0.0;
    if (force && !pcg && h->sl() && !(h->fused())) {
        unsigned long long* d_uni = h->at<unsigned long long>(h->lay.uni);
        FCG_CK(h, cudaMemsetAsync(d_uni, 0, 4 * sizeof(unsigned long long), h->stream));
        force_uniform_kernel<T><<<h->vec_blocks(), 256, 0, h->stream>>>((const T*)k, (const T*)u, h->N, d_uni);
        ++h->launches;
        FCG_CK(h, cudaGetLastError());
        FCG_CK(h, cudaMemcpyAsync(h->h_uni, d_uni, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, h->stream));
        FCG_CK(h, cudaStreamSynchronize(h->stream));
        double kmax, kmin; const unsigned long long b0 = h->h_uni[0], b1 = ~h->h_uni[1];
        std::memcpy(&kmax, &b0, 8); std::memcpy(&kmin, &b1, 8);
        if (h->h_uni[2] == 0 && kmax > 0.0 && kmax == kmin && std::isfinite(kmax)) kappa = kmax;
    }
    if (h->loop_mode == 0) {
        const int var = h->v2() ? 100 + (h->sl() && (!force || kappa > 0.0) ? 1 : 0) : h->row_var();
        const int key = (pcg ? 1 : 0) + 2 * (h->colp() ? 1 : 0) + 4 * h->hints + 1024 * ((h->stagger(0) * 31 + h->stagger(1)) * 31 + h->stagger(2));
        GraphEntry* hit = nullptr;
        for (auto& g : h->graphs)
            if (g.k == k && g.f == f && g.u == u && g.tol == tol && g.maxit == maxit && g.var == var && g.unroll == h->unroll(pcg) && g.pdl == h->pdl() && g.pcg == key && g.force == (force ? 1 : 0) && g.D == D && g.kappa == kappa) { hit = &g; break; }
        if (!hit) {
            if (h->graphs.size() >= 8) {
                size_t lru = 0;
                for (size_t i = 1; i < h->graphs.size(); ++i) if (h->graphs[i].stamp < h->graphs[lru].stamp) lru = i;
                drop_graph(h->graphs[lru]); h->graphs.erase(h->graphs.begin() + lru);
            }
            GraphEntry ge{k, f, u, tol, maxit, var, h->unroll(pcg), h->pdl(), key, force ? 1 : 0, D, kappa, nullptr, nullptr, 0};
            cudaError_t e = build_graph<T>(h, ge);
            if (e != cudaSuccess) {
                // conditional graph nodes unavailable: fall back to direct launches for the rest of this handle's life
                h->err = std::string("graph construction failed (") + cudaGetErrorString(e) + "); using loop mode 1";
                cudaStreamCaptureStatus cst;
                if (cudaStreamIsCapturing(h->cap_stream, &cst) == cudaSuccess && cst != cudaStreamCaptureStatusNone) {
                    cudaGraph_t junk = nullptr; cudaStreamEndCapture(h->cap_stream, &junk);
                }
                drop_graph(ge); cudaGetLastError();
                h->loop_mode = 1;
            } else {
                h->graphs.push_back(ge); hit = &h->graphs.back();
            }
        }
        if (hit) {
            hit->stamp = ++h->stamp;
            FCG_CK(h, cudaGraphLaunch(hit->exec, h->stream));
            if (async) {
                Seq<T> sq{h, h->stream}; sq.pcg = pcg; sq.force = force; sq.D = D; sq.kappa = kappa;
                async->enqueued = 1; async->unroll = hit->unroll;
                async->outside = (kappa > 0.0 ? 1 : 0) + sq.launches_outside_loop(); async->per_iteration = sq.launches_per_iteration();
                return FCG_OK;
            }
            FCG_CK(h, cudaStreamSynchronize(h->stream));
            const long long U = hit->unroll;
            Seq<T> sq{h, h->stream}; sq.pcg = pcg; sq.force = force; sq.D = D; sq.kappa = kappa;
            h->launches = (kappa > 0.0 ? 1 : 0) + sq.launches_outside_loop() + sq.launches_per_iteration() * U * ((h->h_sc->it + U - 1) / U);   // no-op kernels after the stop are launches too
        }
    }
    if (h->loop_mode != 0) {
        Seq<T> s{h, h->stream}; s.pcg = pcg; s.force = force; s.D = D; s.kappa = kappa;
        FCG_CK(h, s.init((const T*)k, (const T*)f, (T*)u, tol, maxit, false, 0ULL));
        FCG_CK(h, cudaMemcpyAsync(h->h_sc, h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
        FCG_CK(h, cudaStreamSynchronize(h->stream));
        while (!h->h_sc->done) {
            for (int c = 0; c < h->chunk; ++c) FCG_CK(h, s.iteration((const T*)k, (T*)u));
            FCG_CK(h, cudaMemcpyAsync(h->h_sc, h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
            FCG_CK(h, cudaStreamSynchronize(h->stream));
        }
        FCG_CK(h, s.finish((T*)u));
        FCG_CK(h, cudaStreamSynchronize(h->stream));
    }
    if (iters) *iters = h->h_sc->it;
    if (relres) *relres = h->h_sc->relres;
    if (h->h_sc->timeout) return fail(h, FCG_CUDA_ERROR, "a pipelined pass gave up waiting on an mbarrier (TMA copy never completed)");
    return h->h_sc->status;
}

template <typename T>
int break_impl(fcg_handle h, void* k, const void* u, const void* t, long long* index, double* ratio, void* fzero = nullptr) {
    break_argmax_kernel<T><<<h->update_blocks(), 256, 0, h->stream>>>(      // whole unrolled trips of 4 vectors per thread
        (T*)k, (const T*)u, (const T*)t, (long long)h->N, h->at<double>(h->lay.brk_r), h->at<long long>(h->lay.brk_i),
        h->at<unsigned int>(h->lay.brk_ticket), h->at<BreakResult>(h->lay.brk_out), (T*)fzero);
    ++h->launches;
    FCG_CK(h, cudaGetLastError());
    FCG_CK(h, cudaMemcpyAsync(h->h_brk, h->at<BreakResult>(h->lay.brk_out), sizeof(BreakResult), cudaMemcpyDeviceToHost, h->stream));
    FCG_CK(h, cudaStreamSynchronize(h->stream));
    if (index) *index = h->h_brk->index;
    if (ratio) *ratio = h->h_brk->ratio;
    return h->h_brk->status;
}

int x_tensor_map(fcg_handle h, const void* X);

template <typename T>
int fft_impl(fcg_handle h, const void* in, void* out, bool inverse) {
    const int L = h->L;
    if (h->v2() && h->fft_direct(inverse)) {
        // two launches: the column pass reads / writes the public layout X[m][n] itself (col2_xpub_kernel)
        Seq<T> s{h, h->stream};
        ColArgs<T> CA{}; CA.mode = inverse ? COL_INV : COL_FWD; CA.Tb = s.Tb(); CA.tw = s.tw(); CA.tmo = &h->sc()->timeout;
        CA.X = (cx<T>*)(inverse ? const_cast<void*>(in) : out);
        if (sizeof(T) == 8) { const int st = x_tensor_map(h, CA.X); if (st != FCG_OK) return st; }
        if (!inverse) {
            FCG_CK(h, s.row_fwd(ROWF_PLAIN, (const T*)in, nullptr));
            FCG_CK(h, h->tab->col2_xpub(&CA, &h->tmap_col, &h->tmap_x, 0, h->stream)); ++h->launches;
        } else {
            FCG_CK(h, h->tab->col2_xpub(&CA, &h->tmap_col, &h->tmap_x, 1, h->stream)); ++h->launches;
            FCG_CK(h, s.row_inv(ROWI_PLAIN, nullptr, nullptr, nullptr, (T*)out, nullptr));
        }
        return FCG_OK;
    }
    if (h->v2()) {
        // pipelined passes on the T2 layout; T2 <-> public half spectrum X[m][n] by one line-wise permutation kernel
        Seq<T> s{h, h->stream};
        ColArgs<T> CA{}; CA.mode = inverse ? COL_INV : COL_FWD; CA.Tb = s.Tb(); CA.tw = s.tw(); CA.tmo = &h->sc()->timeout;
        if (!inverse) {
            FCG_CK(h, s.row_fwd(ROWF_PLAIN, (const T*)in, nullptr));
            FCG_CK(h, h->tab->col2_xform(&CA, &h->tmap_col, 0, h->stream));
            FCG_CK(h, h->tab->t2_export(s.Tb(), out, h->stream));
        } else {
            FCG_CK(h, h->tab->t2_import(in, s.Tb(), h->stream));
            FCG_CK(h, h->tab->col2_xform(&CA, &h->tmap_col, 1, h->stream));
            FCG_CK(h, s.row_inv(ROWI_PLAIN, nullptr, nullptr, nullptr, (T*)out, nullptr));
        }
        return FCG_OK;
    }
    Seq<T> s{h, h->stream, true};       // classic T[n][a] passes + transposing layout kernels
    dim3 blk(32, 8), grd((L / 2 + 31) / 32, (L + 31) / 32);
    if (!inverse) {
        FCG_CK(h, s.row_fwd(ROWF_PLAIN, (const T*)in, nullptr));
        FCG_CK(h, s.col(COL_FWD, false));
        halfspec_export_kernel<T><<<grd, blk, 0, h->stream>>>(s.Tb(), (cx<T>*)out, L);
        FCG_CK(h, cudaGetLastError());
    } else {
        halfspec_import_kernel<T><<<grd, blk, 0, h->stream>>>((const cx<T>*)in, s.Tb(), L);
        FCG_CK(h, cudaGetLastError());
        FCG_CK(h, s.col(COL_INV, false));
        FCG_CK(h, s.row_inv(ROWI_PLAIN, nullptr, nullptr, nullptr, (T*)out, nullptr));
    }
    return FCG_OK;
}

template <typename T>
int apply_impl(fcg_handle h, const void* k, const void* x, void* y, bool force = false) {
    Seq<T> s{h, h->stream}; s.force = force;
    FCG_CK(h, s.row_fwd(ROWF_PLAIN, (const T*)x, nullptr));
    FCG_CK(h, s.col(COL_CONV, false));
    FCG_CK(h, s.row_inv(ROWI_APPLY, (const T*)k, (const T*)x, nullptr, (T*)y, nullptr));
    return FCG_OK;
}

// Per-kernel device times of the CG loop body, measured in sequence (each kernel sees the cache state its
// predecessor leaves, as in a real solve) with CUDA events on the handle's stream.
template <typename T>
int profile_impl(fcg_handle h, const void* k, const void* f, void* u, int iters, double* ms) {
    Seq<T> s{h, h->stream};
    h->launches = 0;
    FCG_CK(h, s.init((const T*)k, (const T*)f, (T*)u, 0.0, 1 << 30, false, 0ULL));
    for (int w = 0; w < 2; ++w) FCG_CK(h, s.iteration((const T*)k, (T*)u));       // warm-up
    EventList ev;
    FCG_CK(h, ev.create((size_t)iters * 5));
    for (int i = 0; i < iters; ++i) {
        cudaEvent_t* e = ev + (size_t)i * 5;
        if (s.sl()) {       // three launches: the residual update is part of P3 (ms[3] = 0)
            FCG_CK(h, cudaEventRecord(e[0], h->stream)); FCG_CK(h, s.it_row_fwd((T*)u));
            FCG_CK(h, cudaEventRecord(e[1], h->stream)); FCG_CK(h, s.it_col_e());
            FCG_CK(h, cudaEventRecord(e[2], h->stream)); FCG_CK(h, s.it_row_inv_f((const T*)k));
            FCG_CK(h, cudaEventRecord(e[3], h->stream));
            FCG_CK(h, cudaEventRecord(e[4], h->stream));
            continue;
        }
        FCG_CK(h, cudaEventRecord(e[0], h->stream)); FCG_CK(h, s.it_row_fwd((T*)u));
        FCG_CK(h, cudaEventRecord(e[1], h->stream)); FCG_CK(h, s.it_col());
        FCG_CK(h, cudaEventRecord(e[2], h->stream)); FCG_CK(h, s.it_row_inv((const T*)k));
        FCG_CK(h, cudaEventRecord(e[3], h->stream)); FCG_CK(h, s.it_update_r());
        FCG_CK(h, cudaEventRecord(e[4], h->stream));
    }
    FCG_CK(h, cudaMemcpyAsync(h->h_sc, h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
    FCG_CK(h, cudaStreamSynchronize(h->stream));
    for (int q = 0; q < 4; ++q) ms[q] = 0.0;
    for (int i = 0; i < iters; ++i)
        for (int q = 0; q < 4; ++q) {
            float t = 0.f;
            FCG_CK(h, cudaEventElapsedTime(&t, ev[(size_t)i * 5 + q], ev[(size_t)i * 5 + q + 1]));
            ms[q] += (double)t / iters;
        }
    return h->h_sc->done ? FCG_NOT_CONVERGED : FCG_OK;       // done would mean the loop kernels exited early
}

// PCG: per-kernel device times of one iteration, ms[0..5] = { P1, P2 (spectrum), P3, r update + row transforms of r,
// P2 (preconditioner), P3 (z, r.z) }; pipelined engine only.
template <typename T>
int profile_pcg_impl(fcg_handle h, const void* k, const void* f, void* u, int iters, double* ms) {
    Seq<T> s{h, h->stream}; s.pcg = true;
    h->launches = 0;
    FCG_CK(h, s.init((const T*)k, (const T*)f, (T*)u, 0.0, 1 << 30, false, 0ULL));
    for (int w = 0; w < 2; ++w) FCG_CK(h, s.iteration((const T*)k, (T*)u));
    EventList ev;
    FCG_CK(h, ev.create((size_t)iters * 7));
    for (int i = 0; i < iters; ++i) {
        cudaEvent_t* e = ev + (size_t)i * 7;
        FCG_CK(h, cudaEventRecord(e[0], h->stream)); FCG_CK(h, s.it_row_fwd((T*)u));
        FCG_CK(h, cudaEventRecord(e[1], h->stream)); FCG_CK(h, s.it_col());
        FCG_CK(h, cudaEventRecord(e[2], h->stream)); FCG_CK(h, s.it_row_inv((const T*)k));
        FCG_CK(h, cudaEventRecord(e[3], h->stream)); FCG_CK(h, s.it_rupd());
        FCG_CK(h, cudaEventRecord(e[4], h->stream)); FCG_CK(h, s.it_col_m());
        FCG_CK(h, cudaEventRecord(e[5], h->stream)); FCG_CK(h, s.it_row_pre());
        FCG_CK(h, cudaEventRecord(e[6], h->stream));
    }
    FCG_CK(h, cudaMemcpyAsync(h->h_sc, h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
    FCG_CK(h, cudaStreamSynchronize(h->stream));
    for (int q = 0; q < 6; ++q) ms[q] = 0.0;
    for (int i = 0; i < iters; ++i)
        for (int q = 0; q < 6; ++q) {
            float t = 0.f;
            FCG_CK(h, cudaEventElapsedTime(&t, ev[(size_t)i * 7 + q], ev[(size_t)i * 7 + q + 1]));
            ms[q] += (double)t / iters;
        }
    return h->h_sc->done ? FCG_NOT_CONVERGED : FCG_OK;
}

template <typename T>
int precond_impl(fcg_handle h, const void* s, double kbar) {
    // m = 1 / (kbar + s) into z (free between solves), then the same preparation as the operator's spectrum
    precond_spectrum_kernel<T><<<h->vec_blocks(), 256, 0, h->stream>>>((const T*)s, h->at<T>(h->lay.z), h->N, (T)kbar);
    FCG_CK(h, cudaGetLastError());
    FCG_CK(h, h->tab->spectrum_prep(h->at<void>(h->lay.z), h->at<void>(h->lay.mhat), h->spectrum_colpos, h->stream));
    FCG_CK(h, cudaStreamSynchronize(h->stream));
    return FCG_OK;
}

// Force formulation, static part: eq. (1c) in closed form, and s = Re F G through the library's own transform
template <typename T>
int green_impl(fcg_handle h, double nu, double E, double a, void* G) {
    green_function_kernel<T><<<h->vec_blocks(), 256, 0, h->stream>>>((T*)G, h->L, (1.0 - nu * nu) / (3.14159265358979323846 * E * a * a), a);
    FCG_CK(h, cudaGetLastError());
    return FCG_OK;
}

template <typename T>
int kernel_spectrum_impl(fcg_handle h, const void* G, void* s) {
    // half spectrum X[m][0..L/2] into r and p (adjacent in the workspace: (L/2+1) L complex <= 2 N reals; free between solves)
    void* X = h->at<void>(h->lay.r);
    int st = fft_impl<T>(h, G, X, false);
    if (st != FCG_OK) return st;
    halfspec_real_expand_kernel<T><<<h->vec_blocks(), 256, 0, h->stream>>>((const cx<T>*)X, (T*)s, h->L);
    FCG_CK(h, cudaGetLastError());
    return FCG_OK;
}

template <typename T>
int twiddle_init(fcg_handle h) {
    const size_t n = (size_t)(h->tab->tw_total > 0 ? h->tab->tw_total : 1);
    std::vector<cx<T>> tw(n);
    h->tab->fill_twiddles(tw.data());
    FCG_CK(h, cudaMemcpyAsync(h->at<void>(h->lay.tw), tw.data(), n * sizeof(cx<T>), cudaMemcpyHostToDevice, h->stream));
    FCG_CK(h, cudaStreamSynchronize(h->stream));
    return FCG_OK;
}

bool supported(int L) { return L >= 16 && L <= 8192 && (L & (L - 1)) == 0; }

// CUtensorMap of T for the tile loads of row_inv2 (driver entry point fetched through the runtime: no -lcuda)
int tensor_map_init(fcg_handle h) {
    typedef CUresult (*EncodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        // no silent 2x cliff: the pipelined passes are the product; the classic ones run only when asked for (FCG_OPT_ENGINE = 1)
        cudaGetLastError();
        h->err = "cuTensorMapEncodeTiled unavailable: the pipelined passes cannot run (FCG_OPT_ENGINE = 1 selects the classic passes)";
        return FCG_OK;
    }
    const cuuint64_t L = (cuuint64_t)h->L, w = (cuuint64_t)h->w, NB = (cuuint64_t)h->tab->v2_nb;
    const CUtensorMapDataType dtp = h->dtype == FCG_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    void* base = h->ws + h->lay.Tb;
    auto enc = reinterpret_cast<EncodeTiled>(fn);
    {   // rows: d0 = one 128-byte line (4 NB reals), d1 = row pair A, d2 = line block m / NB
        const cuuint64_t gdim[3] = {4 * NB, L / 2, L / (2 * NB)};
        const cuuint64_t gstride[2] = {4 * NB * w, (L / 2) * 4 * NB * w};
        const cuuint32_t box[3] = {(cuuint32_t)(4 * NB), 1u, (cuuint32_t)(h->tab->v2_tsub / (int)NB)};
        const cuuint32_t estr[3] = {1u, 1u, 1u};
        CUresult r = enc(&h->tmap_row, dtp, 3, base, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { h->err = "cuTensorMapEncodeTiled (rows) failed (code " + std::to_string((int)r) + ")"; return FCG_CUDA_ERROR; }
    }
    {   // columns: d0 = 2 complex of one row pair (4 reals), d1 = m % NB, d2 = row pair A, d3 = m / NB
        const cuuint64_t gdim[4] = {4, NB, L / 2, L / (2 * NB)};
        const cuuint64_t gstride[3] = {4 * w, 4 * NB * w, (L / 2) * 4 * NB * w};
        const cuuint32_t box[4] = {4u, 1u, (cuuint32_t)h->tab->v2_abox, 1u};
        const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
        CUresult r = enc(&h->tmap_col, dtp, 4, base, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                         CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { h->err = "cuTensorMapEncodeTiled (columns) failed (code " + std::to_string((int)r) + ")"; return FCG_CUDA_ERROR; }
    }
    h->have_tmap = true;
    return FCG_OK;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// FCG_F64: X[m][n] (L rows of L/2+1 complex) as a 3-D tensor {re/im, n, m}: box = one complex x one column x XBOX rows
int x_tensor_map(fcg_handle h, const void* X) {
    if (h->tmap_x_ptr == X) return FCG_OK;
    if ((reinterpret_cast<uintptr_t>(X) & 15u) != 0) return fail(h, FCG_INVALID_ARG, "X must be 16-byte aligned");
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return fail(h, FCG_UNSUPPORTED, "cuTensorMapEncodeTiled unavailable");
    }
    const cuuint64_t L = (cuuint64_t)h->L, XW = L / 2 + 1;
    const cuuint64_t gdim[3] = {2, XW, L};
    const cuuint64_t gstride[2] = {16, XW * 16};
    const cuuint32_t box[3] = {2u, 1u, (cuuint32_t)(L < 256 ? L : 256)};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    if (reinterpret_cast<EncodeTiledFn>(fn)(&h->tmap_x, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(X), gdim, gstride, box, estr,
                                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return fail(h, FCG_CUDA_ERROR, "cuTensorMapEncodeTiled (public half spectrum) failed");
    h->tmap_x_ptr = X;
    return FCG_OK;
}

// tensor maps of one rank's two T2 buffers (same boxes as tensor_map_init, other extents)
int slab_tensor_maps(fcg_handle h) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return fail(h, FCG_UNSUPPORTED, "cuTensorMapEncodeTiled unavailable");
    }
    auto enc = reinterpret_cast<EncodeTiledFn>(fn);
    const cuuint64_t L = (cuuint64_t)h->L, w = (cuuint64_t)h->w, NB = (cuuint64_t)h->tab->v2_nb, Al = (cuuint64_t)h->slab_Al, MBl = (cuuint64_t)h->slab_MBl;
    const CUtensorMapDataType dtp = h->dtype == FCG_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    {   // rows side S: d0 = one 128-byte line, d1 = local row pair, d2 = column block
        const cuuint64_t gdim[3] = {4 * NB, Al, L / (2 * NB)};
        const cuuint64_t gstride[2] = {4 * NB * w, Al * 4 * NB * w};
        const cuuint32_t box[3] = {(cuuint32_t)(4 * NB), 1u, (cuuint32_t)(h->tab->v2_tsub / (int)NB)};
        if (enc(&h->tmap_row_s, dtp, 3, h->ws + h->slab_S, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return fail(h, FCG_CUDA_ERROR, "cuTensorMapEncodeTiled (slab rows) failed");
    }
    {   // columns side = the exchange buffer R itself: d0 = 2 complex of one row pair, d1 = column in block, d2 = local row pair,
        // d3 = local column block, d4 = source rank; a box is one column x boxa row pairs of one source rank
        const cuuint64_t G = (cuuint64_t)h->slab_G;
        const cuuint64_t gdim[5] = {4, NB, Al, MBl, G};
        const cuuint64_t gstride[4] = {4 * w, 4 * NB * w, Al * 4 * NB * w, MBl * Al * 4 * NB * w};
        const cuuint32_t box[5] = {4u, 1u, (cuuint32_t)h->slab_boxa, 1u, 1u};
        const cuuint32_t estr5[5] = {1u, 1u, 1u, 1u, 1u};
        if (enc(&h->tmap_col_s, dtp, 5, h->ws + h->slab_R, gdim, gstride, box, estr5, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return fail(h, FCG_CUDA_ERROR, "cuTensorMapEncodeTiled (slab columns) failed");
    }
    return FCG_OK;
}

// shape algebra of the slab decomposition: pure host arithmetic (also callable without a device: fcg_slab_shape_of)
int slab_shape(int L, int dtype, int G, int rank, fcg_slab_shape* o) {
    if (!supported(L) || (dtype != FCG_F32 && dtype != FCG_F64) || !o) return FCG_INVALID_ARG;
    const PassTable* tab = get_table(L, dtype);
    if (!tab || !tab->v2) return FCG_UNSUPPORTED;
    const int NB = tab->v2_nb, MB = L / (2 * NB);
    if (G < 1 || rank < 0 || rank >= G || MB % G != 0 || (L / 2) % G != 0) return FCG_UNSUPPORTED;
    const size_t w = dtype == FCG_F64 ? 8 : 4;
    o->nranks = G; o->rank = rank; o->columns_per_line = NB; o->column_blocks = MB; o->column_blocks_local = MB / G;
    o->row_pairs_local = (L / 2) / G; o->rows_local = L / G; o->columns_local = (L / 2) / G; o->column0 = rank * ((L / 2) / G);
    o->line_bytes = (size_t)NB * 4 * w;
    o->chunk_bytes = (size_t)(MB / G) * ((L / 2) / G) * o->line_bytes;
    o->buffer_bytes = (size_t)G * o->chunk_bytes;
    return FCG_OK;
}

template <typename T>
int slab_rows_fwd_impl(fcg_handle h, int mode, void* xu) {
    RowFwdArgs<T> A{}; A.mode = mode; A.x = (const T*)xu; A.u = (T*)xu; A.p = h->at<T>(h->lay.p); A.r = h->at<T>(h->lay.r);
    A.Tb = reinterpret_cast<cx<T>*>(h->ws + h->slab_S); A.tw = h->at<cx<T>>(h->lay.tw); A.sc = h->sc(); A.nsm = h->nsm; A.tmo = &h->sc()->timeout;
    A.ntile = h->slab_Al; A.astride = h->slab_Al; A.hints = h->hints; A.stagger_ns = h->stagger(0);
    if (h->slab_peer_maps) {
        A.npeer = h->slab_G; A.prank = h->slab_rank; A.mbl = h->slab_MBl;
        for (int g = 0; g < h->slab_G; ++g) A.peerR[g] = reinterpret_cast<cx<T>*>(h->slab_peerR[g]);
    }
    ++h->launches;
    FCG_CK(h, h->tab->row_fwd2_slab(&A, h->stream));
    return FCG_OK;
}
template <typename T>
int slab_cols_impl(fcg_handle h, void* xch = nullptr) {       // xch: also this rank's share of sum shat |P|^2 (spectral search length)
    ColArgs<T> A{}; A.mode = COL_CONV; A.Tb = reinterpret_cast<cx<T>*>(h->ws + h->slab_R); A.shat = h->at<T>(h->lay.shat); A.tw = h->at<cx<T>>(h->lay.tw);
    A.sc = h->sc(); A.nsm = h->nsm; A.nranks = h->slab_G; A.al = h->slab_Al; A.boxa = h->slab_boxa;
    A.peer_maps = h->slab_peer_maps; A.prank = h->slab_rank; A.mbl = h->slab_MBl; A.tmo = &h->sc()->timeout; A.col0 = h->slab_rank * ((h->L / 2) / h->slab_G);
    const int ncols = (h->L / 2) / h->slab_G;
    A.hints = h->hints; A.stagger_ns = h->stagger(1);
    ++h->launches;
    if (xch) {
        A.partial = h->at<double>(h->lay.partial_col);
        FCG_CK(h, h->tab->col2_slab_e(&A, &h->tmap_col_s, ncols, h->stream));
        ++h->launches;
        slab_energy_kernel<<<1, 256, 0, h->stream>>>(h->at<double>(h->lay.partial_col), ncols, (double*)xch, h->sc());
        FCG_CK(h, cudaGetLastError());
        return FCG_OK;
    }
    FCG_CK(h, h->tab->col2_slab(&A, &h->tmap_col_s, ncols, h->stream));
    return FCG_OK;
}
template <typename T>
int slab_kpp0_impl(fcg_handle h, const void* k, void* xch) {
    const size_t nvec = (h->N / (size_t)h->slab_G) / Vec<T>::W;
    size_t b = (nvec + 255) / 256;
    if (b > (size_t)VEC_BLOCKS_MAX) b = VEC_BLOCKS_MAX;
    ++h->launches;
    cg_kpp0_kernel<T><<<(unsigned)b, 256, 0, h->stream>>>((const T*)k, (const T*)h->at<T>(h->lay.r), nvec, h->at<double>(h->lay.partial_vec), h->sc(), (double*)xch);
    FCG_CK(h, cudaGetLastError());
    return FCG_OK;
}
template <typename T>
int slab_rows_inv_impl(fcg_handle h, int mode, const void* k, const void* v, const void* f, void* xch) {
    RowInvArgs<T> A{}; A.mode = mode; A.tw = h->at<cx<T>>(h->lay.tw); A.k = (const T*)k; A.f = (const T*)f;
    A.v = mode == ROWI_RESID ? (const T*)v : h->at<T>(h->lay.p);
    A.out = mode == ROWI_RESID ? h->at<T>(h->lay.r) : h->at<T>(h->lay.q); A.out2 = mode == ROWI_RESID ? h->at<T>(h->lay.p) : nullptr;
    A.scale = (T)(1.0 / ((double)h->L * (double)h->L)); A.partial = h->at<double>(h->lay.partial_row); A.sc = h->sc(); A.nsm = h->nsm;
    A.tmo = &h->sc()->timeout; A.ntile = h->slab_Al; A.xch = (double*)xch; A.hints = h->hints; A.stagger_ns = h->stagger(2);
    ++h->launches;
    if (mode == ROWI_CGF) {          // q is consumed on the spot: strips k, p, r of the own rows, r in place (fcg_async.cuh, VAR = 5)
        A.f = h->at<T>(h->lay.r); A.out = h->at<T>(h->lay.r); A.out2 = nullptr;
        FCG_CK(h, h->tab->row_inv2_slab_f(&A, &h->tmap_row_s, h->stream));
        return FCG_OK;
    }
    FCG_CK(h, h->tab->row_inv2_slab(&A, &h->tmap_row_s, h->stream));
    return FCG_OK;
}
template <typename T>
int slab_update_r_impl(fcg_handle h, void* xch) {
    const size_t nvec = (h->N / (size_t)h->slab_G) / Vec<T>::W, per = 256 * 4;
    size_t b = (nvec + per - 1) / per;
    if (b > (size_t)VEC_BLOCKS_MAX) b = VEC_BLOCKS_MAX;
    if (b < 1) b = 1;
    ++h->launches;
    cg_update_r_kernel<T><<<(unsigned)b, 256, 0, h->stream>>>(h->at<T>(h->lay.r), (const T*)h->at<T>(h->lay.q), nvec, h->at<double>(h->lay.partial_vec), h->sc(), 0, (double*)xch);
    FCG_CK(h, cudaGetLastError());
    return FCG_OK;
}
template <typename T>
int slab_finish_impl(fcg_handle h, void* u) {
    const size_t nvec = (h->N / (size_t)h->slab_G) / Vec<T>::W;
    size_t b = (nvec + 255) / 256;
    if (b > (size_t)VEC_BLOCKS_MAX) b = VEC_BLOCKS_MAX;
    ++h->launches;
    cg_finish_kernel<T><<<(unsigned)b, 256, 0, h->stream>>>((T*)u, h->at<T>(h->lay.p), nvec, h->sc());
    FCG_CK(h, cudaGetLastError());
    return FCG_OK;
}

}  // namespace

// ================================================================================== C ABI
extern "C" {

const char* fcg_version(void) { return "fcg 0.1 (sm_100a)"; }

size_t fcg_workspace_bytes(int L, fcg_dtype dt) {
    if (!supported(L) || (dt != FCG_F32 && dt != FCG_F64)) return 0;
    return make_layout(L, dt == FCG_F64 ? 8 : 4).total;
}

int fcg_create(int L, fcg_dtype dt, void* workspace, void* cuda_stream, fcg_handle* out) {
    if (!out) return FCG_INVALID_ARG;
    *out = nullptr;
    if (dt != FCG_F32 && dt != FCG_F64) return FCG_INVALID_ARG;
    if (!supported(L)) return FCG_UNSUPPORTED;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return FCG_CUDA_ERROR; }
    fcg_handle h = new fcg_handle_s();
    { int dev = 0, n = 0;
      if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); delete h; return FCG_CUDA_ERROR; }
      h->device = dev;
      if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0) h->nsm = n; }
    h->L = L; h->dtype = dt; h->w = dt == FCG_F64 ? 8 : 4; h->N = (size_t)L * L;
    h->tab = get_table(L, dt);
    h->stream = (cudaStream_t)cuda_stream;
    h->lay = make_layout(L, h->w);
    // bit 6 (T2 stores evict-last) pays while T2 is a quarter of L2 or less, bit 7 (r stores evict-last) while r fits in L2
    h->hints = 63 + (h->N * h->w <= ((size_t)32 << 20) ? 64 : 0) + (h->N * h->w <= ((size_t)128 << 20) ? 128 : 0);
    auto bail = [&](int code) { fcg_destroy(h); return code; };
    if (workspace) { h->ws = (char*)workspace; }
    else {
        if (cudaMalloc((void**)&h->ws, h->lay.total) != cudaSuccess) { cudaGetLastError(); return bail(FCG_CUDA_ERROR); }
        h->own_ws = true;
    }
    if (cudaMallocHost((void**)&h->h_sc, sizeof(Scalars)) != cudaSuccess) return bail(FCG_CUDA_ERROR);
    if (cudaMallocHost((void**)&h->h_brk, sizeof(BreakResult)) != cudaSuccess) return bail(FCG_CUDA_ERROR);
    if (cudaMallocHost((void**)&h->h_uni, 4 * sizeof(unsigned long long)) != cudaSuccess) return bail(FCG_CUDA_ERROR);
    std::memset(h->h_sc, 0, sizeof(Scalars));
    if (cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess) return bail(FCG_CUDA_ERROR);
    if (h->tab->init() != cudaSuccess) return bail(FCG_CUDA_ERROR);
    if (cudaMemsetAsync(h->ws + h->lay.scalars, 0, h->lay.total - h->lay.scalars, h->stream) != cudaSuccess) return bail(FCG_CUDA_ERROR);
    int st = dt == FCG_F64 ? twiddle_init<double>(h) : twiddle_init<float>(h);
    if (st != FCG_OK) return bail(st);
    if (h->tab->v2 && (st = tensor_map_init(h)) != FCG_OK) return bail(st);
    *out = h;
    return FCG_OK;
}

int fcg_destroy(fcg_handle h) {
    if (!h) return FCG_INVALID_ARG;
    DeviceGuard dev_guard_(h->device);
    if (h->stream || h->ws) cudaStreamSynchronize(h->stream);
    for (auto& g : h->graphs) drop_graph(g);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    if (h->own_ws && h->ws) cudaFree(h->ws);
    if (h->h_sc) cudaFreeHost(h->h_sc);
    if (h->h_brk) cudaFreeHost(h->h_brk);
    if (h->h_uni) cudaFreeHost(h->h_uni);
    if (h->pin_stream) cudaStreamSynchronize(h->pin_stream);
    if (h->pout_stream) cudaStreamSynchronize(h->pout_stream);
    for (int s2 = 0; s2 < 2; ++s2) {
        for (void* b : h->pset[s2]) if (b) cudaFree(b);
        if (h->pev_in[s2]) cudaEventDestroy(h->pev_in[s2]);
        if (h->pev_solved[s2]) cudaEventDestroy(h->pev_solved[s2]);
        if (h->pev_out[s2]) cudaEventDestroy(h->pev_out[s2]);
    }
    if (h->pin_stream) cudaStreamDestroy(h->pin_stream);
    if (h->pout_stream) cudaStreamDestroy(h->pout_stream);
    if (h->pres) cudaFreeHost(h->pres);
    if (h->hk) cudaFree(h->hk);
    if (h->hf) cudaFree(h->hf);
    if (h->hu) cudaFree(h->hu);
    if (h->frac_idx) cudaFree(h->frac_idx);
    if (h->frac_it) cudaFree(h->frac_it);
    if (h->frac_ratio) cudaFree(h->frac_ratio);
    if (h->slab_peer_maps) cudaFree(h->slab_peer_maps);
    for (void* b : h->slab_ipc_base) if (b) cudaIpcCloseMemHandle(b);
    cudaGetLastError();
    delete h;
    return FCG_OK;
}

int fcg_set_stream(fcg_handle h, void* cuda_stream) {
    if (!h) return FCG_INVALID_ARG;
    FCG_ENTER_OPT(h);                    // refused while a quasi-static loop is pending: its work is in flight on the old stream
    h->stream = (cudaStream_t)cuda_stream;
    return FCG_OK;
}

int fcg_get_option(fcg_handle h, int option, int* value) {
    if (!h || !value) return FCG_INVALID_ARG;
    switch (option) {                                  // the EFFECTIVE value: automatic choices resolved for this handle's size and dtype
        case FCG_OPT_LOOP_MODE: *value = h->loop_mode; return FCG_OK;
        case FCG_OPT_UNROLL: *value = h->unroll(false); return FCG_OK;
        case FCG_OPT_PDL: *value = h->pdl(); return FCG_OK;
        case FCG_OPT_FUSED: *value = h->fused() ? 1 : 0; return FCG_OK;
        case FCG_OPT_SPECTRAL_ALPHA: *value = h->sl() ? 1 : 0; return FCG_OK;
        case FCG_OPT_COL_PERSISTENT: *value = h->colp() ? 1 : 0; return FCG_OK;
        case FCG_OPT_STAGGER_P1: *value = h->stagger(0); return FCG_OK;
        case FCG_OPT_STAGGER_P2: *value = h->stagger(1); return FCG_OK;
        case FCG_OPT_STAGGER_P3: *value = h->stagger(2); return FCG_OK;
        default: return fail(h, FCG_INVALID_ARG, "fcg_get_option: option has no readable value");
    }
}

int fcg_set_option(fcg_handle h, int option, int value) {
    if (!h) return FCG_INVALID_ARG;
    FCG_ENTER_OPT(h);
    switch (option) {
        case FCG_OPT_LOOP_MODE: if (value != 0 && value != 1) return fail(h, FCG_INVALID_ARG, "loop mode must be 0 or 1"); h->loop_mode = value; return FCG_OK;
        case FCG_OPT_CHUNK: if (value < 1) return fail(h, FCG_INVALID_ARG, "chunk must be >= 1"); h->chunk = value; return FCG_OK;
        case FCG_OPT_ROW_VARIANT:
            if (value >= FCG_NROWVAR || (value >= 0 && !h->tab->row_valid[value])) return fail(h, FCG_INVALID_ARG, "row variant not available for this size");
            h->row_var_opt = value; return FCG_OK;
        case FCG_OPT_FUSED: if (value != 0 && value != 1) return fail(h, FCG_INVALID_ARG, "fused must be 0 or 1"); h->fused_opt = value; return FCG_OK;
        case FCG_OPT_PDL: if (value < -1 || value > 2) return fail(h, FCG_INVALID_ARG, "pdl must be -1, 0, 1 or 2"); h->pdl_opt = value; return FCG_OK;
#ifdef FCG_PROBE
        case FCG_OPT_L2_HINTS: h->hints = value; return FCG_OK;      // measurement build: the probe bits of fcg_async.cuh too
#else
        case FCG_OPT_L2_HINTS: if (value < 0 || value > 255) return fail(h, FCG_INVALID_ARG, "hints must be 0..255"); h->hints = value; return FCG_OK;
#endif
        case FCG_OPT_SPECTRAL_ALPHA: if (value != 0 && value != 1) return fail(h, FCG_INVALID_ARG, "spectral alpha must be 0 or 1"); h->sl_opt = value; return FCG_OK;
        case FCG_OPT_COL_PERSISTENT: if (value < -1 || value > 1) return fail(h, FCG_INVALID_ARG, "col persistent must be -1, 0 or 1"); h->colp_opt = value; return FCG_OK;
        case FCG_OPT_BARRIER_START: h->barrier_start = (unsigned int)value; return FCG_OK;
        case FCG_OPT_FFT_DIRECT: if (value < -1 || value > 1) return fail(h, FCG_INVALID_ARG, "fft direct must be -1, 0 or 1"); h->fft_pub = value; return FCG_OK;
        case FCG_OPT_FUSED_TWO: if (value != 0 && value != 1) return fail(h, FCG_INVALID_ARG, "fused two must be 0 or 1"); h->fused_two = value; return FCG_OK;
        case FCG_OPT_STAGGER_P1: case FCG_OPT_STAGGER_P2: case FCG_OPT_STAGGER_P3:
            if (value < -1 || value > 100000) return fail(h, FCG_INVALID_ARG, "stagger must be -1 (default) or 0..100000 ns");
            h->stag_opt[option - FCG_OPT_STAGGER_P1] = value; return FCG_OK;
        case FCG_OPT_UNROLL: if ((value < 1 && value != -1) || value > 64) return fail(h, FCG_INVALID_ARG, "unroll must be 1..64 or -1"); h->unroll_opt = value; return FCG_OK;
        case FCG_OPT_ENGINE:
            if (value != 0 && value != 1) return fail(h, FCG_INVALID_ARG, "engine must be 0 or 1");
            h->engine_opt = value;
            if (h->have_spectrum && h->spectrum_colpos != (h->v2() ? 1 : 0)) { h->have_spectrum = false; h->have_precond = false; }   // stored layout belongs to the other engine
            return FCG_OK;
    }
    return fail(h, FCG_INVALID_ARG, "unknown option");
}

int fcg_set_spectrum(fcg_handle h, const void* s) {
    if (!h || !s) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    h->spectrum_colpos = h->v2() ? 1 : 0;
    FCG_CK(h, h->tab->spectrum_prep(s, h->at<void>(h->lay.shat), h->spectrum_colpos, h->stream));
    FCG_CK(h, cudaStreamSynchronize(h->stream));      // the caller's array is not referenced after return
    h->have_spectrum = true; h->have_precond = false;
    return FCG_OK;
}

int fcg_apply(fcg_handle h, const void* k, const void* x, void* y) {
    if (!h || !k || !x || !y) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    if (y == k || y == x) return fail(h, FCG_INVALID_ARG, "y must not alias k or x");
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    return h->dtype == FCG_F64 ? apply_impl<double>(h, k, x, y) : apply_impl<float>(h, k, x, y);
}

int fcg_solve(fcg_handle h, const void* k, const void* f, void* u, double tol, int maxit, int* iters_host, double* rel_residual_host) {
    if (!h || !k || !f || !u) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    if (u == k || u == f) return fail(h, FCG_INVALID_ARG, "u must not alias k or f");
    if (misaligned(k) || misaligned(f) || misaligned(u)) return fail(h, FCG_INVALID_ARG, "k, f, u must be 16-byte aligned");
    if (!(tol >= 0.0) || maxit < 0) return fail(h, FCG_INVALID_ARG, "tol must be >= 0 and maxit >= 0");
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    return h->dtype == FCG_F64 ? solve_impl<double>(h, k, f, u, tol, maxit, iters_host, rel_residual_host)
                               : solve_impl<float>(h, k, f, u, tol, maxit, iters_host, rel_residual_host);
}

int fcg_set_preconditioner(fcg_handle h, const void* s, double kbar) {
    if (!h || !s) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    if (!(kbar >= 0.0) || !std::isfinite(kbar)) return fail(h, FCG_INVALID_ARG, "kbar must be finite and >= 0");
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    int st = h->dtype == FCG_F64 ? precond_impl<double>(h, s, kbar) : precond_impl<float>(h, s, kbar);
    if (st == FCG_OK) h->have_precond = true;
    return st;
}

int fcg_pcg_solve(fcg_handle h, const void* k, const void* f, void* u, double tol, int maxit, int* iters_host, double* rel_residual_host) {
    if (!h || !k || !f || !u) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    if (u == k || u == f) return fail(h, FCG_INVALID_ARG, "u must not alias k or f");
    if (misaligned(k) || misaligned(f) || misaligned(u)) return fail(h, FCG_INVALID_ARG, "k, f, u must be 16-byte aligned");
    if (!(tol >= 0.0) || maxit < 0) return fail(h, FCG_INVALID_ARG, "tol must be >= 0 and maxit >= 0");
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    if (!h->have_precond) return fail(h, FCG_NO_SPECTRUM, "fcg_set_preconditioner has not been called");
    return h->dtype == FCG_F64 ? solve_impl<double>(h, k, f, u, tol, maxit, iters_host, rel_residual_host, true)
                               : solve_impl<float>(h, k, f, u, tol, maxit, iters_host, rel_residual_host, true);
}

int fcg_profile_pcg_iteration(fcg_handle h, const void* k, const void* f, void* u, int iters, double* ms_host) {
    if (!h || !k || !f || !u || iters < 1 || !ms_host) return fail(h, FCG_INVALID_ARG, "bad argument");
    FCG_ENTER(h);
    if (!h->have_spectrum || !h->have_precond) return fail(h, FCG_NO_SPECTRUM, "spectrum or preconditioner not set");
    if (!h->v2()) return fail(h, FCG_UNSUPPORTED, "pipelined engine only");
    return h->dtype == FCG_F64 ? profile_pcg_impl<double>(h, k, f, u, iters, ms_host) : profile_pcg_impl<float>(h, k, f, u, iters, ms_host);
}

int fcg_solve_host(fcg_handle h, const void* k_host, const void* f_host, void* u_host, double tol, int maxit,
                   int* iters_host, double* rel_residual_host) {
    if (!h || !k_host || !f_host || !u_host) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    const size_t bytes = h->N * h->w;
    if (!h->hk) { FCG_CK(h, cudaMalloc(&h->hk, bytes)); FCG_CK(h, cudaMalloc(&h->hf, bytes)); FCG_CK(h, cudaMalloc(&h->hu, bytes)); }
    FCG_CK(h, cudaMemcpyAsync(h->hk, k_host, bytes, cudaMemcpyHostToDevice, h->stream));
    FCG_CK(h, cudaMemcpyAsync(h->hf, f_host, bytes, cudaMemcpyHostToDevice, h->stream));
    FCG_CK(h, cudaMemcpyAsync(h->hu, u_host, bytes, cudaMemcpyHostToDevice, h->stream));
    int st = fcg_solve(h, h->hk, h->hf, h->hu, tol, maxit, iters_host, rel_residual_host);
    if (st < 0 && st != FCG_BREAKDOWN) return st;
    FCG_CK(h, cudaMemcpyAsync(u_host, h->hu, bytes, cudaMemcpyDeviceToHost, h->stream));
    FCG_CK(h, cudaStreamSynchronize(h->stream));
    return st;
}

// Pipelined form of fcg_solve_host (include/fcg.h): up to two solves outstanding.  Inputs go up on their own stream into one of two
// staging sets, the solve is enqueued behind them on the handle's stream (one graph launch: nothing blocks), the result comes down
// on a third stream -- so the copies of solve i+1 and of solve i-1 run while solve i computes.
int fcg_solve_host_submit(fcg_handle h, const void* k_host, const void* f_host, void* u_host, double tol, int maxit) {
    if (!h || !k_host || !f_host || !u_host) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    if (!(tol >= 0.0) || maxit < 0) return fail(h, FCG_INVALID_ARG, "tol must be >= 0 and maxit >= 0");
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    if (h->pcount >= 2) return fail(h, FCG_INVALID_ARG, "two solves are outstanding: call fcg_solve_host_wait first");
    const size_t bytes = h->N * h->w;
    if (!h->pin_stream) {
        FCG_CK(h, cudaStreamCreateWithFlags(&h->pin_stream, cudaStreamNonBlocking));
        FCG_CK(h, cudaStreamCreateWithFlags(&h->pout_stream, cudaStreamNonBlocking));
        for (int s2 = 0; s2 < 2; ++s2) {
            FCG_CK(h, cudaEventCreateWithFlags(&h->pev_in[s2], cudaEventDisableTiming));
            FCG_CK(h, cudaEventCreateWithFlags(&h->pev_solved[s2], cudaEventDisableTiming));
            FCG_CK(h, cudaEventCreateWithFlags(&h->pev_out[s2], cudaEventDisableTiming));
        }
        FCG_CK(h, cudaMallocHost((void**)&h->pres, 2 * sizeof(Scalars)));
    }
    const int s2 = (h->phead + h->pcount) % 2;
    for (int v = 0; v < 3; ++v) if (!h->pset[s2][v]) FCG_CK(h, cudaMalloc(&h->pset[s2][v], bytes));
    // (this set's previous solve has been waited for: its inputs were consumed and its result is down)
    FCG_CK(h, cudaMemcpyAsync(h->pset[s2][0], k_host, bytes, cudaMemcpyHostToDevice, h->pin_stream));
    FCG_CK(h, cudaMemcpyAsync(h->pset[s2][1], f_host, bytes, cudaMemcpyHostToDevice, h->pin_stream));
    FCG_CK(h, cudaMemcpyAsync(h->pset[s2][2], u_host, bytes, cudaMemcpyHostToDevice, h->pin_stream));
    FCG_CK(h, cudaEventRecord(h->pev_in[s2], h->pin_stream));
    FCG_CK(h, cudaStreamWaitEvent(h->stream, h->pev_in[s2], 0));
    AsyncSolve as{};
    const int st = h->dtype == FCG_F64
        ? solve_impl<double>(h, h->pset[s2][0], h->pset[s2][1], h->pset[s2][2], tol, maxit, nullptr, nullptr, false, false, 0.0, &as)
        : solve_impl<float>(h, h->pset[s2][0], h->pset[s2][1], h->pset[s2][2], tol, maxit, nullptr, nullptr, false, false, 0.0, &as);
    if (st < 0 && st != FCG_BREAKDOWN) return st;
    h->penq[s2] = as.enqueued; h->pstatus[s2] = st;
    if (as.enqueued) {
        h->punroll[s2] = as.unroll; h->poutside[s2] = as.outside; h->pper[s2] = as.per_iteration;
        FCG_CK(h, cudaMemcpyAsync(&h->pres[s2], h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
    } else {                              // (one-launch kernel or host-driven loop: the solve has run to completion)
        h->pres[s2] = *h->h_sc; h->poutside[s2] = h->launches;
    }
    FCG_CK(h, cudaEventRecord(h->pev_solved[s2], h->stream));
    FCG_CK(h, cudaStreamWaitEvent(h->pout_stream, h->pev_solved[s2], 0));
    FCG_CK(h, cudaMemcpyAsync(u_host, h->pset[s2][2], bytes, cudaMemcpyDeviceToHost, h->pout_stream));
    FCG_CK(h, cudaEventRecord(h->pev_out[s2], h->pout_stream));
    ++h->pcount;
    return FCG_OK;
}

int fcg_solve_host_wait(fcg_handle h, int* iters_host, double* rel_residual_host) {
    if (!h) return FCG_INVALID_ARG;
    FCG_ENTER(h);
    if (h->pcount < 1) return fail(h, FCG_INVALID_ARG, "no fcg_solve_host_submit is outstanding");
    const int s2 = h->phead;
    FCG_CK(h, cudaEventSynchronize(h->pev_out[s2]));
    h->phead ^= 1; --h->pcount;
    const Scalars& r = h->pres[s2];
    if (iters_host) *iters_host = r.it;
    if (rel_residual_host) *rel_residual_host = r.relres;
    if (h->penq[s2]) {
        const long long U = h->punroll[s2];
        h->launches = h->poutside[s2] + h->pper[s2] * U * ((r.it + U - 1) / U);
        if (r.timeout) return fail(h, FCG_CUDA_ERROR, "a pipelined pass gave up waiting on an mbarrier (TMA copy never completed)");
        return r.status;
    }
    h->launches = h->poutside[s2];
    return h->pstatus[s2];
}

int fcg_fft_fwd(fcg_handle h, const void* x, void* X) {
    if (!h || !x || !X) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    return h->dtype == FCG_F64 ? fft_impl<double>(h, x, X, false) : fft_impl<float>(h, x, X, false);
}

int fcg_fft_inv(fcg_handle h, const void* X, void* x) {
    if (!h || !x || !X) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    return h->dtype == FCG_F64 ? fft_impl<double>(h, X, x, true) : fft_impl<float>(h, X, x, true);
}

int fcg_break_step(fcg_handle h, void* k, const void* u, const void* t, long long* index_host, double* ratio_host) {
    if (!h || !k || !u || !t) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    h->launches = 0;
    return h->dtype == FCG_F64 ? break_impl<double>(h, k, u, t, index_host, ratio_host)
                               : break_impl<float>(h, k, u, t, index_host, ratio_host);
}

// device arrays for the per-step results of the fused quasi-static loops
static int frac_reserve(fcg_handle h, int nsteps) {
    if (h->frac_cap >= nsteps) return FCG_OK;
    if (h->frac_idx) cudaFree(h->frac_idx);
    if (h->frac_it) cudaFree(h->frac_it);
    if (h->frac_ratio) cudaFree(h->frac_ratio);
    h->frac_idx = nullptr; h->frac_it = nullptr; h->frac_ratio = nullptr; h->frac_cap = 0;
    FCG_CK(h, cudaMalloc((void**)&h->frac_idx, (size_t)nsteps * sizeof(long long)));
    FCG_CK(h, cudaMalloc((void**)&h->frac_it, (size_t)nsteps * sizeof(int)));
    FCG_CK(h, cudaMalloc((void**)&h->frac_ratio, (size_t)nsteps * sizeof(double)));
    h->frac_cap = nsteps;
    return FCG_OK;
}

// Quasi-static loop in two halves, so that one host thread can keep several handles (streams) busy: begin enqueues (and, where the
// loop is one cooperative kernel, returns at once); end blocks and hands out the results.
static int fracture_begin(fcg_handle h, void* k, const void* f, void* u, const void* t, int nsteps, double tol, int maxit, bool pcg) {
    if (!h || !k || !f || !u || !t || nsteps < 0) return fail(h, FCG_INVALID_ARG, "bad argument");
    FCG_ENTER(h);
    if (pcg && !h->have_precond) return fail(h, FCG_NO_SPECTRUM, "fcg_set_preconditioner has not been called");
    if (h->pend_nsteps >= 0) return fail(h, FCG_INVALID_ARG, "a quasi-static loop is already pending on this handle: call its _end first");
    h->pend_nsteps = -1; h->pend_async = false; h->pend_done = 0; h->pend_status = FCG_OK; h->pend_kind = 0;
    if (h->fused() && h->have_spectrum && nsteps > 0 && tol >= 0.0 && maxit >= 0) {
        // small lattices: the whole quasi-static loop -- every solve and every break step -- is one cooperative kernel
        { const int e0 = frac_reserve(h, nsteps); if (e0 != FCG_OK) return e0; }
        FusedArgs A{};
        A.k = k; A.f = f; A.u = u; A.Tf = h->ws + h->lay.Tb; A.shat = h->ws + h->lay.shat; A.tw = h->ws + h->lay.tw;
        A.partial = h->at<double>(h->lay.partial_row); A.counter = &h->sc()->ticket[3]; A.sc = h->sc(); A.tol = tol; A.maxit = maxit;
        A.mhat = pcg ? h->ws + h->lay.mhat : nullptr;
        A.nsteps = nsteps; A.t = t; A.k_out = k; A.out_index = h->frac_idx; A.out_iters = h->frac_it;
        A.brk_r = h->at<double>(h->lay.brk_r); A.brk_i = h->at<long long>(h->lay.brk_i);
        cudaError_t e = fused_launch(h, A);
        if (e == cudaSuccess) {
            FCG_CK(h, cudaMemcpyAsync(h->h_sc, h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
            h->pend_nsteps = nsteps; h->pend_async = true; h->launches = 1;
            return FCG_OK;
        }
        cudaGetLastError();
        h->err = std::string("cooperative launch failed (") + cudaGetErrorString(e) + "); using the graph path";
        h->fused_opt = 0;
    }
    h->pend_idx.assign((size_t)nsteps, -1); h->pend_it.assign((size_t)nsteps, 0);
    long long total = 0; int done = 0, st = FCG_OK;
    for (int step = 0; step < nsteps; ++step) {
        int it = 0; double rr = 0.0;
        st = pcg ? fcg_pcg_solve(h, k, f, u, tol, maxit, &it, &rr) : fcg_solve(h, k, f, u, tol, maxit, &it, &rr);
        total += h->launches;
        if (st < 0) break;
        long long idx = -1; double ratio = 0.0;
        st = fcg_break_step(h, k, u, t, &idx, &ratio);
        total += h->launches;
        if (st < 0) break;
        h->pend_idx[step] = idx; h->pend_it[step] = it; ++done; st = FCG_OK;
    }
    h->pend_nsteps = nsteps; h->pend_done = done; h->pend_status = st; h->launches = total;
    return st < 0 ? st : FCG_OK;
}

static int fracture_end(fcg_handle h, long long* index_host, int* iters_host, int* steps_done_host) {
    if (!h || !index_host || !iters_host) return fail(h, FCG_INVALID_ARG, "bad argument");
    FCG_ENTER_END(h);
    if (h->pend_nsteps < 0 || h->pend_kind != 0) return fail(h, FCG_INVALID_ARG, "no quasi-static loop of this kind pending on this handle");
    h->pend_nsteps = -1;
    if (h->pend_async) {
        h->pend_async = false;
        FCG_CK(h, cudaStreamSynchronize(h->stream));
        const int done = h->h_sc->steps_done;
        if (done > 0) {
            FCG_CK(h, cudaMemcpyAsync(index_host, h->frac_idx, (size_t)done * sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
            FCG_CK(h, cudaMemcpyAsync(iters_host, h->frac_it, (size_t)done * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
            FCG_CK(h, cudaStreamSynchronize(h->stream));
        }
        if (steps_done_host) *steps_done_host = done;
        if (h->h_sc->status == FCG_CUDA_ERROR) h->err = "fused quasi-static loop: grid barrier timed out";
        return h->h_sc->status < 0 ? h->h_sc->status : FCG_OK;
    }
    for (int i = 0; i < h->pend_done; ++i) { index_host[i] = h->pend_idx[(size_t)i]; iters_host[i] = h->pend_it[(size_t)i]; }
    if (steps_done_host) *steps_done_host = h->pend_done;
    return h->pend_status;
}

static int fracture_impl(fcg_handle h, void* k, const void* f, void* u, const void* t, int nsteps, double tol, int maxit,
                         long long* index_host, int* iters_host, int* steps_done_host, bool pcg) {
    if (!index_host || !iters_host) return fail(h, FCG_INVALID_ARG, "bad argument");
    int st = fracture_begin(h, k, f, u, t, nsteps, tol, maxit, pcg);
    if (st < 0 && (!h || h->pend_nsteps < 0)) return st;
    return fracture_end(h, index_host, iters_host, steps_done_host);
}

int fcg_fracture_begin(fcg_handle h, void* k, const void* f, void* u, const void* t, int nsteps, double tol, int maxit, int use_pcg) {
    return fracture_begin(h, k, f, u, t, nsteps, tol, maxit, use_pcg != 0);
}

int fcg_fracture_end(fcg_handle h, long long* index_host, int* iters_host, int* steps_done_host) {
    return fracture_end(h, index_host, iters_host, steps_done_host);
}

int fcg_fracture(fcg_handle h, void* k, const void* f, void* u, const void* t, int nsteps, double tol, int maxit,
                 long long* index_host, int* iters_host, int* steps_done_host) {
    return fracture_impl(h, k, f, u, t, nsteps, tol, maxit, index_host, iters_host, steps_done_host, false);
}

int fcg_pcg_fracture(fcg_handle h, void* k, const void* f, void* u, const void* t, int nsteps, double tol, int maxit,
                     long long* index_host, int* iters_host, int* steps_done_host) {
    if (h && !h->have_precond) return fail(h, FCG_NO_SPECTRUM, "fcg_set_preconditioner has not been called");
    return fracture_impl(h, k, f, u, t, nsteps, tol, maxit, index_host, iters_host, steps_done_host, true);
}

// ---- the paper's formulation in the bond forces, (I + K G) f = K D (eq. (2))
int fcg_green_function(fcg_handle h, double nu, double E, double a, void* G) {
    if (!h || !G) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    if (!(E > 0.0) || !(a > 0.0) || !std::isfinite(nu) || !std::isfinite(E) || !std::isfinite(a)) return fail(h, FCG_INVALID_ARG, "E and a must be positive and finite, nu finite");
    return h->dtype == FCG_F64 ? green_impl<double>(h, nu, E, a, G) : green_impl<float>(h, nu, E, a, G);
}

int fcg_kernel_spectrum(fcg_handle h, const void* G, void* s) {
    if (!h || !G || !s) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    if (G == s) return fail(h, FCG_INVALID_ARG, "s must not alias G");
    static_assert(ALIGN % 16 == 0, "workspace alignment");
    if (h->lay.p != h->lay.r + h->N * h->w) return fail(h, FCG_UNSUPPORTED, "workspace layout: r and p not adjacent");
    return h->dtype == FCG_F64 ? kernel_spectrum_impl<double>(h, G, s) : kernel_spectrum_impl<float>(h, G, s);
}

int fcg_inverse_spectrum(fcg_handle h, const void* g, void* s) {
    if (!h || !g || !s) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    if (h->dtype == FCG_F64) inverse_spectrum_kernel<double><<<h->vec_blocks(), 256, 0, h->stream>>>((const double*)g, (double*)s, h->N);
    else inverse_spectrum_kernel<float><<<h->vec_blocks(), 256, 0, h->stream>>>((const float*)g, (float*)s, h->N);
    FCG_CK(h, cudaGetLastError());
    return FCG_OK;
}

int fcg_force_rhs(fcg_handle h, const void* k, double D, void* b) {
    if (!h || !k || !b || !std::isfinite(D)) return fail(h, FCG_INVALID_ARG, "null argument or D not finite");
    FCG_ENTER(h);
    if (h->dtype == FCG_F64) scale_kernel<double><<<h->vec_blocks(), 256, 0, h->stream>>>((const double*)k, (double*)b, h->N, D);
    else scale_kernel<float><<<h->vec_blocks(), 256, 0, h->stream>>>((const float*)k, (float*)b, h->N, (float)D);
    FCG_CK(h, cudaGetLastError());
    return FCG_OK;
}

int fcg_force_from_displacement(fcg_handle h, const void* k, double D, const void* u, void* f) {
    if (!h || !k || !u || !f || !std::isfinite(D)) return fail(h, FCG_INVALID_ARG, "null argument or D not finite");
    FCG_ENTER(h);
    if (h->dtype == FCG_F64) force_from_displacement_kernel<double><<<h->vec_blocks(), 256, 0, h->stream>>>((const double*)k, (const double*)u, (double*)f, h->N, D);
    else force_from_displacement_kernel<float><<<h->vec_blocks(), 256, 0, h->stream>>>((const float*)k, (const float*)u, (float*)f, h->N, (float)D);
    FCG_CK(h, cudaGetLastError());
    return FCG_OK;
}

int fcg_force_apply(fcg_handle h, const void* k, const void* x, void* y) {
    if (!h || !k || !x || !y) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    if (y == k || y == x) return fail(h, FCG_INVALID_ARG, "y must not alias k or x");
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    return h->dtype == FCG_F64 ? apply_impl<double>(h, k, x, y, true) : apply_impl<float>(h, k, x, y, true);
}

int fcg_force_solve(fcg_handle h, const void* k, double D, void* f, double tol, int maxit, int* iters_host, double* rel_residual_host) {
    if (!h || !k || !f) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    if (!(tol >= 0.0) || maxit < 0 || !std::isfinite(D)) return fail(h, FCG_INVALID_ARG, "tol must be >= 0, maxit >= 0, D finite");
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    return h->dtype == FCG_F64 ? solve_impl<double>(h, k, nullptr, f, tol, maxit, iters_host, rel_residual_host, false, true, D)
                               : solve_impl<float>(h, k, nullptr, f, tol, maxit, iters_host, rel_residual_host, false, true, D);
}

int fcg_force_break_step(fcg_handle h, void* k, void* f, const void* t, long long* index_host, double* ratio_host) {
    if (!h || !k || !f || !t) return fail(h, FCG_INVALID_ARG, "null argument");
    FCG_ENTER(h);
    h->launches = 0;
    return h->dtype == FCG_F64 ? break_impl<double>(h, k, f, t, index_host, ratio_host, f)
                               : break_impl<float>(h, k, f, t, index_host, ratio_host, f);
}

int fcg_force_fracture(fcg_handle h, void* k, double D, void* f, const void* t, int nsteps, double tol, int maxit,
                       long long* index_host, int* iters_host, double* ratio_host, int* steps_done_host) {
    if (!h || !k || !f || !t || nsteps < 0 || !index_host || !iters_host) return fail(h, FCG_INVALID_ARG, "bad argument");
    FCG_ENTER(h);
    if (!(tol >= 0.0) || maxit < 0 || !std::isfinite(D)) return fail(h, FCG_INVALID_ARG, "tol must be >= 0, maxit >= 0, D finite");
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    if (h->fused() && nsteps > 0) {
        // small lattices: every solve and every break step of the loop in one cooperative kernel (fcg_fused.cuh, FORCE variant)
        { const int e0 = frac_reserve(h, nsteps); if (e0 != FCG_OK) return e0; }
        FusedArgs A{};
        A.form = 1; A.D = D; A.k = k; A.f = nullptr; A.u = f; A.Tf = h->ws + h->lay.Tb; A.shat = h->ws + h->lay.shat; A.tw = h->ws + h->lay.tw;
        A.partial = h->at<double>(h->lay.partial_row); A.counter = &h->sc()->ticket[3]; A.sc = h->sc(); A.tol = tol; A.maxit = maxit;
        A.nsteps = nsteps; A.t = t; A.k_out = k; A.out_index = h->frac_idx; A.out_iters = h->frac_it; A.out_ratio = h->frac_ratio;
        A.brk_r = h->at<double>(h->lay.brk_r); A.brk_i = h->at<long long>(h->lay.brk_i);
        cudaError_t e = fused_launch(h, A);
        if (e == cudaSuccess) {
            FCG_CK(h, cudaMemcpyAsync(h->h_sc, h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
            FCG_CK(h, cudaStreamSynchronize(h->stream));
            h->launches = 1;
            const int done = h->h_sc->steps_done;
            if (done > 0) {
                FCG_CK(h, cudaMemcpyAsync(index_host, h->frac_idx, (size_t)done * sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
                FCG_CK(h, cudaMemcpyAsync(iters_host, h->frac_it, (size_t)done * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
                if (ratio_host) FCG_CK(h, cudaMemcpyAsync(ratio_host, h->frac_ratio, (size_t)done * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
                FCG_CK(h, cudaStreamSynchronize(h->stream));
            }
            if (steps_done_host) *steps_done_host = done;
            if (h->h_sc->status == FCG_CUDA_ERROR) h->err = "fused quasi-static loop: grid barrier timed out";
            return h->h_sc->status < 0 ? h->h_sc->status : FCG_OK;
        }
        cudaGetLastError();
        h->err = std::string("cooperative launch failed (") + cudaGetErrorString(e) + "); using the graph path";
        h->fused_opt = 0;
    }
    long long total = 0; int done = 0, st = FCG_OK;
    for (int step = 0; step < nsteps; ++step) {
        int it = 0; double rr = 0.0;
        st = fcg_force_solve(h, k, D, f, tol, maxit, &it, &rr);
        total += h->launches;
        if (st < 0) break;
        long long idx = -1; double ratio = 0.0;
        st = fcg_force_break_step(h, k, f, t, &idx, &ratio);
        total += h->launches;
        if (st < 0) break;
        index_host[step] = idx; iters_host[step] = it; if (ratio_host) ratio_host[step] = ratio;
        ++done; st = FCG_OK;
    }
    if (steps_done_host) *steps_done_host = done;
    h->launches = total;
    return st < 0 ? st : FCG_OK;
}

// quasi-static loop of the force model through the displacements (reading F7), in two halves like
// fcg_fracture_begin / _end so that one host thread can keep an ensemble of samples (handles on their own streams) in flight
int fcg_force_fracture_displacement_begin(fcg_handle h, void* k, double D, void* u, const void* t, int nsteps, double tol, int maxit, int use_pcg) {
    if (!h || !k || !u || !t || nsteps < 0) return fail(h, FCG_INVALID_ARG, "bad argument");
    FCG_ENTER(h);
    if (!(tol >= 0.0) || maxit < 0 || !std::isfinite(D)) return fail(h, FCG_INVALID_ARG, "tol must be >= 0, maxit >= 0, D finite");
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    if (use_pcg && !h->have_precond) return fail(h, FCG_NO_SPECTRUM, "fcg_set_preconditioner has not been called");
    if (h->pend_nsteps >= 0) return fail(h, FCG_INVALID_ARG, "a quasi-static loop is already pending on this handle: call its _end first");
    h->pend_nsteps = -1; h->pend_async = false; h->pend_done = 0; h->pend_status = FCG_OK; h->pend_kind = 1;
    if (h->fused() && nsteps > 0) {
        // small lattices: the whole loop in one cooperative kernel (fcg_fused.cuh, FORCE = 2)
        { const int e0 = frac_reserve(h, nsteps); if (e0 != FCG_OK) return e0; }
        FusedArgs A{};
        A.form = 2; A.D = D; A.k = k; A.f = nullptr; A.u = u; A.Tf = h->ws + h->lay.Tb; A.shat = h->ws + h->lay.shat; A.tw = h->ws + h->lay.tw;
        A.mhat = use_pcg ? h->ws + h->lay.mhat : nullptr;
        A.partial = h->at<double>(h->lay.partial_row); A.counter = &h->sc()->ticket[3]; A.sc = h->sc(); A.tol = tol; A.maxit = maxit;
        A.nsteps = nsteps; A.t = t; A.k_out = k; A.out_index = h->frac_idx; A.out_iters = h->frac_it; A.out_ratio = h->frac_ratio;
        A.brk_r = h->at<double>(h->lay.brk_r); A.brk_i = h->at<long long>(h->lay.brk_i);
        cudaError_t e = fused_launch(h, A);
        if (e == cudaSuccess) {
            FCG_CK(h, cudaMemcpyAsync(h->h_sc, h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
            h->pend_nsteps = nsteps; h->pend_async = true; h->launches = 1;
            return FCG_OK;
        }
        cudaGetLastError();
        h->err = std::string("cooperative launch failed (") + cudaGetErrorString(e) + "); using the graph path";
        h->fused_opt = 0;
    }
    // larger lattices: the library's own calls in turn, with two scratch vectors (b = K D and the forces); runs to its end here
    const size_t bytes = h->N * h->w;
    if (!h->hk) { FCG_CK(h, cudaMalloc(&h->hk, bytes)); FCG_CK(h, cudaMalloc(&h->hf, bytes)); FCG_CK(h, cudaMalloc(&h->hu, bytes)); }
    void* b = h->hf; void* frc = h->hk;
    h->pend_idx.assign((size_t)nsteps, -1); h->pend_it.assign((size_t)nsteps, 0); h->pend_ratio.assign((size_t)nsteps, 0.0);
    long long total = 0; int done = 0, st = FCG_OK;
    for (int step = 0; step < nsteps; ++step) {
        int it = 0; double rr = 0.0;
        if ((st = fcg_force_rhs(h, k, D, b)) < 0) break;
        st = use_pcg ? fcg_pcg_solve(h, k, b, u, tol, maxit, &it, &rr) : fcg_solve(h, k, b, u, tol, maxit, &it, &rr);
        total += h->launches + 2;
        if (st < 0) break;
        if ((st = fcg_force_from_displacement(h, k, D, u, frc)) < 0) break;
        long long idx = -1; double ratio = 0.0;
        st = fcg_force_break_step(h, k, frc, t, &idx, &ratio);
        total += h->launches;
        if (st < 0) break;
        h->pend_idx[step] = idx; h->pend_it[step] = it; h->pend_ratio[step] = ratio;
        ++done; st = FCG_OK;
    }
    h->pend_nsteps = nsteps; h->pend_done = done; h->pend_status = st; h->launches = total;
    return st < 0 ? st : FCG_OK;
}

int fcg_force_fracture_displacement_end(fcg_handle h, long long* index_host, int* iters_host, double* ratio_host, int* steps_done_host) {
    if (!h || !index_host || !iters_host) return fail(h, FCG_INVALID_ARG, "bad argument");
    FCG_ENTER_END(h);
    if (h->pend_nsteps < 0 || h->pend_kind != 1) return fail(h, FCG_INVALID_ARG, "no quasi-static loop of this kind pending on this handle");
    h->pend_nsteps = -1; h->pend_kind = 0;
    if (h->pend_async) {
        h->pend_async = false;
        FCG_CK(h, cudaStreamSynchronize(h->stream));
        const int done = h->h_sc->steps_done;
        if (done > 0) {
            FCG_CK(h, cudaMemcpyAsync(index_host, h->frac_idx, (size_t)done * sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
            FCG_CK(h, cudaMemcpyAsync(iters_host, h->frac_it, (size_t)done * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
            if (ratio_host) FCG_CK(h, cudaMemcpyAsync(ratio_host, h->frac_ratio, (size_t)done * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
            FCG_CK(h, cudaStreamSynchronize(h->stream));
        }
        if (steps_done_host) *steps_done_host = done;
        if (h->h_sc->status == FCG_CUDA_ERROR) h->err = "fused quasi-static loop: grid barrier timed out";
        return h->h_sc->status < 0 ? h->h_sc->status : FCG_OK;
    }
    for (int i = 0; i < h->pend_done; ++i) {
        index_host[i] = h->pend_idx[(size_t)i]; iters_host[i] = h->pend_it[(size_t)i];
        if (ratio_host) ratio_host[i] = h->pend_ratio[(size_t)i];
    }
    if (steps_done_host) *steps_done_host = h->pend_done;
    return h->pend_status;
}

int fcg_force_fracture_displacement(fcg_handle h, void* k, double D, void* u, const void* t, int nsteps, double tol, int maxit, int use_pcg,
                                    long long* index_host, int* iters_host, double* ratio_host, int* steps_done_host) {
    if (!index_host || !iters_host) return fail(h, FCG_INVALID_ARG, "bad argument");
    if (steps_done_host) *steps_done_host = 0;
    const int st = fcg_force_fracture_displacement_begin(h, k, D, u, t, nsteps, tol, maxit, use_pcg);
    if (st < 0 && (!h || h->pend_nsteps < 0)) return st;
    return fcg_force_fracture_displacement_end(h, index_host, iters_host, ratio_host, steps_done_host);
}

// ---- slab-decomposed CG over several ranks
int fcg_slab_shape_of(int L, fcg_dtype dt, int nranks, int rank, fcg_slab_shape* out) { return slab_shape(L, dt, nranks, rank, out); }

#define FCG_SLAB_ENTER(h)                                                                              \
    if (!(h)) return FCG_INVALID_ARG;                                                                  \
    FCG_ENTER(h);                                                                                      \
    if ((h)->slab_G < 1) return fail((h), FCG_INVALID_ARG, "fcg_slab_configure has not been called")

int fcg_slab_configure(fcg_handle h, int nranks, int rank) {
    if (!h) return FCG_INVALID_ARG;
    FCG_ENTER(h);
    if (!h->v2()) return fail(h, FCG_UNSUPPORTED, "slab decomposition needs the pipelined engine (L >= 256)");
    fcg_slab_shape sh;
    const int st = slab_shape(h->L, h->dtype, nranks, rank, &sh);
    if (st != FCG_OK) return fail(h, st, "slab decomposition: nranks must divide the column blocks L / (2 NB) and the row pairs L / 2");
    h->slab_G = nranks; h->slab_rank = rank; h->slab_Al = sh.row_pairs_local; h->slab_MBl = sh.column_blocks_local; h->slab_bytes = sh.buffer_bytes;
    // This first slice keeps the full-size workspace of fcg_create: S (T2 of the own rows, N w / G bytes) in the T2 region, the exchange
    // buffer R in z, the vector only preconditioned CG uses.  The column pass works on R in place through a 5-D tensor map.
    h->slab_S = h->lay.Tb;
    h->slab_R = h->lay.z;
    h->slab_boxa = h->tab->v2_abox < sh.row_pairs_local ? h->tab->v2_abox : sh.row_pairs_local;
    return slab_tensor_maps(h);
}

// Peer mode: the exchange fused into the passes.  peer_send[g] / peer_recv[g] = device addresses, valid on THIS device, of rank g's
// S and R buffers (its own included): pointers of the other handles for logical ranks on one device, cudaIpcOpenMemHandle'd
// mappings or peer-enabled addresses over NVLink for one process per GPU.
int fcg_slab_set_peers(fcg_handle h, void* const* peer_send_host, void* const* peer_recv_host) {
    FCG_SLAB_ENTER(h);
    if (h->slab_peer_maps) { cudaFree(h->slab_peer_maps); h->slab_peer_maps = nullptr; }
    if (!peer_send_host || !peer_recv_host) return FCG_OK;           // back to the all-to-all mode
    if (h->slab_G > 16) return fail(h, FCG_UNSUPPORTED, "peer mode supports up to 16 ranks");
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return fail(h, FCG_UNSUPPORTED, "cuTensorMapEncodeTiled unavailable");
    }
    auto enc = reinterpret_cast<EncodeTiledFn>(fn);
    const cuuint64_t L = (cuuint64_t)h->L, w = (cuuint64_t)h->w, NB = (cuuint64_t)h->tab->v2_nb, Al = (cuuint64_t)h->slab_Al;
    const CUtensorMapDataType dtp = h->dtype == FCG_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    std::vector<CUtensorMap> maps((size_t)h->slab_G);
    for (int g = 0; g < h->slab_G; ++g) {
        if (!peer_send_host[g] || !peer_recv_host[g] || (reinterpret_cast<uintptr_t>(peer_send_host[g]) & 127u) || (reinterpret_cast<uintptr_t>(peer_recv_host[g]) & 127u))
            return fail(h, FCG_INVALID_ARG, "peer buffers must be non-null and 128-byte aligned");
        // rank g's T2 (rows side): d0 = 2 complex of one row pair, d1 = column in line, d2 = ITS local row pair, d3 = column block (all of them)
        const cuuint64_t gdim[4] = {4, NB, Al, L / (2 * NB)};
        const cuuint64_t gstride[3] = {4 * w, 4 * NB * w, Al * 4 * NB * w};
        const cuuint32_t box[4] = {4u, 1u, (cuuint32_t)h->slab_boxa, 1u};
        const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
        if (enc(&maps[(size_t)g], dtp, 4, peer_send_host[g], gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return fail(h, FCG_CUDA_ERROR, "cuTensorMapEncodeTiled (peer T2) failed");
        h->slab_peerR[g] = peer_recv_host[g];
    }
    FCG_CK(h, cudaMalloc((void**)&h->slab_peer_maps, maps.size() * sizeof(CUtensorMap)));
    FCG_CK(h, cudaMemcpyAsync(h->slab_peer_maps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, h->stream));
    FCG_CK(h, cudaStreamSynchronize(h->stream));
    return FCG_OK;
}

// One process per GPU: the exchange buffers live in the caller's workspace, possibly inside a larger allocation (torch's caching
// allocator), so what is exported is the IPC handle of the ALLOCATION plus the two offsets into it.
struct SlabIpcBlob { cudaIpcMemHandle_t handle; unsigned long long off_send, off_recv; };
static_assert(sizeof(SlabIpcBlob) == FCG_SLAB_IPC_BYTES, "fcg_slab_ipc blob size");

int fcg_slab_ipc_export(fcg_handle h, void* blob_host) {
    FCG_SLAB_ENTER(h);
    if (!blob_host) return fail(h, FCG_INVALID_ARG, "null argument");
    typedef CUresult (*GetRange)(CUdeviceptr*, size_t*, CUdeviceptr);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return fail(h, FCG_UNSUPPORTED, "cuMemGetAddressRange unavailable");
    }
    CUdeviceptr base = 0; size_t size = 0;
    if (reinterpret_cast<GetRange>(fn)(&base, &size, (CUdeviceptr)(uintptr_t)h->ws) != CUDA_SUCCESS) return fail(h, FCG_CUDA_ERROR, "cuMemGetAddressRange failed");
    SlabIpcBlob b{};
    FCG_CK(h, cudaIpcGetMemHandle(&b.handle, (void*)(uintptr_t)base));
    const unsigned long long off = (unsigned long long)((uintptr_t)h->ws - (uintptr_t)base);
    b.off_send = off + h->slab_S; b.off_recv = off + h->slab_R;
    std::memcpy(blob_host, &b, sizeof(b));
    return FCG_OK;
}

int fcg_slab_ipc_open(fcg_handle h, const void* blobs_host) {
    FCG_SLAB_ENTER(h);
    if (!blobs_host) return fail(h, FCG_INVALID_ARG, "null argument");
    if (h->slab_G > 16) return fail(h, FCG_UNSUPPORTED, "peer mode supports up to 16 ranks");
    void* send[16]; void* recv[16];
    for (int g = 0; g < h->slab_G; ++g) {
        if (g == h->slab_rank) { send[g] = h->ws + h->slab_S; recv[g] = h->ws + h->slab_R; continue; }
        SlabIpcBlob b;
        std::memcpy(&b, static_cast<const char*>(blobs_host) + (size_t)g * sizeof(SlabIpcBlob), sizeof(b));
        if (!h->slab_ipc_base[g]) FCG_CK(h, cudaIpcOpenMemHandle(&h->slab_ipc_base[g], b.handle, cudaIpcMemLazyEnablePeerAccess));
        send[g] = static_cast<char*>(h->slab_ipc_base[g]) + b.off_send; recv[g] = static_cast<char*>(h->slab_ipc_base[g]) + b.off_recv;
    }
    return fcg_slab_set_peers(h, send, recv);
}

int fcg_slab_buffers(fcg_handle h, size_t* send_offset, size_t* recv_offset, size_t* bytes) {
    FCG_SLAB_ENTER(h);
    if (!send_offset || !recv_offset || !bytes) return fail(h, FCG_INVALID_ARG, "null argument");
    *send_offset = h->slab_S; *recv_offset = h->slab_R; *bytes = h->slab_bytes;
    return FCG_OK;
}

int fcg_slab_setup(fcg_handle h, double tol, int maxit) {
    FCG_SLAB_ENTER(h);
    if (!(tol >= 0.0) || maxit < 0) return fail(h, FCG_INVALID_ARG, "tol must be >= 0 and maxit >= 0");
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    h->launches = 0;
    SetupArgs sa{tol, maxit, 0, 0ULL, 0};
    cg_setup_kernel<<<1, 32, 0, h->stream>>>(h->sc(), sa); ++h->launches;
    FCG_CK(h, cudaGetLastError());
    return FCG_OK;
}

int fcg_slab_rows_fwd(fcg_handle h, int cg, void* xu) {
    FCG_SLAB_ENTER(h);
    if (!xu) return fail(h, FCG_INVALID_ARG, "null argument");
    const int mode = cg ? ROWF_CG : ROWF_PLAIN;
    return h->dtype == FCG_F64 ? slab_rows_fwd_impl<double>(h, mode, xu) : slab_rows_fwd_impl<float>(h, mode, xu);
}

int fcg_slab_cols(fcg_handle h) {
    FCG_SLAB_ENTER(h);
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    return h->dtype == FCG_F64 ? slab_cols_impl<double>(h) : slab_cols_impl<float>(h);
}

int fcg_slab_cols_energy(fcg_handle h, void* xch) {
    FCG_SLAB_ENTER(h);
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    if (!xch) return fail(h, FCG_INVALID_ARG, "null argument");
    return h->dtype == FCG_F64 ? slab_cols_impl<double>(h, xch) : slab_cols_impl<float>(h, xch);
}

int fcg_slab_kpp0(fcg_handle h, const void* k, void* xch) {
    FCG_SLAB_ENTER(h);
    if (!k || !xch) return fail(h, FCG_INVALID_ARG, "null argument");
    return h->dtype == FCG_F64 ? slab_kpp0_impl<double>(h, k, xch) : slab_kpp0_impl<float>(h, k, xch);
}

int fcg_slab_rows_inv(fcg_handle h, int residual, const void* k, const void* u, const void* f, void* xch) {
    FCG_SLAB_ENTER(h);
    if (residual < 0 || residual > 2) return fail(h, FCG_INVALID_ARG, "residual must be 0, 1 or 2");
    if (!k || !xch || (residual == 1 && (!u || !f))) return fail(h, FCG_INVALID_ARG, "null argument");
    const int mode = residual == 1 ? ROWI_RESID : residual == 2 ? ROWI_CGF : ROWI_CG;
    return h->dtype == FCG_F64 ? slab_rows_inv_impl<double>(h, mode, k, u, f, xch) : slab_rows_inv_impl<float>(h, mode, k, u, f, xch);
}

int fcg_slab_update_r(fcg_handle h, void* xch) {
    FCG_SLAB_ENTER(h);
    if (!xch) return fail(h, FCG_INVALID_ARG, "null argument");
    return h->dtype == FCG_F64 ? slab_update_r_impl<double>(h, xch) : slab_update_r_impl<float>(h, xch);
}

int fcg_slab_scalar(fcg_handle h, int what, const void* xch) {
    FCG_SLAB_ENTER(h);
    if (!xch || what < 0 || what > 5) return fail(h, FCG_INVALID_ARG, "bad argument");
    slab_scalar_kernel<<<1, 32, 0, h->stream>>>(h->sc(), what, (const double*)xch); ++h->launches;
    FCG_CK(h, cudaGetLastError());
    return FCG_OK;
}

int fcg_slab_finish(fcg_handle h, void* u) {
    FCG_SLAB_ENTER(h);
    if (!u) return fail(h, FCG_INVALID_ARG, "null argument");
    return h->dtype == FCG_F64 ? slab_finish_impl<double>(h, u) : slab_finish_impl<float>(h, u);
}

int fcg_slab_poll(fcg_handle h, int* done_host, int* iters_host, double* rel_residual_host, int* status_host) {
    FCG_SLAB_ENTER(h);
    FCG_CK(h, cudaMemcpyAsync(h->h_sc, h->sc(), sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
    FCG_CK(h, cudaStreamSynchronize(h->stream));
    if (done_host) *done_host = h->h_sc->done;
    if (iters_host) *iters_host = h->h_sc->it;
    if (rel_residual_host) *rel_residual_host = h->h_sc->relres;
    if (status_host) *status_host = h->h_sc->status;
    if (h->h_sc->timeout) return fail(h, FCG_CUDA_ERROR, "a pipelined pass gave up waiting on an mbarrier");
    return FCG_OK;
}

// ---- break step without any allocation (include/fcg.h: fcg_break_step_static) -------------------------------------------------
// Scratch of break_argmax_kernel -- one (ratio, index) partial per CTA and the arrival ticket -- in static device memory, so that
// callers who may not allocate (stream capture, serving loops) can run the break step with no handle, workspace or cudaMalloc.
// Every GPU that loads libfcg.so holds these FCG_BREAK_STATIC_SCRATCH_BYTES until the process exits.  In HOST code the array's name
// is only a stand-in: the device address comes from cudaGetSymbolAddress, once per device, with that device current.
}  // extern "C"  (the array, the per-device table and the typed launcher have C++ linkage)
namespace {
constexpr size_t BRK_PR_OFF = 0, BRK_PI_OFF = VEC_BLOCKS_MAX * sizeof(double),
                 BRK_TICKET_OFF = (VEC_BLOCKS_MAX * (sizeof(double) + sizeof(long long)) + 255) / 256 * 256;
static_assert(BRK_TICKET_OFF + 256 == FCG_BREAK_STATIC_SCRATCH_BYTES, "static break-step scratch layout");
}
static __device__ __align__(256) unsigned char g_break_static_scratch[FCG_BREAK_STATIC_SCRATCH_BYTES];
namespace {
constexpr int MAX_DEVICES = 64;
std::atomic<unsigned char*> g_break_static_ptr[MAX_DEVICES];       // device address of the array, per device ordinal (nullptr: not asked yet)
thread_local std::string g_static_err;
int static_fail(int code, const std::string& msg) { g_static_err = msg; return code; }

template <typename T>
cudaError_t break_static_launch(unsigned char* scratch, long long n, void* k, const void* u, const void* t, void* result_dev, cudaStream_t st) {
    // grid as fcg_break_step's: whole unrolled trips of 4 vectors per thread, at most VEC_BLOCKS_MAX CTAs (= the partials' capacity)
    const size_t nvec = (size_t)n / Vec<T>::W, per = 256 * 4;
    size_t b = (nvec + per - 1) / per;
    if (b > (size_t)VEC_BLOCKS_MAX) {
        const size_t trips = (nvec + (size_t)VEC_BLOCKS_MAX * per - 1) / ((size_t)VEC_BLOCKS_MAX * per);
        b = (nvec + per * trips - 1) / (per * trips);
    }
    if (b < 1) b = 1;
    if (b > (size_t)VEC_BLOCKS_MAX) b = VEC_BLOCKS_MAX;
    // the array keeps the last call's contents: the ticket must start at zero (a finished call leaves it there; a call that was
    // aborted may not), the partials are overwritten before they are read
    cudaError_t e = cudaMemsetAsync(scratch + BRK_TICKET_OFF, 0, 2 * sizeof(unsigned int), st);     // ticket + the screen's running maximum
    if (e != cudaSuccess) return e;
    break_argmax_kernel<T><<<(unsigned)b, 256, 0, st>>>((T*)k, (const T*)u, (const T*)t, n, reinterpret_cast<double*>(scratch + BRK_PR_OFF),
                                                        reinterpret_cast<long long*>(scratch + BRK_PI_OFF),
                                                        reinterpret_cast<unsigned int*>(scratch + BRK_TICKET_OFF),
                                                        static_cast<BreakResult*>(result_dev), (T*)nullptr);
    return cudaGetLastError();
}
}  // namespace

extern "C" {

const char* fcg_static_last_error(void) { return g_static_err.c_str(); }

int fcg_break_step_static(fcg_dtype dt, long long n, void* k, const void* u, const void* t, void* result_dev, void* cuda_stream) {
    static_assert(sizeof(BreakResult) == sizeof(fcg_break_result), "fcg_break_result layout");
    if (dt != FCG_F32 && dt != FCG_F64) return static_fail(FCG_INVALID_ARG, "dtype must be FCG_F32 or FCG_F64");
    if (!k || !u || !t || !result_dev) return static_fail(FCG_INVALID_ARG, "null argument");
    if (n < 1) return static_fail(FCG_INVALID_ARG, "n must be >= 1");
    if (n > FCG_BREAK_STATIC_MAX_N)
        return static_fail(FCG_UNSUPPORTED, "n = " + std::to_string(n) + " exceeds FCG_BREAK_STATIC_MAX_N = " + std::to_string((long long)FCG_BREAK_STATIC_MAX_N) +
                                                " (the static scratch is sized for that; use fcg_break_step with a handle beyond it)");
    if (misaligned(k) || misaligned(u) || misaligned(t) || (reinterpret_cast<uintptr_t>(result_dev) & 7u))
        return static_fail(FCG_INVALID_ARG, "k, u, t must be 16-byte aligned, result_dev 8-byte aligned");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) { cudaGetLastError(); return static_fail(FCG_CUDA_ERROR, "no current CUDA device"); }
    unsigned char* scratch = g_break_static_ptr[dev].load(std::memory_order_acquire);
    if (!scratch) {        // set-up, once per device, with that device current: the symbol's DEVICE address (its host-side name is not one)
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_break_static_scratch);
        if (e != cudaSuccess || !p) { cudaGetLastError(); return static_fail(FCG_CUDA_ERROR, std::string("cudaGetSymbolAddress(g_break_static_scratch): ") + cudaGetErrorString(e)); }
        scratch = static_cast<unsigned char*>(p);
        g_break_static_ptr[dev].store(scratch, std::memory_order_release);      // (two threads racing here store the same address)
    }
    const cudaStream_t st = (cudaStream_t)cuda_stream;
    const cudaError_t e = dt == FCG_F64 ? break_static_launch<double>(scratch, n, k, u, t, result_dev, st)
                                        : break_static_launch<float>(scratch, n, k, u, t, result_dev, st);
    if (e != cudaSuccess) return static_fail(FCG_CUDA_ERROR, std::string("fcg_break_step_static: ") + cudaGetErrorString(e));
    return FCG_OK;
}

int fcg_profile_iteration(fcg_handle h, const void* k, const void* f, void* u, int iters, double* ms_host) {
    if (!h || !k || !f || !u || iters < 1 || !ms_host) return fail(h, FCG_INVALID_ARG, "bad argument");
    FCG_ENTER(h);
    if (!h->have_spectrum) return fail(h, FCG_NO_SPECTRUM, "fcg_set_spectrum has not been called");
    return h->dtype == FCG_F64 ? profile_impl<double>(h, k, f, u, iters, ms_host) : profile_impl<float>(h, k, f, u, iters, ms_host);
}

long long fcg_last_launch_count(fcg_handle h) { return h ? h->launches : -1; }

const char* fcg_last_error(fcg_handle h) { return h ? h->err.c_str() : "null handle"; }

}  // extern "C"
