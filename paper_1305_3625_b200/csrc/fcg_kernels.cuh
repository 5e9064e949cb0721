// fcg_kernels.cuh -- __global__ entry points of libfcg.
//   transform passes (templated on plan): row_fwd_kernel, col_kernel, row_inv_kernel, spectrum_prep_kernel
//   BLAS-1 of Listing 2 with device-side reductions and convergence test:
//       cg_setup_kernel, cg_update_r_kernel, cg_finish_kernel
//   break step (BASELINE.json configs[3]): break_argmax_kernel
//   public half-spectrum layout helpers: halfspec_export/import kernels
#pragma once
#include <cuda_runtime.h>
#include "fcg_passes.cuh"
#include "fcg_tma.cuh"

namespace fcg {

constexpr int ST_OK = 0, ST_NOT_CONVERGED = 1, ST_BREAKDOWN = -4;

struct DevRunner {
    template <typename Fn> FCG_HD void operator()(Fn&& f) {
#ifdef __CUDA_ARCH__
        f((int)threadIdx.x);
        __syncthreads();
#else
        (void)f;
#endif
    }
};

#ifdef __CUDACC__
__device__ __forceinline__ void set_cond(const Scalars* sc, bool go) {
    if (sc->use_cond) cudaGraphSetConditional((cudaGraphConditionalHandle)sc->cond, go ? 1u : 0u);
}

// Sum of one double per thread over the CTA, fixed tree (bit-reproducible). Result valid in thread 0.
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* red /* [NV][32] shared */) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int q = 0; q < NV; ++q) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_down_sync(0xffffffffu, v[q], o);
        if (lane == 0) red[q * 32 + w] = v[q];
    }
    __syncthreads();
    if (w == 0) {
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            double x = lane < nw ? red[q * 32 + lane] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
            v[q] = x;
        }
    }
}

// Publish this CTA's partial sums; the last CTA to arrive adds all partials in a fixed order and
// returns true in every one of its threads with the totals in tot[] (valid in thread 0).
template <int NV>
__device__ __forceinline__ bool grid_sum_last(double (&v)[NV], double* partial, unsigned int* ticket,
                                              double* red, double (&tot)[NV]) {
    __shared__ int is_last;
    block_sum<NV>(v, red);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < NV; ++q) partial[(size_t)blockIdx.x * NV + q] = v[q];
        __threadfence();
        const unsigned int t = atomicAdd(ticket, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
#pragma unroll
    for (int q = 0; q < NV; ++q) tot[q] = 0.0;
    for (unsigned int b = threadIdx.x; b < gridDim.x; b += blockDim.x)
#pragma unroll
        for (int q = 0; q < NV; ++q) tot[q] += __ldcg(partial + (size_t)b * NV + q);
    __syncthreads();
    block_sum<NV>(tot, red);
    if (threadIdx.x == 0) *ticket = 0u;
    return true;
}

// ------------------------------------------------------------------------------- transform passes
template <typename T, typename P, int F>
__global__ void __launch_bounds__(F * P::NT) row_fwd_kernel(const RowFwdArgs<T> A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if ((A.mode == ROWF_CG || A.check_done) && A.sc->done) return;
    DevRunner run;
    row_fwd_body<T, P, F>(A, (int)blockIdx.x, reinterpret_cast<cx<T>*>(smem_raw), run);
}

template <typename T, typename P, int COLS>
__global__ void __launch_bounds__(COLS * P::NT) col_kernel(const ColArgs<T> A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (A.sc && A.sc->done) return;
    DevRunner run;
    col_body<T, P, COLS>(A, (int)blockIdx.x, reinterpret_cast<cx<T>*>(smem_raw), run);
}

// scalar step after the residue length r.r is known: count, convergence / maxit, beta.
// PCG keeps rho = r.z: there beta follows from the preconditioner pass (row_inv_reduce_finalize, ROWI_PRECOND).
__device__ __forceinline__ void cg_after_rr(Scalars* sc, double rho_new) {
    const double fn2 = sc->fn2;
    const int it = sc->it + 1;
    sc->it = it;
    if (sqrt(rho_new) <= sc->tol * sqrt(fn2)) { sc->done = 1; sc->status = ST_OK; }
    else if (it >= sc->maxit) { sc->done = 1; sc->status = ST_NOT_CONVERGED; }
    else if (!sc->pcg) sc->beta = rho_new / sc->rho;
    if (sc->pcg) sc->rr = rho_new; else sc->rho = rho_new;
    sc->relres = sqrt(rho_new) / sqrt(fn2);
    set_cond(sc, !sc->done);
}

// Grid-wide reduction of the row pass's partial dot products and the scalar step that follows it:
// search length alpha = rho / p.Ap in the loop, or the initial values after the residual pass.
template <typename T>
__device__ __forceinline__ void row_inv_reduce_finalize(const RowInvArgs<T>& A, double (&acc)[2], double* red) {
    if (A.mode != ROWI_CG && A.mode != ROWI_RESID && A.mode != ROWI_PRECOND && A.mode != ROWI_CGF) return;
    double tot[2];
    if (!grid_sum_last<2>(acc, A.partial, &A.sc->ticket[0], red, tot)) return;
    if (threadIdx.x != 0) return;
    if (A.xch) { A.xch[0] = tot[0]; A.xch[1] = tot[1]; return; }       // slab: this rank's share; the scalar step follows the all-reduce
    Scalars* sc = A.sc;
    if (A.mode == ROWI_CGF) { cg_after_rr(sc, tot[0]); return; }           // fused residual update: r.r is this pass's sum
    if (A.mode == ROWI_CG) {
        const double pq = tot[0];
        sc->pq = pq;
        if (!(pq > 0.0) || !isfinite(pq)) { sc->status = ST_BREAKDOWN; sc->done = 1; sc->alpha = 0.0; }
        else sc->alpha = sc->rho / pq;                                   // search length
    } else if (A.mode == ROWI_PRECOND) {                                 // PCG: rho' = r.z, beta = rho'/rho (first direction: p = z)
        const double rho_new = tot[0];
        if (!(rho_new > 0.0) || !isfinite(rho_new)) { sc->status = ST_BREAKDOWN; sc->done = 1; }
        else { sc->beta = sc->it == 0 ? 0.0 : rho_new / sc->rho; sc->rho = rho_new; }
        set_cond(sc, !sc->done);
    } else {                                                             // set up initial values
        const double rho = tot[0], fn2 = tot[1];
        sc->rho = rho; sc->rr = rho; sc->fn2 = fn2; sc->it = 0; sc->alpha = 0.0; sc->beta = 0.0;
        if (fn2 == 0.0) { sc->zero_u = 1; sc->done = 1; sc->status = ST_OK; sc->rho = 0.0; sc->relres = 0.0; }
        else {
            sc->relres = sqrt(rho) / sqrt(fn2);
            if (sqrt(rho) <= sc->tol * sqrt(fn2)) { sc->done = 1; sc->status = ST_OK; }
            else if (sc->maxit <= 0) { sc->done = 1; sc->status = ST_NOT_CONVERGED; }
        }
        set_cond(sc, !sc->done);
    }
}

template <typename T, typename P, int F>
__global__ void __launch_bounds__(F * P::NT) row_inv_kernel(const RowInvArgs<T> A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[2 * 32];
    if ((A.mode == ROWI_CG || A.mode == ROWI_PRECOND) && A.sc->done) return;
    DevRunner run;
    double acc[2] = {0.0, 0.0};
    row_inv_body<T, P, F>(A, (int)blockIdx.x, reinterpret_cast<cx<T>*>(smem_raw), run, acc);
    row_inv_reduce_finalize<T>(A, acc, red);
}

template <typename T, typename P>
__global__ void spectrum_prep_kernel(const T* __restrict__ s, T* __restrict__ shat, bool colpos) {
    constexpr int L = P::N;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < L * (L / 2); idx += gridDim.x * blockDim.x)
        spectrum_prep_one<T, P>(idx, s, shat, colpos);
}

// Eigenvalues of the spectral preconditioner's inverse: M = kbar I + C  =>  m = 1 / (kbar + s),
// element by element in the working precision (one add, one divide), as the oracle forms it.
template <typename T>
__global__ void __launch_bounds__(256) precond_spectrum_kernel(const T* __restrict__ s, T* __restrict__ m, size_t n, T kbar) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        m[i] = (T)1 / (kbar + s[i]);
}

// ------------------------------------------------------------------------------- CG vector kernels
struct SetupArgs { double tol; int maxit; int use_cond; unsigned long long cond; int pcg; };

#ifdef FCG_MAIN_TU   // non-template kernel: defined in fcg.cu only
__global__ void cg_setup_kernel(Scalars* sc, SetupArgs a) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        sc->rho = 0; sc->pq = 0; sc->alpha = 0; sc->beta = 0; sc->fn2 = 0; sc->relres = 0;
        sc->tol = a.tol; sc->maxit = a.maxit; sc->it = 0; sc->done = 0; sc->status = 0; sc->zero_u = 0;
        sc->use_cond = a.use_cond; sc->cond = a.cond; sc->pcg = a.pcg; sc->rr = 0;
        sc->ticket[0] = sc->ticket[1] = sc->ticket[2] = sc->ticket[3] = 0u;
        sc->kpp = 0; sc->ticket2[0] = sc->ticket2[1] = 0u;
    }
}
#endif

template <typename T> struct Vec;
template <> struct Vec<double> { using type = double2; static constexpr int W = 2; };
template <> struct Vec<float> { using type = float4; static constexpr int W = 4; };

__device__ __forceinline__ void axpy_sq(double2& r, const double2 q, double a, double& acc) {
    r.x = r.x - a * q.x; r.y = r.y - a * q.y;
    acc += r.x * r.x; acc += r.y * r.y;
}
__device__ __forceinline__ void axpy_sq(float4& r, const float4 q, float a, double& acc) {
    r.x = r.x - a * q.x; r.y = r.y - a * q.y; r.z = r.z - a * q.z; r.w = r.w - a * q.w;
    acc += (double)r.x * (double)r.x; acc += (double)r.y * (double)r.y;
    acc += (double)r.z * (double)r.z; acc += (double)r.w * (double)r.w;
}

// residue, residue length (97), update calculation variables (98: beta), check convergence (99)
template <typename T>
__global__ void __launch_bounds__(256) cg_update_r_kernel(T* __restrict__ r, const T* __restrict__ q, size_t nvec,
                                                           double* partial, Scalars* sc, int hints, double* xch = nullptr) {
    __shared__ double red[32];
    using V = typename Vec<T>::type;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");    // programmatic dependent launch (fcg_tma.cuh)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (sc->done) {      // breakdown in this iteration, or (loop mode 1) already finished
        if (blockIdx.x == 0 && threadIdx.x == 0) set_cond(sc, false);
        return;
    }
    const T a = (T)sc->alpha;
    double acc[1] = {0.0};
    // L2 hints (bit 5): q is dead after this pass
    const uint64_t pol_q = (hints & 32) ? tma::policy_evict_first() : tma::policy_evict_normal();
    V* rv = reinterpret_cast<V*>(r);
    const V* qv = reinterpret_cast<const V*>(q);
    // four independent 16-byte loads of r and of q in flight per thread before any use
    constexpr int UN = 4;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + (UN - 1) * stride < nvec; i += UN * stride) {
        V x[UN], y[UN];
#pragma unroll
        for (int c = 0; c < UN; ++c) { x[c] = rv[i + c * stride]; y[c] = tma::ld_hint(qv + i + c * stride, pol_q); }
#pragma unroll
        for (int c = 0; c < UN; ++c) { axpy_sq(x[c], y[c], a, acc[0]); rv[i + c * stride] = x[c]; }
    }
    for (; i < nvec; i += stride) {
        V x = rv[i];
        axpy_sq(x, __ldg(qv + i), a, acc[0]);
        rv[i] = x;
    }
    double tot[1];
    if (!grid_sum_last<1>(acc, partial, &sc->ticket[1], red, tot)) return;
    if (threadIdx.x != 0) return;
    if (xch) { xch[0] = tot[0]; return; }                  // slab: this rank's share of r.r (fcg_slab_scalar after the all-reduce)
    cg_after_rr(sc, tot[0]);
}

// Slab-decomposed CG: the scalar steps of Listing 2 on
// sums that have been all-reduced over the ranks.  Every rank runs this on identical inputs, so alpha, beta, the count and
// the stopping decision are identical everywhere and nothing is broadcast.
//   what = 0: after the residual pass      xch = { r.r, f.f }   -> rho, ||f||^2, early exit
//   what = 1: after the operator           xch = { p.q }        -> alpha (or breakdown)
//   what = 2: after the residual update    xch = { r.r }        -> count, convergence / maxit, beta, rho
#ifdef FCG_MAIN_TU   // non-template kernel: defined in fcg.cu only
__global__ void slab_scalar_kernel(Scalars* sc, int what, const double* xch) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    if (what == 0) {
        const double rho = xch[0], fn2 = xch[1];
        sc->rho = rho; sc->rr = rho; sc->fn2 = fn2; sc->it = 0; sc->alpha = 0.0; sc->beta = 0.0;
        if (fn2 == 0.0) { sc->zero_u = 1; sc->done = 1; sc->status = ST_OK; sc->rho = 0.0; sc->relres = 0.0; }
        else {
            sc->relres = sqrt(rho) / sqrt(fn2);
            if (sqrt(rho) <= sc->tol * sqrt(fn2)) { sc->done = 1; sc->status = ST_OK; }
            else if (sc->maxit <= 0) { sc->done = 1; sc->status = ST_NOT_CONVERGED; }
        }
    } else if (what == 1) {
        if (sc->done) return;
        const double pq = xch[0];
        sc->pq = pq;
        if (!(pq > 0.0) || !isfinite(pq)) { sc->status = ST_BREAKDOWN; sc->done = 1; sc->alpha = 0.0; }
        else sc->alpha = sc->rho / pq;
    } else if (what == 2) {
        if (sc->done) return;
        cg_after_rr(sc, xch[0]);
    } else if (what == 3) {          // spectral search length (DESIGN.md sections 12, 18): start of the recurrence, sum k p^2 with p = r
        sc->kpp = xch[2];
    } else if (what == 4) {          // alpha from the all-reduced spectral sums: p.Ap = sum k p^2 + sum shat |P|^2
        if (sc->done) return;
        const double pq = sc->kpp + xch[0];
        sc->pq = pq;
        if (!(pq > 0.0) || !isfinite(pq)) { sc->status = ST_BREAKDOWN; sc->done = 1; sc->alpha = 0.0; }
        else sc->alpha = sc->rho / pq;
    } else {                         // after the fused last pass: xch = { r'.r', sum k r'^2, sum k r' p }
        if (sc->done) return;
        const double kpp = sc->kpp;
        cg_after_rr(sc, xch[0]);
        if (!sc->done) sc->kpp = xch[1] + 2.0 * sc->beta * xch[2] + sc->beta * sc->beta * kpp;
    }
}
// this rank's share of the spectral half of p.Ap: the column pass's per-column sums, added in a fixed order
__global__ void __launch_bounds__(256) slab_energy_kernel(const double* __restrict__ colsum, int n, double* xch, const Scalars* sc) {
    __shared__ double red[8];
    if (sc->done) return;
    double e = 0.0;
    for (int i = threadIdx.x; i < n; i += 256) e += colsum[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x == 0) {
        e = 0.0;
        for (int w = 0; w < 8; ++w) e += red[w];
        xch[0] = e; xch[1] = 0.0; xch[2] = 0.0; xch[3] = 0.0;
    }
}
#endif

// spectral search length: start value of the recurrence for sum k p^2 -- the first direction is p = r
template <typename T>
__global__ void __launch_bounds__(256) cg_kpp0_kernel(const T* __restrict__ k, const T* __restrict__ r, size_t nvec, double* partial, Scalars* sc,
                                                      double* xch = nullptr) {       // slab: the sum of the own rows goes to xch[2] instead
    __shared__ double red[32];
    using V = typename Vec<T>::type;
    if (sc->done) return;
    double acc[1] = {0.0};
    const V* kv = reinterpret_cast<const V*>(k);
    const V* rv = reinterpret_cast<const V*>(r);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        const V b = __ldg(rv + i);
        const T* bs = reinterpret_cast<const T*>(&b);
        if (k == nullptr) {          // force formulation: unit weights, sum p^2
#pragma unroll
            for (int c = 0; c < Vec<T>::W; ++c) acc[0] += (double)bs[c] * (double)bs[c];
            continue;
        }
        const V a = __ldg(kv + i);
        const T* as = reinterpret_cast<const T*>(&a);
#pragma unroll
        for (int c = 0; c < Vec<T>::W; ++c) acc[0] += (double)as[c] * ((double)bs[c] * (double)bs[c]);
    }
    double tot[1];
    if (!grid_sum_last<1>(acc, partial, &sc->ticket2[0], red, tot)) return;
    if (threadIdx.x == 0) { if (xch) xch[2] = tot[0]; else sc->kpp = tot[0]; }
}

// The force problem through the displacements (reading F7): (K + G^-1) u = K D is fcg_solve / fcg_pcg_solve
// with the spectrum 1 / g and the right-hand side K D; the two element-wise maps around it, one IEEE operation per step.
template <typename T>
__global__ void __launch_bounds__(256) inverse_spectrum_kernel(const T* __restrict__ g, T* __restrict__ s, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) s[i] = (T)1 / g[i];
}
// f = -k (u - D), eq. (1a), as k * (D - u);  b != nullptr: also the right-hand side b = k * D
template <typename T>
__global__ void __launch_bounds__(256) force_from_displacement_kernel(const T* __restrict__ k, const T* __restrict__ u, T* __restrict__ f, size_t n, T D) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) f[i] = k[i] * (D - u[i]);
}
template <typename T>
__global__ void __launch_bounds__(256) scale_kernel(const T* __restrict__ k, T* __restrict__ b, size_t n, T D) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) b[i] = k[i] * D;
}

// Reading F1 checked on the device before a force solve chooses the three-launch iteration: are all k_i in {0, kappa} with kappa > 0,
// and is the start vector zero on the broken bonds?  Doubles >= 0 order like their bit patterns, so max k and min positive k are
// integer atomics: out[0] = bits(max k), out[1] = ~bits(min positive k) (so that a memset to 0 initialises both), out[2] = 1 if any
// k_i is negative or NaN, or f_i != 0 where k_i == 0.
template <typename T>
__global__ void __launch_bounds__(256) force_uniform_kernel(const T* __restrict__ k, const T* __restrict__ f, size_t n, unsigned long long* out) {
    double kmax = 0.0, kmin = INFINITY; unsigned int bad = 0u;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double ki = (double)k[i];
        if (!(ki >= 0.0)) { bad = 1u; continue; }
        if (ki > 0.0) { kmax = fmax(kmax, ki); kmin = fmin(kmin, ki); }
        else if (f[i] != (T)0) bad = 1u;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        kmax = fmax(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
        kmin = fmin(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(out, (unsigned long long)__double_as_longlong(kmax));
        atomicMax(out + 1, ~(unsigned long long)__double_as_longlong(kmin));
        if (bad) atomicOr(out + 2, 1ULL);
    }
}

// last lagged "new x" after the loop has ended; u = 0 when f = 0
template <typename T>
__global__ void __launch_bounds__(256) cg_finish_kernel(T* __restrict__ u, const T* __restrict__ p, size_t nvec, const Scalars* sc) {
    using V = typename Vec<T>::type;
    const int zero = sc->zero_u;
    const T a = (T)sc->alpha;
    if (!zero && a == (T)0) return;
    V* uv = reinterpret_cast<V*>(u);
    const V* pv = reinterpret_cast<const V*>(p);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        V x = uv[i];
        T* xs = reinterpret_cast<T*>(&x);
        if (zero) {
#pragma unroll
            for (int c = 0; c < Vec<T>::W; ++c) xs[c] = (T)0;
        } else {
            const V pp = __ldg(pv + i);
            const T* ps = reinterpret_cast<const T*>(&pp);
#pragma unroll
            for (int c = 0; c < Vec<T>::W; ++c) xs[c] = xs[c] + a * ps[c];
        }
        uv[i] = x;
    }
}

// ------------------------------------------------------------------------------- break step
struct BreakResult { long long index; double ratio; int status; int pad; };

__device__ __forceinline__ bool better(double ra, long long ia, double rb, long long ib) {
    if (ia < 0) return false;
    if (ib < 0) return true;
    return ra > rb || (ra == rb && ia < ib);
}

// Order-preserving key of a float for atomicMax on unsigned: key(a) < key(b) <=> a < b; key 0 lies below every float (the empty maximum)
__device__ __forceinline__ unsigned int float_key(float f) { const unsigned int b = __float_as_uint(f); return (b & 0x80000000u) ? ~b : (b | 0x80000000u); }
__device__ __forceinline__ float key_float(unsigned int k) { return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k); }

// ticket[0]: arrival count of the CTAs;  ticket[1]: key of the grid-wide running maximum of the SCREEN (below); both 0 at launch and
// reset to 0 by the last CTA (the words are part of a 256-byte-aligned scratch block).
//
// The screen.  The rule needs one IEEE double multiply and divide per candidate (~40 fp64-pipe instructions with the conversions:
// 140 us of that pipe at L = 8192 fp32 against 125 us of bytes).  Most candidates are nowhere near the maximum, and that can be
// decided in single precision: a_i = fl32(k_i u_i / t_i) differs from the exact ratio r_i by at most e = 5e-7 relative as long as no
// operand leaves [1e-30, 1e30] (checked; anything outside, NaN, inf takes the exact path) and the quotient is a normal number.  Every
// thread publishes the largest such a_j it has seen among valid candidates (atomicMax on ticket[1]) and skips candidate i when
// a_i < g - |g| 1e-5 for the g it last read: then r_i <= a_i + |a_i| e < a_j - |a_j| e <= r_j (1e-5 > 2 e, either sign; an underflowed
// a_i means |r_i| < 1.2e-38 and is skipped only against g > 2e-30), so i is neither the maximum nor tied with it.  What is
// skipped depends on timing; the result does not: the winner and every candidate tied with it always reach the exact comparison.
template <typename T>
__global__ void __launch_bounds__(256) break_argmax_kernel(T* __restrict__ k, const T* u, const T* __restrict__ t,
                                                            long long n, double* pr, long long* pi, unsigned int* ticket,
                                                            BreakResult* out, T* fzero) {
    // fzero != nullptr: force formulation (reading F2) -- u holds the bond forces, the ratio is f_i / t_i
    // (one IEEE divide), and the broken bond's force is set to zero with its elastic constant (fzero == u)
    __shared__ double sr[32];
    __shared__ long long si[32];
    __shared__ int is_last;
    double br = 0.0; long long bi = -1;
    auto consider = [&](double r, long long i) { if (better(r, i, br, bi)) { br = r; bi = i; } };
    unsigned int* const gkey = ticket + 1;
    float thr = -INFINITY, amax = -INFINITY;          // skip below thr; amax = largest screened value of this thread's valid candidates
    bool have_a = false;
    auto refresh = [&]() {                            // re-read the grid-wide running maximum (relaxed: a stale value only screens less)
        unsigned int g;
        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(g) : "l"(gkey) : "memory");
        if (g == 0u) return;
        const float gm = key_float(g);
        thr = gm == INFINITY ? 3.4028235e38f * (1.0f - 1e-5f) : gm - fabsf(gm) * 1e-5f;
    };
    auto publish = [&]() {
        if (have_a && !(amax < thr)) atomicMax(gkey, float_key(amax));
    };
    // true: candidate i is provably below the maximum (see above); false: take the exact path
    auto screened_out = [&](float kf, float uf, float tf) {
        const float pf = fzero ? uf : kf * uf;
        const float ap = fabsf(pf), at = fabsf(tf);
        if (!(ap > 1e-30f && ap < 1e30f && at > 1e-30f && at < 1e30f)) return false;     // (also NaN)
        const float a = __fdividef(pf, tf);                                                // <= 2 ulp; |tf| < 2^126
        const bool normal = fabsf(a) > 1e-30f;             // (a quotient that underflowed has no relative accuracy, but is known to be tiny)
        if (normal && (!have_a || a > amax)) { amax = a; have_a = true; }                  // only accurate values are published
        return a < thr && (normal || thr > 2e-30f);
    };
    // One sweep over 3 N w bytes: 16-byte loads of k, u, t issued unconditionally, four vectors of each in flight per thread
    // (the scalar form, with u and t loaded behind the k > 0 branch, ran at 2.3 TB/s at L = 2048 fp64 and 1.6 TB/s at L = 8192
    // fp32).  Plain loads, not the read-only path: the last block writes k (and f) at the end.  `better` is a total order, so
    // the order in which candidates are considered does not matter.
    using V = typename Vec<T>::type;
    constexpr int W = Vec<T>::W;
    auto eval = [&](const V& kv, const V& uv, const V& tv, long long i0) {
        const T* ks = reinterpret_cast<const T*>(&kv); const T* us = reinterpret_cast<const T*>(&uv); const T* ts = reinterpret_cast<const T*>(&tv);
#pragma unroll
        for (int c = 0; c < W; ++c) {
            const T ki = ks[c];
            if (!(ki > (T)0)) continue;
            if (screened_out((float)ki, (float)us[c], (float)ts[c])) continue;
            const double load = fzero ? (double)us[c] : (double)ki * (double)us[c];      // l_i = k_i u_i   (one IEEE multiply)
            const double rt = load / (double)ts[c];            // l_i / t_i       (one IEEE divide)
            if (rt != rt) continue;
            consider(rt, i0 + c);
        }
    };
    const V* kvp = reinterpret_cast<const V*>(k); const V* uvp = reinterpret_cast<const V*>(u); const V* tvp = reinterpret_cast<const V*>(t);
    const long long nvec = n / W, stride = (long long)gridDim.x * blockDim.x;
    long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (; v + 3 * stride < nvec; v += 4 * stride) {
        V kk[4], uu[4], tt[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) { kk[c] = kvp[v + c * stride]; uu[c] = uvp[v + c * stride]; tt[c] = tvp[v + c * stride]; }
        refresh();
#pragma unroll
        for (int c = 0; c < 4; ++c) eval(kk[c], uu[c], tt[c], (v + c * stride) * W);
        publish();
    }
    for (; v < nvec; v += stride) {
        const V kk = kvp[v], uu = uvp[v], tt = tvp[v];
        refresh();
        eval(kk, uu, tt, v * W);
        publish();
    }
    for (long long i = nvec * W + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {      // (n not a multiple of W: never for a lattice)
        const T ki = k[i];
        if (!(ki > (T)0)) continue;
        const double rt = (fzero ? (double)u[i] : (double)ki * (double)u[i]) / (double)t[i];
        if (rt != rt) continue;
        consider(rt, i);
    }
    auto warp_red = [&]() {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double r2 = __shfl_down_sync(0xffffffffu, br, o);
            const long long i2 = __shfl_down_sync(0xffffffffu, bi, o);
            consider(r2, i2);
        }
    };
    auto block_red = [&]() {
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        warp_red();
        if (lane == 0) { sr[w] = br; si[w] = bi; }
        __syncthreads();
        if (w == 0) {
            br = lane < (int)(blockDim.x >> 5) ? sr[lane] : 0.0;
            bi = lane < (int)(blockDim.x >> 5) ? si[lane] : -1;
            warp_red();
        }
    };
    block_red();
    if (threadIdx.x == 0) {
        pr[blockIdx.x] = br; pi[blockIdx.x] = bi;
        __threadfence();
        is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    br = 0.0; bi = -1;
    for (unsigned int b = threadIdx.x; b < gridDim.x; b += blockDim.x) consider(__ldcg(pr + b), __ldcg(pi + b));
    __syncthreads();
    block_red();
    if (threadIdx.x == 0) {
        ticket[0] = 0u; ticket[1] = 0u;
        out->index = bi; out->ratio = br; out->status = bi < 0 ? -6 : 0;
        if (bi >= 0) k[bi] = (T)0;
        if (bi >= 0 && fzero) fzero[bi] = (T)0;
    }
}

// ------------------------------------------------------------------------------- force formulation: static kernel
// Real-space Green's function of eq. (1c): G = (1 - nu^2)/(pi E a^2) * integral of 1/r over the a x a square of the
// other bond, in closed form (four-corner sum of x asinh(y/|x|) + y asinh(x/|y|)), minimum-image offsets on the periodic lattice
// (reading F3).  Evaluated in double, rounded once to T.  One thread per offset.
__device__ __forceinline__ double green_corner(double x, double y) { return x * asinh(y / fabs(x)) + y * asinh(x / fabs(y)); }

template <typename T>
__global__ void __launch_bounds__(256) green_function_kernel(T* __restrict__ G, int L, double pref, double a) {
    const double hf = 0.5 * a;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < (long long)L * L; i += (long long)gridDim.x * blockDim.x) {
        const int da = (int)(i / L), db = (int)(i % L);
        const double X = a * (double)(da <= L / 2 ? da : da - L), Y = a * (double)(db <= L / 2 ? db : db - L);
        const double I = green_corner(X + hf, Y + hf) - green_corner(X - hf, Y + hf) - green_corner(X + hf, Y - hf) + green_corner(X - hf, Y - hf);
        G[i] = (T)(pref * I);
    }
}

// s[m][n] = Re X[m][n] over the full L x L plane from the half spectrum X[m][0..L/2] of a real field (X[-m,-n] = conj X[m,n]):
// "the FFT of G is static and performed during initialization"; the imaginary part is dropped like cpyReal does.
template <typename T>
__global__ void __launch_bounds__(256) halfspec_real_expand_kernel(const cx<T>* __restrict__ X, T* __restrict__ s, int L) {
    const int W = L / 2 + 1;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < (long long)L * L; i += (long long)gridDim.x * blockDim.x) {
        const int m = (int)(i / L), n = (int)(i % L);
        s[i] = n <= L / 2 ? X[(size_t)m * W + n].x : X[(size_t)((L - m) % L) * W + (L - n)].x;
    }
}

// ------------------------------------------------------------------------------- public half-spectrum layout
// T2[n][m] (n < L/2, natural m; row 0 = W = Y0 + i YN) <-> X[m][n], n = 0..L/2, row length L/2+1.
template <typename T>
__global__ void halfspec_export_kernel(const cx<T>* __restrict__ T2, cx<T>* __restrict__ X, int L) {
    __shared__ cx<T> tile[32][33];
    const int n0 = blockIdx.x * 32, m0 = blockIdx.y * 32, W = L / 2 + 1;
    for (int j = threadIdx.y; j < 32; j += blockDim.y)
        if (n0 + j < L / 2 && m0 + (int)threadIdx.x < L) tile[j][threadIdx.x] = T2[(size_t)(n0 + j) * L + m0 + threadIdx.x];
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const int m = m0 + j, n = n0 + threadIdx.x;
        if (n > 0 && n < L / 2 && m < L) X[(size_t)m * W + n] = tile[threadIdx.x][j];
    }
    if (blockIdx.x == 0 && threadIdx.y == 0 && m0 + (int)threadIdx.x < L) {        // unpack the n = 0 and n = L/2 columns
        const int m = m0 + threadIdx.x, mm = (L - m) % L;
        const cx<T> a = T2[m], b = T2[mm];
        const T h = (T)0.5;
        X[(size_t)m * W] = mk<T>((a.x + b.x) * h, (a.y - b.y) * h);
        X[(size_t)m * W + L / 2] = mk<T>((a.y + b.y) * h, (b.x - a.x) * h);
    }
}

template <typename T>
__global__ void halfspec_import_kernel(const cx<T>* __restrict__ X, cx<T>* __restrict__ T2, int L) {
    __shared__ cx<T> tile[32][33];
    const int n0 = blockIdx.x * 32, m0 = blockIdx.y * 32, W = L / 2 + 1;
    for (int j = threadIdx.y; j < 32; j += blockDim.y)
        if (m0 + j < L && n0 + (int)threadIdx.x < L / 2) tile[j][threadIdx.x] = X[(size_t)(m0 + j) * W + n0 + threadIdx.x];
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const int n = n0 + j, m = m0 + threadIdx.x;
        if (n > 0 && n < L / 2 && m < L) T2[(size_t)n * L + m] = tile[threadIdx.x][j];
    }
    if (blockIdx.x == 0 && threadIdx.y == 0 && m0 + (int)threadIdx.x < L) {
        const int m = m0 + threadIdx.x;
        const cx<T> x0 = X[(size_t)m * W], xN = X[(size_t)m * W + L / 2];
        T2[m] = mk<T>(x0.x - xN.y, x0.y + xN.x);
    }
}
#endif  // __CUDACC__

}  // namespace fcg
