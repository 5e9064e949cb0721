// tests/emul/emul.cpp -- host replay of libfcg's pass bodies (csrc/fcg_passes.cuh) for CPU-only checks of
// the index algebra: digit reversal, swizzle, two-rows-per-transform packing, the packed n=0/n=L/2 column
// and the fused column pass.  TEST HARNESS ONLY: built by tests/test_host_emulation.py with g++, never part
// of the product library, never used as a fallback.  Each phase of a CTA is executed for tid = 0..NT-1 in
// turn, which is valid because phases are separated by CTA barriers on the device.
#include <cmath>
#include <cstring>
#include <vector>
#include <cuda_runtime.h>
#include "fcg_passes.cuh"
#include "fcg_plans.cuh"

using namespace fcg;

struct HostRunner {
    int nthreads;
    template <typename Fn> void operator()(Fn&& f) { for (int t = 0; t < nthreads; ++t) f(t); }
};

template <typename T, int L>
int run(int what, const T* s, const T* k, const T* x, T* y, T* Tout, int variant)
{
    using P = typename PlanFor<T, L>::type;
    using RS = RowShape<T, P>;
    using CS = ColShape<T, P>;
    const size_t N = (size_t)L * L;
    std::vector<cx<T>> tw(P::TW_TOTAL + 1), Tb(N / 2);
    fill_twiddles<T, P>(tw.data());
    std::vector<T> shat((size_t)(L / 2 + 1) * L);
    for (int idx = 0; idx < L * (L / 2); ++idx) spectrum_prep_one<T, P>(idx, s, shat.data());
    Scalars sc{};
    auto rows = [&](auto V, bool inverse) {
        constexpr int v = decltype(V)::value;
        if constexpr (RS::valid(v)) {
            constexpr int F = RS::F(v);
            std::vector<cx<T>> smem(RS::smem(v) / sizeof(cx<T>));
            HostRunner hr{F * P::NT};
            for (int b = 0; b < L / (2 * F); ++b) {
                if (!inverse) {
                    RowFwdArgs<T> A{}; A.mode = ROWF_PLAIN; A.x = x; A.Tb = Tb.data(); A.tw = tw.data(); A.sc = &sc;
                    row_fwd_body<T, P, F>(A, b, smem.data(), hr);
                } else {
                    RowInvArgs<T> A{}; A.mode = what == 0 ? ROWI_APPLY : ROWI_PLAIN; A.Tb = Tb.data(); A.tw = tw.data();
                    A.k = k; A.v = x; A.out = y; A.scale = (T)(1.0 / ((double)L * L)); A.sc = &sc;
                    double acc[2] = {0, 0};
                    row_inv_body<T, P, F>(A, b, smem.data(), hr, acc);
                }
            }
            return 0;
        }
        return -1;
    };
    auto rows_v = [&](bool inverse) {
        switch (variant) {
            case 0: return rows(std::integral_constant<int, 0>{}, inverse);
            case 1: return rows(std::integral_constant<int, 1>{}, inverse);
            case 2: return rows(std::integral_constant<int, 2>{}, inverse);
            case 3: return rows(std::integral_constant<int, 3>{}, inverse);
        }
        return -1;
    };
    auto cols = [&](int mode) {
        std::vector<cx<T>> smem(CS::smem / sizeof(cx<T>));
        HostRunner hr{CS::COLS * P::NT};
        for (int b = 0; b < (L / 2) / CS::COLS; ++b) {
            ColArgs<T> A{}; A.mode = mode; A.Tb = Tb.data(); A.shat = shat.data(); A.tw = tw.data(); A.sc = nullptr;
            col_body<T, P, CS::COLS>(A, b, smem.data(), hr);
        }
    };
    if (rows_v(false) != 0) return -1;
    if (what == 0) {            // y = k o x + C x
        cols(COL_CONV);
        return rows_v(true);
    }
    if (what == 1) {            // forward transform: Tout[n][m], natural m
        cols(COL_FWD);
        std::memcpy(Tout, Tb.data(), sizeof(cx<T>) * (N / 2));
        return 0;
    }
    // what == 2: round trip through COL_FWD, COL_INV and the plain inverse row pass
    cols(COL_FWD); cols(COL_INV);
    return rows_v(true);
}

template <typename T>
int dispatch(int L, int what, const T* s, const T* k, const T* x, T* y, T* Tout, int variant)
{
    switch (L) {
#define CASE(n) case n: return run<T, n>(what, s, k, x, y, Tout, variant);
        CASE(16) CASE(32) CASE(64) CASE(128) CASE(256) CASE(512) CASE(1024) CASE(2048) CASE(4096) CASE(8192)
#undef CASE
    }
    return -2;
}

extern "C" int emul_run_f64(int L, int what, const double* s, const double* k, const double* x, double* y, double* Tout, int variant)
{ return dispatch<double>(L, what, s, k, x, y, Tout, variant); }
extern "C" int emul_run_f32(int L, int what, const float* s, const float* k, const float* x, float* y, float* Tout, int variant)
{ return dispatch<float>(L, what, s, k, x, y, Tout, variant); }
