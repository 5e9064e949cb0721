// fcg_math.cuh -- complex helpers, in-register radix-2/4/8/16 butterflies, mixed-radix digit
// reversal and the shared-memory swizzle used by every transform pass of libfcg.
//
// Transform convention (include/fcg.h): forward X[k] = sum_j x[j] exp(-2 pi i j k / n),
// DIR = -1; inverse (unnormalised) DIR = +1.
#pragma once
#include <cuda_runtime.h>

#define FCG_HD __host__ __device__ __forceinline__

namespace fcg {

template <typename T> struct Cx;
template <> struct Cx<double> { using type = double2; };
template <> struct Cx<float> { using type = float2; };
template <typename T> using cx = typename Cx<T>::type;

template <typename T> FCG_HD cx<T> mk(T x, T y) { cx<T> r; r.x = x; r.y = y; return r; }
FCG_HD double2 operator+(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
FCG_HD double2 operator-(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
FCG_HD float2 operator+(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
FCG_HD float2 operator-(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

// a * (c + i s)
template <typename C, typename T> FCG_HD C cmul(C a, T c, T s) {
    C r; r.x = a.x * c - a.y * s; r.y = a.x * s + a.y * c; return r;
}
// a * w  and  a * conj(w)
template <typename C> FCG_HD C cmulw(C a, C w) { C r; r.x = a.x * w.x - a.y * w.y; r.y = a.x * w.y + a.y * w.x; return r; }
template <typename C> FCG_HD C cmulwc(C a, C w) { C r; r.x = a.x * w.x + a.y * w.y; r.y = a.y * w.x - a.x * w.y; return r; }
template <int DIR, typename C> FCG_HD C cmul_dir(C a, C w) { return DIR < 0 ? cmulw(a, w) : cmulwc(a, w); }
template <typename C> FCG_HD C cconj(C a) { a.y = -a.y; return a; }
// a * exp(DIR * i * pi/2) : forward (DIR=-1) multiplies by -i, inverse by +i
template <int DIR, typename C> FCG_HD C rot90(C a) {
    C r;
    if (DIR < 0) { r.x = a.y; r.y = -a.x; } else { r.x = -a.y; r.y = a.x; }
    return r;
}
// a * exp(DIR * i * pi/4)
template <int DIR, typename C> FCG_HD C rot45(C a) {
    using T = decltype(a.x);
    const T h = (T)0.70710678118654752440;
    C r;
    if (DIR < 0) { r.x = (a.x + a.y) * h; r.y = (a.y - a.x) * h; }
    else         { r.x = (a.x - a.y) * h; r.y = (a.x + a.y) * h; }
    return r;
}
// a * exp(DIR * i * 3 pi/4)
template <int DIR, typename C> FCG_HD C rot135(C a) {
    using T = decltype(a.x);
    const T h = (T)0.70710678118654752440;
    C r;
    if (DIR < 0) { r.x = (a.y - a.x) * h; r.y = -(a.x + a.y) * h; }
    else         { r.x = -(a.x + a.y) * h; r.y = (a.x - a.y) * h; }
    return r;
}

// ---- in-register DFTs: a[u] <- sum_t a[t] exp(DIR * 2 pi i t u / R), outputs in natural order ------
template <int DIR, typename C> FCG_HD void dft2(C (&a)[2]) { C t = a[0]; a[0] = t + a[1]; a[1] = t - a[1]; }

template <int DIR, typename C> FCG_HD void dft4(C (&a)[4]) {
    C t0 = a[0] + a[2], t1 = a[0] - a[2], t2 = a[1] + a[3], t3 = rot90<DIR>(a[1] - a[3]);
    a[0] = t0 + t2; a[2] = t0 - t2; a[1] = t1 + t3; a[3] = t1 - t3;
}

template <int DIR, typename C> FCG_HD void dft8(C (&a)[8]) {
    C e[4] = {a[0], a[2], a[4], a[6]}, o[4] = {a[1], a[3], a[5], a[7]};
    dft4<DIR>(e); dft4<DIR>(o);
    o[1] = rot45<DIR>(o[1]); o[2] = rot90<DIR>(o[2]); o[3] = rot135<DIR>(o[3]);
#pragma unroll
    for (int u = 0; u < 4; ++u) { a[u] = e[u] + o[u]; a[u + 4] = e[u] - o[u]; }
}

template <int DIR, typename C> FCG_HD void dft16(C (&a)[16]) {
    using T = decltype(a[0].x);
    C e[8], o[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) { e[u] = a[2 * u]; o[u] = a[2 * u + 1]; }
    dft8<DIR>(e); dft8<DIR>(o);
    const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173;   // cos, sin of pi/8
    const T sg = (T)DIR;                                                      // sign of the imaginary part
    o[1] = cmul(o[1], c1, sg * s1);
    o[2] = rot45<DIR>(o[2]);
    o[3] = cmul(o[3], s1, sg * c1);
    o[4] = rot90<DIR>(o[4]);
    o[5] = cmul(o[5], -s1, sg * c1);
    o[6] = rot135<DIR>(o[6]);
    o[7] = cmul(o[7], -c1, sg * s1);
#pragma unroll
    for (int u = 0; u < 8; ++u) { a[u] = e[u] + o[u]; a[u + 8] = e[u] - o[u]; }
}

template <int R, int DIR, typename C> FCG_HD void dftR(C (&a)[R]) {
    if constexpr (R == 2) dft2<DIR>(a);
    else if constexpr (R == 4) dft4<DIR>(a);
    else if constexpr (R == 8) dft8<DIR>(a);
    else if constexpr (R == 16) dft16<DIR>(a);
    else static_assert(R == 2 || R == 4 || R == 8 || R == 16, "unsupported radix");
}

constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v >> 1); }

// ---- transform plan: n = R1*R2*R3*R4 (unused radices = 1), decimation in frequency --------------
// Stage s works on sub-blocks of length m_s = n / (R1..R_{s-1}):
//     b_u = sum_t x[base + j + t*m_s/R_s] w_Rs^{t u};   x[base + u*m_s/R_s + j] = b_u * w_{m_s}^{j u}
// After the last stage position pos = sum_s u_s * (m_s/R_s) holds X[kappa], kappa = u_1 + R1 u_2 + R1 R2 u_3 + ..
// The inverse runs the adjoint stages in reverse order (decimation in time), so a forward followed by
// an inverse needs no reordering pass at all.
template <int N_, int R1_, int R2_, int R3_, int R4_>
struct Plan {
    static constexpr int N = N_, R1 = R1_, R2 = R2_, R3 = R3_, R4 = R4_;
    static_assert(R1_ * R2_ * R3_ * R4_ == N_, "radices must multiply to N");
    static constexpr int S = (R4_ > 1) ? 4 : (R3_ > 1) ? 3 : (R2_ > 1) ? 2 : 1;
    static constexpr int RMAX = (R1_ > R2_ ? R1_ : R2_) > (R3_ > R4_ ? R3_ : R4_) ? (R1_ > R2_ ? R1_ : R2_) : (R3_ > R4_ ? R3_ : R4_);
    static constexpr int NT = N_ / RMAX;                        // threads per transform
    static constexpr int RLAST = (S == 4) ? R4_ : (S == 3) ? R3_ : (S == 2) ? R2_ : R1_;
    static constexpr int radix(int s) { return s == 1 ? R1_ : s == 2 ? R2_ : s == 3 ? R3_ : R4_; }
    static constexpr int prefix(int s) { return s == 1 ? 1 : s == 2 ? R1_ : s == 3 ? R1_ * R2_ : R1_ * R2_ * R3_; }  // R1..R_{s-1}
    static constexpr int mlen(int s) { return N_ / prefix(s); }                                                        // m_s
    // Per-stage twiddle tables, laid out [u-1][j] (u = 1..R-1, j < Q = m_s/R_s) so that consecutive threads
    // (consecutive j) read consecutive entries:  tws[tw_off(s) + (u-1)*Q + j] = exp(-2 pi i j u / m_s).
    static constexpr int tw_count(int s) { return s >= S ? 0 : (radix(s) - 1) * (mlen(s) / radix(s)); }
    static constexpr int tw_off(int s) { return s <= 1 ? 0 : tw_off(s - 1) + tw_count(s - 1); }
    static constexpr int TW_TOTAL = tw_off(S);
    // The spectrum is stored transposed with respect to the last stage's butterflies: position e = g*RLAST + u
    // lives at u*(N/RLAST) + g, so consecutive threads (consecutive g) read consecutive entries.
    static FCG_HD int shat_index(int e) { return (e % RLAST) * (N_ / RLAST) + e / RLAST; }
    // frequency kappa -> position
    static FCG_HD int pos_of(int kappa) {
        int u1 = kappa % R1_, r = kappa / R1_;
        int p = u1 * (N_ / R1_);
        if (S >= 2) { int u2 = r % R2_; r /= R2_; p += u2 * (N_ / (R1_ * R2_)); }
        if (S >= 3) { int u3 = r % R3_; r /= R3_; p += u3 * (N_ / (R1_ * R2_ * R3_)); }
        if (S >= 4) { p += r; }
        return p;
    }
    // position -> frequency
    static FCG_HD int freq_of(int p) {
        int u1 = p / (N_ / R1_); p %= (N_ / R1_);
        int k = u1;
        if (S >= 2) { int u2 = p / (N_ / (R1_ * R2_)); p %= (N_ / (R1_ * R2_)); k += R1_ * u2; }
        if (S >= 3) { int u3 = p / (N_ / (R1_ * R2_ * R3_)); p %= (N_ / (R1_ * R2_ * R3_)); k += R1_ * R2_ * u3; }
        if (S >= 4) { k += R1_ * R2_ * R3_ * p; }
        return k;
    }
};

// Shared-memory swizzle (element units, W = elements per 128 B).  Keeps every stage's accesses spread
// over all banks: stride-1 runs stay within an aligned group, and the last stage's stride-RLAST
// pattern is de-conflicted by XOR-ing the group index into the low bits.
template <typename T, int RLAST> struct Swz {
    static constexpr int W = 128 / (2 * (int)sizeof(T));
    static constexpr int SH = ilog2(W) > ilog2(RLAST) ? ilog2(W) : ilog2(RLAST);
    static constexpr int MASK = (W < RLAST ? W : RLAST) - 1;
    static FCG_HD int at(int e) { return e ^ ((e >> SH) & MASK); }
};

}  // namespace fcg
