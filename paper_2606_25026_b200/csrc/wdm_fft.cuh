// wdm_fft.cuh -- register-resident small DFTs and the shared-memory line-FFT stages.
//
// Every 1-D transform on the hot path is a "forward . pointwise multiply . inverse" sandwich along one
// grid axis (Eq. 18(b),(c): F^-1{ e^{-i eps k^2/2} F{psi} },  F^-1{ -4 pi/k^2 F{rho} }).  That is
// why the forward transform is decimation-in-frequency (natural order in, digit-reversed out) and the
// inverse is its exact adjoint, decimation-in-time (digit-reversed in, natural out): both run IN PLACE on a
// tile of W lines x N points held in shared memory, with no reordering pass, and the pointwise tables are
// simply stored in digit-reversed ("position") order.
//
// A line of N = RA * RB * RM points is transformed by at most three levels of register radix-R
// butterflies (R <= 32): level A (stride N/RA), optional level B, and the middle level RM whose forward and
// inverse butterflies fuse around the multiply without leaving registers.  Tile element (row j, line l)
// lives at smem[j * RS + l]; a half-warp always touches one whole row, so any butterfly stride is free
// of bank conflicts.
//
// The arithmetic here is plain C++ (WDM_HD = __host__ __device__), so the host-side plan code can share the
// digit-reversal helpers; the product only ever runs the sm_100a build.
#pragma once

#include <stdint.h>

#if defined(__CUDACC__)
#define WDM_HD __host__ __device__ __forceinline__
#else
#define WDM_HD inline __attribute__((always_inline))
#endif

namespace wdm {

template <typename T>
struct alignas(2 * sizeof(T)) cx {
    T x, y;
};

template <typename T> WDM_HD cx<T> mk(T a, T b) { cx<T> r; r.x = a; r.y = b; return r; }
template <typename T> WDM_HD cx<T> cadd(cx<T> a, cx<T> b) { return mk<T>(a.x + b.x, a.y + b.y); }
template <typename T> WDM_HD cx<T> csub(cx<T> a, cx<T> b) { return mk<T>(a.x - b.x, a.y - b.y); }
#if defined(__CUDA_ARCH__) && __CUDA_ARCH__ >= 1000 && !defined(WDM_NO_PACKED_ADD)
// sm_100 packed single precision: one issue slot for a complex add
__device__ __forceinline__ cx<float> cadd(cx<float> a, cx<float> b)
{
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(*reinterpret_cast<unsigned long long *>(&a)), "l"(*reinterpret_cast<unsigned long long *>(&b)));
    return *reinterpret_cast<cx<float> *>(&r);
}
__device__ __forceinline__ cx<float> csub(cx<float> a, cx<float> b)
{
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(*reinterpret_cast<unsigned long long *>(&a)), "l"(*reinterpret_cast<unsigned long long *>(&b)));
    return *reinterpret_cast<cx<float> *>(&r);
}
#endif
// a * b
template <typename T> WDM_HD cx<T> cmul(cx<T> a, cx<T> b) { return mk<T>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// a * conj(b)
template <typename T> WDM_HD cx<T> cmulc(cx<T> a, cx<T> b) { return mk<T>(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
template <typename T> WDM_HD cx<T> cscale(cx<T> a, T s) { return mk<T>(a.x * s, a.y * s); }
template <typename T> WDM_HD cx<T> cconj(cx<T> a) { return mk<T>(a.x, -a.y); }

// ---------------------------------------------------------------- compile-time loops

template <int I> struct ic { static constexpr int value = I; };

template <int B, int E, class F>
WDM_HD void static_for(F &&f)
{
    if constexpr (B < E) {
        f(ic<B>{});
        static_for<B + 1, E>(f);
    }
}

constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n / 2); }
constexpr int brev(int x, int R)
{
    int r = 0;
    for (int b = 1; b < R; b <<= 1) { r = (r << 1) | (x & 1); x >>= 1; }
    return r;
}

// cos(2 pi j / 32), j = 0..8, to full double precision
constexpr double kCos32[9] = {1.0,
                              0.98078528040323044912618223613424,
                              0.92387953251128675612818318939679,
                              0.83146961230254523707878837761791,
                              0.70710678118654752440084436210485,
                              0.55557023301960222474283081394853,
                              0.38268343236508977172845998403040,
                              0.19509032201612826784828486847702,
                              0.0};
constexpr double cos32(int j)
{
    j &= 31;
    if (j > 16) j = 32 - j;
    return j <= 8 ? kCos32[j] : -kCos32[16 - j];
}
constexpr double sin32(int j) { return cos32(j - 8); }

// d * omega_M^I with omega_M = exp(-2 pi i / M), I a compile-time constant, 0 <= I < M/2, M | 32
template <typename T, int M, int I>
WDM_HD cx<T> mul_w(cx<T> d)
{
    if constexpr (I == 0) return d;
    else if constexpr (4 * I == M) return mk<T>(d.y, -d.x);
    else if constexpr (8 * I == M) { constexpr T h = (T)kCos32[4]; return mk<T>((d.x + d.y) * h, (d.y - d.x) * h); }
    else if constexpr (8 * I == 3 * M) { constexpr T h = (T)kCos32[4]; return mk<T>((d.y - d.x) * h, -(d.x + d.y) * h); }
    else {
        constexpr T c = (T)cos32(I * (32 / M)), s = (T)sin32(I * (32 / M));
        return mk<T>(d.x * c + d.y * s, d.y * c - d.x * s);
    }
}
// d * conj(omega_M^I)
template <typename T, int M, int I>
WDM_HD cx<T> mul_wc(cx<T> d)
{
    if constexpr (I == 0) return d;
    else if constexpr (4 * I == M) return mk<T>(-d.y, d.x);
    else if constexpr (8 * I == M) { constexpr T h = (T)kCos32[4]; return mk<T>((d.x - d.y) * h, (d.x + d.y) * h); }
    else if constexpr (8 * I == 3 * M) { constexpr T h = (T)kCos32[4]; return mk<T>(-(d.x + d.y) * h, (d.x - d.y) * h); }
    else {
        constexpr T c = (T)cos32(I * (32 / M)), s = (T)sin32(I * (32 / M));
        return mk<T>(d.x * c - d.y * s, d.y * c + d.x * s);
    }
}

// Forward R-point DFT in registers, decimation in frequency: natural order in, X[k] left in v[brev(k)].
template <int R, typename T>
WDM_HD void dif_fwd(cx<T> (&v)[R])
{
    static_for<0, ilog2(R)>([&](auto st) {
        constexpr int half = R >> (decltype(st)::value + 1);
        static_for<0, R / (2 * half)>([&](auto bi) {
            constexpr int blk = decltype(bi)::value * 2 * half;
            static_for<0, half>([&](auto ii) {
                constexpr int i = decltype(ii)::value;
                cx<T> a = v[blk + i], b = v[blk + i + half];
                v[blk + i] = cadd(a, b);
                v[blk + i + half] = mul_w<T, 2 * half, i>(csub(a, b));
            });
        });
    });
}

// Adjoint of dif_fwd (= R * inverse DFT): Y[k] expected in v[brev(k)], natural order out.
template <int R, typename T>
WDM_HD void dit_inv(cx<T> (&v)[R])
{
    static_for<0, ilog2(R)>([&](auto st) {
        constexpr int half = 1 << decltype(st)::value;
        static_for<0, R / (2 * half)>([&](auto bi) {
            constexpr int blk = decltype(bi)::value * 2 * half;
            static_for<0, half>([&](auto ii) {
                constexpr int i = decltype(ii)::value;
                cx<T> a = v[blk + i], b = mul_wc<T, 2 * half, i>(v[blk + i + half]);
                v[blk + i] = cadd(a, b);
                v[blk + i + half] = csub(a, b);
            });
        });
    });
}

// ---------------------------------------------------------------- line-FFT stages
// ld(row) / st(row, value) address one line of the tile (or of global memory); rows are positions along
// the transformed axis.  tw points at the entry for this butterfly's q; entry for output digit s is
// tw[s * m] = omega_M^{q s}  (tables are stored s-major so that lanes with consecutive q read
// consecutive words).

// DIF level: rows rowbase + m*r -> butterfly -> twiddle -> rows rowbase + m*s (natural digit order).
// The _regs form takes the R inputs already in registers (so the caller can issue all loads first).
// The twiddles are fetched into registers BEFORE the butterfly when they fit (R complex values of at most
// 64 bytes' worth of registers... R * sizeof(T) <= 64): a table load placed after the first st() cannot be moved
// above it by the compiler (both may be shared memory), so loading on demand puts one exposed shared-memory
// latency in front of every output.
template <int R, typename T, class ST>
WDM_HD void fwd_level_regs(cx<T> (&v)[R], int rowbase, int m, const cx<T> *tw, ST &&st)
{
    constexpr bool PRE = R * sizeof(T) <= 64;
    constexpr int LOOK = PRE ? R : 4;          // too many to hold: a rolling window, each fetched LOOK outputs ahead of its use
    cx<T> w[R];
    static_for<1, (LOOK < R ? LOOK + 1 : R)>([&](auto s_) { constexpr int s = decltype(s_)::value; w[s] = tw[s * m]; });
    dif_fwd<R>(v);
    static_for<0, R>([&](auto s_) {
        constexpr int s = decltype(s_)::value;
        if constexpr (s > 0 && s + LOOK < R) w[s + LOOK] = tw[(s + LOOK) * m];
        cx<T> y = v[brev(s, R)];
        if constexpr (s > 0) y = cmul(y, w[s]);
        st(rowbase + m * s, y);
    });
}

template <int R, typename T, class LD, class ST>
WDM_HD void fwd_level(int rowbase, int m, const cx<T> *tw, LD &&ld, ST &&st)
{
    cx<T> v[R];
    static_for<0, R>([&](auto r) { v[decltype(r)::value] = ld(rowbase + m * decltype(r)::value); });
    fwd_level_regs<R, T>(v, rowbase, m, tw, st);
}

// adjoint of fwd_level; the _regs form leaves the R outputs (rows rowbase + m*r) in v
template <int R, typename T, class LD>
WDM_HD void inv_level_regs(int rowbase, int m, const cx<T> *tw, LD &&ld, cx<T> (&v)[R])
{
    static_for<0, R>([&](auto s_) {
        constexpr int s = decltype(s_)::value;
        cx<T> y = ld(rowbase + m * s);
        if constexpr (s > 0) y = cmulc(y, tw[s * m]);
        v[brev(s, R)] = y;
    });
    dit_inv<R>(v);
}

template <int R, typename T, class LD, class ST>
WDM_HD void inv_level(int rowbase, int m, const cx<T> *tw, LD &&ld, ST &&st)
{
    cx<T> v[R];
    inv_level_regs<R, T>(rowbase, m, tw, ld, v);
    static_for<0, R>([&](auto r) { st(rowbase + m * decltype(r)::value, v[decltype(r)::value]); });
}

// ---- level stages with the R twiddles of this butterfly already in registers (w[s] = omega^{q s}; w[0] unused).
// A thread whose q is the same for every tile keeps them for the whole kernel.
template <int R, typename T, class ST>
WDM_HD void fwd_level_regs_w(cx<T> (&v)[R], int rowbase, int m, const cx<T> (&w)[R], ST &&st)
{
    dif_fwd<R>(v);
    static_for<0, R>([&](auto s_) {
        constexpr int s = decltype(s_)::value;
        cx<T> y = v[brev(s, R)];
        if constexpr (s > 0) y = cmul(y, w[s]);
        st(rowbase + m * s, y);
    });
}
template <int R, typename T, class LD, class ST>
WDM_HD void fwd_level_w(int rowbase, int m, const cx<T> (&w)[R], LD &&ld, ST &&st)
{
    cx<T> v[R];
    static_for<0, R>([&](auto r) { v[decltype(r)::value] = ld(rowbase + m * decltype(r)::value); });
    dif_fwd<R>(v);
    static_for<0, R>([&](auto s_) {
        constexpr int s = decltype(s_)::value;
        cx<T> y = v[brev(s, R)];
        if constexpr (s > 0) y = cmul(y, w[s]);
        st(rowbase + m * s, y);
    });
}
template <int R, typename T, class LD, class ST>
WDM_HD void inv_level_w(int rowbase, int m, const cx<T> (&w)[R], LD &&ld, ST &&st)
{
    cx<T> v[R];
    static_for<0, R>([&](auto s_) {
        constexpr int s = decltype(s_)::value;
        cx<T> y = ld(rowbase + m * s);
        if constexpr (s > 0) y = cmulc(y, w[s]);
        v[brev(s, R)] = y;
    });
    dit_inv<R>(v);
    static_for<0, R>([&](auto r) { st(rowbase + m * decltype(r)::value, v[decltype(r)::value]); });
}
// Two adjacent lines at once (same q, hence the same twiddles): ld2/st2 move the pair (one 16-byte access for
// complex64), so a level costs half the memory instructions and one set of twiddles.
template <int R, typename T, class LD2, class ST2>
WDM_HD void fwd_level_pair(int rowbase, int m, const cx<T> (&w)[R], LD2 &&ld2, ST2 &&st2)
{
    cx<T> a[R], b[R];
    static_for<0, R>([&](auto r_) { constexpr int r = decltype(r_)::value; ld2(rowbase + m * r, a[r], b[r]); });
    dif_fwd<R>(a);
    dif_fwd<R>(b);
    static_for<0, R>([&](auto s_) {
        constexpr int s = decltype(s_)::value;
        cx<T> ya = a[brev(s, R)], yb = b[brev(s, R)];
        if constexpr (s > 0) { ya = cmul(ya, w[s]); yb = cmul(yb, w[s]); }
        st2(rowbase + m * s, ya, yb);
    });
}
template <int R, typename T, class LD2>
WDM_HD void inv_level_pair_regs(int rowbase, int m, const cx<T> (&w)[R], LD2 &&ld2, cx<T> (&a)[R], cx<T> (&b)[R])
{
    static_for<0, R>([&](auto s_) {
        constexpr int s = decltype(s_)::value;
        cx<T> ya, yb;
        ld2(rowbase + m * s, ya, yb);
        if constexpr (s > 0) { ya = cmulc(ya, w[s]); yb = cmulc(yb, w[s]); }
        a[brev(s, R)] = ya;
        b[brev(s, R)] = yb;
    });
    dit_inv<R>(a);
    dit_inv<R>(b);
}

// middle level, forward . multiply . inverse without leaving registers; mul2(p, a, b) multiplies the values
// at the consecutive positions p (even) and p + 1 in place, so a table lookup can fetch both factors at once
template <int R, typename T, class LD, class ST, class MUL>
WDM_HD void mid_both(int rowbase, LD &&ld, ST &&st, MUL &&mul2)
{
    cx<T> v[R];
    static_for<0, R>([&](auto r) { v[decltype(r)::value] = ld(rowbase + decltype(r)::value); });
    dif_fwd<R>(v);
    static_for<0, R / 2>([&](auto i_) {
        constexpr int i = decltype(i_)::value;
        mul2(rowbase + 2 * i, v[brev(2 * i, R)], v[brev(2 * i + 1, R)]);
    });
    dit_inv<R>(v);
    static_for<0, R>([&](auto r) { st(rowbase + decltype(r)::value, v[decltype(r)::value]); });
}

// same, the R consecutive rows moved as pairs (16-byte shared-memory vectors for complex64)
template <int R, typename T, class LD2, class ST2, class MUL>
WDM_HD void mid_both2(int rowbase, LD2 &&ld2, ST2 &&st2, MUL &&mul2)
{
    cx<T> v[R];
    static_for<0, R / 2>([&](auto i_) { constexpr int i = decltype(i_)::value; ld2(rowbase + 2 * i, v[2 * i], v[2 * i + 1]); });
    dif_fwd<R>(v);
    static_for<0, R / 2>([&](auto i_) {
        constexpr int i = decltype(i_)::value;
        mul2(rowbase + 2 * i, v[brev(2 * i, R)], v[brev(2 * i + 1, R)]);
    });
    dit_inv<R>(v);
    static_for<0, R / 2>([&](auto i_) { constexpr int i = decltype(i_)::value; st2(rowbase + 2 * i, v[2 * i], v[2 * i + 1]); });
}

template <int R, typename T, class LD, class ST>
WDM_HD void mid_fwd(int rowbase, LD &&ld, ST &&st)
{
    cx<T> v[R];
    static_for<0, R>([&](auto r) { v[decltype(r)::value] = ld(rowbase + decltype(r)::value); });
    dif_fwd<R>(v);
    static_for<0, R>([&](auto s_) { constexpr int s = decltype(s_)::value; st(rowbase + s, v[brev(s, R)]); });
}

template <int R, typename T, class LD, class ST>
WDM_HD void mid_inv(int rowbase, LD &&ld, ST &&st)
{
    cx<T> v[R];
    static_for<0, R>([&](auto s_) { constexpr int s = decltype(s_)::value; v[brev(s, R)] = ld(rowbase + s); });
    dit_inv<R>(v);
    static_for<0, R>([&](auto r) { st(rowbase + decltype(r)::value, v[decltype(r)::value]); });
}

// ---------------------------------------------------------------- factorisation of a line

// N = RA * RB * RM (RB = 1: two levels).  W lines per tile, NT threads per compute group, NG groups per CTA
// (NG + 1 tile buffers), MINB resident CTAs per SM.
template <typename T_, int N_, int RA_, int RB_, int RM_, int W_, int NT_, int NG_, int MINB_>
struct LineCfg {
    using T = T_;
    static constexpr int N = N_, RA = RA_, RB = RB_, RM = RM_, W = W_, NT = NT_, NG = NG_, MINB = MINB_;
    static constexpr int mA = N / RA;          // level A: block N, stride mA
    static constexpr int MB = N / RA;          // level B: block MB, stride mB
    static constexpr int mB = MB / RB;
    static_assert(RA * RB * RM == N, "bad factorisation");
    static_assert(RA >= 2 && RM >= 2, "level A and the middle level are always present");
};

// frequency index held at position p after the forward transform (natural digits at every level)
inline int k_of_pos(int p, int RA, int RB, int RM)
{
    int sM = p % RM, sB = (p / RM) % RB, sA = p / (RM * RB);
    return sA + RA * (sB + RB * sM);
}

}  // namespace wdm
