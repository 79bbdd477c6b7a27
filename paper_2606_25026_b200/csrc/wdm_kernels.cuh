// wdm_kernels.cuh -- the fused axis sweeps of one kick-drift-kick step (Eq. 18, Alg. 1 l.5-16).
//
//   psi sweeps (3 per step):  [kick on load] -> FFT -> per-axis kinetic phase -> inverse FFT along one axis.
//       exp(-i mu k^2 dt/2) = prod_axis exp(-i mu k_axis^2 dt/2), each factor acting along one axis only, so
//       Eq. 18(b) needs three tile sweeps instead of six FFT sweeps plus a multiply.
//       The last sweep (x axis) also forms rho = |psi2|^2 (+ particle mesh) in the same tile and writes the
//       real-to-complex x-spectrum of rho (two real lines packed into one complex FFT).
//   Poisson sweeps (4 per step) on the half-spectrum H[kx <= N/2][y][z]: y forward, z forward . Green . inverse
//       (Eq. 18(c), Eq. 23: -4 pi G / k^2, k = 0 zeroed), y inverse, x complex-to-real -> Phi.
//
// Each body is written per thread (tid) and per tile (bid) with WDM_SYNC() as the CTA barrier.
#pragma once

#include "wdm_fft.cuh"

#if defined(__CUDACC__)
#define WDM_DEV __device__ __forceinline__
#define WDM_SYNC() __syncthreads()
#else
#include <cmath>
#define WDM_DEV inline __attribute__((always_inline))
void wdm_host_sync();
#define WDM_SYNC() wdm_host_sync()
#endif

namespace wdm {

// ---------------------------------------------------------------- global memory access helpers
#if defined(__CUDACC__)
WDM_DEV cx<float> ldg(const cx<float> *p) { float2 t = __ldg(reinterpret_cast<const float2 *>(p)); return mk<float>(t.x, t.y); }
WDM_DEV cx<double> ldg(const cx<double> *p) { double2 t = __ldg(reinterpret_cast<const double2 *>(p)); return mk<double>(t.x, t.y); }
WDM_DEV float ldg(const float *p) { return __ldg(p); }
WDM_DEV double ldg(const double *p) { return __ldg(p); }
WDM_DEV unsigned short ldg(const unsigned short *p) { return __ldg(p); }
WDM_DEV cx<float> ldv(const cx<float> *p) { float2 t = *reinterpret_cast<const float2 *>(p); return mk<float>(t.x, t.y); }
WDM_DEV cx<double> ldv(const cx<double> *p) { double2 t = *reinterpret_cast<const double2 *>(p); return mk<double>(t.x, t.y); }
WDM_DEV void stv(cx<float> *p, cx<float> v) { *reinterpret_cast<float2 *>(p) = make_float2(v.x, v.y); }
WDM_DEV void stv(cx<double> *p, cx<double> v) { *reinterpret_cast<double2 *>(p) = make_double2(v.x, v.y); }
WDM_DEV void ld2(const cx<float> *p, cx<float> &a, cx<float> &b) { float4 t = *reinterpret_cast<const float4 *>(p); a = mk<float>(t.x, t.y); b = mk<float>(t.z, t.w); }
WDM_DEV void st2(cx<float> *p, cx<float> a, cx<float> b) { *reinterpret_cast<float4 *>(p) = make_float4(a.x, a.y, b.x, b.y); }
WDM_DEV void ld2(const cx<double> *p, cx<double> &a, cx<double> &b) { a = ldv(p); b = ldv(p + 1); }
WDM_DEV void st2(cx<double> *p, cx<double> a, cx<double> b) { stv(p, a); stv(p + 1, b); }
WDM_DEV void sincos_t(float x, float *s, float *c) { sincosf(x, s, c); }
WDM_DEV void sincos_t(double x, double *s, double *c) { sincos(x, s, c); }
#else
template <typename U> WDM_DEV U ldg(const U *p) { return *p; }
template <typename U> WDM_DEV U ldv(const U *p) { return *p; }
template <typename U> WDM_DEV void stv(U *p, U v) { *p = v; }
template <typename U> WDM_DEV void ld2(const U *p, U &a, U &b) { a = p[0]; b = p[1]; }
template <typename U> WDM_DEV void st2(U *p, U a, U b) { p[0] = a; p[1] = b; }
WDM_DEV void sincos_t(float x, float *s, float *c) { *s = std::sin(x); *c = std::cos(x); }
WDM_DEV void sincos_t(double x, double *s, double *c) { *s = std::sin(x); *c = std::cos(x); }
#endif

// psi * exp(-i theta)
template <typename T>
WDM_DEV cx<T> rotate_neg(cx<T> v, T theta)
{
    T s, c;
    sincos_t(theta, &s, &c);
    return mk<T>(v.x * c + v.y * s, v.y * c - v.x * s);
}

// ---------------------------------------------------------------- parameters

template <typename T>
struct SweepParams {
    cx<T> *data;               // psi (N^3) or H ((N/2+1) N^2), transformed in place
    long long rowStride;       // strided sweeps: elements between consecutive points of the axis
    long long outerStride;     // strided sweeps: elements between consecutive "outer" tiles
    int tilesInner;            // strided sweeps: tiles along the contiguous (z) direction = N / W
    const cx<T> *twA;          // level-A twiddles, s-major: twA[s*mA + q] = exp(-2 pi i q s / N)
    const cx<T> *twB;          // level-B twiddles, s-major over the sub-block
    const cx<T> *phase;        // psi sweeps: exp(-i mu k^2 dt/2)/N in position order
    const T *phi;              // KICK: potential, same shape as psi
    T kick;                    // KICK: theta = phi * kick   (dt/(2 mu) or dt/mu)
    const T *rho_p;            // RHO: particle mesh density or nullptr
    const T *rho_mean;         // RHO: device scalar <rho>, subtracted before the transform (Eq. 23)
    cx<T> *H;                  // RHO / C2R: half spectrum
    T *phi_out;                // C2R: potential out
    const unsigned short *pos_of_k;  // position holding frequency k after a forward transform
    const T *ksq_pos;          // Green: k^2 of the frequency held at a position
    const T *ksq_nat;          // Green: k^2 of frequency index k (natural)
    T green;                   // Green: -4 pi G / N^3
};

enum { AX_STRIDED = 0, AX_CONTIG = 1 };

template <class C, int AX>
struct Tile {
    static constexpr int RS = (AX == AX_CONTIG) ? C::W + 1 : C::W;   // smem row stride (elements)
    long long base, rstride, lstride;
    template <typename T>
    WDM_DEV Tile(const SweepParams<T> &p, int bid)
    {
        if (AX == AX_STRIDED) {
            int outer = bid / p.tilesInner, inner = bid - outer * p.tilesInner;
            base = (long long)outer * p.outerStride + (long long)inner * C::W;
            rstride = p.rowStride;
            lstride = 1;
        } else {
            base = (long long)bid * C::W * C::N;
            rstride = 1;
            lstride = C::N;
        }
    }
    WDM_DEV long long at(int row, int l) const { return base + (long long)row * rstride + (long long)l * lstride; }
};

// thread -> (butterfly g, line l).  Strided tiles: lines fastest (a half-warp owns one 128-byte row).
// Contiguous tiles, when the stage touches global memory: points fastest (a warp reads one pencil).
template <int AX, int NB, int W>
WDM_DEV void split(int b, int &g, int &l)
{
    if (AX == AX_STRIDED) { l = b % W; g = b / W; }
    else { g = b % NB; l = b / NB; }
}

// ---------------------------------------------------------------- in-shared-memory stages (lines fastest)

template <class C, int W, int RS, typename T>
WDM_DEV void smem_fwd_B(cx<T> *S, const cx<T> *twB, int tid)
{
    if constexpr (C::RB > 1) {
        constexpr int NB = C::N / C::RB;
        for (int b = tid; b < NB * W; b += C::NT) {
            int l = b % W, g = b / W, blk = g / C::mB, q = g - blk * C::mB;
            fwd_level<C::RB, T>(blk * C::MB + q, C::mB, twB + q,
                                [&](int row) { return S[row * RS + l]; },
                                [&](int row, cx<T> v) { S[row * RS + l] = v; });
        }
        WDM_SYNC();
    }
}

template <class C, int W, int RS, typename T>
WDM_DEV void smem_inv_B(cx<T> *S, const cx<T> *twB, int tid)
{
    if constexpr (C::RB > 1) {
        constexpr int NB = C::N / C::RB;
        for (int b = tid; b < NB * W; b += C::NT) {
            int l = b % W, g = b / W, blk = g / C::mB, q = g - blk * C::mB;
            inv_level<C::RB, T>(blk * C::MB + q, C::mB, twB + q,
                                [&](int row) { return S[row * RS + l]; },
                                [&](int row, cx<T> v) { S[row * RS + l] = v; });
        }
        WDM_SYNC();
    }
}

// ---------------------------------------------------------------- psi sweep
// DRIFT: FFT . phase . inverse FFT along the axis.  KICK: psi *= exp(-i phi kick) on load.
// RHO (strided x axis only): rho = |psi|^2 (+rho_p) -> packed real-to-complex FFT along x -> H.

template <class C, int AX, bool KICK, bool RHO, bool DRIFT>
WDM_DEV void psi_sweep_body(const SweepParams<typename C::T> &p, int tid, int bid, unsigned char *smem_raw)
{
    using T = typename C::T;
    constexpr int N = C::N, RA = C::RA, RM = C::RM, W = C::W, NT = C::NT, mA = C::mA;
    using TL = Tile<C, AX>;
    constexpr int RS = TL::RS;
    static_assert(!RHO || AX == AX_STRIDED, "the density sweep runs along a strided axis");
    static_assert((mA * W) % NT == 0 || !RHO, "density sweep needs a whole number of butterflies per thread");
    cx<T> *S = reinterpret_cast<cx<T> *>(smem_raw);
    const TL tile(p, bid);
    cx<T> *psi = p.data;
    constexpr int ITER = RHO ? (mA * W) / NT : 1;
    T rho[ITER][RA];

    auto load_psi = [&](int row, int l) {
        long long a = tile.at(row, l);
        cx<T> v = ldv(psi + a);
        if (KICK) v = rotate_neg(v, ldg(p.phi + a) * p.kick);
        return v;
    };

    if constexpr (DRIFT) {
        // level A forward: global -> registers -> shared (all loads of a butterfly are issued before any use)
        for (int b = tid; b < mA * W; b += NT) {
            int q, l;
            split<AX, mA, W>(b, q, l);
            cx<T> v[RA];
            static_for<0, RA>([&](auto r_) { constexpr int r = decltype(r_)::value; v[r] = ldv(psi + tile.at(q + mA * r, l)); });
            if constexpr (KICK) {
                T th[RA];
                static_for<0, RA>([&](auto r_) { constexpr int r = decltype(r_)::value; th[r] = ldg(p.phi + tile.at(q + mA * r, l)); });
                static_for<0, RA>([&](auto r_) { constexpr int r = decltype(r_)::value; v[r] = rotate_neg(v[r], th[r] * p.kick); });
            }
            fwd_level_regs<RA, T>(v, q, mA, p.twA + q, [&](int row, cx<T> y) { S[row * RS + l] = y; });
        }
        WDM_SYNC();
        smem_fwd_B<C, W, RS, T>(S, p.twB, tid);
        // middle level: forward . kinetic phase . inverse
        for (int b = tid; b < (N / RM) * W; b += NT) {
            int l = b % W, g = b / W;
            mid_both<RM, T>(g * RM, [&](int row) { return S[row * RS + l]; },
                            [&](int row, cx<T> v) { S[row * RS + l] = v; },
                            [&](int pos, cx<T> v) { return cmul(v, ldg(p.phase + pos)); });
        }
        WDM_SYNC();
        smem_inv_B<C, W, RS, T>(S, p.twB, tid);
        // level A inverse: shared -> registers -> global
        if constexpr (RHO) {
            static_for<0, ITER>([&](auto it_) {
                constexpr int it = decltype(it_)::value;
                int b = tid + it * NT, q, l;
                split<AX, mA, W>(b, q, l);
                cx<T> v[RA];
                inv_level_regs<RA, T>(q, mA, p.twA + q, [&](int row) { return S[row * RS + l]; }, v);
                static_for<0, RA>([&](auto r_) {
                    constexpr int r = decltype(r_)::value;
                    stv(psi + tile.at(q + mA * r, l), v[r]);
                    rho[it][r] = v[r].x * v[r].x + v[r].y * v[r].y;
                });
            });
        } else {
            for (int b = tid; b < mA * W; b += NT) {
                int q, l;
                split<AX, mA, W>(b, q, l);
                inv_level<RA, T>(q, mA, p.twA + q, [&](int row) { return S[row * RS + l]; },
                                 [&](int row, cx<T> v) { stv(psi + tile.at(row, l), v); });
            }
        }
    } else if constexpr (RHO) {
        static_for<0, ITER>([&](auto it_) {
            constexpr int it = decltype(it_)::value;
            int b = tid + it * NT, q, l;
            split<AX, mA, W>(b, q, l);
            static_for<0, RA>([&](auto r_) {
                constexpr int r = decltype(r_)::value;
                cx<T> v = load_psi(q + mA * r, l);
                rho[it][r] = v.x * v.x + v.y * v.y;
            });
        });
    }

    if constexpr (RHO) {
        // rho tile as N rows x W reals == N rows x W/2 packed complex lines (lines 2l', 2l'+1)
        constexpr int WP = W / 2, RSP = W / 2;
        T *F = reinterpret_cast<T *>(smem_raw);
        if (DRIFT) WDM_SYNC();   // every thread has finished reading the psi tile
        // rho - <rho> (Eq. 23).  <rho> is conserved, so it is measured once per refresh; the k = 0
        // mode is zeroed in the Green's function anyway -- subtracting here only keeps the large mean out of
        // the single-precision partial sums of the low-k modes.
        const T mean = ldg(p.rho_mean);
        static_for<0, ITER>([&](auto it_) {
            constexpr int it = decltype(it_)::value;
            int b = tid + it * NT, q, l;
            split<AX, mA, W>(b, q, l);
            static_for<0, RA>([&](auto r_) {
                constexpr int r = decltype(r_)::value;
                int row = q + mA * r;
                T v = rho[it][r];
                if (p.rho_p) v += ldg(p.rho_p + tile.at(row, l));
                F[row * W + l] = v - mean;
            });
        });
        WDM_SYNC();
        cx<T> *Sp = reinterpret_cast<cx<T> *>(smem_raw);
        for (int b = tid; b < mA * WP; b += NT) {
            int l = b % WP, q = b / WP;
            fwd_level<RA, T>(q, mA, p.twA + q, [&](int row) { return Sp[row * RSP + l]; },
                             [&](int row, cx<T> v) { Sp[row * RSP + l] = v; });
        }
        WDM_SYNC();
        smem_fwd_B<C, WP, RSP, T>(Sp, p.twB, tid);
        for (int b = tid; b < (N / RM) * WP; b += NT) {
            int l = b % WP, g = b / WP;
            mid_fwd<RM, T>(g * RM, [&](int row) { return Sp[row * RSP + l]; },
                           [&](int row, cx<T> v) { Sp[row * RSP + l] = v; });
        }
        WDM_SYNC();
        // Hermitian split of Z = FFT(a + i b):  A_k = (Z_k + conj Z_{N-k})/2,  B_k = (Z_k - conj Z_{N-k})/(2i)
        for (int b = tid; b < (N / 2 + 1) * WP; b += NT) {
            int l = b % WP, k = b / WP;
            int pk = ldg(p.pos_of_k + k), pn = ldg(p.pos_of_k + ((N - k) & (N - 1)));
            cx<T> zk = Sp[pk * RSP + l], zn = Sp[pn * RSP + l];
            const T h = (T)0.5;
            cx<T> A = mk<T>((zk.x + zn.x) * h, (zk.y - zn.y) * h);
            cx<T> B = mk<T>((zk.y + zn.y) * h, (zn.x - zk.x) * h);
            st2(p.H + tile.at(k, 2 * l), A, B);
        }
    }
}

// ---------------------------------------------------------------- Poisson sweeps on the half spectrum

enum { H_Y_FWD = 0, H_Z_GREEN = 1, H_Y_INV = 2 };

template <class C, int MODE>
WDM_DEV void h_sweep_body(const SweepParams<typename C::T> &p, int tid, int bid, unsigned char *smem_raw)
{
    using T = typename C::T;
    constexpr int N = C::N, RA = C::RA, RM = C::RM, W = C::W, NT = C::NT, mA = C::mA;
    constexpr int AX = (MODE == H_Z_GREEN) ? AX_CONTIG : AX_STRIDED;
    using TL = Tile<C, AX>;
    constexpr int RS = TL::RS;
    cx<T> *S = reinterpret_cast<cx<T> *>(smem_raw);
    const TL tile(p, bid);
    cx<T> *H = p.data;

    if constexpr (MODE == H_Y_FWD || MODE == H_Z_GREEN) {
        for (int b = tid; b < mA * W; b += NT) {
            int q, l;
            split<AX, mA, W>(b, q, l);
            fwd_level<RA, T>(q, mA, p.twA + q, [&](int row) { return ldv(H + tile.at(row, l)); },
                             [&](int row, cx<T> v) { S[row * RS + l] = v; });
        }
        WDM_SYNC();
        smem_fwd_B<C, W, RS, T>(S, p.twB, tid);
    }
    if constexpr (MODE == H_Y_FWD) {
        for (int b = tid; b < (N / RM) * W; b += NT) {
            int l = b % W, g = b / W;
            mid_fwd<RM, T>(g * RM, [&](int row) { return S[row * RS + l]; },
                           [&](int row, cx<T> v) { stv(H + tile.at(row, l), v); });
        }
    }
    if constexpr (MODE == H_Z_GREEN) {
        // pencil l of this tile is (kx, y position) = divmod(bid*W + l, N); the y axis is in position order
        for (int b = tid; b < (N / RM) * W; b += NT) {
            int l = b % W, g = b / W;
            int pen = bid * W + l, kx = pen / N, ypos = pen - kx * N;
            T kxy = ldg(p.ksq_nat + kx) + ldg(p.ksq_pos + ypos);
            bool zero_line = (kx == 0 && ypos == 0);
            mid_both<RM, T>(g * RM, [&](int row) { return S[row * RS + l]; },
                            [&](int row, cx<T> v) { S[row * RS + l] = v; },
                            [&](int pos, cx<T> v) {
                                T k2 = kxy + ldg(p.ksq_pos + pos);
                                T gr = (zero_line && pos == 0) ? (T)0 : p.green / k2;
                                return cscale(v, gr);
                            });
        }
        WDM_SYNC();
        smem_inv_B<C, W, RS, T>(S, p.twB, tid);
    }
    if constexpr (MODE == H_Y_INV) {
        for (int b = tid; b < (N / RM) * W; b += NT) {
            int l = b % W, g = b / W;
            mid_inv<RM, T>(g * RM, [&](int row) { return ldv(H + tile.at(row, l)); },
                           [&](int row, cx<T> v) { S[row * RS + l] = v; });
        }
        WDM_SYNC();
        smem_inv_B<C, W, RS, T>(S, p.twB, tid);
    }
    if constexpr (MODE == H_Y_INV || MODE == H_Z_GREEN) {
        for (int b = tid; b < mA * W; b += NT) {
            int q, l;
            split<AX, mA, W>(b, q, l);
            inv_level<RA, T>(q, mA, p.twA + q, [&](int row) { return S[row * RS + l]; },
                             [&](int row, cx<T> v) { stv(H + tile.at(row, l), v); });
        }
    }
}

// complex-to-real inverse along x: H[kx <= N/2][y][z] -> Phi[x][y][z]; lines (2l', 2l'+1) share one FFT
template <class C>
WDM_DEV void c2r_body(const SweepParams<typename C::T> &p, int tid, int bid, unsigned char *smem_raw)
{
    using T = typename C::T;
    constexpr int N = C::N, RA = C::RA, RM = C::RM, W = C::W, NT = C::NT, mA = C::mA;
    constexpr int WP = W / 2, RSP = W / 2;
    cx<T> *Sp = reinterpret_cast<cx<T> *>(smem_raw);
    const Tile<C, AX_STRIDED> tile(p, bid);
    // Z_k = A_k + i B_k,  Z_{N-k} = conj(A_k) + i conj(B_k).  Loads are issued in unrolled batches.
    auto place = [&](int k, int l, cx<T> A, cx<T> B) {
        int pk = ldg(p.pos_of_k + k);
        Sp[pk * RSP + l] = mk<T>(A.x - B.y, A.y + B.x);
        if (k > 0 && k < N / 2) {
            int pn = ldg(p.pos_of_k + (N - k));
            Sp[pn * RSP + l] = mk<T>(A.x + B.y, B.x - A.y);
        }
    };
    constexpr int ITEMS = (N / 2) * WP;              // rows k < N/2
    constexpr int UN = ITEMS % (NT * 8) == 0 ? 8 : (ITEMS % (NT * 4) == 0 ? 4 : (ITEMS % (NT * 2) == 0 ? 2 : 1));
    static_assert(ITEMS % NT == 0 || ITEMS < NT, "pack loop");
    for (int b0 = tid; b0 < ITEMS; b0 += NT * UN) {
        cx<T> A[UN], B[UN];
        static_for<0, UN>([&](auto u_) {
            constexpr int u = decltype(u_)::value;
            int b = b0 + u * NT;
            if (ITEMS >= NT || b < ITEMS) ld2(p.H + tile.at(b / WP, 2 * (b % WP)), A[u], B[u]);
        });
        static_for<0, UN>([&](auto u_) {
            constexpr int u = decltype(u_)::value;
            int b = b0 + u * NT;
            if (ITEMS >= NT || b < ITEMS) place(b / WP, b % WP, A[u], B[u]);
        });
    }
    if (tid < WP) {
        cx<T> A, B;
        ld2(p.H + tile.at(N / 2, 2 * tid), A, B);
        place(N / 2, tid, A, B);
    }
    WDM_SYNC();
    for (int b = tid; b < (N / RM) * WP; b += NT) {
        int l = b % WP, g = b / WP;
        mid_inv<RM, T>(g * RM, [&](int row) { return Sp[row * RSP + l]; },
                       [&](int row, cx<T> v) { Sp[row * RSP + l] = v; });
    }
    WDM_SYNC();
    smem_inv_B<C, WP, RSP, T>(Sp, p.twB, tid);
    for (int b = tid; b < mA * WP; b += NT) {
        int l = b % WP, q = b / WP;
        inv_level<RA, T>(q, mA, p.twA + q, [&](int row) { return Sp[row * RSP + l]; },
                         [&](int row, cx<T> v) {
                             // Re -> line 2l', Im -> line 2l'+1 : one (re, im) pair is two adjacent reals of Phi
                             stv(reinterpret_cast<cx<T> *>(p.phi_out + tile.at(row, 2 * l)), v);
                         });
    }
}

}  // namespace wdm
