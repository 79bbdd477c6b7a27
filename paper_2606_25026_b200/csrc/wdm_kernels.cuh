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
// This header holds what every sweep shares: parameters, tile addressing and memory-access helpers.  The
// kernels themselves (persistent, software-pipelined) are in wdm_pipe.cuh.
#pragma once

#include <cuda.h>          // CUtensorMap (type only: the encoder is fetched through the runtime, no libcuda link)

#include "wdm_fft.cuh"

#define WDM_DEV __device__ __forceinline__

namespace wdm {

// ---------------------------------------------------------------- global memory access helpers
WDM_DEV cx<float> ldg(const cx<float> *p) { float2 t = __ldg(reinterpret_cast<const float2 *>(p)); return mk<float>(t.x, t.y); }
WDM_DEV cx<double> ldg(const cx<double> *p) { double2 t = __ldg(reinterpret_cast<const double2 *>(p)); return mk<double>(t.x, t.y); }
WDM_DEV float ldg(const float *p) { return __ldg(p); }
WDM_DEV double ldg(const double *p) { return __ldg(p); }
WDM_DEV unsigned short ldg(const unsigned short *p) { return __ldg(p); }
WDM_DEV cx<float> ldv(const cx<float> *p) { float2 t = *reinterpret_cast<const float2 *>(p); return mk<float>(t.x, t.y); }
WDM_DEV cx<double> ldv(const cx<double> *p) { double2 t = *reinterpret_cast<const double2 *>(p); return mk<double>(t.x, t.y); }
// (inline PTX: with the plain float2 store ptxas copies already-adjacent register pairs into one scratch pair
// store after store, serialising them on its write-after-read scoreboard.  No "memory" clobber: volatile asm
// statements keep their order among themselves -- barriers, async copies -- and shared-memory accesses may
// still be scheduled across a global store)
WDM_DEV void stv(cx<float> *p, cx<float> v) { asm volatile("st.global.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(v.x), "f"(v.y)); }
WDM_DEV void stv(cx<double> *p, cx<double> v) { *reinterpret_cast<double2 *>(p) = make_double2(v.x, v.y); }
// two adjacent reals (p aligned to both)
WDM_DEV void ld2r(const float *p, float &a, float &b) { float2 t = *reinterpret_cast<const float2 *>(p); a = t.x; b = t.y; }
WDM_DEV void ld2r(const double *p, double &a, double &b) { double2 t = *reinterpret_cast<const double2 *>(p); a = t.x; b = t.y; }
// two adjacent complex64 values to global memory as one 16-byte store (p 16-byte aligned)
WDM_DEV void stg2(cx<float> *p, cx<float> a, cx<float> b)
{
    asm volatile("st.global.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
}
WDM_DEV void stg2(cx<double> *p, cx<double> a, cx<double> b) { stv(p, a); stv(p + 1, b); }
WDM_DEV void ld2(const cx<float> *p, cx<float> &a, cx<float> &b) { float4 t = *reinterpret_cast<const float4 *>(p); a = mk<float>(t.x, t.y); b = mk<float>(t.z, t.w); }
WDM_DEV void st2(cx<float> *p, cx<float> a, cx<float> b) { *reinterpret_cast<float4 *>(p) = make_float4(a.x, a.y, b.x, b.y); }
WDM_DEV void ld2(const cx<double> *p, cx<double> &a, cx<double> &b) { a = ldv(p); b = ldv(p + 1); }
WDM_DEV void st2(cx<double> *p, cx<double> a, cx<double> b) { stv(p, a); stv(p + 1, b); }

// psi * exp(-i theta).  |theta| = |Phi| dt/(2 mu) is far below 1 under the CFL limit (Eq. 26),
// so the single-precision path takes a Taylor branch for |theta| < 1/4 (sin to theta^5, cos to theta^6:
// truncation below 1.3e-8 and 4e-10, under float rounding) and falls back to sincosf only for large phases.
WDM_DEV void sincos_small(float th, float &s, float &c)
{
    float t2 = th * th;
    s = th * fmaf(t2, fmaf(t2, 1.0f / 120.0f, -1.0f / 6.0f), 1.0f);
    c = fmaf(t2, fmaf(t2, fmaf(t2, -1.0f / 720.0f, 1.0f / 24.0f), -0.5f), 1.0f);
}
// large phases are rare: keep the full-range sincosf (with its Payne-Hanek reduction) out of line so the hot
// code stays small and straight
static __device__ __noinline__ float2 sincos_large(float th)
{
    float s, c;
    sincosf(th, &s, &c);
    return make_float2(s, c);
}
WDM_DEV cx<float> rotate_neg(cx<float> v, float th)
{
    float s, c;
    if (fabsf(th) < 0.25f) sincos_small(th, s, c);
    else { float2 sc = sincos_large(th); s = sc.x; c = sc.y; }
    return mk<float>(v.x * c + v.y * s, v.y * c - v.x * s);
}
WDM_DEV cx<double> rotate_neg(cx<double> v, double th)
{
    double s, c;
    sincos(th, &s, &c);
    return mk<double>(v.x * c + v.y * s, v.y * c - v.x * s);
}
// R elements at once (the level-A butterfly of one thread).  Single precision: ONE test on the largest phase of the
// butterfly instead of one per element -- the common path (every phase small) is straight-line code.
template <int R>
WDM_DEV void rotate_neg_all(cx<float> (&v)[R], const float (&th)[R])
{
    float mx = 0.0f;
#pragma unroll
    for (int r = 0; r < R; ++r) mx = fmaxf(mx, fabsf(th[r]));
    if (mx < 0.25f) {
#if defined(__CUDA_ARCH__) && __CUDA_ARCH__ >= 1000 && !defined(WDM_NO_PACKED_ADD)
        // the two polynomials of sincos_small for two phases at a time in packed single precision (the same operations
        // in the same order per phase: identical results, half the issue slots)
        static_assert(R % 2 == 0, "pairs of phases");
        auto pk = [](float a, float b) { unsigned long long r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; };
        auto mul2 = [](unsigned long long a, unsigned long long b) { unsigned long long r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; };
        auto fma2 = [](unsigned long long a, unsigned long long b, unsigned long long c) { unsigned long long r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; };
        const unsigned long long k120 = pk(1.0f / 120.0f, 1.0f / 120.0f), km6 = pk(-1.0f / 6.0f, -1.0f / 6.0f), k1 = pk(1.0f, 1.0f),
                                 km720 = pk(-1.0f / 720.0f, -1.0f / 720.0f), k24 = pk(1.0f / 24.0f, 1.0f / 24.0f), kmh = pk(-0.5f, -0.5f);
#pragma unroll
        for (int r = 0; r < R; r += 2) {
            const unsigned long long t = pk(th[r], th[r + 1]), t2 = mul2(t, t);
            const unsigned long long sp = mul2(t, fma2(t2, fma2(t2, k120, km6), k1));
            const unsigned long long cp = fma2(t2, fma2(t2, fma2(t2, km720, k24), kmh), k1);
            float s0, s1, c0, c1;
            asm("mov.b64 {%0, %1}, %2;" : "=f"(s0), "=f"(s1) : "l"(sp));
            asm("mov.b64 {%0, %1}, %2;" : "=f"(c0), "=f"(c1) : "l"(cp));
            v[r] = mk<float>(v[r].x * c0 + v[r].y * s0, v[r].y * c0 - v[r].x * s0);
            v[r + 1] = mk<float>(v[r + 1].x * c1 + v[r + 1].y * s1, v[r + 1].y * c1 - v[r + 1].x * s1);
        }
#else
#pragma unroll
        for (int r = 0; r < R; ++r) {
            float s, c;
            sincos_small(th[r], s, c);
            v[r] = mk<float>(v[r].x * c + v[r].y * s, v[r].y * c - v[r].x * s);
        }
#endif
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            float2 sc = sincos_large(th[r]);
            v[r] = mk<float>(v[r].x * sc.y + v[r].y * sc.x, v[r].y * sc.y - v[r].x * sc.x);
        }
    }
}
template <int R>
WDM_DEV void rotate_neg_all(cx<double> (&v)[R], const double (&th)[R])
{
#pragma unroll
    for (int r = 0; r < R; ++r) v[r] = rotate_neg(v[r], th[r]);
}
// the general kick of one element (see SweepParams::kick_extra); m = product of the three axis factors or 1
template <typename T>
WDM_DEV cx<T> kick_general(cx<T> v, T phi, T m, T kick, T kd, T ka)
{
    const T a2 = v.x * v.x + v.y * v.y;
    const T th = phi * kick + a2 * (kd + ka * m * m);
    cx<T> r = rotate_neg(v, th);
    return mk<T>(r.x * m, r.y * m);
}

// g / k2 of the Green's function (Eq. 23).  Single precision: one reciprocal (MUFU.RCP, 1 ulp)
// and a multiply instead of the IEEE division sequence -- 2 ulp on a factor whose tolerance is 2e-5.
WDM_DEV float green_over(float g, float k2) { return __fdividef(g, k2); }
WDM_DEV double green_over(double g, double k2) { return g / k2; }

// ---------------------------------------------------------------- parameters

template <typename T>
struct SweepParams {
    cx<T> *data;               // psi (N^3) or H ((N/2+1) N^2), transformed in place
    const cx<T> *twA;          // level-A twiddles, s-major: twA[s*mA + q] = exp(-2 pi i q s / N)
    const cx<T> *twB;          // level-B twiddles, s-major over the sub-block
    const cx<T> *x2tab;        // wdm_x2.cuh (x sweeps on half tiles; tmap2 = the 16-line boxes): 4 tables of N/2 entries, or nullptr
    const cx<T> *phase;        // psi sweeps: exp(-i mu k^2 dt/2)/N in position order
    const T *phi;              // KICK: potential, same shape as psi
    T kick;                    // KICK: theta = phi * kick   (dt/(2 mu) or dt/mu)
    // extra kick terms (Eq. 13-14, Eq. 22; readings G26-G28), used only when kick_extra != 0.  A merged kick is the
    // closing half kick of one step (weight kself_d, then the absorbing layer m) and the opening one of the next
    // (kself_a, on the attenuated field):  psi <- m psi exp(-i (phi kick + |psi|^2 (kself_d + kself_a m^2)))
    int kick_extra;
    T kself_d, kself_a;        // kappa h_d / mu, kappa h_a / mu
    const T *mask;             // 3 N reals, exp(-alpha b(x_axis) dt) along x, y, z; nullptr: no layer in this kick
    const T *phi_ext;          // C2R: static external potential added to Phi on its way out, or nullptr
    const T *rho_p;            // RHO: particle mesh density or nullptr
    const unsigned char *rho_flag;   // RHO: one byte per (y, block of min(16, N) z-cells): 0 = rho_p is zero there, skip its loads
    const T *rho_mean;         // RHO: device scalar <rho>, subtracted before the transform (Eq. 23)
    cx<T> *H;                  // RHO / C2R: half spectrum
    T *phi_out;                // C2R: potential out
    const T *ksq_pos;          // Green: k^2 of the frequency held at a position
    const T *ksq_nat;          // Green: k^2 of frequency index k (natural)
    T green;                   // Green: -4 pi G / N^3
    int kx0;                   // Green: global kx index of the first plane of the array (slab-decomposed runs; else 0)
    // TMA descriptors of the array a strided sweep walks: boxes of (W elements along z) x (<= 256 rows along the
    // sweep axis); tmap2 is the one-row box that fetches row N/2 of the half spectrum in the complex-to-real sweep
    CUtensorMap tmap, tmap2;
    // Per-step diagnostics (the DIAG instantiations only): accumulators of THIS step, and the set the
    // next step will use, zeroed by this launch.  Layout (doubles): [0..2] sum k_a^2 |F_a psi|^2 from the z, y, x sweeps,
    // [3] sum |psi_2|^2, [4] max |psi_2|^2 (bit pattern), [5] sum_k w_kx green(k) |rho~_k|^2, [6] max |Phi| (bit pattern)
    double *diag, *diag_zero;
    // Tiles are handed out in decreasing order.  The y sweep of psi and the z-Green sweep of H run against the direction
    // of the sweep before them (and the y-inverse sweep with the direction of the y-forward one again): each starts on
    // the planes its predecessor wrote last, which are still in the 126 MB L2.
    int reverse;
    unsigned int *ticket;      // tile tickets drawn in this launch (0 when the launch starts)
    unsigned int *ticket_next; // the next launch's counter: this launch zeroes it (launches alternate between two words)
};

// Axis of a sweep over an array [x][y][z] (z contiguous).  The strides are compile-time constants of the
// instantiation (N is), so every global address of a tile is one 64-bit base plus an immediate offset.
enum { AX_Y = 0, AX_CONTIG = 1, AX_X = 2 };
constexpr bool ax_strided(int ax) { return ax != AX_CONTIG; }

// Shared-memory layout of a tile (row = position along the transformed axis, l = line).
//   strided axis   : [row][l], row stride W  -- a half-warp (complex64) reads one whole 128-byte row, so a
//                    butterfly of any stride is free of bank conflicts; filled by 16-byte async copies.
//   contiguous axis: [l][row], line stride N + 16 bytes -- filled by 16-byte async copies straight along
//                    each pencil; level A walks rows with consecutive lanes, the middle level reads its R
//                    consecutive rows as 16-byte vectors with lanes on different lines (the odd line
//                    stride in 16-byte units spreads them over all banks).
template <class C, int AX>
struct Lay {
    using T = typename C::T;
    static constexpr int PAD = 16 / (int)sizeof(cx<T>);
    static constexpr int LS = C::N + PAD;
    static constexpr int RS = C::W;
    static constexpr size_t ELEMS = AX == AX_CONTIG ? (size_t)C::W * LS : (size_t)C::N * RS;
    static constexpr bool VEC2 = AX == AX_CONTIG && sizeof(T) == 4;
    static WDM_DEV int idx(int row, int l) { return AX == AX_CONTIG ? l * LS + row : row * RS + l; }
};

template <class C, int AX>
struct Tile {
    static constexpr long long N = C::N;
    static constexpr long long RSTRIDE = AX == AX_Y ? N : (AX == AX_X ? N * N : 1);   // between points of the axis
    static constexpr long long LSTRIDE = AX == AX_CONTIG ? N : 1;                      // between lines of the tile
    static constexpr int INNER = C::N / C::W;                                          // strided: tiles along z
    long long base;
    template <typename T>
    WDM_DEV Tile(const SweepParams<T> &, int bid) : Tile(bid) {}
    WDM_DEV explicit Tile(int bid)
    {
        if (AX == AX_CONTIG) {
            base = (long long)bid * C::W * C::N;
        } else {
            int outer = bid / INNER, inner = bid - outer * INNER;      // y sweep: outer = x; x sweep: outer = y
            base = (long long)outer * (AX == AX_Y ? N * N : N) + (long long)inner * C::W;
        }
    }
    WDM_DEV long long at(int row, int l) const { return base + (long long)row * RSTRIDE + (long long)l * LSTRIDE; }
};

// thread -> (butterfly g, line l).  Strided tiles: lines fastest (a half-warp owns one 128-byte row).
// Contiguous tiles, when the stage touches global memory: points fastest (a warp reads one pencil).
template <int AX, int NB, int W>
WDM_DEV void split(int b, int &g, int &l)
{
    if (ax_strided(AX)) { l = b % W; g = b / W; }
    else { g = b % NB; l = b / NB; }
}

enum { H_Y_FWD = 0, H_Z_GREEN = 1, H_Y_INV = 2 };

// per-thread accumulators of a DIAG sweep, kept for the whole kernel and reduced once per CTA at its end
struct DiagAcc {
    double s0 = 0.0, s1 = 0.0, mx = 0.0;
};
enum { DIAG_COUNT = 8 };
// block reduction of (s0, s1, mx) over the CTA and one atomic each into d[i0], d[i1], d[imx] (an index < 0: nothing)
__device__ __forceinline__ void diag_flush(double *d, const DiagAcc &a, int i0, int i1, int imx)
{
    __shared__ double r0[32], r1[32], rm[32];
    double s0 = a.s0, s1 = a.s1, mx = a.mx;
    for (int o = 16; o; o >>= 1) {
        s0 += __shfl_down_sync(0xffffffffu, s0, o);
        s1 += __shfl_down_sync(0xffffffffu, s1, o);
        mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
    }
    const int w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if ((threadIdx.x & 31) == 0) { r0[w] = s0; r1[w] = s1; rm[w] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < nw; ++k) { s0 += r0[k]; s1 += r1[k]; mx = fmax(mx, rm[k]); }
        if (i0 >= 0) atomicAdd(d + i0, s0);
        if (i1 >= 0) atomicAdd(d + i1, s1);
        if (imx >= 0) atomicMax(reinterpret_cast<unsigned long long *>(d + imx), (unsigned long long)__double_as_longlong(mx));
    }
}

}  // namespace wdm
