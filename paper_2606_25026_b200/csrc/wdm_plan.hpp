// wdm_plan.hpp -- host-side plan: factorisation of a line and the lookup tables the sweeps read.
// Pure host C++ (no CUDA).  Tables are computed in double and rounded once to the grid precision.
#pragma once

#include <cmath>
#include <cstdint>
#include <vector>

#include "wdm_fft.cuh"

namespace wdm {

struct Fact {
    int N, RA, RB, RM, W, NT, NG, MINB;
};

// One factorisation per (N, dtype): X(N, RA, RB, RM, W, NT, NG, MINB); wdm_sweeps.cu instantiates the same rows.
// complex64 : two levels, radix <= 32 (a radix-32 butterfly is 64 registers of data).
// complex128: radix <= 16 (a radix-16 butterfly is already 64 registers), three levels for N >= 512.
// W lines per tile (128-byte rows where shared memory allows), NT threads per compute group, NG groups and
// NG + 1 tile buffers per CTA, MINB CTAs per SM.
#define WDM_FACT_C64(X)             \
    X(8, 2, 1, 4, 8, 32, 2, 4)      \
    X(16, 4, 1, 4, 16, 64, 2, 4)    \
    X(32, 4, 1, 8, 16, 128, 2, 4)   \
    X(64, 8, 1, 8, 16, 128, 2, 4)   \
    X(128, 8, 1, 16, 16, 128, 2, 2) \
    X(256, 16, 1, 16, 16, 128, 2, 2) \
    X(512, 16, 1, 32, 16, 256, 2, 1) \
    X(1024, 32, 1, 32, 8, 256, 2, 1)
#define WDM_FACT_C128(X)            \
    X(8, 2, 1, 4, 8, 32, 2, 4)      \
    X(16, 4, 1, 4, 8, 32, 2, 4)     \
    X(32, 4, 1, 8, 8, 64, 2, 4)     \
    X(64, 8, 1, 8, 8, 64, 2, 2)     \
    X(128, 8, 1, 16, 8, 64, 2, 2)   \
    X(256, 16, 1, 16, 8, 128, 2, 1) \
    X(512, 8, 8, 8, 8, 256, 2, 1)   \
    X(1024, 8, 8, 16, 4, 256, 1, 1)

inline bool find_fact(int N, int dtype, Fact &f)
{
#define X(n, ra, rb, rm, w, nt, ng, minb) \
    if (N == n) { f = Fact{n, ra, rb, rm, w, nt, ng, minb}; return true; }
    if (dtype == 0) { WDM_FACT_C64(X) }
    else { WDM_FACT_C128(X) }
#undef X
    return false;
}

template <typename T>
struct Tables {
    std::vector<cx<T>> twA, twB;           // s-major twiddles of level A (N entries) and level B (MB entries)
    std::vector<T> ksq_pos, ksq_nat;       // N each
};

inline double wavenumber(int k, int N, double L)
{
    int s = k < N / 2 ? k : k - N;   // reading G4: j >= N/2 maps to j - N
    return 2.0 * M_PI * (double)s / L;
}

template <typename T>
inline cx<T> unit_root(long long num, long long den)   // exp(-2 pi i num/den)
{
    num %= den;
    long double a = -2.0L * 3.14159265358979323846264338327950288L * (long double)num / (long double)den;
    return mk<T>((T)cosl(a), (T)sinl(a));
}

template <typename T>
inline Tables<T> build_tables(const Fact &f, double L)
{
    Tables<T> t;
    const int N = f.N, mA = N / f.RA, MB = N / f.RA, mB = MB / f.RB;
    t.twA.resize(N);
    for (int s = 0; s < f.RA; ++s)
        for (int q = 0; q < mA; ++q) t.twA[s * mA + q] = unit_root<T>((long long)q * s, N);
    t.twB.resize(f.RB > 1 ? MB : 1);
    t.twB[0] = mk<T>(1, 0);
    if (f.RB > 1)
        for (int s = 0; s < f.RB; ++s)
            for (int q = 0; q < mB; ++q) t.twB[s * mB + q] = unit_root<T>((long long)q * s, MB);
    t.ksq_pos.resize(N);
    t.ksq_nat.resize(N);
    for (int p = 0; p < N; ++p) {
        int k = k_of_pos(p, f.RA, f.RB, f.RM);
        double kk = wavenumber(k, N, L);
        t.ksq_pos[p] = (T)(kk * kk);
    }
    for (int k = 0; k < N; ++k) {
        double kk = wavenumber(k, N, L);
        t.ksq_nat[k] = (T)(kk * kk);
    }
    return t;
}

// per-axis kinetic factor exp(-i mu k^2 dt/2) / N in position order (Eq. 18(b); the 1/N is
// the inverse transform's normalisation for this axis)
template <typename T>
inline std::vector<cx<T>> build_phase(const Fact &f, double L, double mu, double dt)
{
    std::vector<cx<T>> ph(f.N);
    for (int p = 0; p < f.N; ++p) {
        double kk = wavenumber(k_of_pos(p, f.RA, f.RB, f.RM), f.N, L);
        double th = -0.5 * mu * kk * kk * dt;
        ph[p] = mk<T>((T)(std::cos(th) / f.N), (T)(std::sin(th) / f.N));
    }
    return ph;
}

// Tables of the half-tile x sweeps (wdm_x2.cuh): a line of N points as two half lines one radix-2 stage apart.
//   static part : [level-A twiddles of the N/2-point transform (s-major): N/2 | w^n = exp(-2 pi i n / N), n < N/2 : N/2]
//   phase part  : the per-axis kinetic factor / N (build_phase) of frequency 2 k' and of 2 k' + 1 at the position of k' in
//                 the N/2-point transform: [even: N/2 | odd: N/2]
template <typename T>
inline std::vector<cx<T>> build_x2_static(int N, const Fact &half)
{
    const int NH = N / 2, mA = NH / half.RA;
    std::vector<cx<T>> t(2 * (size_t)NH);
    for (int s = 0; s < half.RA; ++s)
        for (int q = 0; q < mA; ++q) t[s * mA + q] = unit_root<T>((long long)q * s, NH);
    for (int n = 0; n < NH; ++n) t[NH + n] = unit_root<T>(n, N);
    return t;
}

template <typename T>
inline std::vector<cx<T>> build_x2_phase(int N, const Fact &half, double L, double mu, double dt)
{
    const int NH = N / 2;
    std::vector<cx<T>> t(2 * (size_t)NH);
    for (int p = 0; p < NH; ++p) {
        const int k5 = k_of_pos(p, half.RA, half.RB, half.RM);
        for (int odd = 0; odd < 2; ++odd) {
            const double kk = wavenumber(2 * k5 + odd, N, L), th = -0.5 * mu * kk * kk * dt;
            t[odd * NH + p] = mk<T>((T)(std::cos(th) / N), (T)(std::sin(th) / N));
        }
    }
    return t;
}

}  // namespace wdm
