// wdm_x2.cuh -- the x-direction psi sweep and density sweep of 1024-point complex64 lines on 16-line tiles.
//
// Why a kernel of its own.  Along x every row of a tile lies in a different 2 MB page (rows are N^2 elements = 8 MB
// apart), and the memory system serves about 47 G such rows per second whatever their length up to 128 bytes (measured
// with the sweep skeleton alone -- TMA loads into three 64 KB buffers, stores straight back: 64-byte rows 8 MB apart
// 3.0 TB/s, 128-byte rows 6.0 TB/s; 64-byte rows 8 KB apart 6.7 TB/s).  The generic sweep holds 1024-point lines in
// 64 KB tiles of W = 8 lines: 64-byte rows, and the x sweep (5.65 ms) and the density sweep (7.4 ms) of 1024^3 sat exactly
// on that row rate.  Three 128 KB tiles do not fit in shared memory, so a 16-line tile is kept as TWO 64 KB half tiles,
// rows x < N/2 (A) and x >= N/2 (B), one radix-2 stage apart:
//     u_n = a_n + b_n,  v_n = (a_n - b_n) w^n          (w = exp(-2 pi i / N), n < N/2; formed on the way into the first
//                                                        level: both groups read both buffers, group 0 writes u into A,
//                                                        group 1 writes v into B)
//     even frequencies = FFT_{N/2}(u), odd = FFT_{N/2}(v)  -> kinetic phase -> inverse: group 0 on A, group 1 on B, the
//                                                             paired 512-point stages of the generic sweep, in place
//     a_n = u'_n + conj(w^n) v'_n,  b_n = u'_n - conj(w^n) v'_n     -> 16-byte global stores, 128-byte rows (all 512 threads)
// Per 16-line tile (cycles, developer build with clock64 stamps): loads into the first level 2.7 k, half transforms 10.7 k,
// last cross stage with the 1024 rows of psi stores 5.9 k (the row rate again: 6 cycles per row and SM, and in this
// lock-step CTA nothing else runs meanwhile), packed real-to-complex levels 3.5 k, Hermitian split with 513 rows of H
// 2.2 k: 26 k against 30.6 k for the two 8-line tiles of the generic sweep.
// The k-th half tile of a CTA goes to buffer k mod 3: tile i uses buffers 2i, 2i + 1 (mod 3); when its last reads are
// done, half B of tile i + 1 and half A of tile i + 2 are requested into them (the density sweep, whose tail keeps the
// second buffer, requests that half A at the first barrier of the next tile).  The density sweep forms rho - <rho> from
// the outgoing registers, splits the packed real lines the same way (U = P_a + P_b, V = (P_a - P_b) w^n, both in the
// buffer of B so that A's can be refilled at once), and each group runs the packed 512-point transform and the Hermitian
// split of its half of the spectrum: even rows of H from group 0, odd rows (mirror of k' is N/2 - 1 - k') from group 1 --
// 128-byte rows of H.
#pragma once

#include "wdm_pipe.cuh"

namespace wdm {

template <class C5, bool RHO>
struct X2 {
    using T = typename C5::T;
    static constexpr int NH = C5::N, N2 = 2 * NH, W = C5::W, WP = W / 2, RA = C5::RA, RM = C5::RM, mA = C5::mA, NTG = C5::NT, NT = 2 * NTG;
    static_assert(C5::RB == 1 && C5::NG == 2 && pair_ok<C5>() && sizeof(T) == 4, "paired two-level half transform");
    static_assert((NH * WP) % NT == 0, "whole rounds of the cross stages");
    using L = Lay<C5, AX_X>;
    using PK = Packed<C5>;
    static constexpr int ITEMS = NH * WP / NT;                     // (row, line pair) items per thread in the cross stages
    static constexpr size_t TILE_BYTES = (size_t)NH * W * sizeof(cx<T>);
    static constexpr size_t CTRL = 3 * TILE_BYTES, TAB = CTRL + 64, TOTAL = TAB + 4 * (size_t)NH * sizeof(cx<T>);
    static_assert(2 * PK::ELEMS * sizeof(cx<T>) <= TILE_BYTES, "both packed half spectra in one buffer");
    static constexpr long long RSTRIDE = (long long)N2 * N2;
    static constexpr int INNER = N2 / W;

    static __device__ __forceinline__ void run(const SweepParams<T> &p, int ntiles, unsigned char *smem)
    {
        uint64_t *full = reinterpret_cast<uint64_t *>(smem + CTRL);
        volatile int *tiles = reinterpret_cast<volatile int *>(full + 3);          // tile of sequence number i at [i & 3]
        cx<T> *tw5 = reinterpret_cast<cx<T> *>(smem + TAB), *w2 = tw5 + NH, *phE = w2 + NH, *phO = phE + NH;
        const int tid = threadIdx.x, grp = tid / NTG, gt = tid - grp * NTG, bid = blockIdx.x, stride = gridDim.x;
        auto buf = [&](int j) { return reinterpret_cast<cx<T> *>(smem + (size_t)(j % 3) * TILE_BYTES); };
        // fill number j (half j & 1 of the CTA's tile j / 2) into buffer j mod 3
        auto issue = [&](int j, int t) {
            uint64_t *bar = full + j % 3;
            mbar_expect_tx(bar, (uint32_t)TILE_BYTES);
            const int outer = t / INNER, inner = t - outer * INNER;
#pragma unroll
            for (int k = 0; k < NH / 256; ++k)
                tma_load_3d(buf(j) + (size_t)k * 256 * W, &p.tmap2, inner * 2 * W, outer, (j & 1) * NH + k * 256, bar);
        };
        asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
        if (tid == 0) {
            for (int b = 0; b < 3; ++b) mbar_init(full + b, 1);
            tiles[0] = bid < ntiles ? bid : -1;
            tiles[1] = bid + stride < ntiles ? bid + stride : -1;
        }
        for (int i = tid; i < 4 * NH; i += NT) tw5[i] = p.x2tab[i];              // host-written before any launch
        asm volatile("griddepcontrol.wait;" ::: "memory");
        if (tid == 0 && bid == 0) *p.ticket_next = 0;
        __syncthreads();
        if (tid == 0) {
            if (tiles[0] >= 0) { issue(0, tiles[0]); issue(1, tiles[0]); }
            if (tiles[1] >= 0) issue(2, tiles[1]);
        }
        const int pq = gt / (W / 2), pl = 2 * (gt % (W / 2));         // paired mapping of the half transform's level A
        cx<T> w[RA];
        static_for<1, RA>([&](auto s_) { constexpr int s = decltype(s_)::value; w[s] = tw5[s * mA + pq]; });
        const T mean = RHO ? ldg(p.rho_mean) : (T)0;
        for (int i = 0;; ++i) {
            // tiles[i & 3] was written two tiles ago (or before the loop); every thread has passed a CTA barrier since
            const int t = tiles[i & 3];
            if (t < 0) break;
            unsigned tk = 0;
            if (tid == 0) tk = 2u * stride + atomicAdd(p.ticket, 1u);      // tile i + 2; consumed after the half transforms
            const int jA = 2 * i, jB = 2 * i + 1;
            cx<T> *SA = buf(jA), *SB = buf(jB);
            mbar_wait(full + jA % 3, (jA / 3) & 1);
            mbar_wait(full + jB % 3, (jB / 3) & 1);
            // ---- half transforms: forward, kinetic phase, inverse, in place (group 0: even frequencies in A, group 1: odd in B).
            // The radix-2 stage across the halves, u = a + b or v = (a - b) w^n, is formed on the way into the first level:
            // both groups read both buffers, then each writes its own.
            {
                cx<T> *S = grp ? SB : SA;
                const cx<T> *ph = grp ? phO : phE;
                {
                    cx<T> a[RA], c[RA];
                    static_for<0, RA>([&](auto r_) {
                        constexpr int r = decltype(r_)::value;
                        cx<T> a0, a1, b0, b1;
                        ld2(SA + L::idx(pq + mA * r, pl), a0, a1);
                        ld2(SB + L::idx(pq + mA * r, pl), b0, b1);
                        if (grp == 0) {
                            a[r] = cadd(a0, b0);
                            c[r] = cadd(a1, b1);
                        } else {
                            const cx<T> wn = w2[pq + mA * r];
                            a[r] = cmul(csub(a0, b0), wn);
                            c[r] = cmul(csub(a1, b1), wn);
                        }
                    });
                    if (RHO) fence_proxy_async();      // this thread's reads of the previous tile's packed spectra (buffer of fill 2i - 1)
                    __syncthreads();
                    if (RHO && tid == 0 && i > 0) {
                        const int t1 = tiles[(i + 1) & 3];
                        if (t1 >= 0) issue(2 * i + 2, t1);                     // half A of the next tile, into the buffer the previous tile's tail used
                    }
                    dif_fwd<RA>(a);
                    dif_fwd<RA>(c);
                    static_for<0, RA>([&](auto s_) {
                        constexpr int sdx = decltype(s_)::value;
                        cx<T> ya = a[brev(sdx, RA)], yc = c[brev(sdx, RA)];
                        if constexpr (sdx > 0) { ya = cmul(ya, w[sdx]); yc = cmul(yc, w[sdx]); }
                        st2(S + L::idx(pq + mA * sdx, pl), ya, yc);
                    });
                }
                group_sync(grp, NTG);
                for (int b = gt; b < (NH / RM) * W; b += NTG) {
                    const int l = b % W, g = b / W;
                    mid_both<RM, T>(g * RM, [&](int row) { return S[L::idx(row, l)]; }, [&](int row, cx<T> v) { S[L::idx(row, l)] = v; },
                                    [&](int pos, cx<T> &a, cx<T> &c) {
                                        cx<T> pa, pc;
                                        ld2(ph + pos, pa, pc);
                                        a = cmul(a, pa);
                                        c = cmul(c, pc);
                                    });
                }
                group_sync(grp, NTG);
                cx<T> a[RA], c[RA];
                inv_level_pair_regs<RA, T>(pq, mA, w, [&](int row, cx<T> &x, cx<T> &y) { ld2(S + L::idx(row, pl), x, y); }, a, c);
                static_for<0, RA>([&](auto r_) { constexpr int r = decltype(r_)::value; st2(S + L::idx(pq + mA * r, pl), a[r], c[r]); });
            }
            if (tid == 0) tiles[(i + 2) & 3] = tk < (unsigned)ntiles ? (int)tk : -1;
            __syncthreads();
            // ---- a = u' + conj(w^n) v', b = u' - conj(w^n) v': everything out of the buffers first, then their refills
            cx<T> u0[ITEMS], u1[ITEMS], v0[ITEMS], v1[ITEMS];
#pragma unroll
            for (int it = 0; it < ITEMS; ++it) {
                const int item = it * NT + tid, pr = item % WP, n = item / WP;
                ld2(SA + L::idx(n, 2 * pr), u0[it], u1[it]);
                ld2(SB + L::idx(n, 2 * pr), v0[it], v1[it]);
            }
            fence_proxy_async();
            __syncthreads();
            if (tid == 0) {
                const int t1 = tiles[(i + 1) & 3], t2 = tiles[(i + 2) & 3];
                if (t1 >= 0) issue(2 * i + 3, t1);                       // half B of the next tile, into A's buffer
                if (!RHO && t2 >= 0) issue(2 * i + 4, t2);               // half A of the one after, into B's (the density sweep still needs it)
            }
            const int outer = t / INNER, inner = t - outer * INNER;
            const long long base = (long long)outer * N2 + (long long)inner * W;
            const bool has_rho_p = RHO && p.rho_p != nullptr && p.rho_flag[outer * (N2 / 16) + (inner * W) / 16] != 0;
            cx<T> *Up = SB, *Vp = SB + PK::ELEMS;
#pragma unroll
            for (int it = 0; it < ITEMS; ++it) {
                const int item = it * NT + tid, pr = item % WP, n = item / WP;
                const cx<T> wn = w2[n];
                const cx<T> t0 = cmulc(v0[it], wn), t1 = cmulc(v1[it], wn);
                const cx<T> a0 = cadd(u0[it], t0), a1 = cadd(u1[it], t1), b0 = csub(u0[it], t0), b1 = csub(u1[it], t1);
                cx<T> *gp = p.data + base + (long long)n * RSTRIDE + 2 * pr;
                stg2(gp, a0, a1);
                stg2(gp + (long long)NH * RSTRIDE, b0, b1);
                if constexpr (RHO) {
                    T ra0 = a0.x * a0.x + a0.y * a0.y, ra1 = a1.x * a1.x + a1.y * a1.y;
                    T rb0 = b0.x * b0.x + b0.y * b0.y, rb1 = b1.x * b1.x + b1.y * b1.y;
                    if (has_rho_p) {
                        const T *rp = p.rho_p + base + (long long)n * RSTRIDE + 2 * pr;
                        T e0, e1;
                        ld2r(rp, e0, e1);
                        ra0 += e0; ra1 += e1;
                        ld2r(rp + (long long)NH * RSTRIDE, e0, e1);
                        rb0 += e0; rb1 += e1;
                    }
                    // packed line pr = lines 2 pr (real part), 2 pr + 1 (imaginary part); <rho> leaves with the k = 0 mode only
                    Up[PK::idx(n, pr)] = mk<T>(ra0 + rb0 - 2 * mean, ra1 + rb1 - 2 * mean);
                    Vp[PK::idx(n, pr)] = cmul(mk<T>(ra0 - rb0, ra1 - rb1), wn);
                }
            }
            if constexpr (RHO) {
                __syncthreads();
                cx<T> *Sp = grp ? Vp : Up;
                for (int b = gt; b < mA * WP; b += NTG) {
                    const int l = b % WP, q = b / WP;
                    fwd_level<RA, T>(q, mA, tw5 + q, [&](int row) { return Sp[PK::idxA(q, row - q, l)]; },
                                     [&](int row, cx<T> v) { Sp[PK::idxA(q, row - q, l)] = v; });
                }
                group_sync(grp, NTG);
                for (int b = gt; b < (NH / RM) * WP; b += NTG) {
                    const int l = b % WP, g = b / WP;
                    mid_fwd<RM, T>(g * RM, [&](int row) { return Sp[PK::idxM(g * RM, row - g * RM, l)]; },
                                   [&](int row, cx<T> v) { Sp[PK::idxM(g * RM, row - g * RM, l)] = v; });
                }
                group_sync(grp, NTG);
                // A_k = (Z_k + conj Z_{N-k})/2,  B_k = (Z_k - conj Z_{N-k})/(2i) -> H[k][lines 2l, 2l+1]
                auto emit = [&](int k, int e, int en, int l) {
                    const cx<T> zk = Sp[e], zn = Sp[en];
                    const T h = (T)0.5;
                    st2(p.H + base + (long long)k * RSTRIDE + 2 * l, mk<T>((zk.x + zn.x) * h, (zk.y - zn.y) * h), mk<T>((zk.y + zn.y) * h, (zn.x - zk.x) * h));
                };
                if (grp == 0) {
                    // even k = 2 k': the half transform's own Hermitian pairs (k', NH - k'), k' <= NH/2
                    half_spectrum_items<C5, WP, PK>(gt, [&](int k, int e, int en, int l) { emit(2 * k, e, en, l); });
                    if (gt < WP) {
                        const int e = PK::idx(HalfSpec<C5>::row_of(NH / 2), gt);
                        emit(NH, e, e, gt);
                    }
                } else {
                    // odd k = 2 k' + 1 <= N/2 - 1: N - k = 2 (NH - 1 - k') + 1
                    for (int b = gt; b < (NH / 2) * WP; b += NTG) {
                        const int l = b % WP;
                        int k, row;
                        HalfSpec<C5>::nth(b / WP, k, row);
                        emit(2 * k + 1, PK::idx(row, l), PK::idx(HalfSpec<C5>::row_of(NH - 1 - k), l), l);
                    }
                }
            }
        }
    }
};

}  // namespace wdm
