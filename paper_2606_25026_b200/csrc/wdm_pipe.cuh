// wdm_pipe.cuh -- persistent, software-pipelined form of the axis sweeps (sm_100a).
//
// One CTA per SM.  The CTA is NG "compute groups" of C::NT threads over NG + 1 shared-memory tile buffers; the
// k-th tile of the CTA is transformed by group k % NG inside buffer k % (NG + 1).  The first NG + 1 tiles are
// blockIdx.x + k * gridDim.x, every later one is a ticket from a device-wide counter (fast SMs take more tiles).
// A tile is brought in by TMA -- 3-D tensor boxes for strided tiles, one bulk copy per pencil for contiguous
// tiles -- issued by the first warp of the group that has just finished with the buffer, for the tile NG + 1
// positions ahead, so every load has more than one whole tile-compute time of lead and HBM latency never reaches
// the math.  Results leave through 8 / 16-byte global stores.
//
//   full[b]   mbarrier, count 1: the issuing lane's arrive.expect_tx carries the tile's byte count, the copies
//             complete_tx on it; the consuming group waits on the phase parity (k / NBUF) & 1.
//   issued[b] fills of buffer b started so far; tile_of[b] the tile of the current fill (-1: nothing left).  A
//             parity wait cannot tell a phase from the one two before it, so the consumer's first warp polls
//             issued[b] before the group waits on full[b].
//   group barrier: bar.sync (1 + group), C::NT -- the other group is never stalled by it.
#pragma once

#include "wdm_kernels.cuh"

namespace wdm {

// ---------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, int parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WDM_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WDM_DONE;\n"
        "bra WDM_WAIT;\n"
        "WDM_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// TMA: the mbarrier of a tile buffer has ONE expected arrival -- the issuing thread's arrive.expect_tx with the
// tile's byte count -- and completes when the bulk copies have delivered that many bytes.
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, uint64_t *bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                     smem_u32(dst)),
                 "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// orders this thread's earlier shared-memory accesses (generic proxy) before later bulk copies (async proxy)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void group_sync(int group, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "r"(nthreads) : "memory");
}

// ---------------------------------------------------------------- the pipeline driver
// K provides:  using C;  TILE_BYTES;  AUX;  struct Pre;  issue(p, tile, buf, gt);  prefetch(p, tile, gt, pre);
//              compute(p, tabs, tile, next_tile, buf, gt, grp, pre)

// Lookup tables of the sweep.  A persistent CTA copies them into shared memory ONCE (they are read by every
// butterfly of every tile: from global memory each read is an L1 round trip on the long scoreboard).
template <typename T>
struct Tabs {
    const cx<T> *twA, *twB, *phase;
    const T *ksq_pos;
};
enum { AUX_NONE = 0, AUX_PHASE = 1, AUX_KSQ = 2 };

// Paired mapping of the level-A stages on a strided tile: thread gt owns the butterflies q = gt / (W/2) of
// the two adjacent lines 2 (gt % (W/2)) and + 1 -- 16-byte shared-memory accesses, and ONE set of twiddles,
// which is the same for every tile the thread will ever see: PairTw keeps it in registers for the whole kernel.
template <class C>
constexpr bool pair_ok() { return sizeof(typename C::T) == 4 && C::mA * C::W == 2 * C::NT && C::RA * sizeof(typename C::T) <= 64; }

template <class C, bool ON>
struct PairTw {
    using T = typename C::T;
    cx<T> w[ON ? C::RA : 1];
    __device__ __forceinline__ void setup(const Tabs<T> &tb, int gt)
    {
        if constexpr (ON) {
            const int q = gt / (C::W / 2);
            static_for<1, C::RA>([&](auto s_) { constexpr int s = decltype(s_)::value; w[s] = tb.twA[s * C::mA + q]; });
        }
    }
};
constexpr size_t kMaxSmem = 227 * 1024;

template <class K>
struct PipeSmem {
    using C = typename K::C;
    using T = typename C::T;
    static constexpr size_t CTRL = (size_t)(C::NG + 1) * K::TILE_BYTES;          // mbarriers + issued[]
    static constexpr size_t TWA = CTRL + 64;
    static constexpr size_t TWA_BYTES = (size_t)C::N * sizeof(cx<T>);
    static constexpr size_t TWB_BYTES = C::RB > 1 ? (size_t)C::MB * sizeof(cx<T>) : 0;
    static constexpr size_t AUX_BYTES = K::AUX == AUX_PHASE ? (size_t)C::N * sizeof(cx<T>) : (K::AUX == AUX_KSQ ? (size_t)C::N * sizeof(T) : 0);
    static constexpr bool TW_IN_SMEM = TWA + TWA_BYTES + TWB_BYTES <= kMaxSmem;
    static constexpr size_t AUX_OFF = TWA + (TW_IN_SMEM ? TWA_BYTES + TWB_BYTES : 0);
    static constexpr bool AUX_IN_SMEM = K::AUX != AUX_NONE && AUX_OFF + AUX_BYTES <= kMaxSmem;
    static constexpr size_t TOTAL = AUX_OFF + (AUX_IN_SMEM ? AUX_BYTES : 0);
};

template <class K>
__device__ __forceinline__ void pipe_run(const SweepParams<typename K::C::T> &p, int ntiles, unsigned char *smem)
{
    using C = typename K::C;
    constexpr int NTG = C::NT, NG = C::NG, NBUF = NG + 1;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)NBUF * K::TILE_BYTES);
    // issued[b] = number of fills of buffer b started so far.  A parity wait can only tell the current phase
    // from the one before it, so a consumer that has run ahead first makes sure the fill it needs has been
    // STARTED (which implies the previous phase completed) before waiting on the parity.
    volatile int *issued = reinterpret_cast<volatile int *>(full + NBUF);
    const int tid = threadIdx.x, grp = tid / NTG, gt = tid - grp * NTG;
    const int bid = blockIdx.x, stride = gridDim.x;
    // Tile assignment.  The k-th tile of a CTA is computed by group k % NG in buffer k % NBUF; tile_of[b] is the
    // global tile index of the current fill of buffer b, or -1 when there is nothing left.  The first NBUF tiles
    // are static (bid + k * grid); every later one is a ticket from a device-wide counter, drawn when the tile
    // whose buffer it will take starts computing -- SMs that run faster (the sweeps are memory bound, and not
    // every SM sees the same share of the bandwidth) simply take more tiles.
    volatile int *tile_of = issued + NBUF;
    static_assert(NBUF * (sizeof(uint64_t) + 2 * sizeof(int)) <= 64, "control block");
    const int nstatic = NBUF * stride;
    // Programmatic dependent launch: let the next sweep's CTAs take SMs as this grid's CTAs retire, and do everything
    // that does not depend on the previous kernel (control block, lookup tables: written by the host before any
    // launch) before waiting for it -- the launch latency and this prologue then hide behind the predecessor's tail.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (tid == 0)
        for (int b = 0; b < NBUF; ++b) {
            mbar_init(full + b, 1);
            const int t0 = bid + b * stride;
            tile_of[b] = t0 < ntiles ? (p.reverse ? ntiles - 1 - t0 : t0) : -1;
            issued[b] = 1;
        }
    using SM = PipeSmem<K>;
    using T = typename C::T;
    Tabs<T> tb{p.twA, p.twB, p.phase, p.ksq_pos};
    if constexpr (SM::TW_IN_SMEM) {
        cx<T> *a = reinterpret_cast<cx<T> *>(smem + SM::TWA);
        for (int i = tid; i < C::N; i += NTG * NG) a[i] = p.twA[i];
        tb.twA = a;
        if constexpr (C::RB > 1) {
            cx<T> *b2 = a + C::N;
            for (int i = tid; i < C::MB; i += NTG * NG) b2[i] = p.twB[i];
            tb.twB = b2;
        }
    }
    if constexpr (SM::AUX_IN_SMEM && K::AUX == AUX_PHASE) {
        cx<T> *a = reinterpret_cast<cx<T> *>(smem + SM::AUX_OFF);
        for (int i = tid; i < C::N; i += NTG * NG) a[i] = p.phase[i];
        tb.phase = a;
    }
    if constexpr (SM::AUX_IN_SMEM && K::AUX == AUX_KSQ) {
        T *a = reinterpret_cast<T *>(smem + SM::AUX_OFF);
        for (int i = tid; i < C::N; i += NTG * NG) a[i] = p.ksq_pos[i];
        tb.ksq_pos = a;
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");         // the previous kernel on the stream is complete and visible
    if (tid == 0 && bid == 0) *p.ticket_next = 0;               // the launch before this one has finished with it
    if constexpr (K::DG == 1)
        if (bid == 0 && tid < DIAG_COUNT && p.diag_zero && K::DIAG_ZEROES) p.diag_zero[tid] = 0.0;
    __syncthreads();
    for (int k = 0; k < NBUF; ++k)
        if (k % NG == grp && gt < 32 && tile_of[k] >= 0) K::issue(p, tile_of[k], smem + (size_t)k * K::TILE_BYTES, full + k, gt);
    typename K::Pre pre;
    typename K::Pers pers;
    pers.setup(tb, gt);
    int pre_tile = -1;                                          // tile whose prefetched operands `pre` holds
    for (int k = grp;; k += NG) {
        const int b = k % NBUF;
        unsigned char *buf = smem + (size_t)b * K::TILE_BYTES;
        // one warp polls for the start of this fill (the others would only burn issue slots the other group needs)
        if (gt < 32)
            while (issued[b] < k / NBUF + 1) __nanosleep(100);
        group_sync(grp, NTG);
        const int t = tile_of[b];
        if (t < 0) {
            // nothing left for this group: pass the end mark on to the tile that would have followed in this
            // buffer (its owner may still be waiting for it)
            if (gt == 0) issued[b] = (k + NBUF) / NBUF + 1;
            break;
        }
        unsigned int ticket = 0;
        if (gt == 0) ticket = (unsigned int)nstatic + atomicAdd(p.ticket, 1u);   // consumed after the compute: latency hidden
        mbar_wait(full + b, (k / NBUF) & 1);
        if (pre_tile != t) K::prefetch(p, t, gt, pre);
        // called by compute() before its last stage: fetch what the group's NEXT tile needs into registers, if
        // that tile has been assigned by now
        auto hook = [&]() {
            const int b2 = (k + NG) % NBUF;
            if (issued[b2] >= (k + NG) / NBUF + 1) {
                const int t2 = tile_of[b2];
                if (t2 >= 0) { K::prefetch(p, t2, gt, pre); pre_tile = t2; }
            }
        };
        K::compute(p, tb, t, buf, gt, grp, pre, pers, hook);
        fence_proxy_async();                                    // this thread's accesses to the buffer, before its refill
        group_sync(grp, NTG);                                   // every read of this buffer is done
        if (gt < 32) {
            int tn = (int)__shfl_sync(0xffffffffu, ticket, 0);
            if (tn >= ntiles) tn = -1;
            else if (p.reverse) tn = ntiles - 1 - tn;
            if (gt == 0) {
                tile_of[b] = tn;
                __threadfence_block();
                issued[b] = (k + NBUF) / NBUF + 1;
            }
            if (tn >= 0) K::issue(p, tn, buf, full + b, gt);
        }
    }
    if constexpr (K::DG != 0) {
        __syncthreads();
        K::flush(p, pre);
    }
}

// ---------------------------------------------------------------- shared building blocks

// Asynchronous tile load by the first warp of a group (lane = gt < 32): lane 0 announces the byte count and issues
// the TMA boxes of a strided tile; a contiguous tile is one bulk copy per pencil (its shared-memory lines are
// padded, which a box cannot express), lane l issuing pencils l, l + 32, ....  `bid` is the
// tile index, ROWS the number of points along the sweep axis to fetch, tm1 the one-row box used when ROWS is
// not a multiple of the main box (complex-to-real: N/2 + 1 rows).
template <class C, int AX, int ROWS>
__device__ __forceinline__ void tile_load(cx<typename C::T> *S, const cx<typename C::T> *src, const CUtensorMap *tm, const CUtensorMap *tm1,
                                          int bid, uint64_t *bar, int lane)
{
    using T = typename C::T;
    using L = Lay<C, AX>;
    using TL = Tile<C, AX>;
    constexpr int W = C::W;
    constexpr uint32_t BYTES = (uint32_t)((size_t)ROWS * W * sizeof(cx<T>));
    if (lane == 0) mbar_expect_tx(bar, BYTES);
    if constexpr (ax_strided(AX)) {
        if (lane != 0) return;
        constexpr int EVEN = ROWS & ~1;                                  // ROWS = N, or N/2 + 1
        constexpr int RB = EVEN < 256 ? EVEN : 256;                      // rows per box (as encoded on the host)
        constexpr int FULL = ROWS / RB;
        const int outer = bid / TL::INNER, inner = bid - outer * TL::INNER;
        const int c0 = inner * 2 * W;
#pragma unroll
        for (int k = 0; k < FULL; ++k) {
            if (AX == AX_Y) tma_load_3d(S + (size_t)k * RB * W, tm, c0, k * RB, outer, bar);
            else tma_load_3d(S + (size_t)k * RB * W, tm, c0, outer, k * RB, bar);
        }
        if constexpr (ROWS - FULL * RB > 0) {
            static_assert(ROWS - FULL * RB == 1, "only the half spectrum has an odd row");
            if (AX == AX_Y) tma_load_3d(S + (size_t)FULL * RB * W, tm1, c0, FULL * RB, outer, bar);
            else tma_load_3d(S + (size_t)FULL * RB * W, tm1, c0, outer, FULL * RB, bar);
        }
    } else {
        const TL tile(bid);
        for (int l = lane; l < W; l += 32)
            bulk_load(S + L::idx(0, l), src + tile.at(0, l), (uint32_t)(ROWS * sizeof(cx<T>)), bar);
    }
}

// level B stages with the group barrier
// (IDX maps (row, line) to the shared-memory element index)
template <class C, int W, class IDX, typename T>
__device__ __forceinline__ void g_fwd_B(cx<T> *S, const cx<T> *twB, int gt, int grp, IDX idx)
{
    if constexpr (C::RB > 1) {
        constexpr int NB = C::N / C::RB;
        for (int b = gt; b < NB * W; b += C::NT) {
            int l = b % W, g = b / W, blk = g / C::mB, q = g - blk * C::mB;
            fwd_level<C::RB, T>(blk * C::MB + q, C::mB, twB + q, [&](int row) { return S[idx(row, l)]; },
                                [&](int row, cx<T> v) { S[idx(row, l)] = v; });
        }
        group_sync(grp, C::NT);
    }
}
template <class C, int W, class IDX, typename T>
__device__ __forceinline__ void g_inv_B(cx<T> *S, const cx<T> *twB, int gt, int grp, IDX idx)
{
    if constexpr (C::RB > 1) {
        constexpr int NB = C::N / C::RB;
        for (int b = gt; b < NB * W; b += C::NT) {
            int l = b % W, g = b / W, blk = g / C::mB, q = g - blk * C::mB;
            inv_level<C::RB, T>(blk * C::MB + q, C::mB, twB + q, [&](int row) { return S[idx(row, l)]; },
                                [&](int row, cx<T> v) { S[idx(row, l)] = v; });
        }
        group_sync(grp, C::NT);
    }
}

// Frequencies k < N/2 enumerated so that consecutive indices sit in consecutive shared-memory rows
// (k = sA + RA (sB + RB sM) lives at row (sA RB + sB) RM + sM; k < N/2 <=> sM < RM/2).  Returns k and its row;
// row_of(k) gives the row of any frequency.  All divisors are powers of two.
template <class C>
struct HalfSpec {
    static constexpr int HM = C::RM / 2;
    static __device__ __forceinline__ int row_of(int k)
    {
        int sA = k % C::RA, sB = (k / C::RA) % C::RB, sM = k / (C::RA * C::RB);
        return (sA * C::RB + sB) * C::RM + sM;
    }
    static __device__ __forceinline__ void nth(int kk, int &k, int &row)
    {
        int sM = kk % HM, sAB = kk / HM, sA = sAB / C::RB, sB = sAB % C::RB;
        k = sA + C::RA * (sB + C::RB * sM);
        row = sAB * C::RM + sM;
    }
};

// Packed tile of the real-data transforms: N rows x W/2 complex (two real lines per complex line).  With 64-byte
// rows two rows share a 128-byte bank line; the middle level reads rows a multiple of RM apart from neighbouring
// lanes, which would land in the same half.  Rows whose bit log2(RM) is set therefore swap places with their
// neighbour (row ^ 1): every access pattern of the sweeps (level A: rows q, q + 1; middle: g RM + s, (g+1) RM + s;
// the Hermitian split: consecutive rows) then touches both halves.
// (Measured at 512^3: -2 % on the density sweep.  Through idx() the swizzle costs three integer instructions per
// access, which the latency-bound complex-to-real sweep lost more to than it gained; with idxA / idxM it is free,
// and that sweep's middle level drops its 2-way conflicts: 8.4 M of 29.6 M wavefronts per launch, -5 %.)
template <class C, bool ON = true>
struct Packed {
    using T = typename C::T;
    static constexpr int RSP = C::W / 2;
    static constexpr bool SWZ = ON && RSP * sizeof(cx<T>) == 64 && C::RB == 1;
    // 32-byte rows (W = 8 complex64 / W = 4 complex128: the 1024-point tiles).  The middle level reads rows a multiple of
    // RM apart from neighbouring lanes: RM * 32 bytes apart, i.e. in the same 8 banks -- an 8-way conflict (ncu at 1024^3:
    // 2.4e8 conflicts in 6.4e8 instructions of the complex-to-real sweep, short-scoreboard stalls 9 per issue).  One
    // empty row after every RM rows shifts consecutive blocks by 32 bytes: four blocks cover all banks.
    static constexpr bool PADROW = ON && RSP * sizeof(cx<T>) == 32 && C::RB == 1;
    static constexpr int BLK = (C::RM + (PADROW ? 1 : 0)) * RSP;          // elements from row r to row r + RM
    static constexpr size_t ELEMS = (size_t)(C::N + (PADROW ? C::N / C::RM : 0)) * RSP;
    static __device__ __forceinline__ int idx(int row, int l)
    {
        if constexpr (SWZ) row ^= (row / C::RM) & 1;
        if constexpr (PADROW) row += row / C::RM;
        return row * RSP + l;
    }
    // The same index for the two access patterns of the stages, written so that the swizzle / padding costs nothing per
    // access once the stage is unrolled (d a compile-time constant): two base addresses per thread, the rest
    // immediates.  idxA: row q + d of a level-A butterfly (q < RM, d a multiple of RM; RB == 1 so mA == RM).
    // idxM: row row0 + d of a middle-level butterfly (row0 a multiple of RM, d < RM).
    static __device__ __forceinline__ int idxA(int q, int d, int l)
    {
        if constexpr (SWZ) return ((q ^ ((d / C::RM) & 1)) + d) * RSP + l;
        else if constexpr (PADROW) return (q + d + d / C::RM) * RSP + l;
        else return (q + d) * RSP + l;
    }
    static __device__ __forceinline__ int idxM(int row0, int d, int l)
    {
        if constexpr (SWZ) {
            const int b = ((row0 / C::RM) & 1) * RSP;
            return (row0 + d) * RSP + l + ((d & 1) ? -b : b);
        } else if constexpr (PADROW) return (row0 + row0 / C::RM + d) * RSP + l;
        else return (row0 + d) * RSP + l;
    }
};

// The frequencies k < N/2 of the packed lines, spread over a group's threads: item b = gt + i NT is packed line
// b % WP, frequency number b / WP (HalfSpec::nth).  f(k, e, en, l): e / en = shared-memory element (PK::idx) of
// frequency k / of its mirror N - k in line l.  When the group's stride NT / WP is an even multiple DA of RM/2 (and
// RB == 1), item i of a thread is frequency k0 + DA i, at rows a fixed distance apart, and so is its mirror from
// i = 1 on (an even DA also keeps the swizzle bit of Packed the same): the indices are formed once per tile and
// every later item is an immediate offset -- the index arithmetic was 40 % of the complex-to-real sweep's
// instructions (ncu, profiles/r1e).
template <class C, int WP, class PK, class F>
__device__ __forceinline__ void half_spectrum_items(int gt, F &&f)
{
    constexpr int NT = C::NT, HM = C::RM / 2, ITEMS = (C::N / 2) * WP;
    constexpr bool FAST = C::RB == 1 && NT % WP == 0 && (NT / WP) % (2 * HM) == 0 && ITEMS % NT == 0 && ITEMS / NT <= 16;
    if constexpr (FAST) {
        constexpr int DA = NT / WP / HM, ITERS = ITEMS / NT, STEP = DA * PK::BLK;
        static_assert(ITERS * DA == C::RA && PK::RSP == WP, "item i of a thread is frequency k0 + DA i");
        const int l = gt % WP, kk0 = gt / WP, sM = kk0 % HM, sA0 = kk0 / HM;
        const int k0 = sA0 + C::RA * sM;
        const int e0 = PK::idx(sA0 * C::RM + sM, l);
        const int en0 = PK::idx(HalfSpec<C>::row_of((C::N - k0) & (C::N - 1)), l);
        // k = sA + RA sM with sA > 0:  N - k = (RA - sA) + RA (RM - 1 - sM)
        const int en1 = PK::idx((C::RA - sA0 - DA) * C::RM + (C::RM - 1 - sM), l);
        f(k0, e0, en0, l);
        static_for<1, ITERS>([&](auto i_) {
            constexpr int i = decltype(i_)::value;
            f(k0 + DA * i, e0 + i * STEP, en1 - (i - 1) * STEP, l);
        });
    } else {
        for (int b = gt; b < ITEMS; b += NT) {
            int l = b % WP, k, pk;
            HalfSpec<C>::nth(b / WP, k, pk);
            f(k, PK::idx(pk, l), PK::idx(HalfSpec<C>::row_of((C::N - k) & (C::N - 1)), l), l);
        }
    }
}

struct NoPre { DiagAcc d; };

constexpr size_t align128(size_t x) { return (x + 127) & ~(size_t)127; }

// ---------------------------------------------------------------- psi sweep
// DRIFT: FFT . per-axis kinetic phase . inverse FFT (Eq. 18(b)).  KICK: psi *= exp(-i Phi kick) as the tile
// leaves shared memory for the first butterfly (Eq. 18(a),(d)); the Phi values of the NEXT tile are fetched
// into registers before the current tile's last stage.  RHO (x axis): rho - <rho> = |psi2|^2 (+ rho_p) - <rho>
// formed from the outgoing registers, packed real-to-complex FFT along x in the same buffer -> H.
// KICK: 0 none, 1 plain potential kick, 2 with the extra terms of SweepParams::kick_extra (a separate
// instantiation, so the plain kernel carries none of their code or registers).
// DG_: 0 no diagnostics; 1 accumulate the per-step diagnostics on the way (sum k^2 |F psi|^2 of this axis in the middle
// level -- the drift multiplies the spectrum by unit-modulus factors, so each axis sweep sees the kinetic energy of
// its own axis; with RHO also sum and max of |psi_2|^2 from the outgoing registers); 2 measure only: forward transform,
// accumulate, nothing written (the on-demand kinetic energy of wdm_get_diagnostics).
template <class C_, int AX, int KICK, bool RHO, bool DRIFT, int DG_ = 0>
struct PsiK {
    static constexpr int DG = DG_;
    static constexpr bool DIAG_ZEROES = AX == AX_CONTIG;        // the z sweep opens a step
    static_assert(DG_ != 2 || (KICK == 0 && !RHO && DRIFT), "measure-only sweeps are plain forward transforms");
    using C = C_;
    using T = typename C::T;
    using TL = Tile<C, AX>;
    using L = Lay<C, AX>;
    static constexpr int N = C::N, RA = C::RA, RM = C::RM, W = C::W, NTG = C::NT, mA = C::mA;
    static constexpr int ITER = (mA * W) / NTG;
    static_assert((mA * W) % NTG == 0, "whole number of level-A butterflies per thread");
    // The density sweep runs along x: the outermost index of the single-GPU layout (AX_X), or the MIDDLE index of the
    // transposed slab psi^T[y_loc][x][z] of a slab-decomposed run (AX_Y; the half spectrum is then H^T[y_loc][kx][z],
    // (N/2 + 1) N elements per outer index -- see wdm_dist.cu)
    static_assert(!RHO || ax_strided(AX), "the density sweep runs along a strided axis");
    static constexpr size_t TILE_BYTES = align128(L::ELEMS * sizeof(cx<T>));
    static constexpr int AUX = DRIFT ? AUX_PHASE : AUX_NONE;
    // Potential values prefetched across tiles (into registers, during the previous tile's last stage): those of
    // the thread's FIRST level-A butterfly only.  The rest are loaded at the top of the tile's first phase and
    // arrive while the first butterfly computes -- half the registers held through the radix-32 middle level.
    static constexpr int PF = 1;
    struct Pre { T th[KICK ? PF : 1][KICK ? RA : 1]; DiagAcc d; };
    static __device__ __forceinline__ void flush(const SweepParams<T> &p, const Pre &pre)
    {
        diag_flush(p.diag, pre.d, AX == AX_CONTIG ? 0 : (AX == AX_Y ? 1 : 2), RHO ? 3 : -1, RHO ? 4 : -1);
    }
    static constexpr bool PAIR = ax_strided(AX) && pair_ok<C>();
    // the density sweep is short of registers at the end of its last psi stage (two lines of outputs, their
    // |psi|^2 and the twiddles): it fetches the twiddles where it needs them instead of keeping them
    static constexpr bool KEEP_TW = PAIR && !RHO;
    using Pers = PairTw<C, KEEP_TW>;

    // (first warp of the group, lane = gt)
    static __device__ __forceinline__ void issue(const SweepParams<T> &p, int t, unsigned char *buf, uint64_t *bar, int lane)
    {
        tile_load<C, AX, N>(reinterpret_cast<cx<T> *>(buf), p.data, &p.tmap, &p.tmap2, t, bar, lane);
    }
    static __device__ __forceinline__ void prefetch(const SweepParams<T> &p, int t, int gt, Pre &pre)
    {
        if constexpr (KICK) {
            const TL tile(p, t);
            static_for<0, (PF < ITER ? PF : ITER)>([&](auto it_) {
                constexpr int it = decltype(it_)::value;
                int q, l;
                split<AX, mA, W>(gt + it * NTG, q, l);
                const T *gp = p.phi + tile.at(q, l);
                static_for<0, RA>([&](auto r_) {
                    constexpr int r = decltype(r_)::value;
                    pre.th[it][r] = ldg(gp + (long long)(mA * r) * TL::RSTRIDE);
                });
            });
        }
    }
    template <class HOOK>
    static __device__ __forceinline__ void compute(const SweepParams<T> &p, const Tabs<T> &tb, int t, unsigned char *buf, int gt,
                                                   int grp, Pre &pre, const Pers &pers, HOOK &&hook)
    {
        cx<T> *S = reinterpret_cast<cx<T> *>(buf);
        const TL tile(p, t);
        cx<T> *psi = p.data;
        T rho[RHO ? ITER : 1][RHO ? RA : 1];
        const int pq = gt / (W / 2), pl = 2 * (gt % (W / 2));      // paired mapping: butterfly q of lines pl, pl + 1
        // level-A twiddles of butterfly pq: the kernel-long copy, or fetched now
        auto twiddles = [&](cx<T> (&w)[RA]) {
            static_for<1, RA>([&](auto s_) {
                constexpr int s = decltype(s_)::value;
                if constexpr (KEEP_TW) w[s] = pers.w[s];
                else w[s] = tb.twA[s * mA + pq];
            });
        };
        if constexpr (DRIFT) {
            if constexpr (PAIR) {
                cx<T> w[RA];
                twiddles(w);
                fwd_level_pair<RA, T>(pq, mA, w, [&](int row, cx<T> &a, cx<T> &c) { ld2(S + L::idx(row, pl), a, c); },
                                      [&](int row, cx<T> a, cx<T> c) { st2(S + L::idx(row, pl), a, c); });
            } else {
                T late[(KICK != 0 && ITER > PF) ? ITER - PF : 1][KICK != 0 ? RA : 1];
                if constexpr (KICK != 0)
                    static_for<PF, ITER>([&](auto it_) {
                        constexpr int it = decltype(it_)::value;
                        int q, l;
                        split<AX, mA, W>(gt + it * NTG, q, l);
                        const T *gp = p.phi + tile.at(q, l);
                        static_for<0, RA>([&](auto r_) { constexpr int r = decltype(r_)::value; late[it - PF][r] = ldg(gp + (long long)(mA * r) * TL::RSTRIDE); });
                    });
                static_for<0, ITER>([&](auto it_) {
                    constexpr int it = decltype(it_)::value;
                    int q, l;
                    split<AX, mA, W>(gt + it * NTG, q, l);
                    cx<T> v[RA];
                    static_for<0, RA>([&](auto r_) { constexpr int r = decltype(r_)::value; v[r] = S[L::idx(q + mA * r, l)]; });
                    auto th = [&](auto r_) -> T {
                        constexpr int r = decltype(r_)::value;
                        if constexpr (KICK == 0) return (T)0;
                        else if constexpr (it < PF) return pre.th[it][r];
                        else return late[it - PF][r];
                    };
                    if constexpr (KICK != 0) {
                        if constexpr (KICK == 2) {
                            // self-interaction and / or absorbing layer: the pencil of line l is (x, y) = divmod(t W + l, N)
                            T mxy = (T)1;
                            if (p.mask) {
                                const int pen = t * W + l, x = pen / N, y = pen - x * N;
                                mxy = ldg(p.mask + x) * ldg(p.mask + N + y);
                            }
                            static_for<0, RA>([&](auto r_) {
                                constexpr int r = decltype(r_)::value;
                                const T m = p.mask ? mxy * ldg(p.mask + 2 * N + q + mA * r) : (T)1;
                                v[r] = kick_general(v[r], th(r_), m, p.kick, p.kself_d, p.kself_a);
                            });
                        } else {
                            T ph[RA];
                            static_for<0, RA>([&](auto r_) { constexpr int r = decltype(r_)::value; ph[r] = th(r_) * p.kick; });
                            rotate_neg_all<RA>(v, ph);
                        }
                    }
                    fwd_level_regs<RA, T>(v, q, mA, tb.twA + q, [&](int row, cx<T> y) { S[L::idx(row, l)] = y; });
                });
            }
            group_sync(grp, NTG);
            auto idx = [](int row, int l) { return L::idx(row, l); };
            g_fwd_B<C, W>(S, tb.twB, gt, grp, idx);
            T tsum = (T)0;                                 // this tile's share of sum k^2 |F psi|^2 (DG)
            if constexpr (DG == 2) {
                for (int b = gt; b < (N / RM) * W; b += NTG) {
                    int l = b % W, g = b / W;
                    mid_fwd<RM, T>(g * RM, [&](int row) { return S[L::idx(row, l)]; },
                                   [&](int row, cx<T> v) { tsum += ldg(p.ksq_pos + row) * (v.x * v.x + v.y * v.y); });
                }
                pre.d.s0 += (double)tsum;
                return;
            }
            for (int b = gt; b < (N / RM) * W; b += NTG) {
                int l = b % W, g = b / W;
                auto mul = [&](int pos, cx<T> &a, cx<T> &c) {
                    if constexpr (DG == 1) {
                        T ka, kc;
                        ld2r(p.ksq_pos + pos, ka, kc);
                        tsum += ka * (a.x * a.x + a.y * a.y) + kc * (c.x * c.x + c.y * c.y);
                    }
                    cx<T> pa, pc;
                    ld2(tb.phase + pos, pa, pc);          // both kinetic factors in one 16-byte load
                    a = cmul(a, pa);
                    c = cmul(c, pc);
                };
                if constexpr (L::VEC2)
                    mid_both2<RM, T>(g * RM, [&](int row, cx<T> &a, cx<T> &c) { ld2(S + L::idx(row, l), a, c); },
                                     [&](int row, cx<T> a, cx<T> c) { st2(S + L::idx(row, l), a, c); }, mul);
                else
                    mid_both<RM, T>(g * RM, [&](int row) { return S[L::idx(row, l)]; },
                                    [&](int row, cx<T> v) { S[L::idx(row, l)] = v; }, mul);
            }
            if constexpr (DG == 1) pre.d.s0 += (double)tsum;
            group_sync(grp, NTG);
            g_inv_B<C, W>(S, tb.twB, gt, grp, idx);
            hook();
            if constexpr (PAIR) {
                cx<T> a[RA], c[RA];
                {
                    cx<T> w[RA];
                    twiddles(w);
                    inv_level_pair_regs<RA, T>(pq, mA, w, [&](int row, cx<T> &x, cx<T> &y) { ld2(S + L::idx(row, pl), x, y); }, a, c);
                }
                cx<T> *gp = psi + tile.at(pq, pl);
                static_for<0, RA>([&](auto r_) {
                    constexpr int r = decltype(r_)::value;
                    stg2(gp + (long long)(mA * r) * TL::RSTRIDE, a[r], c[r]);
                    if constexpr (RHO) {
                        rho[0][r] = a[r].x * a[r].x + a[r].y * a[r].y;
                        rho[1][r] = c[r].x * c[r].x + c[r].y * c[r].y;
                    }
                });
            } else {
                static_for<0, ITER>([&](auto it_) {
                    constexpr int it = decltype(it_)::value;
                    int q, l;
                    split<AX, mA, W>(gt + it * NTG, q, l);
                    cx<T> v[RA];
                    inv_level_regs<RA, T>(q, mA, tb.twA + q, [&](int row) { return S[L::idx(row, l)]; }, v);
                    cx<T> *gp = psi + tile.at(q, l);
                    static_for<0, RA>([&](auto r_) {
                        constexpr int r = decltype(r_)::value;
                        stv(gp + (long long)(mA * r) * TL::RSTRIDE, v[r]);
                        if constexpr (RHO) rho[it][r] = v[r].x * v[r].x + v[r].y * v[r].y;
                    });
                });
            }
        } else if constexpr (RHO) {
            if constexpr (PAIR) {
                static_for<0, RA>([&](auto r_) {
                    constexpr int r = decltype(r_)::value;
                    cx<T> a, c;
                    ld2(S + L::idx(pq + mA * r, pl), a, c);
                    rho[0][r] = a.x * a.x + a.y * a.y;
                    rho[1][r] = c.x * c.x + c.y * c.y;
                });
            } else {
                static_for<0, ITER>([&](auto it_) {
                    constexpr int it = decltype(it_)::value;
                    int q, l;
                    split<AX, mA, W>(gt + it * NTG, q, l);
                    static_for<0, RA>([&](auto r_) {
                        constexpr int r = decltype(r_)::value;
                        cx<T> v = S[L::idx(q + mA * r, l)];
                        rho[it][r] = v.x * v.x + v.y * v.y;
                    });
                });
            }
        }
        if constexpr (RHO && DG == 1) {
            // mass and peak density of psi_2 (Alg. 1 l.12; the maxima feed Eq. 26) from the registers
            T rs = (T)0, rm = (T)0;
            static_for<0, (PAIR ? 2 : ITER)>([&](auto it_) {
                static_for<0, RA>([&](auto r_) {
                    const T v = rho[decltype(it_)::value][decltype(r_)::value];
                    rs += v;
                    rm = fmax(rm, v);
                });
            });
            pre.d.s1 += (double)rs;
            pre.d.mx = fmax(pre.d.mx, (double)rm);
        }
        if constexpr (RHO) {
            // rho tile as N rows x W reals == N rows x W/2 packed complex lines (lines 2l', 2l'+1)
            constexpr int WP = W / 2;
            T *F = reinterpret_cast<T *>(buf);
            group_sync(grp, NTG);                       // every thread has finished reading the psi tile
            // rho - <rho> (Eq. 23).  <rho> is conserved, so it is measured once per refresh; k = 0 is
            // zeroed in the Green's function anyway -- subtracting here only keeps the large mean out of the
            // single-precision partial sums of the low-k modes.
            const T mean = ldg(p.rho_mean);
            cx<T> *Sp = reinterpret_cast<cx<T> *>(buf);
            // particle mass reaches only a small part of the mesh (a thin disc: ~10 % of the tiles); the deposit flags the
            // (y, z-block) columns it touched and every other tile skips the loads (rho_p is zero there)
            constexpr int FB = N < 16 ? N : 16;
            const bool has_rho_p = p.rho_p != nullptr && p.rho_flag[(t / TL::INNER) * (N / FB) + ((t % TL::INNER) * W) / FB] != 0;
            if constexpr (PAIR) {
                // the pair (pl, pl + 1) at rows pq + mA r IS packed line pl / 2 at the rows of this thread's own
                // level-A butterfly of the real-to-complex transform: straight from registers
                const T *gp = has_rho_p ? p.rho_p + tile.at(pq, pl) : nullptr;
                cx<T> v[RA];
                static_for<0, RA>([&](auto r_) {
                    constexpr int r = decltype(r_)::value;
                    T va = rho[0][r], vc = rho[1][r];
                    if (gp) {
                        cx<T> e = ldg(reinterpret_cast<const cx<T> *>(gp + (long long)(mA * r) * TL::RSTRIDE));
                        va += e.x;
                        vc += e.y;
                    }
                    v[r] = mk<T>(va - mean, vc - mean);
                });
                cx<T> w[RA];
                twiddles(w);
                fwd_level_regs_w<RA, T>(v, pq, mA, w, [&](int row, cx<T> y) { Sp[Packed<C>::idxA(pq, row - pq, pl / 2)] = y; });
            } else {
                static_for<0, ITER>([&](auto it_) {
                    constexpr int it = decltype(it_)::value;
                    int q, l;
                    split<AX, mA, W>(gt + it * NTG, q, l);
                    const T *gp = has_rho_p ? p.rho_p + tile.at(q, l) : nullptr;
                    static_for<0, RA>([&](auto r_) {
                        constexpr int r = decltype(r_)::value;
                        int row = q + mA * r;
                        T v = rho[it][r];
                        if (gp) v += ldg(gp + (long long)(mA * r) * TL::RSTRIDE);
                        F[2 * Packed<C>::idxA(q, mA * r, l / 2) + (l & 1)] = v - mean;
                    });
                });
                group_sync(grp, NTG);
                for (int b = gt; b < mA * WP; b += NTG) {
                    int l = b % WP, q = b / WP;
                    fwd_level<RA, T>(q, mA, tb.twA + q, [&](int row) { return Sp[Packed<C>::idxA(q, row - q, l)]; },
                                     [&](int row, cx<T> v) { Sp[Packed<C>::idxA(q, row - q, l)] = v; });
                }
            }
            group_sync(grp, NTG);
            g_fwd_B<C, WP>(Sp, tb.twB, gt, grp, [](int row, int l) { return Packed<C>::idx(row, l); });
            for (int b = gt; b < (N / RM) * WP; b += NTG) {
                int l = b % WP, g = b / WP;
                mid_fwd<RM, T>(g * RM, [&](int row) { return Sp[Packed<C>::idxM(g * RM, row - g * RM, l)]; },
                               [&](int row, cx<T> v) { Sp[Packed<C>::idxM(g * RM, row - g * RM, l)] = v; });
            }
            group_sync(grp, NTG);
            // Hermitian split of Z = FFT(a + i b):  A_k = (Z_k + conj Z_{N-k})/2,  B_k = (Z_k - conj Z_{N-k})/(2i)
            // row k of the half spectrum, line 2l of this tile
            const long long hbase = AX == AX_X ? tile.base : (long long)(t / TL::INNER) * ((long long)(N / 2 + 1) * N) + (long long)(t % TL::INNER) * W;
            auto emit = [&](int k, int e, int en, int l) {
                cx<T> zk = Sp[e], zn = Sp[en];
                const T h = (T)0.5;
                cx<T> A = mk<T>((zk.x + zn.x) * h, (zk.y - zn.y) * h);
                cx<T> B = mk<T>((zk.y + zn.y) * h, (zn.x - zk.x) * h);
                st2(p.H + hbase + (long long)k * TL::RSTRIDE + 2 * l, A, B);
            };
            half_spectrum_items<C, WP, Packed<C>>(gt, emit);
            if (gt < WP) {
                const int e = Packed<C>::idx(HalfSpec<C>::row_of(N / 2), gt);
                emit(N / 2, e, e, gt);
            }
        }
    }
};

// ---------------------------------------------------------------- Poisson sweeps on the half spectrum
template <class C_, int MODE, int DG_ = 0>
struct HK {
    static constexpr int DG = DG_;                              // 1 (Green sweep only): W = 1/2 sum rho Phi, spectrally
    static constexpr bool DIAG_ZEROES = false;
    static_assert(DG_ == 0 || MODE == H_Z_GREEN, "only the Green sweep accumulates");
    using C = C_;
    using T = typename C::T;
    static constexpr int AX = (MODE == H_Z_GREEN) ? AX_CONTIG : AX_Y;
    using TL = Tile<C, AX>;
    using L = Lay<C, AX>;
    static constexpr int N = C::N, RA = C::RA, RM = C::RM, W = C::W, NTG = C::NT, mA = C::mA;
    static constexpr size_t TILE_BYTES = align128(L::ELEMS * sizeof(cx<T>));
    static constexpr int AUX = MODE == H_Z_GREEN ? AUX_KSQ : AUX_NONE;
    using Pre = NoPre;
    static __device__ __forceinline__ void flush(const SweepParams<T> &p, const Pre &pre) { diag_flush(p.diag, pre.d, 5, -1, -1); }
    static constexpr bool PAIR = ax_strided(AX) && pair_ok<C>();
    using Pers = PairTw<C, PAIR>;
    // (first warp of the group, lane = gt)
    static __device__ __forceinline__ void issue(const SweepParams<T> &p, int t, unsigned char *buf, uint64_t *bar, int lane)
    {
        tile_load<C, AX, N>(reinterpret_cast<cx<T> *>(buf), p.data, &p.tmap, &p.tmap2, t, bar, lane);
    }
    static __device__ __forceinline__ void prefetch(const SweepParams<T> &, int, int, Pre &) {}
    template <class HOOK>
    static __device__ __forceinline__ void compute(const SweepParams<T> &p, const Tabs<T> &tb, int t, unsigned char *buf, int gt, int grp, Pre &pre,
                                                   const Pers &pers, HOOK &&)
    {
        cx<T> *S = reinterpret_cast<cx<T> *>(buf);
        const TL tile(p, t);
        cx<T> *H = p.data;
        const int pq = gt / (W / 2), pl = 2 * (gt % (W / 2));      // paired mapping (see PairTw)
        auto ldS = [&](int l) { return [S, l](int row) { return S[L::idx(row, l)]; }; };
        auto stS = [&](int l) { return [S, l](int row, cx<T> v) { S[L::idx(row, l)] = v; }; };
        auto idx = [](int row, int l) { return L::idx(row, l); };
        if constexpr (MODE == H_Y_FWD || MODE == H_Z_GREEN) {
            if constexpr (PAIR) {
                fwd_level_pair<RA, T>(pq, mA, pers.w, [&](int row, cx<T> &a, cx<T> &c) { ld2(S + L::idx(row, pl), a, c); },
                                      [&](int row, cx<T> a, cx<T> c) { st2(S + L::idx(row, pl), a, c); });
            } else {
                for (int b = gt; b < mA * W; b += NTG) {
                    int q, l;
                    split<AX, mA, W>(b, q, l);
                    fwd_level<RA, T>(q, mA, tb.twA + q, ldS(l), stS(l));
                }
            }
            group_sync(grp, NTG);
            g_fwd_B<C, W>(S, tb.twB, gt, grp, idx);
        }
        if constexpr (MODE == H_Y_FWD) {
            for (int b = gt; b < (N / RM) * W; b += NTG) {
                int l = b % W, g = b / W;
                cx<T> *gp = H + tile.at(g * RM, l);
                mid_fwd<RM, T>(g * RM, ldS(l), [&](int row, cx<T> v) { stv(gp + (long long)(row - g * RM) * TL::RSTRIDE, v); });
            }
        }
        if constexpr (MODE == H_Z_GREEN) {
            // pencil l of this tile is (kx, y position) = divmod(t*W + l, N); the y axis is in position order
            for (int b = gt; b < (N / RM) * W; b += NTG) {
                int l = b % W, g = b / W;
                int pen = t * W + l, kx = pen / N, ypos = pen - kx * N;
                kx += p.kx0;                                   // first kx-plane of this rank's slab (0 on a single GPU)
                T kxy = ldg(p.ksq_nat + kx) + tb.ksq_pos[ypos];
                bool zero_line = (kx == 0 && ypos == 0);
                T wsum = (T)0;
                auto mul = [&](int pos, cx<T> &a, cx<T> &c) {
                    T ka, kc;
                    ld2r(tb.ksq_pos + pos, ka, kc);
                    T ga = (zero_line && pos == 0) ? (T)0 : green_over(p.green, kxy + ka);
                    const T gc = green_over(p.green, kxy + kc);
                    if constexpr (DG == 1) wsum += ga * (a.x * a.x + a.y * a.y) + gc * (c.x * c.x + c.y * c.y);
                    a = cscale(a, ga);
                    c = cscale(c, gc);
                };
                if constexpr (L::VEC2)
                    mid_both2<RM, T>(g * RM, [&](int row, cx<T> &a, cx<T> &c) { ld2(S + L::idx(row, l), a, c); },
                                     [&](int row, cx<T> a, cx<T> c) { st2(S + L::idx(row, l), a, c); }, mul);
                else
                    mid_both<RM, T>(g * RM, ldS(l), stS(l), mul);
                // conj(rho~_k) Phi~_k over the FULL spectrum: rows 0 < kx < N/2 stand for their mirrors too
                if constexpr (DG == 1) pre.d.s0 += (double)wsum * ((kx == 0 || kx == N / 2) ? 1.0 : 2.0);
            }
            group_sync(grp, NTG);
            g_inv_B<C, W>(S, tb.twB, gt, grp, idx);
        }
        if constexpr (MODE == H_Y_INV) {
            for (int b = gt; b < (N / RM) * W; b += NTG) {
                int l = b % W, g = b / W;
                mid_inv<RM, T>(g * RM, ldS(l), stS(l));
            }
            group_sync(grp, NTG);
            g_inv_B<C, W>(S, tb.twB, gt, grp, idx);
        }
        if constexpr (MODE == H_Y_INV || MODE == H_Z_GREEN) {
            if constexpr (PAIR) {
                cx<T> a[RA], c[RA];
                inv_level_pair_regs<RA, T>(pq, mA, pers.w, [&](int row, cx<T> &x, cx<T> &y) { ld2(S + L::idx(row, pl), x, y); }, a, c);
                cx<T> *gp = H + tile.at(pq, pl);
                static_for<0, RA>([&](auto r_) { constexpr int r = decltype(r_)::value; stg2(gp + (long long)(mA * r) * TL::RSTRIDE, a[r], c[r]); });
            } else {
                for (int b = gt; b < mA * W; b += NTG) {
                    int q, l;
                    split<AX, mA, W>(b, q, l);
                    cx<T> *gp = H + tile.at(q, l);
                    inv_level<RA, T>(q, mA, tb.twA + q, ldS(l), [&](int row, cx<T> v) { stv(gp + (long long)(row - q) * TL::RSTRIDE, v); });
                }
            }
        }
    }
};

// complex-to-real inverse along x: H[kx <= N/2][y][z] -> Phi[x][y][z]; lines (2l', 2l'+1) share one FFT.
// Buffer = [packed tile: N rows x W/2 complex][raw tile: N/2+1 rows x W complex, filled by the async copies].
// EXT: add the static external potential on the way out (SweepParams::phi_ext != nullptr), a separate instantiation
// AXR: the axis of the transform -- AX_X on a single GPU; AX_Y for the transposed slab H^T[y_loc][kx][z] ->
// Phi^T[y_loc][x][z] of a slab-decomposed run.
template <class C_, bool EXT = false, int DG_ = 0, int AXR = AX_X>
struct C2RK {
    static constexpr int DG = DG_;                              // 1: max |Phi_total| from the outgoing registers
    static constexpr bool DIAG_ZEROES = false;
    using C = C_;
    using T = typename C::T;
    using TL = Tile<C, AXR>;
    static constexpr int N = C::N, RA = C::RA, RM = C::RM, W = C::W, NTG = C::NT, mA = C::mA;
    static constexpr int WP = W / 2, RSP = W / 2;
    using PK = Packed<C, true>;
    static constexpr size_t PACKED_BYTES = align128(PK::ELEMS * sizeof(cx<T>));
    static constexpr size_t TILE_BYTES = PACKED_BYTES + align128((size_t)(N / 2 + 1) * W * sizeof(cx<T>));
    static constexpr int AUX = AUX_NONE;
    using Pre = NoPre;
    static __device__ __forceinline__ void flush(const SweepParams<T> &p, const Pre &pre) { diag_flush(p.diag, pre.d, -1, -1, 6); }
    static constexpr bool PAIR = pair_ok<C>();          // packed line gt % (W/2), butterfly gt / (W/2): the PairTw twiddles
    using Pers = PairTw<C, PAIR>;
    static __device__ __forceinline__ void issue(const SweepParams<T> &p, int t, unsigned char *buf, uint64_t *bar, int lane)
    {
        tile_load<C, AXR, N / 2 + 1>(reinterpret_cast<cx<T> *>(buf + PACKED_BYTES), p.H, &p.tmap, &p.tmap2, t, bar, lane);
    }
    static __device__ __forceinline__ void prefetch(const SweepParams<T> &, int, int, Pre &) {}
    template <class HOOK>
    static __device__ __forceinline__ void compute(const SweepParams<T> &p, const Tabs<T> &tb, int t, unsigned char *buf, int gt, int grp, Pre &pre,
                                                   const Pers &pers, HOOK &&)
    {
        cx<T> *Sp = reinterpret_cast<cx<T> *>(buf);
        const cx<T> *R = reinterpret_cast<const cx<T> *>(buf + PACKED_BYTES);
        T pmax = (T)0;
        const TL tile(p, t);
        // Z_k = A_k + i B_k,  Z_{N-k} = conj(A_k) + i conj(B_k)
        // Rows kx = 0 and kx = N/2 are the x-spectrum of REAL lines at a self-mirrored frequency: real in exact
        // arithmetic.  What rounding leaves in their imaginary parts (Hermitian asymmetry of the y, z transforms,
        // amplified by 1/k^2 at low k) must not enter: B's would land on line 2l', A's on line 2l'+1 -- with opposite
        // signs on adjacent z, i.e. folded onto the mode at the z-Nyquist mirror (measured at 512^3 complex64: 2e-3 of
        // the coefficient of (0, 0, 255), N^2-growing).  As in any complex-to-real transform they are ignored.
        auto place = [&](int k, int e, int en, int l) {
            cx<T> A, B;
            ld2(R + k * W + 2 * l, A, B);
            if (k == 0 || k == N / 2) A.y = B.y = (T)0;
            Sp[e] = mk<T>(A.x - B.y, A.y + B.x);
            if (k > 0 && k < N / 2) Sp[en] = mk<T>(A.x + B.y, B.x - A.y);
        };
        half_spectrum_items<C, WP, PK>(gt, place);
        if (gt < WP) {
            const int e = PK::idx(HalfSpec<C>::row_of(N / 2), gt);
            place(N / 2, e, e, gt);
        }
        group_sync(grp, NTG);
        for (int b = gt; b < (N / RM) * WP; b += NTG) {
            int l = b % WP, g = b / WP;
            mid_inv<RM, T>(g * RM, [&](int row) { return Sp[PK::idxM(g * RM, row - g * RM, l)]; },
                           [&](int row, cx<T> v) { Sp[PK::idxM(g * RM, row - g * RM, l)] = v; });
        }
        group_sync(grp, NTG);
        g_inv_B<C, WP>(Sp, tb.twB, gt, grp, [](int row, int l) { return PK::idx(row, l); });
        for (int b = gt; b < mA * WP; b += NTG) {
            int l = b % WP, q = b / WP;
            T *gp = p.phi_out + tile.at(q, 2 * l);
            const T *ge = EXT ? p.phi_ext + tile.at(q, 2 * l) : nullptr;           // Phi_total = Phi_DM + Phi_ext (Alg. 1 l.15)
            auto out = [&](int row, cx<T> v) {
                // Re -> line 2l', Im -> line 2l'+1: one (re, im) pair is two adjacent reals of Phi
                if constexpr (EXT) {
                    cx<T> e = ldg(reinterpret_cast<const cx<T> *>(ge + (long long)(row - q) * TL::RSTRIDE));
                    v.x += e.x;
                    v.y += e.y;
                }
                if constexpr (DG == 1) pmax = fmax(pmax, fmax(fabs(v.x), fabs(v.y)));
                stv(reinterpret_cast<cx<T> *>(gp + (long long)(row - q) * TL::RSTRIDE), v);
            };
            if constexpr (PAIR) inv_level_w<RA, T>(q, mA, pers.w, [&](int row) { return Sp[PK::idxA(q, row - q, l)]; }, out);
            else inv_level<RA, T>(q, mA, tb.twA + q, [&](int row) { return Sp[PK::idxA(q, row - q, l)]; }, out);
        }
        if constexpr (DG == 1) pre.d.mx = fmax(pre.d.mx, (double)pmax);
    }
};

// Complex-to-real sweep IN PLACE, for tiles too large to hold a packed copy beside the half spectrum (1024-point lines:
// with the copy only W = 8 fits three times in shared memory -- 32-byte rows of Phi, 64-byte rows of H, and half of a
// group idle in every stage).  Here the tile buffer is the half spectrum alone, W = 16, and every stage has one
// butterfly per thread.  Two facts make it work (N = RA RM, RA = RM, two real lines 2l, 2l+1 per complex line l):
//   * frequency k = g + RA sM sits at position (g, sM) of the inverse transform, and its mirror N - k at position
//     (RA - g, RM - 1 - sM).  The first stage of thread (l, g) needs Z_k of block g: sM < RM/2 from the rows k <= N/2 of
//     its own block (Z_k = A_k + i B_k), the others from the rows of block RA - g (Z_{N-k} = conj A_k + i conj B_k): the
//     Hermitian unsplit happens in the registers that feed the butterfly, 32 conflict-free 16-byte loads per thread.
//   * its RM outputs (g, r) go back as 16-byte pairs (r, r + RM/2) over the rows g + RA r of its own block -- rows the
//     thread of block RA - g has read as well, hence one group barrier between the loads and the stores.  The last
//     stage of thread (l, q) then finds (s, q), s < RA, in RA consecutive rows, in half q / (RM/2) of the pair; a warp
//     holds q and q + RM/2 together, so its 8-byte loads cover whole 128-byte rows.
// Rows k = 0 and k = N/2 drop their imaginary parts as in C2RK (reading G33).
template <class C_, bool EXT, int DG_ = 0, int AXR = AX_X>
struct C2RI {
    static constexpr int DG = DG_;
    static constexpr bool DIAG_ZEROES = false;
    using C = C_;
    using T = typename C::T;
    using TL = Tile<C, AXR>;
    static constexpr int N = C::N, RA = C::RA, RM = C::RM, W = C::W, NTG = C::NT, mA = C::mA, WP = W / 2, HM = RM / 2;
    static_assert(C::RB == 1 && NTG == WP * RA && (mA * WP) % NTG == 0, "one first-stage butterfly per thread, whole rounds of the last stage");
    static constexpr size_t TILE_BYTES = align128((size_t)(N / 2 + 1) * W * sizeof(cx<T>));
    static constexpr int AUX = AUX_NONE;
    using Pre = NoPre;
    struct Pers {
        __device__ __forceinline__ void setup(const Tabs<T> &, int) {}
    };
    static __device__ __forceinline__ void flush(const SweepParams<T> &p, const Pre &pre) { diag_flush(p.diag, pre.d, -1, -1, 6); }
    static __device__ __forceinline__ void issue(const SweepParams<T> &p, int t, unsigned char *buf, uint64_t *bar, int lane)
    {
        tile_load<C, AXR, N / 2 + 1>(reinterpret_cast<cx<T> *>(buf), p.H, &p.tmap, &p.tmap2, t, bar, lane);
    }
    static __device__ __forceinline__ void prefetch(const SweepParams<T> &, int, int, Pre &) {}
    template <class HOOK>
    static __device__ __forceinline__ void compute(const SweepParams<T> &p, const Tabs<T> &tb, int t, unsigned char *buf, int gt, int grp, Pre &pre,
                                                   const Pers &, HOOK &&)
    {
        cx<T> *R = reinterpret_cast<cx<T> *>(buf);
        const int l = gt % WP;
        const TL tile(p, t);
        {
            const int g = gt / WP;
            cx<T> *ra = R + g * W + 2 * l;
            const cx<T> *rb = R + (RA - g) * W + 2 * l;
            cx<T> v[RM];
            static_for<0, HM>([&](auto i_) {
                constexpr int i = decltype(i_)::value;
                cx<T> A, B;
                ld2(ra + i * RA * W, A, B);                                  // k = g + RA i
                if (i == 0 && g == 0) A.y = B.y = (T)0;                      // k = 0
                v[brev(i, RM)] = mk<T>(A.x - B.y, A.y + B.x);
                ld2(rb + i * RA * W, A, B);                                  // k' = RA - g + RA i, for N - k' = g + RA (RM - 1 - i)
                if (i == HM - 1 && g == 0) A.y = B.y = (T)0;                 // k' = N/2
                v[brev(RM - 1 - i, RM)] = mk<T>(A.x + B.y, B.x - A.y);
            });
            dit_inv<RM>(v);
            group_sync(grp, NTG);                                            // every thread has read its rows
            static_for<0, HM>([&](auto r_) {
                constexpr int r = decltype(r_)::value;
                st2(ra + r * RA * W, v[r], v[r + HM]);
            });
        }
        group_sync(grp, NTG);
        T pmax = (T)0;
        for (int b = gt; b < mA * WP; b += NTG) {
            const int t2 = b / WP, q = (t2 & 1) * HM + (t2 >> 1);
            const cx<T> *src = R + (RA * (q % HM)) * W + 2 * l + q / HM;
            T *gp = p.phi_out + tile.at(q, 2 * l);
            const T *ge = EXT ? p.phi_ext + tile.at(q, 2 * l) : nullptr;           // Phi_total = Phi_DM + Phi_ext (Alg. 1 l.15)
            auto out = [&](int row, cx<T> v) {
                // Re -> line 2l, Im -> line 2l+1: one (re, im) pair is two adjacent reals of Phi
                if constexpr (EXT) {
                    cx<T> e = ldg(reinterpret_cast<const cx<T> *>(ge + (long long)(row - q) * TL::RSTRIDE));
                    v.x += e.x;
                    v.y += e.y;
                }
                if constexpr (DG == 1) pmax = fmax(pmax, fmax(fabs(v.x), fabs(v.y)));
                stv(reinterpret_cast<cx<T> *>(gp + (long long)(row - q) * TL::RSTRIDE), v);
            };
            inv_level<RA, T>(q, mA, tb.twA + q, [&](int row) { return src[((row - q) / mA) * W]; }, out);
        }
        if constexpr (DG == 1) pre.d.mx = fmax(pre.d.mx, (double)pmax);
    }
};

}  // namespace wdm
