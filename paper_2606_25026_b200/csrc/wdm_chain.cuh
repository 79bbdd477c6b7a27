// wdm_chain.cuh -- several axis sweeps of the same array chained through the L2 cache in ONE persistent kernel.
//
// Two consecutive sweeps of Eq. 18(b) (z then y on psi) and the three middle sweeps of the Poisson solve
// (y forward, z forward . Green . inverse, y inverse on the half spectrum; Eq. 18(c), Eq. 23) each touch a
// whole x-plane of the array and nothing else: plane u (N x N elements, contiguous, 2 MB at 512^2 complex64)
// is a closed unit for all of them.  Run as separate launches, every sweep streams the array HBM -> SM ->
// HBM.  Here stage s + 1 of plane u runs `lag` planes behind stage s, while the plane stage s wrote is still
// in the 126 MB L2: only the first stage reads HBM and only the last stage's lines are ever written back
// (a dirty line that is overwritten in L2 never reaches DRAM).
//
// Position sequence.  Slot sigma holds, for every stage s with 0 <= sigma - s*lag < units, the TPU tiles of
// (stage s, plane sigma - s*lag), stage-major.  Positions are numbered over VALID tiles only (the ramps at both
// ends are shorter slots), CTA c owns positions c, c + grid, ... and runs them through the same three-buffer
// asynchronous pipeline as pipe_run.  A tile of stage s >= 1 is not requested before all TPU tiles of
// (s - 1, same plane) have been stored: every finished tile bumps a per-(stage, plane) counter with release
// semantics; lane 0 of the requesting warp spins on it with acquire loads before the warp issues the TMA copies.
//
// Progress: dependencies always point to smaller positions; a group blocks only while REQUESTING position
// g + (NBUF - NG) * grid, g its own next tile, and what it waits for lies more than (NBUF - NG) * grid
// positions back (the launcher refuses a lag that does not guarantee it), i.e. before g -- so the smallest
// unfinished position is never held up.  All CTAs must be co-resident: cooperative launch.
#pragma once

#include "wdm_pipe.cuh"

namespace wdm {

template <typename T, int NS>
struct ChainParams {
    SweepParams<T> p[NS];
    unsigned int *done;          // (NS - 1) x units completion counters, monotone across launches
    unsigned int target;         // value a complete plane's counter has reached in this launch
    int units, tpu_log2, lag, total, nseg;
    int seg_pos[2 * NS + 1], seg_slot[2 * NS], seg_lo[2 * NS], seg_v[2 * NS];
};

// host: segments of the position sequence (constant set of valid stages within a segment)
template <typename T, int NS>
inline void chain_plan(ChainParams<T, NS> &cp, int units, int tpu, int lag)
{
    cp.units = units; cp.lag = lag;
    cp.tpu_log2 = 0;
    while ((1 << cp.tpu_log2) < tpu) ++cp.tpu_log2;
    int br[2 * NS], nb = 0;
    for (int s = 0; s < NS; ++s) { br[nb++] = s * lag; br[nb++] = s * lag + units; }
    for (int i = 0; i < nb; ++i)
        for (int j = i + 1; j < nb; ++j)
            if (br[j] < br[i]) { int t = br[i]; br[i] = br[j]; br[j] = t; }
    int pos = 0;
    cp.nseg = 0;
    for (int i = 0; i + 1 < nb; ++i) {
        if (br[i] == br[i + 1]) continue;
        int lo = -1, v = 0;
        for (int s = 0; s < NS; ++s)
            if (br[i] >= s * lag && br[i] < s * lag + units) { if (lo < 0) lo = s; ++v; }
        if (v == 0) continue;
        cp.seg_pos[cp.nseg] = pos; cp.seg_slot[cp.nseg] = br[i]; cp.seg_lo[cp.nseg] = lo; cp.seg_v[cp.nseg] = v;
        ++cp.nseg;
        pos += (br[i + 1] - br[i]) * v * tpu;
    }
    for (int i = cp.nseg; i < 2 * NS; ++i) { cp.seg_pos[i] = 0x7fffffff; cp.seg_slot[i] = 0; cp.seg_lo[i] = 0; cp.seg_v[i] = 1; }
    cp.seg_pos[2 * NS] = 0x7fffffff;
    cp.total = pos;
}

// smallest distance, in positions, between a tile and the last tile it depends on: the worst case is the
// first dependent plane, because the slots before `lag` hold one stage only
inline int chain_min_distance(int tpu, int lag) { return lag * tpu + 1; }

#if defined(__CUDACC__)

struct TileRef { int stage, unit, tile; };

template <typename T, int NS>
__device__ __forceinline__ TileRef chain_decode(const ChainParams<T, NS> &cp, int g)
{
    int k = 0;
#pragma unroll
    for (int i = 1; i < 2 * NS; ++i)
        if (g >= cp.seg_pos[i]) k = i;
    const int rel = g - cp.seg_pos[k], per = cp.seg_v[k] << cp.tpu_log2;
    const int ds = rel / per, r = rel - ds * per;
    TileRef t;
    t.stage = cp.seg_lo[k] + (r >> cp.tpu_log2);
    t.unit = cp.seg_slot[k] + ds - t.stage * cp.lag;
    t.tile = (t.unit << cp.tpu_log2) + (r & ((1 << cp.tpu_log2) - 1));
    return t;
}

__device__ __forceinline__ unsigned int ld_acquire(const unsigned int *p)
{
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add(unsigned int *p, unsigned int v)
{
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <int I, class K0, class... KS> struct StageAt { using type = typename StageAt<I - 1, KS...>::type; };
template <class K0, class... KS> struct StageAt<0, K0, KS...> { using type = K0; };

template <class... KS>
struct ChainSmem {
    using K0 = typename StageAt<0, KS...>::type;
    using C = typename K0::C;
    using T = typename C::T;
    static constexpr int NS = sizeof...(KS);
    static constexpr size_t cmax(size_t a, size_t b) { return a > b ? a : b; }
    static constexpr size_t fold_tile() { size_t m = 0; ((m = cmax(m, KS::TILE_BYTES)), ...); return m; }
    static constexpr int fold_aux() { int a = AUX_NONE; ((a = (a == AUX_NONE ? KS::AUX : a)), ...); return a; }
    static constexpr size_t TILE_BYTES = fold_tile();
    static constexpr int AUX = fold_aux();
    static_assert(((KS::AUX == AUX_NONE || KS::AUX == AUX) && ...), "stages of a chain share one auxiliary table");
    static constexpr size_t CTRL = (size_t)(C::NG + 1) * TILE_BYTES;
    static constexpr size_t TWA = CTRL + 64;
    static constexpr size_t TWA_BYTES = (size_t)C::N * sizeof(cx<T>);
    static constexpr size_t TWB_BYTES = C::RB > 1 ? (size_t)C::MB * sizeof(cx<T>) : 0;
    static constexpr size_t AUX_BYTES = AUX == AUX_PHASE ? (size_t)C::N * sizeof(cx<T>) : (AUX == AUX_KSQ ? (size_t)C::N * sizeof(T) : 0);
    static constexpr bool TW_IN_SMEM = TWA + TWA_BYTES + TWB_BYTES <= kMaxSmem;
    static constexpr size_t AUX_OFF = TWA + (TW_IN_SMEM ? TWA_BYTES + TWB_BYTES : 0);
    static constexpr bool AUX_IN_SMEM = AUX != AUX_NONE && AUX_OFF + AUX_BYTES <= kMaxSmem;
    static constexpr size_t TOTAL = AUX_OFF + (AUX_IN_SMEM ? AUX_BYTES : 0);
};

// f(K{}) for the stage's kernel type; `stage` is uniform over the calling group
template <int I, int NS, class F>
__device__ __forceinline__ void chain_dispatch(int stage, F &f)
{
    if constexpr (I + 1 == NS) {
        f(ic<I>{});
    } else {
        if (stage == I) f(ic<I>{});
        else chain_dispatch<I + 1, NS>(stage, f);
    }
}

template <class... KS>
__device__ __forceinline__ void chain_run(const ChainParams<typename StageAt<0, KS...>::type::C::T, (int)sizeof...(KS)> &cp, unsigned char *smem)
{
    using SM = ChainSmem<KS...>;
    using K0 = typename SM::K0;
    using C = typename SM::C;
    using T = typename C::T;
    constexpr int NS = SM::NS, NTG = C::NT, NG = C::NG, NBUF = NG + 1;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)NBUF * SM::TILE_BYTES);
    volatile int *issued = reinterpret_cast<volatile int *>(full + NBUF);
    const int tid = threadIdx.x, grp = tid / NTG, gt = tid - grp * NTG;
    const int bid = blockIdx.x, stride = gridDim.x;
    const int J = (cp.total - bid + stride - 1) / stride;
    if (tid == 0)
        for (int b = 0; b < NBUF; ++b) { mbar_init(full + b, 1); issued[b] = (b < J) ? 1 : 0; }
    const SweepParams<T> &p0 = cp.p[0];
    Tabs<T> tb{p0.twA, p0.twB, p0.phase, p0.ksq_pos};
    if constexpr (SM::TW_IN_SMEM) {
        cx<T> *a = reinterpret_cast<cx<T> *>(smem + SM::TWA);
        for (int i = tid; i < C::N; i += NTG * NG) a[i] = p0.twA[i];
        tb.twA = a;
        if constexpr (C::RB > 1) {
            cx<T> *b2 = a + C::N;
            for (int i = tid; i < C::MB; i += NTG * NG) b2[i] = p0.twB[i];
            tb.twB = b2;
        }
    }
    if constexpr (SM::AUX_IN_SMEM && SM::AUX == AUX_PHASE) {
        cx<T> *a = reinterpret_cast<cx<T> *>(smem + SM::AUX_OFF);
        for (int i = tid; i < C::N; i += NTG * NG) a[i] = p0.phase[i];
        tb.phase = a;
    }
    if constexpr (SM::AUX_IN_SMEM && SM::AUX == AUX_KSQ) {
        T *a = reinterpret_cast<T *>(smem + SM::AUX_OFF);
        for (int i = tid; i < C::N; i += NTG * NG) a[i] = p0.ksq_pos[i];
        tb.ksq_pos = a;
    }
    __syncthreads();

    // request tile number j of this CTA into buffer b: the FIRST WARP of the group (gt < 32) -- lane 0 waits for
    // the planes the tile depends on, then the warp issues the bulk copies; the other warps go on to their next tile
    auto request = [&](int j, int b) {
        const TileRef r = chain_decode(cp, bid + j * stride);
        if (r.stage > 0) {
            if (gt == 0) {
                const unsigned int *ctr = cp.done + (size_t)(r.stage - 1) * cp.units + r.unit;
                while ((int)(ld_acquire(ctr) - cp.target) < 0) __nanosleep(100);
            }
            __syncwarp();
            asm volatile("fence.proxy.async;" ::: "memory");       // acquired (generic proxy) before the bulk reads (async proxy)
        }
        unsigned char *buf = smem + (size_t)b * SM::TILE_BYTES;
        auto go = [&](auto i_) {
            constexpr int I = decltype(i_)::value;
            using K = typename StageAt<I, KS...>::type;
            K::issue(cp.p[I], r.tile, buf, full + b, gt);
        };
        chain_dispatch<0, NS>(r.stage, go);
    };

    // first round of fills: a group requests its own first tile now and the rest of the round only after it
    // has computed that tile (a group must never wait on a dependency while it sits on an uncomputed tile
    // that the dependency may, transitively, need)
    if (grp < J && gt < 32) request(grp, grp);
    typename K0::Pre pre;
    auto prefetch_for = [&](int j) {
        if (j < J) {
            const TileRef r = chain_decode(cp, bid + j * stride);
            if (r.stage == 0) K0::prefetch(cp.p[0], r.tile, gt, pre);
        }
    };
    prefetch_for(grp);
    for (int j = grp; j < J; j += NG) {
        const int b = j % NBUF;
        unsigned char *buf = smem + (size_t)b * SM::TILE_BYTES;
        const TileRef r = chain_decode(cp, bid + j * stride);
        // one warp polls for the start of this fill (the others would only burn issue slots the other group needs)
        if (gt < 32)
            while (issued[b] < j / NBUF + 1) __nanosleep(100);
        group_sync(grp, NTG);
        mbar_wait(full + b, (j / NBUF) & 1);
        auto hook = [&]() { prefetch_for(j + NG); };
        auto go = [&](auto i_) {
            constexpr int I = decltype(i_)::value;
            using K = typename StageAt<I, KS...>::type;
            typename K::Pers pers;          // (level-A twiddles: fetched per tile here, the stages differ)
            pers.setup(tb, gt);
            if constexpr (I == 0) {
                K::compute(cp.p[I], tb, r.tile, buf, gt, grp, pre, pers, hook);
            } else {
                typename K::Pre none;
                K::compute(cp.p[I], tb, r.tile, buf, gt, grp, none, pers, hook);
            }
        };
        chain_dispatch<0, NS>(r.stage, go);
        fence_proxy_async();
        group_sync(grp, NTG);                                   // buffer free; every store of the tile issued
        if (gt < 32) {
            // release: the group's stores (ordered before this thread by the barrier) are visible before the count
            if (gt == 0 && r.stage < NS - 1) red_release_add(cp.done + (size_t)r.stage * cp.units + r.unit, 1u);
            if (j < NG)
                for (int jj = j + NG; jj < NBUF && jj < J; jj += NG) request(jj, jj);
            if (j + NBUF < J) {
                if (gt == 0) issued[b] = (j + NBUF) / NBUF + 1;
                request(j + NBUF, b);
            }
        }
    }
}

#endif  // __CUDACC__

}  // namespace wdm
