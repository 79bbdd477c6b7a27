// wdm_sweeps.cu -- __global__ wrappers of the pipelined sweeps for ONE (dtype, N), selected at compile time
// with -DWDM_DTYPE={0,1} -DWDM_N=<N>.  build.py compiles this file once per supported size.
#include "wdm_internal.hpp"
#include "wdm_chain.cuh"

#ifndef WDM_DTYPE
#error "compile with -DWDM_DTYPE=0|1 -DWDM_N=<N>"
#endif

namespace wdm {
namespace {

#if WDM_DTYPE == 0
using Real = float;
#define WDM_FACT_LIST WDM_FACT_C64
#else
using Real = double;
#define WDM_FACT_LIST WDM_FACT_C128
#endif

// pick the row of the factorisation table with n == WDM_N
template <int NN> struct CfgOf;
#define X(n, ra, rb, rm, w, nt, ng, minb) \
    template <> struct CfgOf<n> { using type = LineCfg<Real, n, ra, rb, rm, w, nt, ng, minb>; };
WDM_FACT_LIST(X)
#undef X
using C = CfgOf<WDM_N>::type;
using P = SweepParams<Real>;

constexpr int kThreads = C::NT * C::NG;
constexpr int kTilesGrid = C::N * C::N / C::W;                 // tiles of an N^3 array
constexpr int kTilesHalf = (C::N / 2 + 1) * C::N / C::W;       // tiles of the half spectrum
int g_ctas = 0;                                                // persistent grid: SMs x MINB

template <class K>
__global__ void __launch_bounds__(kThreads, C::MINB) k_pipe(const __grid_constant__ P p, const int ntiles)
{
    extern __shared__ __align__(128) unsigned char smem[];
    pipe_run<K>(p, ntiles, smem);
}

template <class K> constexpr size_t smem_of() { return PipeSmem<K>::TOTAL; }

template <class... KS>
__global__ void __launch_bounds__(kThreads, C::MINB) k_chain(const __grid_constant__ ChainParams<Real, (int)sizeof...(KS)> cp)
{
    extern __shared__ __align__(128) unsigned char smem[];
    chain_run<KS...>(cp, smem);
}

template <class K>
cudaError_t optin()
{
    return cudaFuncSetAttribute(k_pipe<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_of<K>());
}

template <class K>
cudaError_t launch(const void *pp, int ntiles, cudaStream_t s)
{
    int grid = ntiles < g_ctas ? ntiles : g_ctas;
    // programmatic stream serialization: the kernel may start while its predecessor drains; it orders itself with
    // griddepcontrol.wait (pipe_run) before touching anything the predecessor wrote
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = smem_of<K>();
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k_pipe<K>, *static_cast<const P *>(pp), ntiles);
}

constexpr int kTilesPerPlane = C::N / C::W;                     // every chained stage: N / W tiles per x-plane
int g_chain_ctas = 0;                                           // co-resident CTAs of the chained kernels

template <class... KS>
cudaError_t chain_optin(int sms)
{
    auto *f = k_chain<KS...>;
    cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ChainSmem<KS...>::TOTAL);
    if (e != cudaSuccess) return e;
    int occ = 0;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, f, kThreads, ChainSmem<KS...>::TOTAL)) != cudaSuccess) return e;
    if (occ > C::MINB) occ = C::MINB;
    if (occ * sms < g_chain_ctas) g_chain_ctas = occ * sms;
    return cudaSuccess;
}

template <class... KS>
cudaError_t chain_launch(ChainParams<Real, (int)sizeof...(KS)> &cp, int planes, const ChainCtl *ctl, cudaStream_t s)
{
    chain_plan(cp, planes, kTilesPerPlane, ctl->lag);
    cp.done = ctl->done;
    cp.target = ctl->target;
    int grid = cp.total < g_chain_ctas ? cp.total : g_chain_ctas;
    if (grid <= 0 || chain_min_distance(kTilesPerPlane, ctl->lag < planes ? ctl->lag : planes) <= grid) return cudaErrorInvalidConfiguration;
    void *args[] = {&cp};
    return cudaLaunchCooperativeKernel((void *)k_chain<KS...>, dim3(grid), dim3(kThreads), args, ChainSmem<KS...>::TOTAL, s);
}

using PsiZKick = PsiK<C, AX_CONTIG, 1, false, true>;
using PsiZKickX = PsiK<C, AX_CONTIG, 2, false, true>;
using PsiZ = PsiK<C, AX_CONTIG, 0, false, true>;
using PsiS = PsiK<C, AX_Y, 0, false, true>;
using PsiX = PsiK<C, AX_X, 0, false, true>;
using PsiXRho = PsiK<C, AX_X, 0, true, true>;
using RhoOnly = PsiK<C, AX_X, 0, true, false>;
using HYF = HK<C, H_Y_FWD>;
using HZG = HK<C, H_Z_GREEN>;
using HYI = HK<C, H_Y_INV>;
using C2R = C2RK<C, false>;
using C2RExt = C2RK<C, true>;
// the same sweeps accumulating the per-step diagnostics (wdm_set_step_diagnostics), and the forward-only sweeps that
// measure the spectral kinetic energy on demand (wdm_get_diagnostics)
using PsiZKickD = PsiK<C, AX_CONTIG, 1, false, true, 1>;
using PsiZKickXD = PsiK<C, AX_CONTIG, 2, false, true, 1>;
using PsiZD = PsiK<C, AX_CONTIG, 0, false, true, 1>;
using PsiSD = PsiK<C, AX_Y, 0, false, true, 1>;
using PsiXD = PsiK<C, AX_X, 0, false, true, 1>;
using PsiXRhoD = PsiK<C, AX_X, 0, true, true, 1>;
using HZGD = HK<C, H_Z_GREEN, 1>;
using C2RD = C2RK<C, false, 1>;
using C2RExtD = C2RK<C, true, 1>;
using PsiZM = PsiK<C, AX_CONTIG, 0, false, true, 2>;
using PsiSM = PsiK<C, AX_Y, 0, false, true, 2>;
using PsiXM = PsiK<C, AX_X, 0, false, true, 2>;

cudaError_t init()
{
    int dev = 0, sms = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    g_ctas = sms * C::MINB;
#define OPT(K) if ((e = optin<K>()) != cudaSuccess) return e;
    OPT(PsiZKick) OPT(PsiZKickX) OPT(C2RExt) OPT(PsiZ) OPT(PsiS) OPT(PsiX) OPT(PsiXRho) OPT(RhoOnly) OPT(HYF) OPT(HZG) OPT(HYI) OPT(C2R)
    OPT(PsiZKickD) OPT(PsiZKickXD) OPT(PsiZD) OPT(PsiSD) OPT(PsiXD) OPT(PsiXRhoD) OPT(HZGD) OPT(C2RD) OPT(C2RExtD) OPT(PsiZM) OPT(PsiSM) OPT(PsiXM)
#undef OPT
    g_chain_ctas = g_ctas;
    if ((e = chain_optin<PsiZKick, PsiS>(sms)) != cudaSuccess) return e;
    if ((e = chain_optin<PsiZ, PsiS>(sms)) != cudaSuccess) return e;
    if ((e = chain_optin<HYF, HZG, HYI>(sms)) != cudaSuccess) return e;
    return cudaSuccess;
}

// lag (in planes) between consecutive stages: large enough that a tile's dependencies were stored before the
// pipeline wants to request it (NBUF tiles per CTA are in flight), as small as possible beyond that so the
// planes in transit stay in L2.  0: chaining is pointless or unsafe for this size.
int chain_lag(int stages, int planes, int requested)
{
    const int tiles = planes * kTilesPerPlane * stages;
    const int grid = tiles < g_chain_ctas ? tiles : g_chain_ctas;
    if (g_chain_ctas <= 0 || planes < 4) return 0;
    int safe = grid / kTilesPerPlane + 1;                                   // lag * tpu + 1 > grid
    int lag = requested;
    if (lag <= 0) {
        int inflight = (C::NG + 1) * grid;                                  // measured optimum: about twice the tiles in flight
        lag = 2 * inflight / (kTilesPerPlane * stages) + 1;
        if (lag > planes / 2) lag = planes / 2;                             // small grids: keep the stages overlapped
    }
    if (lag < safe) lag = safe;
    if (lag >= planes) return 0;
    return lag;
}

cudaError_t psi_zy(const void *pz, const void *py, int kick, const ChainCtl *ctl, cudaStream_t s)
{
    ChainParams<Real, 2> cp;
    cp.p[0] = *static_cast<const P *>(pz);
    cp.p[1] = *static_cast<const P *>(py);
    return kick ? chain_launch<PsiZKick, PsiS>(cp, C::N, ctl, s) : chain_launch<PsiZ, PsiS>(cp, C::N, ctl, s);
}
cudaError_t h_yzy(const void *py, const void *pz, const ChainCtl *ctl, cudaStream_t s)
{
    ChainParams<Real, 3> cp;
    cp.p[0] = *static_cast<const P *>(py);
    cp.p[1] = *static_cast<const P *>(pz);
    cp.p[2] = *static_cast<const P *>(py);
    return chain_launch<HYF, HZG, HYI>(cp, C::N / 2 + 1, ctl, s);
}

// diag: 0 plain, 1 accumulate the per-step diagnostics, 2 (psi sweeps without kick only) measure, write nothing
cudaError_t psi_z(const void *pp, int kick, int diag, cudaStream_t s)
{
    if (diag == 2) return launch<PsiZM>(pp, kTilesGrid, s);
    if (diag == 1) return kick == 2 ? launch<PsiZKickXD>(pp, kTilesGrid, s) : (kick ? launch<PsiZKickD>(pp, kTilesGrid, s) : launch<PsiZD>(pp, kTilesGrid, s));
    return kick == 2 ? launch<PsiZKickX>(pp, kTilesGrid, s) : (kick ? launch<PsiZKick>(pp, kTilesGrid, s) : launch<PsiZ>(pp, kTilesGrid, s));
}
cudaError_t psi_strided(const void *pp, int along_x, int diag, cudaStream_t s)
{
    if (diag == 2) return along_x ? launch<PsiXM>(pp, kTilesGrid, s) : launch<PsiSM>(pp, kTilesGrid, s);
    if (diag == 1) return along_x ? launch<PsiXD>(pp, kTilesGrid, s) : launch<PsiSD>(pp, kTilesGrid, s);
    return along_x ? launch<PsiX>(pp, kTilesGrid, s) : launch<PsiS>(pp, kTilesGrid, s);
}
cudaError_t psi_x_rho(const void *pp, int drift, int diag, cudaStream_t s)
{
    if (diag == 1 && drift) return launch<PsiXRhoD>(pp, kTilesGrid, s);
    return drift ? launch<PsiXRho>(pp, kTilesGrid, s) : launch<RhoOnly>(pp, kTilesGrid, s);
}
cudaError_t h_y_fwd(const void *pp, cudaStream_t s) { return launch<HYF>(pp, kTilesHalf, s); }
cudaError_t h_z_green(const void *pp, int diag, cudaStream_t s) { return diag == 1 ? launch<HZGD>(pp, kTilesHalf, s) : launch<HZG>(pp, kTilesHalf, s); }
cudaError_t h_y_inv(const void *pp, cudaStream_t s) { return launch<HYI>(pp, kTilesHalf, s); }
cudaError_t c2r(const void *pp, int diag, cudaStream_t s)
{
    const bool ext = static_cast<const P *>(pp)->phi_ext != nullptr;
    if (diag == 1) return ext ? launch<C2RExtD>(pp, kTilesGrid, s) : launch<C2RD>(pp, kTilesGrid, s);
    return ext ? launch<C2RExt>(pp, kTilesGrid, s) : launch<C2R>(pp, kTilesGrid, s);
}

const SweepTable kTable = {Fact{C::N, C::RA, C::RB, C::RM, C::W, C::NT, C::NG, C::MINB}, WDM_DTYPE, init, psi_z,
                           psi_strided, psi_x_rho, h_y_fwd, h_z_green, h_y_inv, c2r, chain_lag, psi_zy, h_yzy};

}  // namespace

#define WDM_CAT3(a, b, c) a##b##_##c
#define WDM_TABLE_NAME(d, n) WDM_CAT3(sweep_table_, d, n)
const SweepTable *WDM_TABLE_NAME(WDM_DTYPE, WDM_N)() { return &kTable; }

}  // namespace wdm
