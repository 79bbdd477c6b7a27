// wdm_sweeps.cu -- __global__ wrappers of the pipelined sweeps for ONE (dtype, N), selected at compile time
// with -DWDM_DTYPE={0,1} -DWDM_N=<N>.  build.py compiles this file once per supported size.
#include "wdm_internal.hpp"
#include "wdm_pipe.cuh"
#if WDM_DTYPE == 0 && WDM_N == 1024
#include "wdm_x2.cuh"
#endif

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

// x-direction psi sweep and density sweep on half tiles (wdm_x2.cuh): 1024-point complex64 lines
#if WDM_DTYPE == 0 && WDM_N == 1024
#define WDM_HAVE_X2 1
using C5 = LineCfg<Real, 512, 16, 1, 32, 16, 256, 2, 1>;
constexpr int kX2W = C5::W, kTilesX2 = C::N * C::N / C5::W;
static_assert(kThreads == 512 && C::MINB == 1, "launch shape of the half-tile sweeps");

template <bool RHO>
__global__ void __launch_bounds__(512, 1) k_x2(const __grid_constant__ P p, const int ntiles)
{
    extern __shared__ __align__(128) unsigned char smem[];
    X2<C5, RHO>::run(p, ntiles, smem);
}

template <bool RHO>
cudaError_t launch_x2(const void *pp, cudaStream_t s)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(kTilesX2 < g_ctas ? kTilesX2 : g_ctas);
    cfg.blockDim = dim3(512);
    cfg.dynamicSmemBytes = X2<C5, RHO>::TOTAL;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k_x2<RHO>, *static_cast<const P *>(pp), kTilesX2);
}
#else
#define WDM_HAVE_X2 0
constexpr int kX2W = 0;
#endif

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
// complex-to-real sweep: in place where the tile buffer then holds twice the lines of the packed-copy form (W = 16 instead
// of 8 for 1024-point complex64 lines, 32 instead of 16 for 512-point ones)
#if WDM_DTYPE == 0 && WDM_N == 1024
using CR = LineCfg<Real, 1024, 32, 1, 32, 16, 256, 2, 1>;
template <bool EXT, int DG> using C2RSel = C2RI<CR, EXT, DG>;
#elif WDM_DTYPE == 0 && WDM_N == 512
using CR = LineCfg<Real, 512, 16, 1, 32, 32, 256, 2, 1>;
template <bool EXT, int DG> using C2RSel = C2RI<CR, EXT, DG>;
#else
using CR = C;
template <bool EXT, int DG> using C2RSel = C2RK<C, EXT, DG>;
#endif
static_assert(CR::NT * CR::NG == kThreads && CR::MINB == C::MINB, "one launch shape for every sweep of a size");
constexpr int kTilesC2R = CR::N * CR::N / CR::W;
using C2R = C2RSel<false, 0>;
using C2RExt = C2RSel<true, 0>;
// the same sweeps accumulating the per-step diagnostics (wdm_set_step_diagnostics), and the forward-only sweeps that
// measure the spectral kinetic energy on demand (wdm_get_diagnostics)
using PsiZKickD = PsiK<C, AX_CONTIG, 1, false, true, 1>;
using PsiZKickXD = PsiK<C, AX_CONTIG, 2, false, true, 1>;
using PsiZD = PsiK<C, AX_CONTIG, 0, false, true, 1>;
using PsiSD = PsiK<C, AX_Y, 0, false, true, 1>;
using PsiXD = PsiK<C, AX_X, 0, false, true, 1>;
using PsiXRhoD = PsiK<C, AX_X, 0, true, true, 1>;
using HZGD = HK<C, H_Z_GREEN, 1>;
using C2RD = C2RSel<false, 1>;
using C2RExtD = C2RSel<true, 1>;
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
#if WDM_HAVE_X2
    if ((e = cudaFuncSetAttribute(k_x2<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)X2<C5, false>::TOTAL)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_x2<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)X2<C5, true>::TOTAL)) != cudaSuccess) return e;
#endif
    return cudaSuccess;
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
#if WDM_HAVE_X2
    if (along_x && diag == 0 && static_cast<const P *>(pp)->x2tab) return launch_x2<false>(pp, s);
#endif
    if (diag == 2) return along_x ? launch<PsiXM>(pp, kTilesGrid, s) : launch<PsiSM>(pp, kTilesGrid, s);
    if (diag == 1) return along_x ? launch<PsiXD>(pp, kTilesGrid, s) : launch<PsiSD>(pp, kTilesGrid, s);
    return along_x ? launch<PsiX>(pp, kTilesGrid, s) : launch<PsiS>(pp, kTilesGrid, s);
}
cudaError_t psi_x_rho(const void *pp, int drift, int diag, cudaStream_t s)
{
#if WDM_HAVE_X2
    if (drift && diag == 0 && static_cast<const P *>(pp)->x2tab) return launch_x2<true>(pp, s);
#endif
    if (diag == 1 && drift) return launch<PsiXRhoD>(pp, kTilesGrid, s);
    return drift ? launch<PsiXRho>(pp, kTilesGrid, s) : launch<RhoOnly>(pp, kTilesGrid, s);
}
cudaError_t h_y_fwd(const void *pp, cudaStream_t s) { return launch<HYF>(pp, kTilesHalf, s); }
cudaError_t h_z_green(const void *pp, int diag, cudaStream_t s) { return diag == 1 ? launch<HZGD>(pp, kTilesHalf, s) : launch<HZG>(pp, kTilesHalf, s); }
cudaError_t h_y_inv(const void *pp, cudaStream_t s) { return launch<HYI>(pp, kTilesHalf, s); }
cudaError_t c2r(const void *pp, int diag, cudaStream_t s)
{
    const bool ext = static_cast<const P *>(pp)->phi_ext != nullptr;
    if (diag == 1) return ext ? launch<C2RExtD>(pp, kTilesC2R, s) : launch<C2RD>(pp, kTilesC2R, s);
    return ext ? launch<C2RExt>(pp, kTilesC2R, s) : launch<C2R>(pp, kTilesC2R, s);
}

// ---- slab-decomposed runs (wdm_dist.cu): the same sweeps on slab-shaped arrays, tile count given by the caller; the
// distributed axis x is the middle index of the transposed slabs, so its sweeps are AX_Y instantiations
using PsiTRho = PsiK<C, AX_Y, 0, true, true>;
using RhoOnlyT = PsiK<C, AX_Y, 0, true, false>;
using C2RT = C2RK<C, false, 0, AX_Y>;
cudaError_t dist_init()
{
    cudaError_t e;
    if ((e = optin<PsiTRho>()) != cudaSuccess) return e;
    if ((e = optin<RhoOnlyT>()) != cudaSuccess) return e;
    return optin<C2RT>();
}
cudaError_t dist_psi_z(const void *pp, int kick, int ntiles, cudaStream_t s) { return kick ? launch<PsiZKick>(pp, ntiles, s) : launch<PsiZ>(pp, ntiles, s); }
cudaError_t dist_psi_y(const void *pp, int ntiles, cudaStream_t s) { return launch<PsiS>(pp, ntiles, s); }
cudaError_t dist_psi_x_rho(const void *pp, int drift, int ntiles, cudaStream_t s)
{
    return drift ? launch<PsiTRho>(pp, ntiles, s) : launch<RhoOnlyT>(pp, ntiles, s);
}
cudaError_t dist_h_y(const void *pp, int inverse, int ntiles, cudaStream_t s) { return inverse ? launch<HYI>(pp, ntiles, s) : launch<HYF>(pp, ntiles, s); }
cudaError_t dist_h_z_green(const void *pp, int ntiles, cudaStream_t s) { return launch<HZG>(pp, ntiles, s); }
cudaError_t dist_c2r(const void *pp, int ntiles, cudaStream_t s) { return launch<C2RT>(pp, ntiles, s); }

const SweepTable kTable = {Fact{C::N, C::RA, C::RB, C::RM, C::W, C::NT, C::NG, C::MINB}, WDM_DTYPE, CR::W, kX2W, init, psi_z,
                           psi_strided, psi_x_rho, h_y_fwd, h_z_green, h_y_inv, c2r,
                           dist_init, dist_psi_z, dist_psi_y, dist_psi_x_rho, dist_h_y, dist_h_z_green, dist_c2r};

}  // namespace

#define WDM_CAT3(a, b, c) a##b##_##c
#define WDM_TABLE_NAME(d, n) WDM_CAT3(sweep_table_, d, n)
const SweepTable *WDM_TABLE_NAME(WDM_DTYPE, WDM_N)() { return &kTable; }

}  // namespace wdm
