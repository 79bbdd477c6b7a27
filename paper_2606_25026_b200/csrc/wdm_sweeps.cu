// wdm_sweeps.cu -- __global__ wrappers of the pipelined sweeps for ONE (dtype, N), selected at compile time
// with -DWDM_DTYPE={0,1} -DWDM_N=<N>.  build.py compiles this file once per supported size.
#include "wdm_internal.hpp"
#include "wdm_pipe.cuh"

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
    k_pipe<K><<<grid, kThreads, smem_of<K>(), s>>>(*static_cast<const P *>(pp), ntiles);
    return cudaGetLastError();
}

using PsiZKick = PsiK<C, AX_CONTIG, true, false, true>;
using PsiZ = PsiK<C, AX_CONTIG, false, false, true>;
using PsiS = PsiK<C, AX_STRIDED, false, false, true>;
using PsiXRho = PsiK<C, AX_STRIDED, false, true, true>;
using RhoOnly = PsiK<C, AX_STRIDED, false, true, false>;
using HYF = HK<C, H_Y_FWD>;
using HZG = HK<C, H_Z_GREEN>;
using HYI = HK<C, H_Y_INV>;
using C2R = C2RK<C>;

cudaError_t init()
{
    int dev = 0, sms = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    g_ctas = sms * C::MINB;
#define OPT(K) if ((e = optin<K>()) != cudaSuccess) return e;
    OPT(PsiZKick) OPT(PsiZ) OPT(PsiS) OPT(PsiXRho) OPT(RhoOnly) OPT(HYF) OPT(HZG) OPT(HYI) OPT(C2R)
#undef OPT
    return cudaSuccess;
}

cudaError_t psi_z(const void *pp, int kick, cudaStream_t s)
{
    return kick ? launch<PsiZKick>(pp, kTilesGrid, s) : launch<PsiZ>(pp, kTilesGrid, s);
}
cudaError_t psi_strided(const void *pp, cudaStream_t s) { return launch<PsiS>(pp, kTilesGrid, s); }
cudaError_t psi_x_rho(const void *pp, int drift, cudaStream_t s)
{
    return drift ? launch<PsiXRho>(pp, kTilesGrid, s) : launch<RhoOnly>(pp, kTilesGrid, s);
}
cudaError_t h_y_fwd(const void *pp, cudaStream_t s) { return launch<HYF>(pp, kTilesHalf, s); }
cudaError_t h_z_green(const void *pp, cudaStream_t s) { return launch<HZG>(pp, kTilesHalf, s); }
cudaError_t h_y_inv(const void *pp, cudaStream_t s) { return launch<HYI>(pp, kTilesHalf, s); }
cudaError_t c2r(const void *pp, cudaStream_t s) { return launch<C2R>(pp, kTilesGrid, s); }

const SweepTable kTable = {Fact{C::N, C::RA, C::RB, C::RM, C::W, C::NT, C::NG, C::MINB}, WDM_DTYPE, init, psi_z,
                           psi_strided, psi_x_rho, h_y_fwd, h_z_green, h_y_inv, c2r};

}  // namespace

#define WDM_CAT3(a, b, c) a##b##_##c
#define WDM_TABLE_NAME(d, n) WDM_CAT3(sweep_table_, d, n)
const SweepTable *WDM_TABLE_NAME(WDM_DTYPE, WDM_N)() { return &kTable; }

}  // namespace wdm
