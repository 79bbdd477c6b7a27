// wdm_sweeps.cu -- __global__ wrappers of the sweep bodies for ONE (dtype, N), selected at compile time
// with -DWDM_DTYPE={0,1} -DWDM_N=<N>.  build.py compiles this file once per supported size.
#include "wdm_internal.hpp"
#include "wdm_kernels.cuh"

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
#define X(n, ra, rb, rm, w, nt, minb) \
    template <> struct CfgOf<n> { using type = LineCfg<Real, n, ra, rb, rm, w, nt, minb>; };
WDM_FACT_LIST(X)
#undef X
using C = CfgOf<WDM_N>::type;
using P = SweepParams<Real>;

constexpr size_t kSmemStrided = (size_t)C::N * C::W * sizeof(cx<Real>);
constexpr size_t kSmemContig = (size_t)C::N * (C::W + 1) * sizeof(cx<Real>);

template <int AX, bool KICK, bool RHO, bool DRIFT>
__global__ void __launch_bounds__(C::NT, C::MINB) k_psi(const __grid_constant__ P p)
{
    extern __shared__ __align__(16) unsigned char smem[];
    psi_sweep_body<C, AX, KICK, RHO, DRIFT>(p, threadIdx.x, blockIdx.x, smem);
}

template <int MODE>
__global__ void __launch_bounds__(C::NT, C::MINB) k_h(const __grid_constant__ P p)
{
    extern __shared__ __align__(16) unsigned char smem[];
    h_sweep_body<C, MODE>(p, threadIdx.x, blockIdx.x, smem);
}

__global__ void __launch_bounds__(C::NT, C::MINB) k_c2r(const __grid_constant__ P p)
{
    extern __shared__ __align__(16) unsigned char smem[];
    c2r_body<C>(p, threadIdx.x, blockIdx.x, smem);
}

constexpr int kTilesGrid = C::N * C::N / C::W;                 // tiles of an N^3 array
constexpr int kTilesHalf = (C::N / 2 + 1) * C::N / C::W;       // tiles of the half spectrum

template <class K>
cudaError_t optin(K kernel, size_t smem)
{
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}

cudaError_t init()
{
    cudaError_t e;
#define OPT(k, s) if ((e = optin(k, s)) != cudaSuccess) return e;
    OPT((k_psi<AX_CONTIG, true, false, true>), kSmemContig)
    OPT((k_psi<AX_CONTIG, false, false, true>), kSmemContig)
    OPT((k_psi<AX_STRIDED, false, false, true>), kSmemStrided)
    OPT((k_psi<AX_STRIDED, false, true, true>), kSmemStrided)
    OPT((k_psi<AX_STRIDED, false, true, false>), kSmemStrided)
    OPT((k_h<H_Y_FWD>), kSmemStrided)
    OPT((k_h<H_Z_GREEN>), kSmemContig)
    OPT((k_h<H_Y_INV>), kSmemStrided)
    OPT(k_c2r, kSmemStrided)
#undef OPT
    return cudaSuccess;
}

cudaError_t psi_z(const void *pp, int kick, cudaStream_t s)
{
    const P &p = *static_cast<const P *>(pp);
    if (kick) k_psi<AX_CONTIG, true, false, true><<<kTilesGrid, C::NT, kSmemContig, s>>>(p);
    else k_psi<AX_CONTIG, false, false, true><<<kTilesGrid, C::NT, kSmemContig, s>>>(p);
    return cudaGetLastError();
}

cudaError_t psi_strided(const void *pp, cudaStream_t s)
{
    k_psi<AX_STRIDED, false, false, true><<<kTilesGrid, C::NT, kSmemStrided, s>>>(*static_cast<const P *>(pp));
    return cudaGetLastError();
}

cudaError_t psi_x_rho(const void *pp, int drift, cudaStream_t s)
{
    const P &p = *static_cast<const P *>(pp);
    if (drift) k_psi<AX_STRIDED, false, true, true><<<kTilesGrid, C::NT, kSmemStrided, s>>>(p);
    else k_psi<AX_STRIDED, false, true, false><<<kTilesGrid, C::NT, kSmemStrided, s>>>(p);
    return cudaGetLastError();
}

cudaError_t h_y_fwd(const void *pp, cudaStream_t s)
{
    k_h<H_Y_FWD><<<kTilesHalf, C::NT, kSmemStrided, s>>>(*static_cast<const P *>(pp));
    return cudaGetLastError();
}
cudaError_t h_z_green(const void *pp, cudaStream_t s)
{
    k_h<H_Z_GREEN><<<kTilesHalf, C::NT, kSmemContig, s>>>(*static_cast<const P *>(pp));
    return cudaGetLastError();
}
cudaError_t h_y_inv(const void *pp, cudaStream_t s)
{
    k_h<H_Y_INV><<<kTilesHalf, C::NT, kSmemStrided, s>>>(*static_cast<const P *>(pp));
    return cudaGetLastError();
}
cudaError_t c2r(const void *pp, cudaStream_t s)
{
    k_c2r<<<kTilesGrid, C::NT, kSmemStrided, s>>>(*static_cast<const P *>(pp));
    return cudaGetLastError();
}

const SweepTable kTable = {Fact{C::N, C::RA, C::RB, C::RM, C::W, C::NT, C::MINB}, WDM_DTYPE, init, psi_z, psi_strided,
                           psi_x_rho, h_y_fwd, h_z_green, h_y_inv, c2r};

}  // namespace

#define WDM_CAT3(a, b, c) a##b##_##c
#define WDM_TABLE_NAME(d, n) WDM_CAT3(sweep_table_, d, n)
const SweepTable *WDM_TABLE_NAME(WDM_DTYPE, WDM_N)() { return &kTable; }

}  // namespace wdm
