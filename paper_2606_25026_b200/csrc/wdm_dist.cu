// wdm_dist.cu -- slab-decomposed kick-drift-kick step: the local half of a multi-GPU run (the
// paper lists a distributed FFT as future work).  See include/wdm_dist.h for the contract.
//
// World of P ranks, N divisible by P, xl = N / P.  Rank r owns the x-planes [r xl, (r+1) xl).  Every axis sweep couples
// a whole line, so the distributed axis has to be gathered before it is swept: the state is kept TRANSPOSED,
//     psi^T[y_l][x][z], Phi^T[y_l][x][z], H^T[y_l][kx][z]      (y_l < xl local, x / kx complete, z contiguous)
// in which the x transforms are plain middle-axis (AX_Y) sweeps and the z sweeps and the kick are local; only the y
// sweeps need the x-slab form psi[x_l][y][z] / H[kx_l][y][z].  One step is five phases of local kernels separated by
// four all-to-all exchanges of equal-sized blocks (two of psi, two of the half spectrum), which the CALLER performs
// between phases (torch.distributed.all_to_all_single over NCCL; a device-to-device copy in the single-GPU emulation
// of the tests):
//     S1  z sweep with the kick on psi^T                         pack -> exchange
//     S2  unpack -> psi x-slab, y sweep                          pack -> exchange
//     S3  unpack -> psi^T, x sweep + rho + real-to-complex -> H^T    pack -> exchange
//     S4  unpack -> H kx-slab, y forward, z Green, y inverse     pack -> exchange
//     S5  unpack -> H^T, complex-to-real along x -> Phi^T
// The sweeps are the single-GPU kernels on slab-shaped arrays (fewer tiles); pack / unpack are line-copy kernels whose
// index maps (dist_copy_plan) are exported for the CPU test.  The kx-planes (N/2 + 1 of them) are dealt out in blocks of
// kxb = ceil((N/2 + 1) / P); the last block(s) are partly or wholly padding.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/wdm_dist.h"
#include "wdm_internal.hpp"
#include "wdm_kernels.cuh"

namespace wdm {

// dst line (i0 d0 + i1 d1 + i2 d2) <- src line (i0 s0 + i1 s1 + i2 s2) for i0 < n0, i1 < n1, i2 < n2; a line is N complex.
// kmul > 0: only where i0 kmul + i[ksel] < klim (kx-planes beyond N/2 are padding).
struct CopyPlan {
    long long n0, n1, n2, s0, s1, s2, d0, d1, d2, kmul, ksel, klim;
};

enum { CP_PSI_T2X_PACK = 0, CP_PSI_T2X_UNPACK, CP_PSI_X2T_PACK, CP_PSI_X2T_UNPACK,
       CP_H_T2K_PACK, CP_H_T2K_UNPACK, CP_H_K2T_PACK, CP_H_K2T_UNPACK, CP_COUNT };

static CopyPlan dist_copy_plan(int N, int P, int op)
{
    const long long xl = N / P, NH = N / 2 + 1, kxb = (NH + P - 1) / P;
    switch (op) {
    // psi^T[y_l][x][z] -> blocks by the rank that owns x: send[d][y_l][x_l]
    case CP_PSI_T2X_PACK:   return {P, xl, xl, /*src*/ xl, N, 1, /*dst*/ xl * xl, xl, 1, 0, 0, 0};
    // recv[s][y_l'][x_l] -> psi[x_l][s xl + y_l'][z]
    case CP_PSI_T2X_UNPACK: return {P, xl, xl, xl * xl, xl, 1, xl, 1, N, 0, 0, 0};
    // psi[x_l][y][z] -> send[d][x_l][y_l]
    case CP_PSI_X2T_PACK:   return {P, xl, xl, xl, N, 1, xl * xl, xl, 1, 0, 0, 0};
    // recv[s][x_l'][y_l] -> psi^T[y_l][s xl + x_l'][z]
    case CP_PSI_X2T_UNPACK: return {P, xl, xl, xl * xl, xl, 1, xl, 1, N, 0, 0, 0};
    // H^T[y_l][kx][z] -> send[d][y_l][kx_l], kx = d kxb + kx_l
    case CP_H_T2K_PACK:     return {P, xl, kxb, kxb, NH, 1, xl * kxb, kxb, 1, kxb, 2, NH};
    // recv[s][y_l'][kx_l] -> H[kx_l][s xl + y_l'][z]
    case CP_H_T2K_UNPACK:   return {P, xl, kxb, xl * kxb, kxb, 1, xl, 1, N, 0, 0, 0};
    // H[kx_l][y][z] -> send[d][kx_l][y_l]
    case CP_H_K2T_PACK:     return {P, kxb, xl, xl, N, 1, kxb * xl, xl, 1, 0, 0, 0};
    // recv[s][kx_l'][y_l] -> H^T[y_l][s kxb + kx_l'][z]
    case CP_H_K2T_UNPACK:   return {P, kxb, xl, kxb * xl, xl, 1, kxb, 1, NH, kxb, 1, NH};
    }
    return {};
}

// one warp per line, 16-byte vectors
__global__ void __launch_bounds__(256) k_copy_lines(const uint4 *__restrict__ src, uint4 *__restrict__ dst, CopyPlan cp, int vec_per_line)
{
    const long long nlines = cp.n0 * cp.n1 * cp.n2;
    const int lane = threadIdx.x & 31;
    for (long long ln = blockIdx.x * (long long)(blockDim.x >> 5) + (threadIdx.x >> 5); ln < nlines; ln += (long long)gridDim.x * (blockDim.x >> 5)) {
        const long long i2 = ln % cp.n2, i1 = (ln / cp.n2) % cp.n1, i0 = ln / (cp.n2 * cp.n1);
        if (cp.kmul > 0 && i0 * cp.kmul + (cp.ksel == 1 ? i1 : i2) >= cp.klim) continue;
        const uint4 *s = src + (i0 * cp.s0 + i1 * cp.s1 + i2 * cp.s2) * vec_per_line;
        uint4 *d = dst + (i0 * cp.d0 + i1 * cp.d1 + i2 * cp.d2) * vec_per_line;
        for (int v = lane; v < vec_per_line; v += 32) d[v] = s[v];
    }
}

template <typename T>
__global__ void k_dist_kick(cx<T> *psi, const T *phi, T coef, size_t n)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        stv(psi + i, rotate_neg(ldv(psi + i), ldg(phi + i) * coef));
}

// partial[b] = sum over this block's share of |psi|^2 (fixed order, as in wdm.cu)
template <typename T>
__global__ void __launch_bounds__(256) k_dist_sum(const cx<T> *psi, size_t n, double *partial)
{
    __shared__ double part[8];
    double s = 0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        cx<T> v = ldv(psi + i);
        s += (double)v.x * v.x + (double)v.y * v.y;
    }
    for (int d = 16; d; d >>= 1) s += __shfl_down_sync(0xffffffffu, s, d);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0;
        for (int w = 0; w < 8; ++w) t += part[w];
        partial[blockIdx.x] = t;
    }
}

}  // namespace wdm

using namespace wdm;

struct wdm_dist {
    int N = 0, dtype = 0, rank = 0, P = 1, xl = 0, NH = 0, kxb = 0, nkx = 0;
    double L = 0, mu = 0, G = 0;
    const SweepTable *tab = nullptr;
    cudaStream_t stream = nullptr;
    size_t slab = 0;                          // N^3 / P elements
    void *psiT = nullptr, *psiX = nullptr, *HT = nullptr, *HK = nullptr, *phiT = nullptr;
    void *twA = nullptr, *twB = nullptr, *phase = nullptr, *ksq_pos = nullptr, *ksq_nat = nullptr, *mean = nullptr;
    double *partial = nullptr;
    unsigned int *tickets = nullptr;
    void *send = nullptr, *recv = nullptr;    // caller's exchange buffers
    CUtensorMap tm_psiT, tm_psiX, tm_HK, tm_HT, tm_HT1;
    int ticket_parity = 0;
    double phase_dt = 0;
    bool phase_valid = false, have_psi = false, in_T = false, phi_valid = false;
    std::string err;
};

static std::string g_dist_err;

static int dfail(wdm_dist *d, int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (d) d->err = buf;
    else g_dist_err = buf;
    return code;
}

#define DCU(d, call)                                                                                    \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) return dfail(d, WDM_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));    \
    } while (0)

static size_t dcs(const wdm_dist *d) { return d->dtype == WDM_C64 ? 8 : 16; }
static size_t drs(const wdm_dist *d) { return d->dtype == WDM_C64 ? 4 : 8; }

// ---------------------------------------------------------------- create / destroy

static int dalloc(wdm_dist *d, void **out, size_t bytes)
{
    cudaError_t e = cudaMalloc(out, bytes ? bytes : 16);
    if (e != cudaSuccess) { cudaGetLastError(); *out = nullptr; return dfail(d, WDM_ENOMEM, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e)); }
    return WDM_OK;
}

template <typename T>
static int dist_upload_tables(wdm_dist *d)
{
    Tables<T> t = build_tables<T>(d->tab->fact, d->L);
    DCU(d, cudaMemcpyAsync(d->twA, t.twA.data(), t.twA.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, d->stream));
    DCU(d, cudaMemcpyAsync(d->twB, t.twB.data(), t.twB.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, d->stream));
    DCU(d, cudaMemcpyAsync(d->ksq_pos, t.ksq_pos.data(), t.ksq_pos.size() * sizeof(T), cudaMemcpyHostToDevice, d->stream));
    DCU(d, cudaMemcpyAsync(d->ksq_nat, t.ksq_nat.data(), t.ksq_nat.size() * sizeof(T), cudaMemcpyHostToDevice, d->stream));
    DCU(d, cudaStreamSynchronize(d->stream));
    return WDM_OK;
}

static void dist_free(wdm_dist *d)
{
    void *ps[] = {d->psiT, d->psiX, d->HT, d->HK, d->phiT, d->twA, d->twB, d->phase, d->ksq_pos, d->ksq_nat, d->mean, d->partial, d->tickets};
    for (void *p : ps)
        if (p) cudaFree(p);
    delete d;
}

extern "C" int wdm_dist_create(wdm_dist **out, int N, double L, double hbar_over_m, double G, int dtype, int rank, int world)
{
    if (!out) return dfail(nullptr, WDM_EINVAL, "null output pointer");
    *out = nullptr;
    if (!(L > 0) || !(hbar_over_m > 0) || !(G >= 0)) return dfail(nullptr, WDM_EINVAL, "need L > 0, hbar_over_m > 0, G >= 0");
    if (dtype != WDM_C64 && dtype != WDM_C128) return dfail(nullptr, WDM_EINVAL, "dtype must be WDM_C64 or WDM_C128");
    if (N < 8 || N > 1024 || (N & (N - 1))) return dfail(nullptr, WDM_EUNSUPPORTED, "N must be a power of two in [8, 1024], got %d", N);
    if (world < 1 || rank < 0 || rank >= world) return dfail(nullptr, WDM_EINVAL, "need 0 <= rank < world");
    const SweepTable *tab = sweep_table(dtype, N);
    if (!tab) return dfail(nullptr, WDM_EUNSUPPORTED, "no kernels built for N = %d", N);
    // a slab must hold whole tiles of every sweep: xl = N / world a multiple of the tile width W (psi^T tiles are
    // (y_l, z-block) pairs and pencil groups; the x-slab form has xl planes)
    if (N % world || (N / world) < 1) return dfail(nullptr, WDM_EUNSUPPORTED, "world = %d must divide N = %d", world, N);
    wdm_dist *d = new wdm_dist();
    d->N = N; d->dtype = dtype; d->rank = rank; d->P = world; d->xl = N / world; d->NH = N / 2 + 1;
    d->kxb = (d->NH + world - 1) / world;
    d->nkx = d->NH - rank * d->kxb;
    if (d->nkx > d->kxb) d->nkx = d->kxb;
    if (d->nkx < 0) d->nkx = 0;
    d->L = L; d->mu = hbar_over_m; d->G = G; d->tab = tab;
    d->slab = (size_t)N * N * d->xl;
    auto bail = [&](int code) { g_dist_err = d->err; dist_free(d); return code; };
    cudaError_t e = tab->init();
    if (e == cudaSuccess) e = tab->dist_init();
    if (e != cudaSuccess) return bail(dfail(d, WDM_ECUDA, "kernel attribute setup: %s", cudaGetErrorString(e)));
    const size_t cs = dcs(d), rs = drs(d);
    int rc;
    if ((rc = dalloc(d, &d->psiT, d->slab * cs)) || (rc = dalloc(d, &d->psiX, d->slab * cs)) ||
        (rc = dalloc(d, &d->HT, (size_t)d->xl * d->NH * N * cs)) || (rc = dalloc(d, &d->HK, (size_t)d->kxb * N * N * cs)) ||
        (rc = dalloc(d, &d->phiT, d->slab * rs)) || (rc = dalloc(d, &d->twA, N * cs)) || (rc = dalloc(d, &d->twB, N * cs)) ||
        (rc = dalloc(d, &d->phase, N * cs)) || (rc = dalloc(d, &d->ksq_pos, N * rs)) || (rc = dalloc(d, &d->ksq_nat, N * rs)) ||
        (rc = dalloc(d, &d->mean, 64)) || (rc = dalloc(d, (void **)&d->partial, 1024 * sizeof(double))) ||
        (rc = dalloc(d, (void **)&d->tickets, 8 * sizeof(unsigned int))))
        return bail(rc);
    if (cudaMemset(d->tickets, 0, 8 * sizeof(unsigned int)) != cudaSuccess || cudaMemset(d->mean, 0, 64) != cudaSuccess ||
        cudaMemset(d->phiT, 0, d->slab * rs) != cudaSuccess)
        return bail(dfail(d, WDM_ECUDA, "cudaMemset failed"));
    rc = dtype == WDM_C64 ? dist_upload_tables<float>(d) : dist_upload_tables<double>(d);
    if (rc) return bail(rc);
    const int W = tab->fact.W, rows = N < 256 ? N : 256, hrows = (N / 2) < 256 ? N / 2 : 256;
    int t;
    if ((t = encode_tmap(dtype, N, W, d->psiT, N, d->xl, 1, rows, &d->tm_psiT)) || (t = encode_tmap(dtype, N, W, d->psiX, N, d->xl, 1, rows, &d->tm_psiX)) ||
        (t = encode_tmap(dtype, N, W, d->HK, N, d->kxb, 1, rows, &d->tm_HK)) || (t = encode_tmap(dtype, N, W, d->HT, d->NH, d->xl, 1, hrows, &d->tm_HT)) ||
        (t = encode_tmap(dtype, N, W, d->HT, d->NH, d->xl, 1, 1, &d->tm_HT1)))
        return bail(dfail(d, WDM_ECUDA, "cuTensorMapEncodeTiled failed (%d)", t));
    *out = d;
    return WDM_OK;
}

extern "C" int wdm_dist_destroy(wdm_dist *d)
{
    if (!d) return WDM_OK;
    cudaStreamSynchronize(d->stream);
    dist_free(d);
    return WDM_OK;
}

extern "C" int wdm_dist_set_stream(wdm_dist *d, void *s)
{
    if (!d) return WDM_EINVAL;
    if ((cudaStream_t)s != d->stream) DCU(d, cudaStreamSynchronize(d->stream));
    d->stream = (cudaStream_t)s;
    return WDM_OK;
}

extern "C" int wdm_dist_exchange_bytes(wdm_dist *d, size_t *bytes_out)
{
    if (!d || !bytes_out) return WDM_EINVAL;
    const size_t psi = (size_t)d->xl * d->xl * d->N * dcs(d), h = (size_t)d->xl * d->kxb * d->N * dcs(d);
    *bytes_out = (psi > h ? psi : h) * d->P;
    return WDM_OK;
}

extern "C" int wdm_dist_set_buffers(wdm_dist *d, void *send_dev, void *recv_dev)
{
    if (!d) return WDM_EINVAL;
    if (!send_dev || !recv_dev || send_dev == recv_dev) return dfail(d, WDM_EINVAL, "need two distinct exchange buffers");
    d->send = send_dev;
    d->recv = recv_dev;
    return WDM_OK;
}

extern "C" int wdm_dist_copy_plan(int N, int world, int op, long long *out12)
{
    if (!out12 || op < 0 || op >= CP_COUNT || world < 1 || N % world) return WDM_EINVAL;
    CopyPlan cp = dist_copy_plan(N, world, op);
    memcpy(out12, &cp, sizeof cp);
    return WDM_OK;
}

extern "C" int wdm_dist_set_psi(wdm_dist *d, const void *psi_xslab_dev)
{
    if (!d) return WDM_EINVAL;
    if (!psi_xslab_dev) return dfail(d, WDM_EINVAL, "null psi");
    DCU(d, cudaMemcpyAsync(d->psiX, psi_xslab_dev, d->slab * dcs(d), cudaMemcpyDeviceToDevice, d->stream));
    d->have_psi = true;
    d->in_T = false;
    d->phi_valid = false;
    return WDM_OK;
}

extern "C" const char *wdm_dist_last_error(const wdm_dist *d) { return d ? d->err.c_str() : g_dist_err.c_str(); }

// ---------------------------------------------------------------- phases

template <typename T>
static int dist_phase_table(wdm_dist *d, double dt)
{
    if (d->phase_valid && d->phase_dt == dt) return WDM_OK;
    std::vector<cx<T>> ph = build_phase<T>(d->tab->fact, d->L, d->mu, dt);
    DCU(d, cudaMemcpyAsync(d->phase, ph.data(), ph.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, d->stream));
    DCU(d, cudaStreamSynchronize(d->stream));
    d->phase_dt = dt;
    d->phase_valid = true;
    return WDM_OK;
}

template <typename T>
static SweepParams<T> dist_params(wdm_dist *d)
{
    SweepParams<T> p{};
    p.twA = (const cx<T> *)d->twA;
    p.twB = (const cx<T> *)d->twB;
    p.phase = (const cx<T> *)d->phase;
    p.ksq_pos = (const T *)d->ksq_pos;
    p.ksq_nat = (const T *)d->ksq_nat;
    p.green = (T)(-4.0 * M_PI * d->G / ((double)d->N * d->N * d->N));
    p.kx0 = d->rank * d->kxb;
    p.H = (cx<T> *)d->HT;
    p.phi = (const T *)d->phiT;
    p.phi_out = (T *)d->phiT;
    p.rho_mean = (const T *)((const unsigned char *)d->mean + 16);
    p.ticket = d->tickets + d->ticket_parity;
    p.ticket_next = d->tickets + (d->ticket_parity ^ 1);
    d->ticket_parity ^= 1;
    return p;
}

static int dist_copy(wdm_dist *d, int op, const void *src, void *dst)
{
    const CopyPlan cp = dist_copy_plan(d->N, d->P, op);
    const long long nlines = cp.n0 * cp.n1 * cp.n2;
    if (nlines == 0) return WDM_OK;
    const int vec = (int)((size_t)d->N * dcs(d) / 16);
    long long blocks = (nlines + 7) / 8;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_copy_lines<<<(unsigned)blocks, 256, 0, d->stream>>>((const uint4 *)src, (uint4 *)dst, cp, vec);
    DCU(d, cudaGetLastError());
    return WDM_OK;
}

static size_t psi_block_bytes(const wdm_dist *d) { return (size_t)d->xl * d->xl * d->N * dcs(d); }
static size_t h_block_bytes(const wdm_dist *d) { return (size_t)d->xl * d->kxb * d->N * dcs(d); }

// The Poisson half shared by the refresh and the step: H^T (just written by the density sweep) -> Phi^T in three phases
template <typename T>
static int dist_poisson_phase(wdm_dist *d, int which, size_t *xbytes)
{
    const int N = d->N, W = d->tab->fact.W;
    int rc;
    if (which == 0) {           // pack H^T for the kx-slab owners
        if ((rc = dist_copy(d, CP_H_T2K_PACK, d->HT, d->send))) return rc;
        *xbytes = h_block_bytes(d);
    } else if (which == 1) {    // kx-slab: y forward, z Green, y inverse
        if ((rc = dist_copy(d, CP_H_T2K_UNPACK, d->recv, d->HK))) return rc;
        const int nt = d->nkx * N / W;
        if (nt > 0) {
            SweepParams<T> p = dist_params<T>(d);
            p.data = (cx<T> *)d->HK;
            p.tmap = d->tm_HK;
            DCU(d, d->tab->dist_h_y(&p, 0, nt, d->stream));
            p = dist_params<T>(d); p.data = (cx<T> *)d->HK; p.tmap = d->tm_HK;
            DCU(d, d->tab->dist_h_z_green(&p, nt, d->stream));
            p = dist_params<T>(d); p.data = (cx<T> *)d->HK; p.tmap = d->tm_HK;
            DCU(d, d->tab->dist_h_y(&p, 1, nt, d->stream));
        }
        if ((rc = dist_copy(d, CP_H_K2T_PACK, d->HK, d->send))) return rc;
        *xbytes = h_block_bytes(d);
    } else {                    // back in H^T: complex-to-real along x
        if ((rc = dist_copy(d, CP_H_K2T_UNPACK, d->recv, d->HT))) return rc;
        SweepParams<T> p = dist_params<T>(d);
        p.tmap = d->tm_HT;
        p.tmap2 = d->tm_HT1;
        DCU(d, d->tab->dist_c2r(&p, d->xl * N / W, d->stream));
        d->phi_valid = true;
        *xbytes = 0;
    }
    return WDM_OK;
}

template <typename T>
static int dist_phase_impl(wdm_dist *d, int phase, double dt, double kick_dt, size_t *xbytes)
{
    const int N = d->N, W = d->tab->fact.W, nt = d->xl * N / W;
    int rc;
    *xbytes = 0;
    switch (phase) {
    case WDM_DIST_R1:           // psi x-slab (as set) -> transposed form
        if (!d->have_psi) return dfail(d, WDM_ESTATE, "wdm_dist_set_psi has not been called");
        if ((rc = dist_copy(d, CP_PSI_X2T_PACK, d->psiX, d->send))) return rc;
        *xbytes = psi_block_bytes(d);
        return WDM_OK;
    case WDM_DIST_R2: {         // psi^T; rho - <rho> and its x-spectrum (the mean was set by wdm_dist_set_mean)
        if ((rc = dist_copy(d, CP_PSI_X2T_UNPACK, d->recv, d->psiT))) return rc;
        d->in_T = true;
        if (!(d->G > 0)) { d->phi_valid = true; return WDM_OK; }        // Phi^T stays zero
        SweepParams<T> p = dist_params<T>(d);
        p.data = (cx<T> *)d->psiT;
        p.tmap = d->tm_psiT;
        DCU(d, d->tab->dist_psi_x_rho(&p, 0, nt, d->stream));
        return dist_poisson_phase<T>(d, 0, xbytes);
    }
    case WDM_DIST_S1: {         // kick on load + z sweep, in the transposed form
        if (!d->in_T || !d->phi_valid) return dfail(d, WDM_ESTATE, "the potential is stale: run the refresh phases first");
        if ((rc = dist_phase_table<T>(d, dt))) return rc;
        SweepParams<T> p = dist_params<T>(d);
        p.data = (cx<T> *)d->psiT;
        p.kick = (T)(kick_dt / d->mu);
        DCU(d, d->tab->dist_psi_z(&p, (d->G > 0 && kick_dt != 0.0) ? 1 : 0, nt, d->stream));
        if ((rc = dist_copy(d, CP_PSI_T2X_PACK, d->psiT, d->send))) return rc;
        *xbytes = psi_block_bytes(d);
        return WDM_OK;
    }
    case WDM_DIST_S2: {         // x-slab: y sweep
        if ((rc = dist_copy(d, CP_PSI_T2X_UNPACK, d->recv, d->psiX))) return rc;
        SweepParams<T> p = dist_params<T>(d);
        p.data = (cx<T> *)d->psiX;
        p.tmap = d->tm_psiX;
        DCU(d, d->tab->dist_psi_y(&p, nt, d->stream));
        if ((rc = dist_copy(d, CP_PSI_X2T_PACK, d->psiX, d->send))) return rc;
        *xbytes = psi_block_bytes(d);
        return WDM_OK;
    }
    case WDM_DIST_S3: {         // transposed form: x sweep + density + real-to-complex
        if ((rc = dist_copy(d, CP_PSI_X2T_UNPACK, d->recv, d->psiT))) return rc;
        SweepParams<T> p = dist_params<T>(d);
        p.data = (cx<T> *)d->psiT;
        p.tmap = d->tm_psiT;
        if (d->G > 0) {
            DCU(d, d->tab->dist_psi_x_rho(&p, 1, nt, d->stream));
            return dist_poisson_phase<T>(d, 0, xbytes);
        }
        DCU(d, d->tab->dist_psi_y(&p, nt, d->stream));          // G = 0: the x transform alone (middle axis of psi^T)
        return WDM_OK;
    }
    case WDM_DIST_S4: case WDM_DIST_R3:
        return dist_poisson_phase<T>(d, 1, xbytes);
    case WDM_DIST_S5: case WDM_DIST_R4:
        return dist_poisson_phase<T>(d, 2, xbytes);
    case WDM_DIST_KICK:         // closing half kick of a call (elementwise; kicks inside a call are merged into S1)
        if (d->G > 0 && kick_dt != 0.0) {
            k_dist_kick<T><<<148 * 8, 256, 0, d->stream>>>((cx<T> *)d->psiT, (const T *)d->phiT, (T)(kick_dt / d->mu), d->slab);
            DCU(d, cudaGetLastError());
        }
        return WDM_OK;
    case WDM_DIST_G1:           // getter: transposed form -> x-slab
        if (!d->in_T) return WDM_OK;
        if ((rc = dist_copy(d, CP_PSI_T2X_PACK, d->psiT, d->send))) return rc;
        *xbytes = psi_block_bytes(d);
        return WDM_OK;
    case WDM_DIST_G2:
        if (!d->in_T) return WDM_OK;
        return dist_copy(d, CP_PSI_T2X_UNPACK, d->recv, d->psiX);
    }
    return dfail(d, WDM_EINVAL, "unknown phase %d", phase);
}

extern "C" int wdm_dist_phase(wdm_dist *d, int phase, double dt, double kick_dt, size_t *exchange_bytes_per_peer)
{
    if (!d || !exchange_bytes_per_peer) return WDM_EINVAL;
    if (!std::isfinite(dt) || !std::isfinite(kick_dt)) return dfail(d, WDM_EINVAL, "dt must be finite");
    if (!d->send || !d->recv) return dfail(d, WDM_ESTATE, "wdm_dist_set_buffers has not been called");
    return d->dtype == WDM_C64 ? dist_phase_impl<float>(d, phase, dt, kick_dt, exchange_bytes_per_peer)
                               : dist_phase_impl<double>(d, phase, dt, kick_dt, exchange_bytes_per_peer);
}

// sum |psi|^2 over this rank's slab (host value; synchronises).  The caller all-reduces it and hands the global mean
// density to wdm_dist_set_mean before the refresh phases.
extern "C" int wdm_dist_local_sum(wdm_dist *d, double *sum_out)
{
    if (!d || !sum_out) return WDM_EINVAL;
    if (!d->have_psi) return dfail(d, WDM_ESTATE, "wdm_dist_set_psi has not been called");
    const void *psi = d->in_T ? d->psiT : d->psiX;
    const int nb = (int)std::min<size_t>(592, (d->slab + 255) / 256);
    if (d->dtype == WDM_C64) k_dist_sum<float><<<nb, 256, 0, d->stream>>>((const cx<float> *)psi, d->slab, d->partial);
    else k_dist_sum<double><<<nb, 256, 0, d->stream>>>((const cx<double> *)psi, d->slab, d->partial);
    double h[592];
    DCU(d, cudaMemcpyAsync(h, d->partial, nb * sizeof(double), cudaMemcpyDeviceToHost, d->stream));
    DCU(d, cudaStreamSynchronize(d->stream));
    double s = 0;
    for (int i = 0; i < nb; ++i) s += h[i];
    *sum_out = s;
    return WDM_OK;
}

extern "C" int wdm_dist_set_mean(wdm_dist *d, double mean_density)
{
    if (!d) return WDM_EINVAL;
    if (d->dtype == WDM_C64) { float m = (float)mean_density; DCU(d, cudaMemcpyAsync((unsigned char *)d->mean + 16, &m, sizeof m, cudaMemcpyHostToDevice, d->stream)); }
    else { double m = mean_density; DCU(d, cudaMemcpyAsync((unsigned char *)d->mean + 16, &m, sizeof m, cudaMemcpyHostToDevice, d->stream)); }
    DCU(d, cudaStreamSynchronize(d->stream));
    return WDM_OK;
}

// copy out this rank's x-planes of psi (valid after phases G1, exchange, G2) / its Phi^T[y_l][x][z] slab
extern "C" int wdm_dist_get_psi(wdm_dist *d, void *psi_xslab_out_dev)
{
    if (!d || !psi_xslab_out_dev) return WDM_EINVAL;
    if (!d->have_psi) return dfail(d, WDM_ESTATE, "wdm_dist_set_psi has not been called");
    DCU(d, cudaMemcpyAsync(psi_xslab_out_dev, d->psiX, d->slab * dcs(d), cudaMemcpyDeviceToDevice, d->stream));
    return WDM_OK;
}

extern "C" int wdm_dist_get_potential_t(wdm_dist *d, void *phi_t_out_dev)
{
    if (!d || !phi_t_out_dev) return WDM_EINVAL;
    if (!d->phi_valid) return dfail(d, WDM_ESTATE, "the potential is stale: run the refresh phases first");
    DCU(d, cudaMemcpyAsync(phi_t_out_dev, d->phiT, d->slab * drs(d), cudaMemcpyDeviceToDevice, d->stream));
    return WDM_OK;
}
