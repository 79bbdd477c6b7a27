// wdm.cu -- host logic and C ABI of libwdm.so (see include/wdm.h for the contract).
//
// One wdm_step(nsteps, dt) enqueues, per step, on the context's stream:
//   [particles: gather -grad Phi, kick, drift, wrap, deposit]            (wdm_particles.cu)
//   psi sweep z  (kick on load: half kick at the first step, merged full kick afterwards; reading G21)
//   psi sweep y
//   psi sweep x + rho = |psi|^2 + rho_p + real-to-complex x-spectrum -> H
//   H sweep y forward, H sweep z forward . Green . inverse, H sweep y inverse, x complex-to-real -> Phi
// The closing half kick of the call stays pending: the next wdm_step folds it into its opening kick, a read of the
// state applies it (flush_pending).  Nothing synchronises with the host.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "../../include/wdm.h"

#include "wdm_internal.hpp"
#include "wdm_kernels.cuh"
#include "wdm_particles.hpp"

namespace wdm {

#define X(n, ra, rb, rm, w, nt, ng, minb) const SweepTable *sweep_table_0_##n();
WDM_FACT_C64(X)
#undef X
#define X(n, ra, rb, rm, w, nt, ng, minb) const SweepTable *sweep_table_1_##n();
WDM_FACT_C128(X)
#undef X

const SweepTable *sweep_table(int dtype, int N)
{
#define X(n, ra, rb, rm, w, nt, ng, minb) if (dtype == 0 && N == n) return sweep_table_0_##n();
    WDM_FACT_C64(X)
#undef X
#define X(n, ra, rb, rm, w, nt, ng, minb) if (dtype == 1 && N == n) return sweep_table_1_##n();
    WDM_FACT_C128(X)
#undef X
    return nullptr;
}

// ---------------------------------------------------------------- elementwise kernels (not on the per-step path)

template <typename T>
__global__ void k_kick(cx<T> *psi, const T *phi, T coef, size_t n)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        stv(psi + i, rotate_neg(ldv(psi + i), ldg(phi + i) * coef));
}

// general form (extra kick terms, see SweepParams::kick_extra); mask = 3 N axis factors or nullptr
template <typename T>
__global__ void k_kick_general(cx<T> *psi, const T *phi, T coef, T kd, T ka, const T *mask, int N, size_t n)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        T m = (T)1;
        if (mask) {
            const size_t z = i % N, y = (i / N) % N, x = i / ((size_t)N * N);
            m = ldg(mask + x) * ldg(mask + N + y) * ldg(mask + 2 * N + z);
        }
        stv(psi + i, kick_general(ldv(psi + i), ldg(phi + i), m, coef, kd, ka));
    }
}

template <typename T>
__global__ void k_density(const cx<T> *psi, const T *rho_p, T *out, size_t n)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        cx<T> v = ldv(psi + i);
        T r = v.x * v.x + v.y * v.y;
        if (rho_p) r += rho_p[i];
        out[i] = r;
    }
}

// <rho> = (sum |psi|^2)/N^3 + (sum m_p)/L^3 in double, in a FIXED order (per-thread strided sums, warp shuffles, one
// partial per block, then one block over the partials): no atomics, so the mean -- and with it every bit of a pure SPE
// run -- is reproducible from run to run.
constexpr int kSumBlocks = 148 * 4;

__device__ __forceinline__ double block_sum_256(double s)
{
    __shared__ double part[8];
    for (int d = 16; d; d >>= 1) s += __shfl_down_sync(0xffffffffu, s, d);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    double t = 0;
    if (threadIdx.x == 0)
        for (int w = 0; w < 8; ++w) t += part[w];
    __syncthreads();
    return t;          // valid in thread 0
}

template <typename T>
__global__ void __launch_bounds__(256) k_sum_density(const cx<T> *psi, size_t n, double *partial)
{
    double s = 0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        cx<T> v = ldv(psi + i);
        s += (double)v.x * v.x + (double)v.y * v.y;
    }
    s = block_sum_256(s);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

template <typename T>
__global__ void __launch_bounds__(256) k_sum_mass(const T *mass, long long n, double *partial)
{
    double s = 0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) s += mass[i];
    s = block_sum_256(s);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// acc[slot] = sum of partial[0 .. nb) (one block of 256 threads)
__global__ void __launch_bounds__(256) k_sum_partials(const double *partial, int nb, double *acc, int slot)
{
    double s = 0;
    for (int i = threadIdx.x; i < nb; i += 256) s += partial[i];
    s = block_sum_256(s);
    if (threadIdx.x == 0) acc[slot] = s;
}

template <typename T>
__global__ void k_finish_mean(const double *acc, double inv_cells, double extra_mass, double inv_volume, T *mean)
{
    *mean = (T)(acc[0] * inv_cells + (acc[1] + extra_mass) * inv_volume);
}

// Diagnostics of Sect. 3.5-3.6 in one pass over (psi, Phi): per cell rho, rho Phi, the momentum
// density mu Im(psi* grad psi) and grad sqrt(rho) by the central differences of Eq. 21 (periodic).
// acc[0..3] = sum rho, sum rho Phi, sum |rho v|^2 / (2 rho), sum mu^2/2 |grad sqrt rho|^2;  mx[0..1] = bit
// patterns of max rho and max |Phi| as doubles (non-negative doubles order like their bit patterns).
template <typename T>
__global__ void __launch_bounds__(256) k_diag(const cx<T> *__restrict__ psi, const T *__restrict__ phi, int N, double mu, double inv2dx,
                                              double *acc, unsigned long long *mx)
{
    const size_t n = (size_t)N * N * N;
    const int M = N - 1;
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0, m0 = 0, m1 = 0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int z = (int)(i % N), y = (int)((i / N) % N), x = (int)(i / ((size_t)N * N));
        const cx<T> p = ldg(psi + i);
        const double pr = p.x, pi = p.y, rho = pr * pr + pi * pi, f = ldg(phi + i);
        const size_t nb[3][2] = {{((size_t)((x + 1) & M) * N + y) * N + z, ((size_t)((x - 1) & M) * N + y) * N + z},
                                 {((size_t)x * N + ((y + 1) & M)) * N + z, ((size_t)x * N + ((y - 1) & M)) * N + z},
                                 {((size_t)x * N + y) * N + ((z + 1) & M), ((size_t)x * N + y) * N + ((z - 1) & M)}};
        double j2 = 0, g2 = 0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const cx<T> u = ldg(psi + nb[a][0]), d = ldg(psi + nb[a][1]);
            const double gr = ((double)u.x - (double)d.x) * inv2dx, gi = ((double)u.y - (double)d.y) * inv2dx;
            const double j = mu * (pr * gi - pi * gr);                               // Im(conj(p) * grad)
            const double gs = (sqrt((double)u.x * u.x + (double)u.y * u.y) - sqrt((double)d.x * d.x + (double)d.y * d.y)) * inv2dx;
            j2 += j * j;
            g2 += gs * gs;
        }
        s0 += rho;
        s1 += rho * f;
        if (rho > 0) s2 += 0.5 * j2 / rho;
        s3 += 0.5 * mu * mu * g2;
        m0 = fmax(m0, rho);
        m1 = fmax(m1, fabs(f));
    }
    for (int d = 16; d; d >>= 1) {
        s0 += __shfl_down_sync(0xffffffffu, s0, d); s1 += __shfl_down_sync(0xffffffffu, s1, d);
        s2 += __shfl_down_sync(0xffffffffu, s2, d); s3 += __shfl_down_sync(0xffffffffu, s3, d);
        m0 = fmax(m0, __shfl_down_sync(0xffffffffu, m0, d)); m1 = fmax(m1, __shfl_down_sync(0xffffffffu, m1, d));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(acc, s0); atomicAdd(acc + 1, s1); atomicAdd(acc + 2, s2); atomicAdd(acc + 3, s3);
        atomicMax(mx, (unsigned long long)__double_as_longlong(m0));
        atomicMax(mx + 1, (unsigned long long)__double_as_longlong(m1));
    }
}

enum Slot { S_PSI_Z, S_PSI_Y, S_PSI_X_RHO, S_H_Y_FWD, S_H_Z_GREEN, S_H_Y_INV, S_C2R, S_KICK, S_PART_PUSH,
            S_PART_DEPOSIT, S_PART_SORT, S_MISC, S_PART_CLEAR, S_COUNT };
static const char *kSlotNames[S_COUNT] = {"psi_sweep_z_kick", "psi_sweep_y", "psi_sweep_x_rho_r2c", "poisson_y_fwd",
                                          "poisson_z_green", "poisson_y_inv", "poisson_x_c2r", "kick_elementwise",
                                          "particle_gather_kick_drift", "particle_cic_deposit", "particle_cell_sort",
                                          "misc", "particle_mesh_clear"};

}  // namespace wdm

using namespace wdm;

struct wdm_ctx {
    int N = 0, dtype = 0;
    double L = 0, mu = 0, G = 0;
    size_t n = 0, nH = 0;
    const SweepTable *tab = nullptr;
    cudaStream_t stream = nullptr;
    // memory
    bool owns = true;
    unsigned char *ws = nullptr;
    size_t ws_bytes = 0, ws_used = 0;
    std::vector<void *> owned;
    void *psi = nullptr, *phi = nullptr, *H = nullptr;
    void *rho_mean = nullptr;   // [0..1] double accumulators, then the mean as T at byte offset 16
    void *twA = nullptr, *twB = nullptr, *phase = nullptr, *ksq_pos = nullptr, *ksq_nat = nullptr;
    void *x2tab = nullptr;                    // tables of the half-tile x sweeps (tab->x2_w != 0): 2 N complex, the second half follows dt
    double phase_dt = 0;
    bool phase_valid = false, have_psi = false, stale = true;
    // particle variants (wdm_set_particle_mode; reading G29)
    int nsub = 1;
    bool pstatic = false;
    // extra kick terms (wdm_set_kick_terms; readings G26-G28)
    double kappa = 0, alpha = 0;
    int absorb_nb = 50;
    const void *phi_ext = nullptr;            // library-owned copy of the caller's N^3 reals (phi_ext_buf) or nullptr
    void *phi_ext_buf = nullptr;              // cudaMalloc'ed on the first wdm_set_kick_terms with an external potential
    // per-step diagnostics accumulated inside the sweeps (wdm_set_step_diagnostics): three sets of DIAG_COUNT doubles on the
    // device -- two used by alternate steps (a step's z sweep zeroes the other set), one for the on-demand measurement
    bool step_diag = false, step_diag_valid = false;
    double *diag_dev = nullptr;
    int diag_set = 0, diag_last = 0;
    // deterministic deposit (wdm_set_deposit_mode): N^3 64-bit accumulators, cudaMalloc'ed on first use; upper bound of
    // the total particle mass (0 = not measured for the current particle set)
    bool deposit_fixed = false;
    unsigned long long *deposit_acc = nullptr;
    double deposit_mass = 0;
    void *mask = nullptr;                     // 3 N axis factors exp(-alpha b dt) for mask_dt
    double mask_dt = 0;
    bool mask_valid = false;
    // TMA descriptors (see SweepParams): psi along y / x, H along y / x, H single row along x
    CUtensorMap tm_psi_y, tm_psi_x, tm_h_y, tm_h_x, tm_h_x1, tm_psi_x2;
    unsigned int *tickets = nullptr;          // two tile-ticket words used by alternate sweep launches
    int ticket_parity = 0;
    int l2_reverse = 1;                       // see SweepParams::reverse (WDM_L2_REVERSE=0 switches it off for A/B runs)
    // closing half kicks not applied yet (dt of the call that owes them; 0 = none): they merge with the opening
    // half kick of the next wdm_step, or are applied when the state is read or a parameter changes
    double pend_psi = 0, pend_part = 0;
    ParticleState part;
    void *part_pool = nullptr;      // owned contexts: the current particle pool (replaced by a larger one on demand)
    long long max_particles = -1;   // -1: unbounded (cudaMalloc on demand)
    // instrumentation
    long long launches = 0;
    bool profiling = false;
    std::vector<cudaEvent_t> ev;    // pairs
    std::vector<int> ev_slot;
    size_t ev_used = 0;
    double slot_ms[S_COUNT] = {0};
    long long slot_n[S_COUNT] = {0};
    std::string err;
};

static std::string g_create_err = "";

static int fail(wdm_ctx *c, int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (c) c->err = buf;
    else g_create_err = buf;
    return code;
}

#define CU(c, call)                                                                                     \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) return fail(c, WDM_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));     \
    } while (0)

static size_t csize(int dtype) { return dtype == WDM_C64 ? 8 : 16; }
static size_t rsize(int dtype) { return dtype == WDM_C64 ? 4 : 8; }
static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

static size_t grid_bytes(int N, int dtype, long long max_particles)
{
    size_t n = (size_t)N * N * N, nH = (size_t)(N / 2 + 1) * N * N, c = csize(dtype), r = rsize(dtype);
    size_t b = align_up(n * c) + align_up(n * r) + align_up(nH * c);
    b += 3 * align_up((size_t)N * c) + 2 * align_up((size_t)N * r) + align_up((size_t)N * 2) + 256;
    b += align_up((size_t)(2 * N + 2 + 8) * sizeof(unsigned int)) + align_up((size_t)3 * N * r) + align_up(3 * DIAG_COUNT * sizeof(double));
    b += align_up((size_t)2 * N * c);                                  // tables of the half-tile x sweeps (where built)
    if (max_particles > 0) b += align_up(n * r) + particle_bytes(N, dtype, max_particles);
    return b + 4096;
}

static int ctx_alloc(wdm_ctx *c, void **out, size_t bytes)
{
    bytes = align_up(bytes ? bytes : 1);
    if (c->owns) {
        void *p = nullptr;
        cudaError_t e = cudaMalloc(&p, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); return fail(c, WDM_ENOMEM, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e)); }
        c->owned.push_back(p);
        *out = p;
    } else {
        if (c->ws_used + bytes > c->ws_bytes) return fail(c, WDM_ENOMEM, "workspace too small: need %zu more bytes", c->ws_used + bytes - c->ws_bytes);
        *out = c->ws + c->ws_used;
        c->ws_used += bytes;
    }
    return WDM_OK;
}

// ---------------------------------------------------------------- instrumentation

static int prof_flush(wdm_ctx *c)
{
    if (c->ev_used == 0) return WDM_OK;
    CU(c, cudaStreamSynchronize(c->stream));
    for (size_t i = 0; i < c->ev_used; ++i) {
        float ms = 0;
        CU(c, cudaEventElapsedTime(&ms, c->ev[2 * i], c->ev[2 * i + 1]));
        c->slot_ms[c->ev_slot[i]] += ms;
        c->slot_n[c->ev_slot[i]] += 1;
    }
    c->ev_used = 0;
    return WDM_OK;
}

// NVTX range per launch, named like the kernel-statistics slot ("NVTX ranges per sweep"): switched on
// by WDM_NVTX=1 in the environment; the header-only NVTX v3 costs one predictable branch when no tool is attached.
static bool nvtx_on()
{
    static const bool on = [] { const char *e = getenv("WDM_NVTX"); return e && atoi(e) != 0; }();
    return on;
}

// Brackets one launch with events when profiling is on.  A failing event call switches profiling off for the
// context and leaves the text in wdm_last_error (the launch itself is unaffected; its own status is checked by CU).
struct Timed {
    wdm_ctx *c;
    int slot;
    bool on;
    size_t idx = 0;
    static bool ok(wdm_ctx *c, cudaError_t e, const char *what)
    {
        if (e == cudaSuccess) return true;
        fail(c, WDM_ECUDA, "profiling switched off: %s: %s", what, cudaGetErrorString(e));
        c->profiling = false;
        c->ev_used = 0;
        return false;
    }
    Timed(wdm_ctx *c_, int slot_) : c(c_), slot(slot_), on(c_->profiling)
    {
        c->launches++;
        if (nvtx_on()) nvtxRangePushA(kSlotNames[slot]);
        if (!on) return;
        if (c->ev_used * 2 >= c->ev.size()) {
            if (c->ev.size() >= 2 * 8192) {
                if (prof_flush(c) != WDM_OK) { c->profiling = on = false; return; }
            } else {
                cudaEvent_t a = nullptr, b = nullptr;
                if (!ok(c, cudaEventCreate(&a), "cudaEventCreate")) { on = false; return; }
                if (!ok(c, cudaEventCreate(&b), "cudaEventCreate")) { cudaEventDestroy(a); on = false; return; }
                c->ev.push_back(a); c->ev.push_back(b); c->ev_slot.push_back(0);
            }
        }
        idx = c->ev_used++;
        c->ev_slot[idx] = slot;
        if (!ok(c, cudaEventRecord(c->ev[2 * idx], c->stream), "cudaEventRecord")) on = false;
    }
    ~Timed()
    {
        if (on) ok(c, cudaEventRecord(c->ev[2 * idx + 1], c->stream), "cudaEventRecord");
        if (nvtx_on()) nvtxRangePop();
    }
};

// ---------------------------------------------------------------- TMA descriptors

// (the encoder itself is in wdm_internal.hpp: encode_tmap)
static int make_tmap(wdm_ctx *c, CUtensorMap *out, void *base, int nx, int axis, int rows, int W = 0)
{
    const int rc = encode_tmap(c->dtype, c->N, W ? W : c->tab->fact.W, base, c->N, nx, axis, rows, out);
    if (rc == -1) return fail(c, WDM_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
    if (rc != 0) return fail(c, WDM_ECUDA, "cuTensorMapEncodeTiled failed (%d) for N = %d axis %d rows %d", rc, c->N, axis, rows);
    return WDM_OK;
}

static int box_rows(int n) { return n < 256 ? n : 256; }

static int make_tmaps(wdm_ctx *c)
{
    const int N = c->N;
    int rc;
    if ((rc = make_tmap(c, &c->tm_psi_y, c->psi, N, 1, box_rows(N))) || (rc = make_tmap(c, &c->tm_psi_x, c->psi, N, 2, box_rows(N))) ||
        (rc = make_tmap(c, &c->tm_h_y, c->H, N / 2 + 1, 1, box_rows(N))) ||
        (rc = make_tmap(c, &c->tm_h_x, c->H, N / 2 + 1, 2, box_rows(N / 2), c->tab->c2r_w)) ||          // the complex-to-real sweep's tiles
        (rc = make_tmap(c, &c->tm_h_x1, c->H, N / 2 + 1, 2, 1, c->tab->c2r_w)))
        return rc;
    if (c->tab->x2_w && (rc = make_tmap(c, &c->tm_psi_x2, c->psi, N, 2, 256, c->tab->x2_w))) return rc;
    return WDM_OK;
}

// ---------------------------------------------------------------- tables

template <typename T>
static int upload_tables(wdm_ctx *c)
{
    Tables<T> t = build_tables<T>(c->tab->fact, c->L);
    CU(c, cudaMemcpyAsync(c->twA, t.twA.data(), t.twA.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(c->twB, t.twB.data(), t.twB.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, c->stream));
    std::vector<cx<T>> x2;
    if (c->tab->x2_w) {
        Fact half;
        if (!find_fact(c->N / 2, c->dtype, half)) return fail(c, WDM_EUNSUPPORTED, "no factorisation for the half line");
        x2 = build_x2_static<T>(c->N, half);
        CU(c, cudaMemcpyAsync(c->x2tab, x2.data(), x2.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, c->stream));
    }
    CU(c, cudaMemcpyAsync(c->ksq_pos, t.ksq_pos.data(), t.ksq_pos.size() * sizeof(T), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(c->ksq_nat, t.ksq_nat.data(), t.ksq_nat.size() * sizeof(T), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));   // host vectors die here
    return WDM_OK;
}

template <typename T>
static int ensure_phase(wdm_ctx *c, double dt)
{
    if (c->phase_valid && c->phase_dt == dt) return WDM_OK;
    std::vector<cx<T>> ph = build_phase<T>(c->tab->fact, c->L, c->mu, dt);
    CU(c, cudaMemcpyAsync(c->phase, ph.data(), ph.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, c->stream));
    std::vector<cx<T>> x2;
    if (c->tab->x2_w) {
        Fact half;
        if (!find_fact(c->N / 2, c->dtype, half)) return fail(c, WDM_EUNSUPPORTED, "no factorisation for the half line");
        x2 = build_x2_phase<T>(c->N, half, c->L, c->mu, dt);
        CU(c, cudaMemcpyAsync((cx<T> *)c->x2tab + c->N, x2.data(), x2.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, c->stream));
    }
    CU(c, cudaStreamSynchronize(c->stream));
    c->phase_dt = dt;
    c->phase_valid = true;
    return WDM_OK;
}

// axis factors of the absorbing layer, exp(-alpha b(x_i) dt) with b(x) = 2 - tanh((x + L/2)/w) + tanh((x - L/2)/w),
// w = L/nb (Eq. 22): the same table along x, y and z of the cubic box
template <typename T>
static int ensure_mask(wdm_ctx *c, double dt)
{
    if (!(c->alpha > 0) || (c->mask_valid && c->mask_dt == dt)) return WDM_OK;
    const int N = c->N;
    std::vector<T> m(3 * (size_t)N);
    const double w = c->L / (double)c->absorb_nb;
    for (int i = 0; i < N; ++i) {
        const double x = -0.5 * c->L + (c->L / N) * i;
        const double b = 2.0 - std::tanh((x + 0.5 * c->L) / w) + std::tanh((x - 0.5 * c->L) / w);
        m[i] = m[N + i] = m[2 * N + i] = (T)std::exp(-c->alpha * b * dt);
    }
    CU(c, cudaMemcpyAsync(c->mask, m.data(), m.size() * sizeof(T), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    c->mask_dt = dt;
    c->mask_valid = true;
    return WDM_OK;
}

// Tile-ticket counters of the sweeps: two words used by alternate launches (a launch draws from one and zeroes the
// other for its successor on the stream).  Call once per sweep launch, right before it.
template <typename T>
static void take_ticket(wdm_ctx *c, SweepParams<T> &p)
{
    unsigned int *base = c->tickets;
    p.ticket = base + c->ticket_parity;
    p.ticket_next = base + (c->ticket_parity ^ 1);
    c->ticket_parity ^= 1;
}

template <typename T>
static SweepParams<T> base_params(wdm_ctx *c)
{
    SweepParams<T> p{};
    const int N = c->N;
    p.twA = (const cx<T> *)c->twA;
    p.twB = (const cx<T> *)c->twB;
    p.x2tab = (const cx<T> *)c->x2tab;
    p.phase = (const cx<T> *)c->phase;
    p.ksq_pos = (const T *)c->ksq_pos;
    p.ksq_nat = (const T *)c->ksq_nat;
    p.green = (T)(-4.0 * M_PI * c->G / ((double)N * N * N));
    p.H = (cx<T> *)c->H;
    p.phi = (const T *)c->phi;
    p.phi_out = (T *)c->phi;
    p.rho_p = c->part.n > 0 ? (const T *)c->part.rho_p : nullptr;
    p.rho_flag = c->part.flag;
    p.rho_mean = (const T *)((const unsigned char *)c->rho_mean + 16);
    p.phi_ext = (const T *)c->phi_ext;
    p.diag = c->diag_dev + c->diag_set * DIAG_COUNT;
    p.diag_zero = c->diag_dev + (c->diag_set ^ 1) * DIAG_COUNT;
    return p;
}

// ---------------------------------------------------------------- the step

// rho (from the current psi and particle mesh) -> Phi.  drift: also do the x-axis part of Eq. 18(b).
template <typename T>
static int density_poisson(wdm_ctx *c, bool drift, int dg = 0)
{
    const long long N = c->N;
    {
        SweepParams<T> p = base_params<T>(c);
        p.data = (cx<T> *)c->psi;
        p.tmap = c->tm_psi_x;
        p.tmap2 = c->tm_psi_x2;
        take_ticket(c, p);
        Timed t(c, S_PSI_X_RHO);
        CU(c, c->tab->psi_x_rho(&p, drift ? 1 : 0, dg, c->stream));
    }
    SweepParams<T> p = base_params<T>(c);
    p.data = (cx<T> *)c->H;
    p.tmap = c->tm_h_y;
    { take_ticket(c, p); Timed t(c, S_H_Y_FWD); CU(c, c->tab->h_y_fwd(&p, c->stream)); }
    p.reverse = c->l2_reverse;
    { take_ticket(c, p); Timed t(c, S_H_Z_GREEN); CU(c, c->tab->h_z_green(&p, dg, c->stream)); }
    p.reverse = 0;
    { take_ticket(c, p); Timed t(c, S_H_Y_INV); CU(c, c->tab->h_y_inv(&p, c->stream)); }
    p.tmap = c->tm_h_x;
    p.tmap2 = c->tm_h_x1;
    { take_ticket(c, p); Timed t(c, S_C2R); CU(c, c->tab->c2r(&p, dg, c->stream)); }
    return WDM_OK;
}

template <typename T>
static int particles_deposit(wdm_ctx *c)
{
    if (c->part.n == 0) return WDM_OK;
    if (c->deposit_fixed) {
        if (!c->deposit_acc) {
            cudaError_t e = cudaMalloc(&c->deposit_acc, c->n * sizeof(unsigned long long));
            if (e != cudaSuccess) { cudaGetLastError(); c->deposit_acc = nullptr; return fail(c, WDM_ENOMEM, "cudaMalloc of the fixed-point deposit mesh (%zu bytes): %s", c->n * 8, cudaGetErrorString(e)); }
            CU(c, cudaMemsetAsync(c->deposit_acc, 0, c->n * sizeof(unsigned long long), c->stream));
        }
        if (c->deposit_mass == 0) {
            // bound of the total mass, needed once per particle set for the fixed-point scale (host synchronisation)
            if (!c->part.has_mass) c->deposit_mass = fabs(c->part.mass_scalar) * (double)c->part.n;
            else {
                double *acc = (double *)c->rho_mean, h[2];
                const int nb = (int)std::min<long long>(148, (c->part.n + 255) / 256);
                k_sum_mass<T><<<nb, 256, 0, c->stream>>>((const T *)c->part.mass, c->part.n, (double *)c->H);
                k_sum_partials<<<1, 256, 0, c->stream>>>((const double *)c->H, nb, acc, 1);
                CU(c, cudaMemcpyAsync(h, acc, 16, cudaMemcpyDeviceToHost, c->stream));
                CU(c, cudaStreamSynchronize(c->stream));
                c->deposit_mass = fabs(h[1]) * 1.001;          // the scale is a power of two: the last bits of this sum do not matter
            }
            if (!(c->deposit_mass > 0)) c->deposit_mass = 1.0;
        }
        Timed t(c, S_PART_DEPOSIT);
        c->launches += 1;
        CU(c, particle_deposit_fixed(c->part, c->N, c->L, c->dtype, c->deposit_acc, c->deposit_mass, c->stream));
        return WDM_OK;
    }
    if (c->part.mesh_cleared) c->part.mesh_cleared = false;          // the push kernel before this cleared the flagged columns
    else { Timed t(c, S_PART_CLEAR); CU(c, particle_mesh_clear(c->part, c->N, c->dtype, c->stream)); }
    Timed t(c, S_PART_DEPOSIT);
    CU(c, particle_deposit(c->part, c->N, c->L, c->dtype, c->stream));
    return WDM_OK;
}

template <typename T>
static int refresh(wdm_ctx *c)
{
    if (!c->have_psi) return fail(c, WDM_ESTATE, "wdm_set_psi has not been called");
    if (!c->stale) return WDM_OK;
    if (c->G > 0) {
        {   // <rho> of the current state (conserved afterwards): see the density sweep.  Block partials go to the head
            // of H, which is dead until the density sweep writes it
            double *acc = (double *)c->rho_mean, *partial = (double *)c->H;
            Timed t(c, S_MISC);
            CU(c, cudaMemsetAsync(acc, 0, 16, c->stream));
            int nb = (int)std::min<size_t>(kSumBlocks, (c->n + 255) / 256);
            k_sum_density<T><<<nb, 256, 0, c->stream>>>((const cx<T> *)c->psi, c->n, partial);
            k_sum_partials<<<1, 256, 0, c->stream>>>(partial, nb, acc, 0);
            double extra = 0;
            if (c->part.n > 0) {
                if (c->part.has_mass) {
                    nb = (int)std::min<long long>(148, (c->part.n + 255) / 256);
                    k_sum_mass<T><<<nb, 256, 0, c->stream>>>((const T *)c->part.mass, c->part.n, partial);
                    k_sum_partials<<<1, 256, 0, c->stream>>>(partial, nb, acc, 1);
                } else extra = c->part.mass_scalar * (double)c->part.n;
            }
            k_finish_mean<T><<<1, 1, 0, c->stream>>>(acc, 1.0 / (double)c->n, extra, 1.0 / (c->L * c->L * c->L),
                                                      (T *)((unsigned char *)c->rho_mean + 16));
            CU(c, cudaGetLastError());
        }
        int rc = particles_deposit<T>(c);
        if (rc) return rc;
        rc = density_poisson<T>(c, false);
        if (rc) return rc;
    } else {
        Timed t(c, S_MISC);
        if (c->phi_ext) CU(c, cudaMemcpyAsync(c->phi, c->phi_ext, c->n * sizeof(T), cudaMemcpyDeviceToDevice, c->stream));
        else CU(c, cudaMemsetAsync(c->phi, 0, c->n * sizeof(T), c->stream));
    }
    c->stale = false;
    return WDM_OK;
}

// Apply the closing half kick(s) a previous wdm_step left pending (psi: half kick with Phi, then the absorbing layer;
// particles: v += a dt/(2 nsub)).  Phi and the kick parameters must still be the ones of that step.
template <typename T>
static int flush_pending(wdm_ctx *c, bool psi, bool part)
{
    const bool layer = c->alpha > 0;
    if (psi && c->pend_psi != 0.0) {
        const double dt = c->pend_psi;
        int rc = ensure_mask<T>(c, dt);
        if (rc) return rc;
        Timed t(c, S_KICK);
        if (c->kappa != 0.0 || layer)
            k_kick_general<T><<<148 * 8, 256, 0, c->stream>>>((cx<T> *)c->psi, (const T *)c->phi, (T)(0.5 * dt / c->mu),
                                                                (T)(c->kappa * 0.5 * dt / c->mu), (T)0, layer ? (const T *)c->mask : nullptr,
                                                                c->N, c->n);
        else
            k_kick<T><<<148 * 8, 256, 0, c->stream>>>((cx<T> *)c->psi, (const T *)c->phi, (T)(0.5 * dt / c->mu), c->n);
        CU(c, cudaGetLastError());
        c->pend_psi = 0.0;
    }
    if (part && c->pend_part != 0.0) {
        Timed t(c, S_PART_PUSH);
        CU(c, particle_push(c->part, c->N, c->L, c->dtype, c->phi, 0.5 * c->pend_part / c->nsub, 0.0, 1, false, c->stream));
        c->pend_part = 0.0;
    }
    return WDM_OK;
}

template <typename T>
static int step_impl(wdm_ctx *c, int nsteps, double dt)
{
    int rc = refresh<T>(c);
    if (rc || nsteps == 0) return rc;
    // a pending closing kick merges with this call's opening kick only if both use the same dt (one table of
    // absorbing-layer factors, one sub-step size)
    if ((c->pend_psi != 0.0 && c->pend_psi != dt) || (c->pend_part != 0.0 && c->pend_part != dt))
        if ((rc = flush_pending<T>(c, true, true))) return rc;
    rc = ensure_phase<T>(c, dt);
    if (rc) return rc;
    rc = ensure_mask<T>(c, dt);
    if (rc) return rc;
    const long long N = c->N;
    const bool grav = c->G > 0;
    const bool have_phi = grav || c->phi_ext != nullptr;                 // particles and psi feel a potential
    const bool layer = c->alpha > 0;
    const bool kicks = have_phi || c->kappa != 0.0 || layer;
    const int dg = c->step_diag ? 1 : 0;                  // the accumulating instantiations
    if (dg) CU(c, cudaMemsetAsync(c->diag_dev + c->diag_set * DIAG_COUNT, 0, DIAG_COUNT * sizeof(double), c->stream));
    for (int s = 0; s < nsteps; ++s) {
        // merged closing (h_d, of the previous step -- possibly of the previous call) + opening (h_a) half kicks
        // (G21); the absorbing layer sits between them
        const double hd = s == 0 ? 0.5 * c->pend_psi : 0.5 * dt, ha = 0.5 * dt, kdt = hd + ha;
        const double hd_p = s == 0 ? 0.5 * c->pend_part : 0.5 * dt;
        if (c->part.n > 0 && !c->pstatic) {
            // v += a(Phi^n, x^n) kdt/nsub ; nsub x { x += v dt/nsub ; wrap ; [kick] } ; then deposit x^{n+1}  (G14-G16, G29)
            { Timed t(c, S_PART_PUSH); CU(c, particle_push(c->part, c->N, c->L, c->dtype, c->phi, have_phi ? (hd_p + ha) / c->nsub : 0.0, dt, c->nsub, grav && !c->deposit_fixed, c->stream)); }
            if (particle_sort_due(c->part)) { Timed t(c, S_PART_SORT); c->launches += 2; CU(c, particle_resort(c->part, c->N, c->L, c->dtype, c->stream)); }
            if (grav) { rc = particles_deposit<T>(c); if (rc) return rc; }
        }
        {
            SweepParams<T> pz = base_params<T>(c), py = base_params<T>(c);
            pz.data = (cx<T> *)c->psi;
            pz.kick = (T)(kdt / c->mu);
            pz.kself_d = (T)(c->kappa * hd / c->mu);
            pz.kself_a = (T)(c->kappa * ha / c->mu);
            pz.mask = layer && hd != 0.0 ? (const T *)c->mask : nullptr;
            pz.kick_extra = (c->kappa != 0.0 || pz.mask != nullptr) ? 1 : 0;
            py.data = (cx<T> *)c->psi;
            py.tmap = c->tm_psi_y;
            py.reverse = c->l2_reverse;
            { take_ticket(c, pz); Timed t(c, S_PSI_Z); CU(c, c->tab->psi_z(&pz, kicks ? (pz.kick_extra ? 2 : 1) : 0, dg, c->stream)); }
            { take_ticket(c, py); Timed t(c, S_PSI_Y); CU(c, c->tab->psi_strided(&py, 0, dg, c->stream)); }
        }
        c->pend_psi = 0.0;
        c->pend_part = 0.0;
        if (grav) {
            rc = density_poisson<T>(c, true, dg);
            if (rc) return rc;
        } else {
            SweepParams<T> p = base_params<T>(c);
            p.data = (cx<T> *)c->psi;
            p.tmap = c->tm_psi_x;
            p.tmap2 = c->tm_psi_x2;
            take_ticket(c, p);
            Timed t(c, S_PSI_Y);
            CU(c, c->tab->psi_strided(&p, 1, dg, c->stream));
        }
        if (dg) { c->diag_last = c->diag_set; c->diag_set ^= 1; c->step_diag_valid = true; }
    }
    // the closing half kicks (and the last absorbing layer) stay pending: the next wdm_step merges them into its
    // opening kick; a read of the state or a change of parameters applies them first (flush_pending)
    c->pend_psi = kicks ? dt : 0.0;
    c->pend_part = (have_phi && c->part.n > 0 && !c->pstatic) ? dt : 0.0;
    return WDM_OK;
}

static int do_flush(wdm_ctx *c, bool psi, bool part)
{
    return c->dtype == WDM_C64 ? flush_pending<float>(c, psi, part) : flush_pending<double>(c, psi, part);
}

// ---------------------------------------------------------------- C ABI

static int check_args(int N, double L, double mu, double G, int dtype)
{
    if (!(L > 0) || !(mu > 0) || !(G >= 0)) return fail(nullptr, WDM_EINVAL, "need L > 0, hbar_over_m > 0, G >= 0");
    if (dtype != WDM_C64 && dtype != WDM_C128) return fail(nullptr, WDM_EINVAL, "dtype must be WDM_C64 or WDM_C128");
    if (N < 8 || N > 1024 || (N & (N - 1))) return fail(nullptr, WDM_EUNSUPPORTED, "N must be a power of two in [8, 1024], got %d", N);
    return WDM_OK;
}

extern "C" int wdm_workspace_bytes(int N, int dtype, long long max_particles, size_t *bytes_out)
{
    if (!bytes_out || max_particles < 0) return fail(nullptr, WDM_EINVAL, "null output or negative max_particles");
    int rc = check_args(N, 1.0, 1.0, 0.0, dtype);
    if (rc) return rc;
    *bytes_out = grid_bytes(N, dtype, max_particles);
    return WDM_OK;
}

static int create_common(wdm_ctx **out, int N, double L, double mu, double G, int dtype, long long max_particles,
                         void *ws, size_t ws_bytes, bool owns)
{
    if (!out) return fail(nullptr, WDM_EINVAL, "null output pointer");
    *out = nullptr;
    int rc = check_args(N, L, mu, G, dtype);
    if (rc) return rc;
    wdm_ctx *c = new wdm_ctx();
    c->N = N; c->dtype = dtype; c->L = L; c->mu = mu; c->G = G;
    c->n = (size_t)N * N * N; c->nH = (size_t)(N / 2 + 1) * N * N;
    c->owns = owns; c->ws = (unsigned char *)ws; c->ws_bytes = ws_bytes;
    c->max_particles = owns ? -1 : max_particles;
    c->tab = sweep_table(dtype, N);
    auto bail = [&](int code) {
        g_create_err = c->err;
        for (void *p : c->owned) cudaFree(p);
        delete c;
        return code;
    };
    if (!c->tab) return bail(fail(c, WDM_EUNSUPPORTED, "no kernels built for N = %d", N));
    if (!owns) {
        size_t mis = (size_t)((uintptr_t)ws & 255);
        if (!ws) return bail(fail(c, WDM_EINVAL, "null workspace"));
        if (mis) { c->ws += 256 - mis; c->ws_bytes -= (256 - mis) < ws_bytes ? (256 - mis) : ws_bytes; }
        if (ws_bytes < grid_bytes(N, dtype, max_particles)) return bail(fail(c, WDM_ENOMEM, "workspace of %zu bytes < required %zu", ws_bytes, grid_bytes(N, dtype, max_particles)));
    }
    cudaError_t e = c->tab->init();
    if (e != cudaSuccess) return bail(fail(c, WDM_ECUDA, "kernel attribute setup: %s", cudaGetErrorString(e)));
    size_t cs = csize(dtype), rs = rsize(dtype);
    if ((rc = ctx_alloc(c, &c->psi, c->n * cs)) || (rc = ctx_alloc(c, &c->phi, c->n * rs)) ||
        (rc = ctx_alloc(c, &c->H, c->nH * cs)) || (rc = ctx_alloc(c, &c->twA, N * cs)) ||
        (rc = ctx_alloc(c, &c->twB, N * cs)) || (rc = ctx_alloc(c, &c->phase, N * cs)) ||
        (rc = ctx_alloc(c, &c->ksq_pos, N * rs)) || (rc = ctx_alloc(c, &c->ksq_nat, N * rs)) ||
        (rc = ctx_alloc(c, &c->rho_mean, 64)) ||
        (rc = ctx_alloc(c, (void **)&c->tickets, 8 * sizeof(unsigned int))) ||
        (rc = ctx_alloc(c, &c->mask, (size_t)3 * N * rs)) || (c->tab->x2_w && (rc = ctx_alloc(c, &c->x2tab, (size_t)2 * N * cs))) || (rc = ctx_alloc(c, (void **)&c->diag_dev, 3 * DIAG_COUNT * sizeof(double))))
        return bail(rc);
    if (cudaMemset(c->tickets, 0, 8 * sizeof(unsigned int)) != cudaSuccess)
        return bail(fail(c, WDM_ECUDA, "cudaMemset of the ticket words failed"));
    if (const char *env = getenv("WDM_L2_REVERSE")) c->l2_reverse = atoi(env) != 0;
    rc = dtype == WDM_C64 ? upload_tables<float>(c) : upload_tables<double>(c);
    if (rc) return bail(rc);
    if ((rc = make_tmaps(c))) return bail(rc);
    if (!owns && max_particles > 0) {
        void *rho_p = nullptr, *pm = nullptr;
        if ((rc = ctx_alloc(c, &rho_p, c->n * rs)) || (rc = ctx_alloc(c, &pm, particle_bytes(N, dtype, max_particles)))) return bail(rc);
        particle_bind(c->part, N, dtype, max_particles, rho_p, pm);
    }
    *out = c;
    return WDM_OK;
}

extern "C" int wdm_create(wdm_ctx **out, int N, double L, double hbar_over_m, double G, int dtype)
{
    return create_common(out, N, L, hbar_over_m, G, dtype, 0, nullptr, 0, true);
}

extern "C" int wdm_create_ws(wdm_ctx **out, int N, double L, double hbar_over_m, double G, int dtype,
                             long long max_particles, void *workspace_dev, size_t workspace_bytes)
{
    if (max_particles < 0) return fail(nullptr, WDM_EINVAL, "negative max_particles");
    return create_common(out, N, L, hbar_over_m, G, dtype, max_particles, workspace_dev, workspace_bytes, false);
}

extern "C" int wdm_destroy(wdm_ctx *c)
{
    if (!c) return WDM_OK;
    cudaStreamSynchronize(c->stream);
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    for (void *p : c->owned) cudaFree(p);
    if (c->phi_ext_buf) cudaFree(c->phi_ext_buf);
    if (c->deposit_acc) cudaFree(c->deposit_acc);
    delete c;
    return WDM_OK;
}

extern "C" int wdm_set_stream(wdm_ctx *c, void *s)
{
    if (!c) return WDM_EINVAL;
    int rc = prof_flush(c);
    if (rc) return rc;
    if ((cudaStream_t)s != c->stream) {
        // work already enqueued on the old stream (wdm_step is asynchronous) must precede anything on the new one
        cudaEvent_t e;
        CU(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        cudaError_t e1 = cudaEventRecord(e, c->stream), e2 = e1 == cudaSuccess ? cudaStreamWaitEvent((cudaStream_t)s, e, 0) : e1;
        cudaEventDestroy(e);
        if (e2 != cudaSuccess) return fail(c, WDM_ECUDA, "ordering the new stream after the old one: %s", cudaGetErrorString(e2));
    }
    c->stream = (cudaStream_t)s;
    return WDM_OK;
}

static int set_psi(wdm_ctx *c, const void *psi, cudaMemcpyKind kind)
{
    if (!c) return WDM_EINVAL;
    if (!psi) return fail(c, WDM_EINVAL, "null psi");
    // the particles still owe the closing half kick of the last step (with the old Phi); psi's is moot
    int rcf = do_flush(c, false, true);
    if (rcf) return rcf;
    c->pend_psi = 0.0;
    CU(c, cudaMemcpyAsync(c->psi, psi, c->n * csize(c->dtype), kind, c->stream));
    c->have_psi = true;
    c->stale = true;
    return WDM_OK;
}
extern "C" int wdm_set_psi(wdm_ctx *c, const void *p) { return set_psi(c, p, cudaMemcpyDeviceToDevice); }
extern "C" int wdm_set_psi_host(wdm_ctx *c, const void *p) { return set_psi(c, p, cudaMemcpyHostToDevice); }

static int set_particles(wdm_ctx *c, long long n, const void *pos, const void *vel, const void *mass, double ms,
                         cudaMemcpyKind kind)
{
    if (!c) return WDM_EINVAL;
    if (n < 0 || (n > 0 && (!pos || !vel))) return fail(c, WDM_EINVAL, "bad particle arguments");
    if (c->max_particles >= 0 && n > c->max_particles) return fail(c, WDM_ENOMEM, "%lld particles > max_particles %lld of the workspace", n, c->max_particles);
    {   // psi still owes the closing half kick of the last step (with the old Phi); the old particles' is moot
        int rcf = do_flush(c, true, false);
        if (rcf) return rcf;
        c->pend_part = 0.0;
    }
    if (c->owns && n > c->part.capacity) {
        size_t rs = rsize(c->dtype);
        void *rho_p = c->part.rho_p, *pm = nullptr;
        int rc;
        if (!rho_p && (rc = ctx_alloc(c, &rho_p, c->n * rs))) return rc;
        if ((rc = ctx_alloc(c, &pm, particle_bytes(c->N, c->dtype, n)))) return rc;
        particle_bind(c->part, c->N, c->dtype, n, rho_p, pm);
        if (c->part_pool) {
            // the smaller pool is not needed any more: release it once the stream has passed everything that used it
            CU(c, cudaStreamSynchronize(c->stream));
            for (size_t i = 0; i < c->owned.size(); ++i)
                if (c->owned[i] == c->part_pool) { c->owned.erase(c->owned.begin() + i); break; }
            cudaFree(c->part_pool);
        }
        c->part_pool = pm;
    }
    c->launches += 3;
    c->deposit_mass = 0;
    cudaError_t e = particle_set(c->part, c->N, c->L, c->dtype, n, pos, vel, mass, ms, kind == cudaMemcpyHostToDevice, c->stream);
    if (e != cudaSuccess) return fail(c, WDM_ECUDA, "particle_set: %s", cudaGetErrorString(e));
    c->stale = true;
    return WDM_OK;
}
extern "C" int wdm_set_particles(wdm_ctx *c, long long n, const void *pos, const void *vel, const void *mass, double ms)
{
    return set_particles(c, n, pos, vel, mass, ms, cudaMemcpyDeviceToDevice);
}
extern "C" int wdm_set_particles_host(wdm_ctx *c, long long n, const void *pos, const void *vel, const void *mass, double ms)
{
    return set_particles(c, n, pos, vel, mass, ms, cudaMemcpyHostToDevice);
}

extern "C" int wdm_step(wdm_ctx *c, int nsteps, double dt)
{
    if (!c) return WDM_EINVAL;
    if (nsteps < 0 || !std::isfinite(dt)) return fail(c, WDM_EINVAL, "nsteps must be >= 0 and dt finite");
    return c->dtype == WDM_C64 ? step_impl<float>(c, nsteps, dt) : step_impl<double>(c, nsteps, dt);
}

static int do_refresh(wdm_ctx *c) { return c->dtype == WDM_C64 ? refresh<float>(c) : refresh<double>(c); }

static int get_grid(wdm_ctx *c, void *out, int what, cudaMemcpyKind kind)
{
    if (!c) return WDM_EINVAL;
    if (!out) return fail(c, WDM_EINVAL, "null output");
    if (!c->have_psi) return fail(c, WDM_ESTATE, "wdm_set_psi has not been called");
    if (what != 1) {                 // psi, or the density (the absorbing layer of a pending kick changes |psi|)
        int rcf = do_flush(c, true, false);
        if (rcf) return rcf;
    }
    if (what == 0) {
        CU(c, cudaMemcpyAsync(out, c->psi, c->n * csize(c->dtype), kind, c->stream));
    } else {
        int rc = do_refresh(c);
        if (rc) return rc;
        if (what == 1) {
            CU(c, cudaMemcpyAsync(out, c->phi, c->n * rsize(c->dtype), kind, c->stream));
        } else {
            // density is not kept (its spectrum is overwritten by the Poisson solve): recompute, via H as scratch
            void *dst = kind == cudaMemcpyDeviceToDevice ? out : c->H;
            const void *rp = c->part.n > 0 && c->G > 0 ? c->part.rho_p : nullptr;
            if (rp == nullptr && c->part.n > 0) {   // G = 0 never deposits: do it now
                int r2 = c->dtype == WDM_C64 ? particles_deposit<float>(c) : particles_deposit<double>(c);
                if (r2) return r2;
                rp = c->part.rho_p;
            }
            {
                Timed t(c, S_MISC);
                if (c->dtype == WDM_C64) k_density<float><<<148 * 8, 256, 0, c->stream>>>((const cx<float> *)c->psi, (const float *)rp, (float *)dst, c->n);
                else k_density<double><<<148 * 8, 256, 0, c->stream>>>((const cx<double> *)c->psi, (const double *)rp, (double *)dst, c->n);
                CU(c, cudaGetLastError());
            }
            if (dst != out) CU(c, cudaMemcpyAsync(out, dst, c->n * rsize(c->dtype), kind, c->stream));
        }
    }
    if (kind == cudaMemcpyDeviceToHost) CU(c, cudaStreamSynchronize(c->stream));
    return WDM_OK;
}
extern "C" int wdm_get_psi(wdm_ctx *c, void *o) { return get_grid(c, o, 0, cudaMemcpyDeviceToDevice); }
extern "C" int wdm_get_potential(wdm_ctx *c, void *o) { return get_grid(c, o, 1, cudaMemcpyDeviceToDevice); }
extern "C" int wdm_get_density(wdm_ctx *c, void *o) { return get_grid(c, o, 2, cudaMemcpyDeviceToDevice); }
extern "C" int wdm_get_psi_host(wdm_ctx *c, void *o) { return get_grid(c, o, 0, cudaMemcpyDeviceToHost); }
extern "C" int wdm_get_potential_host(wdm_ctx *c, void *o) { return get_grid(c, o, 1, cudaMemcpyDeviceToHost); }
extern "C" int wdm_get_density_host(wdm_ctx *c, void *o) { return get_grid(c, o, 2, cudaMemcpyDeviceToHost); }

static int get_particles(wdm_ctx *c, void *pos, void *vel, bool host)
{
    if (!c) return WDM_EINVAL;
    {
        int rcf = do_flush(c, false, true);
        if (rcf) return rcf;
    }
    if (c->part.n > 0) {
        c->launches += 1;
        cudaError_t e = particle_get(c->part, c->dtype, pos, vel, host, c->stream);
        if (e != cudaSuccess) return fail(c, WDM_ECUDA, "particle_get: %s", cudaGetErrorString(e));
    }
    if (host) CU(c, cudaStreamSynchronize(c->stream));
    return WDM_OK;
}
extern "C" int wdm_get_particles(wdm_ctx *c, void *pos, void *vel) { return get_particles(c, pos, vel, false); }
extern "C" int wdm_get_particles_host(wdm_ctx *c, void *pos, void *vel) { return get_particles(c, pos, vel, true); }

extern "C" int wdm_run_host(wdm_ctx *c, const void *psi_in, int nsteps, double dt, void *psi_out)
{
    int rc = wdm_set_psi_host(c, psi_in);
    if (rc) return rc;
    if ((rc = wdm_step(c, nsteps, dt))) return rc;
    return wdm_get_psi_host(c, psi_out);
}

extern "C" int wdm_launch_count(wdm_ctx *c, long long *out)
{
    if (!c || !out) return WDM_EINVAL;
    *out = c->launches;
    return WDM_OK;
}

extern "C" int wdm_set_particle_mode(wdm_ctx *c, int substeps, int is_static)
{
    if (!c) return WDM_EINVAL;
    if (substeps < 1) return fail(c, WDM_EINVAL, "substeps must be >= 1");
    int rcf = do_flush(c, true, true);
    if (rcf) return rcf;
    c->nsub = substeps;
    c->pstatic = is_static != 0;
    return WDM_OK;
}

extern "C" int wdm_set_assignment(wdm_ctx *c, int order)
{
    if (!c) return WDM_EINVAL;
    if (order != 2 && order != 3) return fail(c, WDM_EINVAL, "assignment order must be 2 (cloud-in-cell) or 3 (triangular-shaped cloud)");
    int rcf = do_flush(c, true, true);       // a pending closing half kick belongs to the scheme it was computed with
    if (rcf) return rcf;
    if (c->part.order != order) {
        c->part.order = order;
        c->stale = true;                     // the particles' share of the Poisson source changes
    }
    return WDM_OK;
}

extern "C" int wdm_set_deposit_mode(wdm_ctx *c, int deterministic)
{
    if (!c) return WDM_EINVAL;
    if (deterministic != 0 && deterministic != 1) return fail(c, WDM_EINVAL, "deterministic must be 0 or 1");
    int rcf = do_flush(c, true, true);
    if (rcf) return rcf;
    if (c->deposit_fixed != (deterministic != 0)) {
        c->deposit_fixed = deterministic != 0;
        c->stale = true;                     // the mesh is re-deposited with the other arithmetic
    }
    return WDM_OK;
}

extern "C" int wdm_get_assignment(wdm_ctx *c, int *order)
{
    if (!c || !order) return WDM_EINVAL;
    *order = c->part.order;
    return WDM_OK;
}

// sum k_a^2 |F_a psi|^2 of the current psi for a = z, y, x into acc[0..2] (forward-only sweeps, psi untouched)
template <typename T>
static int measure_kinetic(wdm_ctx *c, double *acc)
{
    for (int a = 0; a < 3; ++a) {
        SweepParams<T> p = base_params<T>(c);
        p.data = (cx<T> *)c->psi;
        p.diag = acc;
        p.diag_zero = nullptr;
        p.tmap = a == 1 ? c->tm_psi_y : c->tm_psi_x;
        take_ticket(c, p);
        Timed t(c, S_MISC);
        CU(c, a == 0 ? c->tab->psi_z(&p, 0, 2, c->stream) : c->tab->psi_strided(&p, a == 2 ? 1 : 0, 2, c->stream));
    }
    return WDM_OK;
}

extern "C" int wdm_get_diagnostics(wdm_ctx *c, double *out_host)
{
    if (!c) return WDM_EINVAL;
    if (!out_host) return fail(c, WDM_EINVAL, "null output");
    int rc = do_refresh(c);
    if (rc) return rc;
    if ((rc = do_flush(c, true, false))) return rc;
    // scratch: the 64-byte block of the <rho> accumulators is free between refreshes except for the mean at byte 16;
    // use the first 48 bytes of the head of H instead (H is dead outside a Poisson solve)
    double *acc = (double *)c->H;
    unsigned long long *mx = (unsigned long long *)(acc + 4);
    {
        Timed t(c, S_MISC);
        CU(c, cudaMemsetAsync(acc, 0, 6 * sizeof(double), c->stream));
        const double inv2dx = 0.5 * c->N / c->L;
        if (c->dtype == WDM_C64) k_diag<float><<<148 * 8, 256, 0, c->stream>>>((const cx<float> *)c->psi, (const float *)c->phi, c->N, c->mu, inv2dx, acc, mx);
        else k_diag<double><<<148 * 8, 256, 0, c->stream>>>((const cx<double> *)c->psi, (const double *)c->phi, c->N, c->mu, inv2dx, acc, mx);
        CU(c, cudaGetLastError());
    }
    double h[6];
    CU(c, cudaMemcpyAsync(h, acc, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    const double dx = c->L / c->N, dV = dx * dx * dx;
    double maxrho, maxphi;
    memcpy(&maxrho, &h[4], 8);
    memcpy(&maxphi, &h[5], 8);
    out_host[0] = h[0] * dV; out_host[1] = maxrho; out_host[2] = maxphi;
    out_host[3] = h[1] * dV; out_host[4] = h[2] * dV; out_host[5] = h[3] * dV;
    double dtm = 4.0 / (3.0 * M_PI) * dx * dx / c->mu;                                       // Eq. 26
    if (maxphi > 0 && 2.0 * M_PI * c->mu / maxphi < dtm) dtm = 2.0 * M_PI * c->mu / maxphi;
    if (c->kappa != 0 && maxrho > 0 && 2.0 * M_PI * c->mu / (fabs(c->kappa) * maxrho) < dtm) dtm = 2.0 * M_PI * c->mu / (fabs(c->kappa) * maxrho);
    out_host[6] = 0.5 * dtm;
    // spectral kinetic energy of the current psi: three forward-only sweeps (one per axis) that write nothing
    {
        double *m = c->diag_dev + 2 * DIAG_COUNT;
        CU(c, cudaMemsetAsync(m, 0, DIAG_COUNT * sizeof(double), c->stream));
        rc = c->dtype == WDM_C64 ? measure_kinetic<float>(c, m) : measure_kinetic<double>(c, m);
        if (rc) return rc;
        double t[3];
        CU(c, cudaMemcpyAsync(t, m, sizeof t, cudaMemcpyDeviceToHost, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
        const double f = 0.5 * c->mu * c->mu * dV / c->N;
        out_host[7] = f * (t[0] + t[1] + t[2]);
    }
    out_host[8] = 0.5 * out_host[3];
    out_host[9] = out_host[7] + out_host[8];
    out_host[10] = out_host[11] = 0;
    return WDM_OK;
}

extern "C" int wdm_set_step_diagnostics(wdm_ctx *c, int on)
{
    if (!c) return WDM_EINVAL;
    c->step_diag = on != 0;
    c->step_diag_valid = false;
    return WDM_OK;
}

extern "C" int wdm_get_step_diagnostics(wdm_ctx *c, double *out_host)
{
    if (!c) return WDM_EINVAL;
    if (!out_host) return fail(c, WDM_EINVAL, "null output");
    if (!c->step_diag_valid) return fail(c, WDM_ESTATE, "no step has run since wdm_set_step_diagnostics(ctx, 1)");
    double d[DIAG_COUNT];
    CU(c, cudaMemcpyAsync(d, c->diag_dev + c->diag_last * DIAG_COUNT, sizeof d, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    const double dx = c->L / c->N, dV = dx * dx * dx, f = 0.5 * c->mu * c->mu * dV / c->N;
    out_host[0] = d[3] * dV;
    out_host[1] = d[4];                      // maxima travel as bit patterns of non-negative doubles
    out_host[2] = d[6];
    out_host[5] = f * d[2]; out_host[6] = f * d[1]; out_host[7] = f * d[0];
    out_host[3] = out_host[5] + out_host[6] + out_host[7];
    out_host[4] = 0.5 * dV * d[5];
    return WDM_OK;
}

extern "C" int wdm_set_kick_terms(wdm_ctx *c, double kappa, const void *phi_ext_dev, double absorb_alpha, int absorb_nb)
{
    if (!c) return WDM_EINVAL;
    if (!std::isfinite(kappa) || !std::isfinite(absorb_alpha) || !(absorb_alpha >= 0) || (absorb_alpha > 0 && absorb_nb < 1))
        return fail(c, WDM_EINVAL, "need a finite kappa, absorb_alpha >= 0 and absorb_nb >= 1");
    int rcf = do_flush(c, true, true);           // pending closing kicks belong to the old terms
    if (rcf) return rcf;
    if (phi_ext_dev) {
        // copied: the caller's buffer may be freed or changed after this call returns (stream-ordered copy)
        if (!c->phi_ext_buf) {
            cudaError_t e = cudaMalloc(&c->phi_ext_buf, c->n * rsize(c->dtype));
            if (e != cudaSuccess) { cudaGetLastError(); c->phi_ext_buf = nullptr; return fail(c, WDM_ENOMEM, "cudaMalloc of the external potential copy (%zu bytes): %s", c->n * rsize(c->dtype), cudaGetErrorString(e)); }
        }
        CU(c, cudaMemcpyAsync(c->phi_ext_buf, phi_ext_dev, c->n * rsize(c->dtype), cudaMemcpyDeviceToDevice, c->stream));
    }
    c->kappa = kappa;
    c->phi_ext = phi_ext_dev ? c->phi_ext_buf : nullptr;
    c->alpha = absorb_alpha;
    c->absorb_nb = absorb_nb;
    c->mask_valid = false;
    c->stale = true;                 // Phi_total changes with the external term
    return WDM_OK;
}

extern "C" int wdm_set_profiling(wdm_ctx *c, int on)
{
    if (!c) return WDM_EINVAL;
    int rc = prof_flush(c);
    c->profiling = on != 0;
    return rc;
}

extern "C" int wdm_kernel_stats(wdm_ctx *c, int *n_inout, const char **names, long long *launches, double *ms)
{
    if (!c || !n_inout) return WDM_EINVAL;
    int rc = prof_flush(c);
    if (rc) return rc;
    int cap = *n_inout;
    *n_inout = S_COUNT;
    for (int i = 0; i < S_COUNT && i < cap; ++i) {
        if (names) names[i] = kSlotNames[i];
        if (launches) launches[i] = c->slot_n[i];
        if (ms) ms[i] = c->slot_ms[i];
    }
    for (int i = 0; i < S_COUNT; ++i) { c->slot_n[i] = 0; c->slot_ms[i] = 0; }
    return WDM_OK;
}

extern "C" const char *wdm_last_error(const wdm_ctx *c) { return c ? c->err.c_str() : g_create_err.c_str(); }
