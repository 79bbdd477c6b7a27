// wdm_particles.cu -- particle kernels (see wdm_particles.hpp).
//
// Particles are kept sorted by mesh tile (TS^3 cells, tile-major) with a counting sort, redone every
// kResortInterval pushes: a disc particle moves 1e-3..1e-2 cells per step, so the order stays useful for
// hundreds of steps.  Correctness never depends on the order: the deposit falls back to global atomics
// for any node outside the CTA's shared-memory box.
#include <cstdint>

#include "wdm_particles.hpp"

namespace wdm {
namespace {

constexpr int TS = 8;                 // tile edge in cells
constexpr int BOX = 2 * TS + 1;       // shared accumulator box edge in nodes
constexpr int CHUNK = 1024;           // sorted particles per deposit CTA
constexpr int kResortInterval = 64;

__host__ __device__ inline int ntiles1(int N) { return N >= TS ? N / TS : 1; }

template <typename T>
struct Cic {
    int i0[3];
    T f[3];
};

// u = (x + L/2)/dx, i0 = floor(u) (wrapped), f = u - floor(u)   (reading G12)
template <typename T>
__device__ __forceinline__ Cic<T> cic_of(const T *x, T half_L, T inv_dx, int N)
{
    Cic<T> c;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        T u = (x[a] + half_L) * inv_dx;
        T fl = floor(u);
        int i = (int)fl;
        c.f[a] = u - fl;
        i %= N;
        if (i < 0) i += N;
        c.i0[a] = i;
    }
    return c;
}

// Assignment stencil of one particle: ORDER nodes per axis starting at `base` (wrapped), weights w[axis][0..ORDER).
//   ORDER 2, cloud-in-cell (G12):        base = floor(u),           w = (1 - f, f),  f = u - floor(u)
//   ORDER 3, triangular-shaped cloud (G30): base = floor(u + 1/2) - 1,  w = ((1/2 - d)^2 / 2, 3/4 - d^2, (1/2 + d)^2 / 2),
//            d = u - floor(u + 1/2) in [-1/2, 1/2)
template <typename T, int ORDER>
struct Asg {
    int base[3];
    T w[3][ORDER];
};

template <typename T, int ORDER>
__device__ __forceinline__ Asg<T, ORDER> asg_of(const T *x, T half_L, T inv_dx, int N)
{
    static_assert(ORDER == 2 || ORDER == 3, "cloud-in-cell or triangular-shaped cloud");
    Asg<T, ORDER> s;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        T u = (x[a] + half_L) * inv_dx;
        int i;
        if constexpr (ORDER == 2) {
            T fl = floor(u);
            T f = u - fl;
            i = (int)fl;
            s.w[a][0] = (T)1 - f;
            s.w[a][1] = f;
        } else {
            T fl = floor(u + (T)0.5);
            T d = u - fl;
            i = (int)fl - 1;
            s.w[a][0] = (T)0.5 * ((T)0.5 - d) * ((T)0.5 - d);
            s.w[a][1] = (T)0.75 - d * d;
            s.w[a][2] = (T)0.5 * ((T)0.5 + d) * ((T)0.5 + d);
        }
        i %= N;
        if (i < 0) i += N;
        s.base[a] = i;
    }
    return s;
}

__device__ __forceinline__ int tile_key(const int *i0, int N)
{
    int nt = ntiles1(N);
    int tx = i0[0] / TS, ty = i0[1] / TS, tz = i0[2] / TS;
    if (N < TS) return 0;
    return (tx * nt + ty) * nt + tz;
}

template <typename T>
__device__ __forceinline__ T wrap_pos(T x, T L)
{
    T half = (T)0.5 * L;
    T y = x - L * floor((x + half) / L);
    if (y >= half) y -= L;
    if (y < -half) y += L;
    return y;
}

template <typename T>
__global__ void k_ingest(const T *pos_in, const T *vel_in, T *pos, T *vel, int *orig, long long n, T L)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        pos[3 * i + a] = wrap_pos(pos_in[3 * i + a], L);
        vel[3 * i + a] = vel_in[3 * i + a];
    }
    orig[i] = (int)i;
}

template <typename T>
__global__ void k_keys(const T *pos, int *key, int *bin, long long n, int N, T L)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    T x[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
    Cic<T> c = cic_of<T>(x, (T)0.5 * L, (T)N / L, N);
    int k = tile_key(c.i0, N);
    key[i] = k;
    atomicAdd(bin + k, 1);
}

// exclusive scan of bin[0..nb) in place (one CTA), also copied to cursor = bin + nb + 1
__global__ void k_scan(int *bin, int nb)
{
    __shared__ int warp_sum[32];
    __shared__ int carry;
    int *cursor = bin + nb + 1;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += blockDim.x) {
        int i = base + threadIdx.x;
        int v = i < nb ? bin[i] : 0, x = v;
        int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        for (int d = 1; d < 32; d <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
        if (lane == 31) warp_sum[w] = x;
        __syncthreads();
        if (w == 0) {
            int s = lane < (blockDim.x >> 5) ? warp_sum[lane] : 0, t = s;
            for (int d = 1; d < 32; d <<= 1) { int y = __shfl_up_sync(0xffffffffu, t, d); if (lane >= d) t += y; }
            warp_sum[lane] = t - s;
        }
        __syncthreads();
        int excl = carry + warp_sum[w] + x - v;
        if (i < nb) { bin[i] = excl; cursor[i] = excl; }
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = excl + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) bin[nb] = carry;
}

template <typename T>
__global__ void k_scatter(const T *pos, const T *vel, const T *mass, const int *orig, const int *key, int *cursor,
                          T *pos2, T *vel2, T *mass2, int *orig2, long long n)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    int d = atomicAdd(cursor + key[i], 1);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        pos2[3 * (long long)d + a] = pos[3 * i + a];
        vel2[3 * (long long)d + a] = vel[3 * i + a];
    }
    if (mass) mass2[d] = mass[i];
    orig2[d] = orig[i];
}

// a = sum_nodes w * (phi[node+e] - phi[node-e]) per axis (the caller scales by -1/(2 dx)): gather of the
// central-difference gradient (Eq. 21) with the deposit's weights (G13, G30)
template <typename T, int ORDER>
__device__ __forceinline__ void gather_grad(const T *__restrict__ phi, const T (&x)[3], int N, T L, T (&a)[3])
{
    const T inv_dx = (T)N / L;
    Asg<T, ORDER> c = asg_of<T, ORDER>(x, (T)0.5 * L, inv_dx, N);
    const int M = N - 1;
    // indices base-1 .. base+ORDER along each axis
    int ix[ORDER + 2], iy[ORDER + 2], iz[ORDER + 2];
#pragma unroll
    for (int d = 0; d < ORDER + 2; ++d) {
        ix[d] = (c.base[0] + d - 1) & M;
        iy[d] = (c.base[1] + d - 1) & M;
        iz[d] = (c.base[2] + d - 1) & M;
    }
    a[0] = a[1] = a[2] = (T)0;
#pragma unroll
    for (int bx = 0; bx < ORDER; ++bx)
#pragma unroll
        for (int by = 0; by < ORDER; ++by)
#pragma unroll
            for (int bz = 0; bz < ORDER; ++bz) {
                T w = c.w[0][bx] * c.w[1][by] * c.w[2][bz];
                size_t X = ix[bx + 1], Y = iy[by + 1], Z = iz[bz + 1];
                T gx = __ldg(phi + ((size_t)ix[bx + 2] * N + Y) * N + Z) - __ldg(phi + ((size_t)ix[bx] * N + Y) * N + Z);
                T gy = __ldg(phi + (X * N + iy[by + 2]) * N + Z) - __ldg(phi + (X * N + iy[by]) * N + Z);
                T gz = __ldg(phi + (X * N + Y) * N + iz[bz + 2]) - __ldg(phi + (X * N + Y) * N + iz[bz]);
                a[0] += w * gx; a[1] += w * gy; a[2] += w * gz;
            }
}

// v += a(x) kick_dt ; then nsub drifts of drift_dt / nsub, wrapped, with a full kick of that size (gathered at the
// new position, in the same potential) between two drifts (several N-body sub-steps per SPE step)
template <typename T, int ORDER>
__global__ void k_push(T *pos, T *vel, const T *__restrict__ phi, long long n, int N, T L, T kick_dt, T drift_dt, int nsub)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    T x[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
    T v[3] = {vel[3 * i], vel[3 * i + 1], vel[3 * i + 2]};
    const T g = -(T)0.5 * (T)N / L;
    bool kicked = false;
    if (kick_dt != (T)0) {
        T a[3];
        gather_grad<T, ORDER>(phi, x, N, L, a);
#pragma unroll
        for (int d = 0; d < 3; ++d) v[d] += a[d] * (g * kick_dt);
        kicked = true;
    }
    if (drift_dt != (T)0) {
        const T h = drift_dt / (T)nsub;
        for (int j = 1; j <= nsub; ++j) {
#pragma unroll
            for (int d = 0; d < 3; ++d) x[d] = wrap_pos(x[d] + v[d] * h, L);
            if (j < nsub) {
                T a[3];
                gather_grad<T, ORDER>(phi, x, N, L, a);
#pragma unroll
                for (int d = 0; d < 3; ++d) v[d] += a[d] * (g * h);
                kicked = true;
            }
        }
#pragma unroll
        for (int d = 0; d < 3; ++d) pos[3 * i + d] = x[d];
    }
    if (kicked) {
#pragma unroll
        for (int d = 0; d < 3; ++d) vel[3 * i + d] = v[d];
    }
}

// Deposit: each CTA takes CHUNK consecutive (tile-sorted) particles and accumulates into a BOX^3-node
// shared-memory box anchored at the tile of its first particle (one node lower for the three-point cloud, whose
// stencil starts one node below the nearest node); nodes outside the box go straight to global memory.
// Particles of a warp with the same stencil are combined first (warp-aggregated atomics).
template <typename T, int ORDER>
__global__ void __launch_bounds__(256) k_deposit(const T *__restrict__ pos, const T *__restrict__ mass, T mass_scalar,
                                                 T *rho, long long n, int N, T L)
{
    constexpr int NW = ORDER * ORDER * ORDER;
    __shared__ T box[BOX * BOX * BOX];
    __shared__ int org[3];
    const long long start = (long long)blockIdx.x * CHUNK;
    const long long end = start + CHUNK < n ? start + CHUNK : n;
    const T inv_dx = (T)N / L, inv_vol = inv_dx * inv_dx * inv_dx, half_L = (T)0.5 * L;
    for (int j = threadIdx.x; j < BOX * BOX * BOX; j += blockDim.x) box[j] = (T)0;
    if (threadIdx.x == 0) {
        T x[3] = {pos[3 * start], pos[3 * start + 1], pos[3 * start + 2]};
        Cic<T> c = cic_of<T>(x, half_L, inv_dx, N);
#pragma unroll
        for (int a = 0; a < 3; ++a) org[a] = (c.i0[a] / TS) * TS - (ORDER - 2);
    }
    __syncthreads();
    const int M = N - 1;
    for (long long base = start; base < end; base += blockDim.x) {
        long long i = base + threadIdx.x;
        bool active = i < end;
        Asg<T, ORDER> c;
        T m = (T)0;
        int cell = -1;
        if (active) {
            T x[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
            c = asg_of<T, ORDER>(x, half_L, inv_dx, N);
            m = (mass ? mass[i] : mass_scalar) * inv_vol;
            cell = (c.base[0] * N + c.base[1]) * N + c.base[2];
        }
        // combine the lanes whose stencils coincide: the group leader deposits the summed weights
        unsigned peers = __match_any_sync(0xffffffffu, cell);
        int leader = __ffs(peers) - 1;
        int lane = threadIdx.x & 31;
        T w[NW];
#pragma unroll
        for (int q = 0; q < NW; ++q) {
            int bx = q / (ORDER * ORDER), by = (q / ORDER) % ORDER, bz = q % ORDER;
            w[q] = active ? m * c.w[0][bx] * c.w[1][by] * c.w[2][bz] : (T)0;
        }
        if (peers != (1u << lane)) {
            // tree-free reduction inside each peer group: walk the group mask
#pragma unroll
            for (int q = 0; q < NW; ++q) {
                T acc = (T)0;
                unsigned rem = peers;
                while (rem) {
                    int src = __ffs(rem) - 1;
                    rem &= rem - 1;
                    acc += __shfl_sync(peers, w[q], src);
                }
                w[q] = acc;
            }
        }
        if (active && lane == leader) {
            int rx = (c.base[0] - org[0]) & M, ry = (c.base[1] - org[1]) & M, rz = (c.base[2] - org[2]) & M;
            bool inside = rx <= BOX - ORDER && ry <= BOX - ORDER && rz <= BOX - ORDER;
#pragma unroll
            for (int q = 0; q < NW; ++q) {
                int bx = q / (ORDER * ORDER), by = (q / ORDER) % ORDER, bz = q % ORDER;
                if (inside) atomicAdd(&box[((rx + bx) * BOX + ry + by) * BOX + rz + bz], w[q]);
                else atomicAdd(rho + ((size_t)((c.base[0] + bx) & M) * N + ((c.base[1] + by) & M)) * N + ((c.base[2] + bz) & M), w[q]);
            }
        }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < BOX * BOX * BOX; j += blockDim.x) {
        T v = box[j];
        if (v != (T)0) {
            int rz = j % BOX, ry = (j / BOX) % BOX, rx = j / (BOX * BOX);
            atomicAdd(rho + ((size_t)((org[0] + rx) & M) * N + ((org[1] + ry) & M)) * N + ((org[2] + rz) & M), v);
        }
    }
}

template <typename T>
__global__ void k_unsort(const T *pos, const T *vel, const int *orig, T *pos_out, T *vel_out, long long n)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    long long d = orig[i];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (pos_out) pos_out[3 * d + a] = pos[3 * i + a];
        if (vel_out) vel_out[3 * d + a] = vel[3 * i + a];
    }
}

inline size_t al(size_t x) { return (x + 255) & ~(size_t)255; }
inline int nbins(int N) { int t = ntiles1(N); return t * t * t; }
inline unsigned blocks(long long n, int b) { return (unsigned)((n + b - 1) / b); }

template <typename T>
cudaError_t resort(ParticleState &ps, int N, double L, cudaStream_t s)
{
    const long long n = ps.n;
    const int nb = nbins(N);
    cudaError_t e = cudaMemsetAsync(ps.bin, 0, sizeof(int) * (2 * (size_t)nb + 2), s);
    if (e != cudaSuccess) return e;
    k_keys<T><<<blocks(n, 256), 256, 0, s>>>((const T *)ps.pos, ps.key, ps.bin, n, N, (T)L);
    k_scan<<<1, 1024, 0, s>>>(ps.bin, nb);
    k_scatter<T><<<blocks(n, 256), 256, 0, s>>>((const T *)ps.pos, (const T *)ps.vel, ps.has_mass ? (const T *)ps.mass : nullptr,
                                                ps.orig, ps.key, ps.bin + nb + 1, (T *)ps.pos2, (T *)ps.vel2,
                                                (T *)ps.mass2, ps.orig2, n);
    std::swap(ps.pos, ps.pos2);
    std::swap(ps.vel, ps.vel2);
    std::swap(ps.mass, ps.mass2);
    std::swap(ps.orig, ps.orig2);
    ps.steps_since_sort = 0;
    return cudaGetLastError();
}

template <typename T>
cudaError_t set_impl(ParticleState &ps, int N, double L, long long n, const void *pos, const void *vel, const void *mass,
                     double mass_scalar, bool from_host, cudaStream_t s)
{
    ps.n = n;
    ps.has_mass = mass != nullptr;
    ps.mass_scalar = mass_scalar;
    if (n == 0) return cudaSuccess;
    cudaMemcpyKind kind = from_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    cudaError_t e;
    // stage the caller's arrays in the second buffers, then wrap + index into the first
    if ((e = cudaMemcpyAsync(ps.pos2, pos, sizeof(T) * 3 * n, kind, s)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(ps.vel2, vel, sizeof(T) * 3 * n, kind, s)) != cudaSuccess) return e;
    if (mass && (e = cudaMemcpyAsync(ps.mass, mass, sizeof(T) * n, kind, s)) != cudaSuccess) return e;
    k_ingest<T><<<blocks(n, 256), 256, 0, s>>>((const T *)ps.pos2, (const T *)ps.vel2, (T *)ps.pos, (T *)ps.vel, ps.orig, n, (T)L);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    return resort<T>(ps, N, L, s);
}

}  // namespace

size_t particle_bytes(int N, int dtype, long long cap)
{
    size_t r = dtype == 0 ? 4 : 8, c = (size_t)(cap > 0 ? cap : 1);
    return 4 * al(3 * c * r) + 2 * al(c * r) + 3 * al(c * 4) + al(sizeof(int) * (2 * (size_t)nbins(N) + 2)) + 256;
}

void particle_bind(ParticleState &ps, int N, int dtype, long long cap, void *rho_p, void *pool)
{
    size_t r = dtype == 0 ? 4 : 8, c = (size_t)(cap > 0 ? cap : 1);
    unsigned char *p = (unsigned char *)pool;
    auto take = [&](size_t bytes) { void *q = p; p += al(bytes); return q; };
    ps.rho_p = rho_p;
    ps.pos = take(3 * c * r); ps.vel = take(3 * c * r); ps.pos2 = take(3 * c * r); ps.vel2 = take(3 * c * r);
    ps.mass = take(c * r); ps.mass2 = take(c * r);
    ps.orig = (int *)take(c * 4); ps.orig2 = (int *)take(c * 4); ps.key = (int *)take(c * 4);
    ps.bin = (int *)take(sizeof(int) * (2 * (size_t)nbins(N) + 2));
    ps.capacity = cap;
    ps.n = 0;
}

cudaError_t particle_set(ParticleState &ps, int N, double L, int dtype, long long n, const void *pos, const void *vel,
                         const void *mass, double mass_scalar, bool from_host, cudaStream_t s)
{
    return dtype == 0 ? set_impl<float>(ps, N, L, n, pos, vel, mass, mass_scalar, from_host, s)
                      : set_impl<double>(ps, N, L, n, pos, vel, mass, mass_scalar, from_host, s);
}

cudaError_t particle_push(ParticleState &ps, int N, double L, int dtype, const void *phi, double kick_dt, double drift_dt,
                          int nsub, cudaStream_t s)
{
    if (ps.n == 0) return cudaSuccess;
    if (nsub < 1) nsub = 1;
    const unsigned g = blocks(ps.n, 128);
    if (dtype == 0 && ps.order == 2) k_push<float, 2><<<g, 128, 0, s>>>((float *)ps.pos, (float *)ps.vel, (const float *)phi, ps.n, N, (float)L, (float)kick_dt, (float)drift_dt, nsub);
    else if (dtype == 0) k_push<float, 3><<<g, 128, 0, s>>>((float *)ps.pos, (float *)ps.vel, (const float *)phi, ps.n, N, (float)L, (float)kick_dt, (float)drift_dt, nsub);
    else if (ps.order == 2) k_push<double, 2><<<g, 128, 0, s>>>((double *)ps.pos, (double *)ps.vel, (const double *)phi, ps.n, N, L, kick_dt, drift_dt, nsub);
    else k_push<double, 3><<<g, 128, 0, s>>>((double *)ps.pos, (double *)ps.vel, (const double *)phi, ps.n, N, L, kick_dt, drift_dt, nsub);
    if (drift_dt != 0.0) ++ps.steps_since_sort;
    return cudaGetLastError();
}

bool particle_sort_due(const ParticleState &ps) { return ps.n > 0 && ps.steps_since_sort >= kResortInterval; }

cudaError_t particle_resort(ParticleState &ps, int N, double L, int dtype, cudaStream_t s)
{
    if (ps.n == 0) return cudaSuccess;
    return dtype == 0 ? resort<float>(ps, N, L, s) : resort<double>(ps, N, L, s);
}

cudaError_t particle_deposit(ParticleState &ps, int N, double L, int dtype, cudaStream_t s)
{
    if (ps.n == 0) return cudaSuccess;
    unsigned g = blocks(ps.n, CHUNK);
    const float *mf = ps.has_mass ? (const float *)ps.mass : nullptr;
    const double *md = ps.has_mass ? (const double *)ps.mass : nullptr;
    if (dtype == 0 && ps.order == 2) k_deposit<float, 2><<<g, 256, 0, s>>>((const float *)ps.pos, mf, (float)ps.mass_scalar, (float *)ps.rho_p, ps.n, N, (float)L);
    else if (dtype == 0) k_deposit<float, 3><<<g, 256, 0, s>>>((const float *)ps.pos, mf, (float)ps.mass_scalar, (float *)ps.rho_p, ps.n, N, (float)L);
    else if (ps.order == 2) k_deposit<double, 2><<<g, 256, 0, s>>>((const double *)ps.pos, md, ps.mass_scalar, (double *)ps.rho_p, ps.n, N, L);
    else k_deposit<double, 3><<<g, 256, 0, s>>>((const double *)ps.pos, md, ps.mass_scalar, (double *)ps.rho_p, ps.n, N, L);
    return cudaGetLastError();
}

cudaError_t particle_get(ParticleState &ps, int dtype, void *pos_out, void *vel_out, bool to_host, cudaStream_t s)
{
    if (ps.n == 0 || (!pos_out && !vel_out)) return cudaSuccess;
    const long long n = ps.n;
    size_t r = dtype == 0 ? 4 : 8;
    void *dp = to_host ? ps.pos2 : pos_out, *dv = to_host ? ps.vel2 : vel_out;
    if (to_host && !pos_out) dp = nullptr;
    if (to_host && !vel_out) dv = nullptr;
    if (dtype == 0) k_unsort<float><<<blocks(n, 256), 256, 0, s>>>((const float *)ps.pos, (const float *)ps.vel, ps.orig, (float *)dp, (float *)dv, n);
    else k_unsort<double><<<blocks(n, 256), 256, 0, s>>>((const double *)ps.pos, (const double *)ps.vel, ps.orig, (double *)dp, (double *)dv, n);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (to_host) {
        if (pos_out && (e = cudaMemcpyAsync(pos_out, dp, 3 * n * r, cudaMemcpyDeviceToHost, s)) != cudaSuccess) return e;
        if (vel_out && (e = cudaMemcpyAsync(vel_out, dv, 3 * n * r, cudaMemcpyDeviceToHost, s)) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace wdm
