// wdm_particles.cu -- particle kernels (see wdm_particles.hpp).
//
// Particles are kept sorted by mesh tile (TS^3 cells, tile-major) and, inside a tile, by cell: a counting sort over
// the tiles, then one CTA per tile sorting its segment by the 512 local cells in shared memory.  Redone every
// kResortInterval pushes: a disc particle moves 1e-3..1e-2 cells per step, so the order stays useful for
// hundreds of steps.  With neighbouring lanes in the same or adjacent cells the 32 scattered Phi loads of a gather
// fall into one or two sectors per instruction (the gather was bound by L1 wavefronts: 48 loads x ~32 sectors per
// warp), and the lanes of a warp that share a stencil combine their weights before touching shared memory.
// Correctness never depends on the order: the deposit falls back to global atomics for any node outside the
// CTA's shared-memory box.
#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>
#include <type_traits>

#include "../../include/wdm_static.h"
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

// Second level of the sort: CTA t orders the particles of tile t (the segment [bin[t], bin[t+1]) of the tile-sorted
// arrays) by their cell inside the tile -- histogram of the TS^3 local cells in shared memory, exclusive scan,
// scatter into the other buffer set.  Empty tiles exit at once.
template <typename T>
__global__ void __launch_bounds__(256) k_cellsort(const T *pos, const T *vel, const T *mass, const int *orig, const int *bin,
                                                  T *pos2, T *vel2, T *mass2, int *orig2, int N, T L)
{
    constexpr int NC = TS * TS * TS;
    __shared__ int hist[NC];
    __shared__ int wsum[8];
    const int t = blockIdx.x;
    const int beg = bin[t], end = bin[t + 1];
    if (end <= beg) return;
    const T half_L = (T)0.5 * L, inv_dx = (T)N / L;
    auto local_cell = [&](int i) {
        T x[3] = {pos[3 * (long long)i], pos[3 * (long long)i + 1], pos[3 * (long long)i + 2]};
        Cic<T> c = cic_of<T>(x, half_L, inv_dx, N);
        return ((c.i0[0] % TS) * TS + (c.i0[1] % TS)) * TS + (c.i0[2] % TS);
    };
    if (end - beg == 1) {                       // the common case in the outskirts: nothing to order
        if (threadIdx.x == 0) {
#pragma unroll
            for (int a = 0; a < 3; ++a) { pos2[3 * (long long)beg + a] = pos[3 * (long long)beg + a]; vel2[3 * (long long)beg + a] = vel[3 * (long long)beg + a]; }
            if (mass) mass2[beg] = mass[beg];
            orig2[beg] = orig[beg];
        }
        return;
    }
    for (int j = threadIdx.x; j < NC; j += blockDim.x) hist[j] = 0;
    __syncthreads();
    for (int i = beg + threadIdx.x; i < end; i += blockDim.x) atomicAdd(&hist[local_cell(i)], 1);
    __syncthreads();
    {   // exclusive scan of hist[0..512): two entries per thread
        const int j = 2 * threadIdx.x, a0 = hist[j], a1 = hist[j + 1];
        int x = a0 + a1;
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        for (int d = 1; d < 32; d <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
        if (lane == 31) wsum[w] = x;
        __syncthreads();
        int base = 0;
        for (int k = 0; k < w; ++k) base += wsum[k];
        const int excl = base + x - (a0 + a1);
        hist[j] = excl;
        hist[j + 1] = excl + a0;
    }
    __syncthreads();
    for (int i = beg + threadIdx.x; i < end; i += blockDim.x) {
        const long long d = beg + atomicAdd(&hist[local_cell(i)], 1);
#pragma unroll
        for (int a = 0; a < 3; ++a) { pos2[3 * d + a] = pos[3 * (long long)i + a]; vel2[3 * d + a] = vel[3 * (long long)i + a]; }
        if (mass) mass2[d] = mass[i];
        orig2[d] = orig[i];
    }
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
    if constexpr (ORDER == 2) {
        // cloud-in-cell: the 48 central-difference operands are 32 distinct nodes of the 4^3 neighbourhood (those with at
        // most one coordinate outside the cell); load each once, 32-bit offsets (N^3 <= 2^30)
        int ox[4], oy[4];
#pragma unroll
        for (int d = 0; d < 4; ++d) { ox[d] = ix[d] * N * N; oy[d] = iy[d] * N; }
        T f[4][4][4];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if ((i == 0 || i == 3) + (j == 0 || j == 3) + (k == 0 || k == 3) <= 1) f[i][j][k] = __ldg(phi + (ox[i] + oy[j] + iz[k]));
#pragma unroll
        for (int p = 1; p <= 2; ++p)
#pragma unroll
            for (int q = 1; q <= 2; ++q) {
                a[0] += c.w[1][p - 1] * c.w[2][q - 1] * (c.w[0][0] * (f[2][p][q] - f[0][p][q]) + c.w[0][1] * (f[3][p][q] - f[1][p][q]));
                a[1] += c.w[0][p - 1] * c.w[2][q - 1] * (c.w[1][0] * (f[p][2][q] - f[p][0][q]) + c.w[1][1] * (f[p][3][q] - f[p][1][q]));
                a[2] += c.w[0][p - 1] * c.w[1][q - 1] * (c.w[2][0] * (f[p][q][2] - f[p][q][0]) + c.w[2][1] * (f[p][q][3] - f[p][q][1]));
            }
        return;
    }
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
__global__ void k_push(T *pos, T *vel, const T *__restrict__ phi, long long n, int N, T L, T kick_dt, T drift_dt, int nsub,
                       T *mesh, unsigned char *flag, int nflag, int fb)
{
    // Clear duty (mesh != nullptr): the particle mesh must be zero before the deposit that follows this kernel, and
    // nothing here reads it -- CTA b < nflag zeroes flagged column b (see k_mesh_clear) on its way, which saves a launch.
    if (mesh && (int)blockIdx.x < nflag && flag[blockIdx.x]) {
        const int b = blockIdx.x, nfb = N / fb, y = b / nfb, z0 = (b - y * nfb) * fb;
        for (int i = threadIdx.x; i < N * fb; i += blockDim.x) mesh[((size_t)(i / fb) * N + y) * N + z0 + i % fb] = (T)0;
        __syncthreads();
        if (threadIdx.x == 0) flag[b] = 0;
    }
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
                                                 T *rho, unsigned char *flag, long long n, int N, T L)
{
    // flag[y * (N / FB) + z / FB] = 1 for every block of FB z-cells of a y-row that receives mass (see mesh_flag_block)
    const int fb = mesh_flag_block(N), nfb = N / fb;
    constexpr int NW = ORDER * ORDER * ORDER;
    // Single precision: the box holds 32-bit FIXED-POINT sums.  Shared-memory atomics are native only for 32-bit integers
    // (ATOMS.ADD); a float atomicAdd compiles to a compare-and-swap spin loop (ATOMS.CAST.SPIN), which retries whenever
    // the leaders of several warps hit the same node of a dense cell.  The scale maps the largest sum the chunk can
    // produce -- all its particles on one node -- onto 2^31; one unit is 5e-7 of a single particle's m / dx^3, below the
    // float rounding of the sums it replaces.  Double precision keeps the (compare-and-swap) double sums.
    constexpr bool FIXED = sizeof(T) == 4;
    using BoxT = typename std::conditional<FIXED, int, T>::type;
    __shared__ BoxT box[BOX * BOX * BOX];
    __shared__ int org[3];
    __shared__ T smax[8];
    const long long start = (long long)blockIdx.x * CHUNK;
    const long long end = start + CHUNK < n ? start + CHUNK : n;
    const T inv_dx = (T)N / L, inv_vol = inv_dx * inv_dx * inv_dx, half_L = (T)0.5 * L;
    for (int j = threadIdx.x; j < BOX * BOX * BOX; j += blockDim.x) box[j] = (BoxT)0;
    T scale = (T)1, inv_scale = (T)1;
    if constexpr (FIXED) {
        T mmax = fabs(mass_scalar);
        if (mass) {                                            // largest |mass| of the chunk
            mmax = (T)0;
            for (long long i = start + threadIdx.x; i < end; i += blockDim.x) mmax = fmax(mmax, fabs(mass[i]));
            for (int d = 16; d; d >>= 1) mmax = fmax(mmax, __shfl_down_sync(0xffffffffu, mmax, d));
            if ((threadIdx.x & 31) == 0) smax[threadIdx.x >> 5] = mmax;
            __syncthreads();
            mmax = smax[0];
            for (int w = 1; w < (int)(blockDim.x >> 5); ++w) mmax = fmax(mmax, smax[w]);
        }
        const T bound = (T)CHUNK * mmax * inv_vol;
        scale = bound > (T)0 ? (T)2147480000.0 / bound : (T)0;
        inv_scale = bound > (T)0 ? bound / (T)2147480000.0 : (T)0;
    }
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
        // Combine the lanes whose stencils coincide.  The particles are sorted by cell, so lanes with the same stencil
        // form RUNS of consecutive lanes: a segmented reduction (5 shuffle steps per weight) leaves the run's sum in its
        // first lane, which deposits it.  (A cell that shows up in two separate runs -- particles that drifted since the
        // last sort -- is simply deposited twice.)
        const int lane = threadIdx.x & 31;
        const int prev = __shfl_up_sync(0xffffffffu, cell, 1);
        const bool head = lane == 0 || prev != cell;
        const unsigned heads = __ballot_sync(0xffffffffu, head);
        const unsigned above = lane == 31 ? 0u : heads & ~((2u << lane) - 1u);       // run heads in the lanes after this one
        const int run_end = above ? __ffs(above) - 1 : 32;                         // first lane of the next run
        const int leader = head ? lane : -1;
        T w[NW];
#pragma unroll
        for (int q = 0; q < NW; ++q) {
            int bx = q / (ORDER * ORDER), by = (q / ORDER) % ORDER, bz = q % ORDER;
            w[q] = active ? m * c.w[0][bx] * c.w[1][by] * c.w[2][bz] : (T)0;
        }
        if (heads != 0xffffffffu) {
#pragma unroll
            for (int q = 0; q < NW; ++q) {
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const T v = __shfl_down_sync(0xffffffffu, w[q], d);
                    if (lane + d < run_end) w[q] += v;
                }
            }
        }
        if (active && lane == leader) {
            int rx = (c.base[0] - org[0]) & M, ry = (c.base[1] - org[1]) & M, rz = (c.base[2] - org[2]) & M;
            bool inside = rx <= BOX - ORDER && ry <= BOX - ORDER && rz <= BOX - ORDER;
#pragma unroll
            for (int q = 0; q < NW; ++q) {
                int bx = q / (ORDER * ORDER), by = (q / ORDER) % ORDER, bz = q % ORDER;
                if (inside) {
                    if constexpr (FIXED) atomicAdd(&box[((rx + bx) * BOX + ry + by) * BOX + rz + bz], __float2int_rn(w[q] * scale));
                    else atomicAdd(&box[((rx + bx) * BOX + ry + by) * BOX + rz + bz], w[q]);
                } else {
                    const int gy = (c.base[1] + by) & M, gz = (c.base[2] + bz) & M;
                    atomicAdd(rho + ((size_t)((c.base[0] + bx) & M) * N + gy) * N + gz, w[q]);
                    flag[gy * nfb + gz / fb] = 1;
                }
            }
        }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < BOX * BOX * BOX; j += blockDim.x) {
        const BoxT vb = box[j];
        if (vb != (BoxT)0) {
            const T v = FIXED ? (T)vb * inv_scale : (T)vb;
            int rz = j % BOX, ry = (j / BOX) % BOX, rx = j / (BOX * BOX);
            const int gy = (org[1] + ry) & M, gz = (org[2] + rz) & M;
            atomicAdd(rho + ((size_t)((org[0] + rx) & M) * N + gy) * N + gz, v);
            flag[gy * nfb + gz / fb] = 1;
        }
    }
}

// Deterministic deposit (debugging mode, SURVEY.md "Determinism"): every weight is rounded ONCE to a 64-bit fixed-point
// number (scale = a power of two chosen from the total mass, so that the sum of everything fits) and accumulated with
// integer atomics -- integer addition is associative, so the mesh is bit-identical from run to run whatever the order
// of the particles, the warps or the sort.  Costs 8 bytes per cell of extra memory and a conversion pass.
template <typename T, int ORDER>
__global__ void __launch_bounds__(256) k_deposit_fixed(const T *__restrict__ pos, const T *__restrict__ mass, T mass_scalar,
                                                       unsigned long long *acc, long long n, int N, T L, double scale)
{
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const T inv_dx = (T)N / L, inv_vol = inv_dx * inv_dx * inv_dx;
    const T x[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
    const Asg<T, ORDER> c = asg_of<T, ORDER>(x, (T)0.5 * L, inv_dx, N);
    const T m = (mass ? mass[i] : mass_scalar) * inv_vol;
    const int M = N - 1;
#pragma unroll
    for (int bx = 0; bx < ORDER; ++bx)
#pragma unroll
        for (int by = 0; by < ORDER; ++by)
#pragma unroll
            for (int bz = 0; bz < ORDER; ++bz) {
                const T w = m * c.w[0][bx] * c.w[1][by] * c.w[2][bz];          // the same product as k_deposit
                const long long q = __double2ll_rn((double)w * scale);
                atomicAdd(acc + ((size_t)((c.base[0] + bx) & M) * N + ((c.base[1] + by) & M)) * N + ((c.base[2] + bz) & M),
                          (unsigned long long)q);
            }
}

// rho = acc / scale, acc = 0 (whole mesh)
template <typename T>
__global__ void k_fixed_to_mesh(unsigned long long *acc, T *rho, size_t n, double inv_scale)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const long long v = (long long)acc[i];
        rho[i] = (T)((double)v * inv_scale);
        if (v) acc[i] = 0;
    }
}

// Zero the flagged parts of the particle mesh and the flags: block b = (y, z-block) covers rho[x][y][zb*FB .. +FB) for
// every x.  One CTA per flag; unflagged blocks (a thin disc flags ~10 % of them) cost one byte load.
template <typename T>
__global__ void __launch_bounds__(128) k_mesh_clear(T *rho, unsigned char *flag, int N, int fb)
{
    const int b = blockIdx.x, nfb = N / fb;
    if (!flag[b]) return;
    const int y = b / nfb, z0 = (b - y * nfb) * fb;
    // fb reals per x-row: threads cover (x, z) pairs, fb consecutive threads on one row
    for (int i = threadIdx.x; i < N * fb; i += blockDim.x) {
        const int x = i / fb, z = z0 + i % fb;
        rho[((size_t)x * N + y) * N + z] = (T)0;
    }
    __syncthreads();
    if (threadIdx.x == 0) flag[b] = 0;
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
    if (N >= TS) {
        // tile-sorted set 2 -> tile- and cell-sorted set 1
        k_cellsort<T><<<nb, 256, 0, s>>>((const T *)ps.pos2, (const T *)ps.vel2, ps.has_mass ? (const T *)ps.mass2 : nullptr, ps.orig2,
                                         ps.bin, (T *)ps.pos, (T *)ps.vel, (T *)ps.mass, ps.orig, N, (T)L);
    } else {
        std::swap(ps.pos, ps.pos2);
        std::swap(ps.vel, ps.vel2);
        std::swap(ps.mass, ps.mass2);
        std::swap(ps.orig, ps.orig2);
    }
    ps.steps_since_sort = 0;
    return cudaGetLastError();
}

template <typename T>
cudaError_t set_impl(ParticleState &ps, int N, double L, long long n, const void *pos, const void *vel, const void *mass,
                     double mass_scalar, bool from_host, cudaStream_t s)
{
    // the particle set is committed only when every copy and launch has been accepted; a failure leaves none
    ps.n = 0;
    if (n == 0) { ps.has_mass = false; ps.mass_scalar = mass_scalar; return cudaSuccess; }
    cudaMemcpyKind kind = from_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    cudaError_t e;
    // stage the caller's arrays in the second buffers, then wrap + index into the first
    if ((e = cudaMemcpyAsync(ps.pos2, pos, sizeof(T) * 3 * n, kind, s)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(ps.vel2, vel, sizeof(T) * 3 * n, kind, s)) != cudaSuccess) return e;
    if (mass && (e = cudaMemcpyAsync(ps.mass, mass, sizeof(T) * n, kind, s)) != cudaSuccess) return e;
    k_ingest<T><<<blocks(n, 256), 256, 0, s>>>((const T *)ps.pos2, (const T *)ps.vel2, (T *)ps.pos, (T *)ps.vel, ps.orig, n, (T)L);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    ps.n = n;
    ps.has_mass = mass != nullptr;
    ps.mass_scalar = mass_scalar;
    if ((e = resort<T>(ps, N, L, s)) != cudaSuccess) ps.n = 0;
    return e;
}

}  // namespace

size_t particle_bytes(int N, int dtype, long long cap)
{
    size_t r = dtype == 0 ? 4 : 8, c = (size_t)(cap > 0 ? cap : 1);
    return 4 * al(3 * c * r) + 2 * al(c * r) + 3 * al(c * 4) + al(sizeof(int) * (2 * (size_t)nbins(N) + 2)) + al((size_t)N * N) + 256;
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
    ps.flag = (unsigned char *)take((size_t)N * N);
    ps.mesh_clean = false;
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
                          int nsub, bool clear_mesh, cudaStream_t s)
{
    if (ps.n == 0) return cudaSuccess;
    if (nsub < 1) nsub = 1;
    const int fb = mesh_flag_block(N), nflag = N * (N / fb);
    unsigned g = blocks(ps.n, 128);
    // the sparse clear rides along only when the mesh is known to be clean outside the flagged columns
    const bool clr = clear_mesh && ps.mesh_clean && ps.rho_p != nullptr;
    if (clr && g < (unsigned)nflag) g = (unsigned)nflag;
    void *mesh = clr ? ps.rho_p : nullptr;
    if (dtype == 0 && ps.order == 2) k_push<float, 2><<<g, 128, 0, s>>>((float *)ps.pos, (float *)ps.vel, (const float *)phi, ps.n, N, (float)L, (float)kick_dt, (float)drift_dt, nsub, (float *)mesh, ps.flag, nflag, fb);
    else if (dtype == 0) k_push<float, 3><<<g, 128, 0, s>>>((float *)ps.pos, (float *)ps.vel, (const float *)phi, ps.n, N, (float)L, (float)kick_dt, (float)drift_dt, nsub, (float *)mesh, ps.flag, nflag, fb);
    else if (ps.order == 2) k_push<double, 2><<<g, 128, 0, s>>>((double *)ps.pos, (double *)ps.vel, (const double *)phi, ps.n, N, L, kick_dt, drift_dt, nsub, (double *)mesh, ps.flag, nflag, fb);
    else k_push<double, 3><<<g, 128, 0, s>>>((double *)ps.pos, (double *)ps.vel, (const double *)phi, ps.n, N, L, kick_dt, drift_dt, nsub, (double *)mesh, ps.flag, nflag, fb);
    if (drift_dt != 0.0) ++ps.steps_since_sort;
    ps.mesh_cleared = clr;
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
    if (dtype == 0 && ps.order == 2) k_deposit<float, 2><<<g, 256, 0, s>>>((const float *)ps.pos, mf, (float)ps.mass_scalar, (float *)ps.rho_p, ps.flag, ps.n, N, (float)L);
    else if (dtype == 0) k_deposit<float, 3><<<g, 256, 0, s>>>((const float *)ps.pos, mf, (float)ps.mass_scalar, (float *)ps.rho_p, ps.flag, ps.n, N, (float)L);
    else if (ps.order == 2) k_deposit<double, 2><<<g, 256, 0, s>>>((const double *)ps.pos, md, ps.mass_scalar, (double *)ps.rho_p, ps.flag, ps.n, N, L);
    else k_deposit<double, 3><<<g, 256, 0, s>>>((const double *)ps.pos, md, ps.mass_scalar, (double *)ps.rho_p, ps.flag, ps.n, N, L);
    return cudaGetLastError();
}

cudaError_t particle_deposit_fixed(ParticleState &ps, int N, double L, int dtype, unsigned long long *acc, double total_mass,
                                   cudaStream_t s)
{
    if (ps.n == 0) return cudaSuccess;
    // the largest possible cell value is total_mass / dx^3; leave two bits of head room below 2^62
    const double dx = L / N, top = total_mass / (dx * dx * dx);
    int ex = 0;
    frexp(top > 0 ? top : 1.0, &ex);
    const double scale = ldexp(1.0, 60 - ex);
    const unsigned g = blocks(ps.n, 256);
    const float *mf = ps.has_mass ? (const float *)ps.mass : nullptr;
    const double *md = ps.has_mass ? (const double *)ps.mass : nullptr;
    if (dtype == 0 && ps.order == 2) k_deposit_fixed<float, 2><<<g, 256, 0, s>>>((const float *)ps.pos, mf, (float)ps.mass_scalar, acc, ps.n, N, (float)L, scale);
    else if (dtype == 0) k_deposit_fixed<float, 3><<<g, 256, 0, s>>>((const float *)ps.pos, mf, (float)ps.mass_scalar, acc, ps.n, N, (float)L, scale);
    else if (ps.order == 2) k_deposit_fixed<double, 2><<<g, 256, 0, s>>>((const double *)ps.pos, md, ps.mass_scalar, acc, ps.n, N, L, scale);
    else k_deposit_fixed<double, 3><<<g, 256, 0, s>>>((const double *)ps.pos, md, ps.mass_scalar, acc, ps.n, N, L, scale);
    const size_t n3 = (size_t)N * N * N;
    if (dtype == 0) k_fixed_to_mesh<float><<<148 * 8, 256, 0, s>>>(acc, (float *)ps.rho_p, n3, 1.0 / scale);
    else k_fixed_to_mesh<double><<<148 * 8, 256, 0, s>>>(acc, (double *)ps.rho_p, n3, 1.0 / scale);
    // the whole mesh was rewritten: every block counts as touched (a later sparse clear then zeroes all of it)
    cudaError_t e = cudaMemsetAsync(ps.flag, 1, (size_t)N * (N / mesh_flag_block(N)), s);
    if (e != cudaSuccess) return e;
    ps.mesh_clean = true;
    return cudaGetLastError();
}

cudaError_t particle_mesh_clear(ParticleState &ps, int N, int dtype, cudaStream_t s)
{
    const int fb = mesh_flag_block(N), nflag = N * (N / fb);
    if (ps.mesh_cleared) { ps.mesh_cleared = false; return cudaSuccess; }      // the preceding push did it
    if (!ps.mesh_clean) {
        // first use (or a mesh of unknown content): everything, once
        cudaError_t e = cudaMemsetAsync(ps.rho_p, 0, (size_t)N * N * N * (dtype == 0 ? 4 : 8), s);
        if (e == cudaSuccess) e = cudaMemsetAsync(ps.flag, 0, (size_t)nflag, s);
        if (e == cudaSuccess) ps.mesh_clean = true;
        return e;
    }
    if (dtype == 0) k_mesh_clear<float><<<nflag, 128, 0, s>>>((float *)ps.rho_p, ps.flag, N, fb);
    else k_mesh_clear<double><<<nflag, 128, 0, s>>>((double *)ps.rho_p, ps.flag, N, fb);
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

// ---------------------------------------------------------------- wdm_deposit_static (include/wdm_static.h)
// The deterministic deposit with its accumulator mesh in a file-scope array instead of allocated memory: for
// callers that must not allocate.  Every GPU that loads the library holds these 2 MiB until the process exits; every
// call on a GPU shares them (overlapping calls race, see the header).
//
// In HOST code `g_static_acc` is only a stand-in for the symbol, not a device address: the address the kernels get is
// looked up with cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned long long g_static_acc[WDM_STATIC_MAX_CELLS];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
unsigned long long *g_static_ptr[kMaxDevices] = {};      // device address of g_static_acc on device d, once looked up
thread_local char g_static_err[512] = "";               // fixed buffer: not even the error path allocates

int sfail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_static_err, sizeof g_static_err, fmt, ap);
    va_end(ap);
    return code;
}

// set-up: the scratch address on the CURRENT device (cached per device)
int static_scratch(unsigned long long **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return sfail(WDM_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return sfail(WDM_EUNSUPPORTED, "device ordinal %d outside [0, %d)", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        unsigned long long *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_static_acc);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return sfail(WDM_ECUDA, "cudaGetSymbolAddress of the static deposit scratch on device %d: %s", dev, cudaGetErrorString(e));
        }
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return WDM_OK;
}

}  // namespace

extern "C" size_t wdm_static_scratch_bytes(void) { return sizeof(unsigned long long) * WDM_STATIC_MAX_CELLS; }

extern "C" const char *wdm_static_last_error(void) { return g_static_err; }

extern "C" int wdm_deposit_static(const void *pos_dev, const void *mass_dev, double mass_scalar, long long n, int N, double L,
                                  int dtype, int order, double total_mass, void *rho_out_dev, void *cuda_stream)
{
    using namespace wdm;
    if (dtype != WDM_C64 && dtype != WDM_C128) return sfail(WDM_EINVAL, "dtype must be WDM_C64 or WDM_C128, got %d", dtype);
    if (order != 2 && order != 3) return sfail(WDM_EINVAL, "assignment order must be 2 (cloud-in-cell) or 3 (triangular-shaped cloud), got %d", order);
    if (n < 0 || n > 0x7fffffffll * 256) return sfail(WDM_EINVAL, "particle count %lld out of range", n);
    if (!(L > 0) || !std::isfinite(L)) return sfail(WDM_EINVAL, "L must be positive and finite");
    if (!(total_mass > 0) || !std::isfinite(total_mass)) return sfail(WDM_EINVAL, "total_mass must be positive and finite (an upper bound of sum |m_i|)");
    if (!std::isfinite(mass_scalar)) return sfail(WDM_EINVAL, "mass_scalar must be finite");
    if (N < 8 || (N & (N - 1)) != 0) return sfail(WDM_EUNSUPPORTED, "N must be a power of two >= 8, got %d", N);
    if (N > WDM_STATIC_MAX_N)
        return sfail(WDM_EUNSUPPORTED, "N = %d: N^3 cells exceed the static scratch (%llu cells, N <= %d); use a wdm_ctx with wdm_set_deposit_mode",
                     N, (unsigned long long)WDM_STATIC_MAX_CELLS, WDM_STATIC_MAX_N);
    if (!rho_out_dev || (n > 0 && !pos_dev)) return sfail(WDM_EINVAL, "null pointer");

    unsigned long long *acc = nullptr;
    if (int rc = static_scratch(&acc)) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t n3 = (size_t)N * N * N;
    // the array keeps whatever the last call (possibly a failed or a differently sized one) left in it
    cudaError_t e = cudaMemsetAsync(acc, 0, n3 * sizeof(unsigned long long), s);
    if (e != cudaSuccess) return sfail(WDM_ECUDA, "cudaMemsetAsync of the static scratch: %s", cudaGetErrorString(e));
    // the same scale as particle_deposit_fixed: the largest possible cell value is total_mass / dx^3, two bits of head room
    const double dx = L / N, top = total_mass / (dx * dx * dx);
    int ex = 0;
    frexp(top, &ex);
    const double scale = ldexp(1.0, 60 - ex);
    if (n > 0) {
        const unsigned g = blocks(n, 256);
        if (dtype == WDM_C64 && order == 2) k_deposit_fixed<float, 2><<<g, 256, 0, s>>>((const float *)pos_dev, (const float *)mass_dev, (float)mass_scalar, acc, n, N, (float)L, scale);
        else if (dtype == WDM_C64) k_deposit_fixed<float, 3><<<g, 256, 0, s>>>((const float *)pos_dev, (const float *)mass_dev, (float)mass_scalar, acc, n, N, (float)L, scale);
        else if (order == 2) k_deposit_fixed<double, 2><<<g, 256, 0, s>>>((const double *)pos_dev, (const double *)mass_dev, mass_scalar, acc, n, N, L, scale);
        else k_deposit_fixed<double, 3><<<g, 256, 0, s>>>((const double *)pos_dev, (const double *)mass_dev, mass_scalar, acc, n, N, L, scale);
        if ((e = cudaGetLastError()) != cudaSuccess) return sfail(WDM_ECUDA, "deposit kernel launch: %s", cudaGetErrorString(e));
    }
    const unsigned gc = blocks((long long)n3, 256);
    if (dtype == WDM_C64) k_fixed_to_mesh<float><<<gc, 256, 0, s>>>(acc, (float *)rho_out_dev, n3, 1.0 / scale);
    else k_fixed_to_mesh<double><<<gc, 256, 0, s>>>(acc, (double *)rho_out_dev, n3, 1.0 / scale);
    if ((e = cudaGetLastError()) != cudaSuccess) return sfail(WDM_ECUDA, "conversion kernel launch: %s", cudaGetErrorString(e));
    return WDM_OK;
}
