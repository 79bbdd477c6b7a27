// wdm_particles.hpp -- N-body particles coupled through the shared potential:
// cloud-in-cell deposit into the Poisson source, CIC gather of the central-difference gradient
// (Eq. 21), kick-drift-kick leapfrog with the wave field's dt (readings G11-G16).
#pragma once
#include <cuda_runtime.h>
#include <cstddef>

namespace wdm {

struct ParticleState {
    long long n = 0, capacity = 0;
    void *rho_p = nullptr;                   // N^3 reals: particle mass density on the mesh
    void *pos = nullptr, *vel = nullptr;     // (n,3) reals, kept sorted by mesh tile
    void *pos2 = nullptr, *vel2 = nullptr;   // sort double buffers
    void *mass = nullptr, *mass2 = nullptr;  // n reals (per-particle masses) -- unused when has_mass == false
    int *orig = nullptr, *orig2 = nullptr;   // caller's index of each sorted particle
    int *key = nullptr;                      // tile key per particle
    int *bin = nullptr;                      // (ntiles + 1) counters / offsets, then a cursor copy
    // rho_p is zero wherever its flag is clear: flag[y * (N / FB) + z / FB], FB = mesh_flag_block(N), marks the blocks of
    // FB z-cells (for every x) that hold deposited mass.  The deposit sets flags, the clear zeroes flagged blocks only,
    // and the density sweep reads rho_p only for flagged tiles.
    unsigned char *flag = nullptr;
    bool mesh_clean = false;                 // false: content unknown, the next clear zeroes the whole mesh
    bool mesh_cleared = false;               // the last push also cleared the flagged columns: the next clear is a no-op
    bool has_mass = false;
    double mass_scalar = 0.0;
    int steps_since_sort = 0;
    int order = 2;                           // 2: cloud-in-cell (G12-G13), 3: triangular-shaped cloud (G30)
};

size_t particle_bytes(int N, int dtype, long long capacity);
void particle_bind(ParticleState &ps, int N, int dtype, long long capacity, void *rho_p, void *pool);
cudaError_t particle_set(ParticleState &ps, int N, double L, int dtype, long long n, const void *pos, const void *vel,
                         const void *mass, double mass_scalar, bool from_host, cudaStream_t s);
// v += a(phi, x) * kick_dt ; then nsub drifts of drift_dt / nsub (wrapped into [-L/2, L/2)) with a kick of that
// size, gathered at the new position, between two drifts
// clear_mesh: also zero the flagged columns of rho_p (the caller deposits next; see particle_mesh_clear)
cudaError_t particle_push(ParticleState &ps, int N, double L, int dtype, const void *phi, double kick_dt,
                          double drift_dt, int nsub, bool clear_mesh, cudaStream_t s);
// the tile order is kResortInterval drifts old: re-sort (counting sort by mesh tile) before the next deposit
bool particle_sort_due(const ParticleState &ps);
cudaError_t particle_resort(ParticleState &ps, int N, double L, int dtype, cudaStream_t s);
// z-cells per flag (a multiple of every sweep's tile width W <= 16)
inline __host__ __device__ int mesh_flag_block(int N) { return N < 16 ? N : 16; }
// rho_p = 0 (only where the flags say mass was deposited, once the mesh is known to be clean)
cudaError_t particle_mesh_clear(ParticleState &ps, int N, int dtype, cudaStream_t s);
// rho_p += deposit of the particles' mass with the scheme ps.order (the caller zeroes rho_p)
cudaError_t particle_deposit(ParticleState &ps, int N, double L, int dtype, cudaStream_t s);
// the same deposit accumulated in 64-bit fixed point (acc: N^3 zeroed words, left zeroed): bit-reproducible; writes the
// WHOLE mesh rho_p, no clear needed.  total_mass bounds the sum of all particle masses.
cudaError_t particle_deposit_fixed(ParticleState &ps, int N, double L, int dtype, unsigned long long *acc, double total_mass,
                                   cudaStream_t s);
cudaError_t particle_get(ParticleState &ps, int dtype, void *pos_out, void *vel_out, bool to_host, cudaStream_t s);

}  // namespace wdm
