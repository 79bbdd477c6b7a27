/*
 * wdm.h -- C ABI of libwdm.so: the B200 (sm_100a) split-step Schroedinger-Poisson + CIC particle step.
 *
 * One context = one periodic N^3 box.  Every call returns a WDM_* code; no exception crosses the
 * boundary.  Pointers named *_dev are DEVICE pointers (e.g. torch.Tensor.data_ptr()), pointers named
 * *_host are HOST pointers (pinned memory makes the copies asynchronous).  The caller owns every
 * buffer it passes; the library copies in/out on the context's stream and owns only its internal
 * state.  PAPER.md below is the paper text (arxiv/paper_2606_25026); G<n> are the readings listed in
 * DESIGN.md.
 *
 * Layout: grid arrays have shape (N, N, N) in C order, index (ix, iy, iz) <-> grid point
 * x = -L/2 + ix*dx etc. with dx = L/N (Eq. 20; reading G1), iz contiguous.
 * Complex values are interleaved (re, im).  For dtype WDM_C64 complex = 2 x float32 and every real
 * array / particle array is float32; for WDM_C128 complex = 2 x float64 and reals are float64 (G23).
 * Particle pos/vel are (n, 3) C order, columns x, y, z.
 */
#ifndef WDM_H
#define WDM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wdm_ctx wdm_ctx; /* opaque, owned by the library */

enum { WDM_C64 = 0, WDM_C128 = 1 };
enum {
    WDM_OK = 0,
    WDM_EINVAL = 1,       /* null pointer, L <= 0, hbar_over_m <= 0, G < 0, n < 0, nsteps < 0, non-finite dt, bad dtype */
    WDM_EUNSUPPORTED = 2, /* N not a power of two or outside [8, 1024] (powers of two)  */
    WDM_ENOMEM = 3,       /* device allocation failed / caller workspace too small                     */
    WDM_ECUDA = 4,        /* a CUDA call failed; text in wdm_last_error                                */
    WDM_ESTATE = 5        /* wdm_step / wdm_get_* before wdm_set_psi                                   */
};

/* Bytes of device workspace a context needs (psi, Phi, the Poisson half-spectrum, tables and, if
 * max_particles > 0, the particle mesh and particle arrays).  Lets the caller take ALL device memory
 * from its own allocator (PyTorch) and hand it to wdm_create_ws. */
int wdm_workspace_bytes(int N, int dtype, long long max_particles, size_t *bytes_out);

/* Create a context for the SPE  i psi_t = -(mu/2) lap psi + (1/mu) Phi psi,  lap Phi = 4 pi G rho,
 * rho = |psi|^2 + particles, mu = hbar_over_m (Eq. 1-2 PAPER.md:47-58 with |psi|^2 the mass density,
 * G6; Eq. 9-10 PAPER.md:96-103 when mu = 1).  wdm_create allocates with cudaMalloc on the current
 * device; wdm_create_ws carves everything out of caller memory (256-byte aligned, at least
 * wdm_workspace_bytes; must outlive the context).  *out is NULL on failure. */
int wdm_create(wdm_ctx **out, int N, double L, double hbar_over_m, double G, int dtype);
int wdm_create_ws(wdm_ctx **out, int N, double L, double hbar_over_m, double G, int dtype,
                  long long max_particles, void *workspace_dev, size_t workspace_bytes);
int wdm_destroy(wdm_ctx *ctx);

/* All later work of this context is enqueued on `cuda_stream` (a cudaStream_t, e.g.
 * torch.cuda.current_stream().cuda_stream; NULL = the legacy default stream).  The new stream is first made to
 * wait (event) for everything the context has already enqueued on the old one, so a change is always safe. */
int wdm_set_stream(wdm_ctx *ctx, void *cuda_stream);

/* Copy in the wave function, N^3 interleaved complex of the context dtype.  Marks Phi stale (G8). */
int wdm_set_psi(wdm_ctx *ctx, const void *psi_dev);
int wdm_set_psi_host(wdm_ctx *ctx, const void *psi_host);

/* Copy in n particles (n = 0 removes them).  Positions are wrapped into [-L/2, L/2) (G16).
 * mass_dev: n reals, or NULL for the equal mass `mass_scalar`.  Particle mass enters the Poisson
 * source through a cloud-in-cell deposit and particles feel the CIC-interpolated central-difference
 * gradient of the shared potential (Eq. 21; G11-G13).  A context made
 * by wdm_create_ws accepts at most its max_particles. */
int wdm_set_particles(wdm_ctx *ctx, long long n, const void *pos_dev, const void *vel_dev,
                      const void *mass_dev, double mass_scalar);
int wdm_set_particles_host(wdm_ctx *ctx, long long n, const void *pos_host, const void *vel_host,
                           const void *mass_host, double mass_scalar);

/* Advance nsteps kick-drift-kick steps of size dt (Eq. 17-18; Alg. 1 l.5-16
 * PAPER.md:247-267; particles: leapfrog KDK sharing dt, G14-G15).  nsteps >= 0; dt may be negative
 * (time reversal).  If Phi is stale it is first recomputed from the current (psi, x); nsteps = 0 does
 * only that.  After the call psi, x, v are at the same time level and Phi / rho are the ones consistent
 * with them -- as seen through every wdm_get_*: the closing half kicks of the last step (and its absorbing
 * layer) are kept pending and folded into the opening kick of the next wdm_step with the same dt, or applied
 * by the next call that reads the state, changes dt or changes a parameter (so a loop of wdm_step(1, dt)
 * costs no extra pass over psi).  Asynchronous: no host synchronisation. */
int wdm_step(wdm_ctx *ctx, int nsteps, double dt);

/* Whole user call with HOST buffers: copy psi in, wdm_step(nsteps, dt), copy psi out, synchronise. */
int wdm_run_host(wdm_ctx *ctx, const void *psi_in_host, int nsteps, double dt, void *psi_out_host);

/* Copy out (stream-ordered for *_dev; the *_host forms synchronise the stream before returning).
 * density  : |psi|^2 + CIC particle mass density, the Poisson source before mean removal (G22)
 * potential: zero-mean Phi (Eq. 23, k = 0 mode zeroed, G3)
 * particles: pos (wrapped) and vel, either may be NULL; particles come back in the caller's order. */
int wdm_get_psi(wdm_ctx *ctx, void *psi_out_dev);
int wdm_get_density(wdm_ctx *ctx, void *rho_out_dev);
int wdm_get_potential(wdm_ctx *ctx, void *phi_out_dev);
int wdm_get_particles(wdm_ctx *ctx, void *pos_out_dev, void *vel_out_dev);
int wdm_get_psi_host(wdm_ctx *ctx, void *psi_out_host);
int wdm_get_density_host(wdm_ctx *ctx, void *rho_out_host);
int wdm_get_potential_host(wdm_ctx *ctx, void *phi_out_host);
int wdm_get_particles_host(wdm_ctx *ctx, void *pos_out_host, void *vel_out_host);

/* Extra terms of the potential kick (generalised equation, Eq. 13-14) and the absorbing
 * layer (Eq. 22; Alg. 1 l.15-18).  All act inside the fused kick: no extra pass over psi.
 *   kappa        local self-interaction, V += kappa |psi|^2 (potential units, like Phi; any sign)
 *   phi_ext_dev  static external potential, N^3 reals in the layout of Phi, or NULL.  COPIED (stream-ordered) into
 *                library-owned memory (one cudaMalloc of N^3 reals on first use, also for wdm_create_ws contexts;
 *                WDM_ENOMEM if it fails): the caller may free or change its buffer once the stream has passed
 *                the call.  It is added to the Poisson
 *                potential (Phi_total = Phi_DM + Phi_ext): psi and the particles feel the sum, and
 *                wdm_get_potential returns the sum.
 *   absorb_alpha, absorb_nb   after every step psi *= exp(-alpha (b(x) + b(y) + b(z)) dt) with
 *                b(x) = 2 - tanh((x + L/2)/w) + tanh((x - L/2)/w), w = L/absorb_nb; alpha = 0: off.
 * Defaults: 0, NULL, 0.  Marks the potential stale (recomputed by the next step / get). */
int wdm_set_kick_terms(wdm_ctx *ctx, double kappa, const void *phi_ext_dev, double absorb_alpha, int absorb_nb);

/* Particle variants.  substeps >= 1: leapfrog sub-steps of dt/substeps per wave step, all in the
 * potential of the start of the step, the acceleration re-gathered at every new position; the half kicks that open
 * and close a wave step use the potentials of its two ends (substeps = 1 is the default scheme).  is_static != 0
 * (":particles_static"): the particles never move; their mass stays in the Poisson source.  Default: 1, 0. */
int wdm_set_particle_mode(wdm_ctx *ctx, int substeps, int is_static);

/* Mass-assignment / force-interpolation scheme of the particles ("interpolated from the grid to particle
 * positions", scheme not given; DESIGN reading G30).  order = 2: cloud-in-cell,
 * 8 nodes, weights (1 - f, f) per axis (default).  order = 3: triangular-shaped cloud, 27 nodes: with j the node
 * nearest to the particle and d in [-1/2, 1/2) its offset from it in cells, weights (1/2 - d)^2/2, 3/4 - d^2,
 * (1/2 + d)^2/2 on nodes j-1, j, j+1 per axis.  The same weights deposit the mass into the Poisson source and gather
 * the central-difference gradient of Eq. 21.  Any other order: WDM_EINVAL.  A change marks the
 * potential stale (recomputed by the next step / get).  wdm_get_assignment writes the current order to *order. */
int wdm_set_assignment(wdm_ctx *ctx, int order);
int wdm_get_assignment(wdm_ctx *ctx, int *order);

/* Arithmetic of the particle deposit.  0 (default): partial sums per chunk of 1024 sorted particles in shared memory
 * (complex64: 32-bit fixed point, one unit = 5e-7 of the chunk's largest particle mass / dx^3; complex128: double),
 * added to the mesh with floating-point atomics -- the sum over the particles of a node depends on their order, so the
 * coupled result is reproducible only to rounding (1e-7 relative in complex64).  1: every weight is rounded once to 64-bit fixed point (a power-of-two scale chosen from the
 * total particle mass) and accumulated with integer atomics: the mesh, hence the whole coupled run, is bit-identical from
 * run to run (a debugging mode: 8 bytes per cell of extra device memory, cudaMalloc'ed on first use -- WDM_ENOMEM if that
 * fails -- a conversion pass per step, and one host synchronisation per particle set).  Either way the deposit is the
 * cloud-in-cell / triangular-shaped-cloud sum of PAPER.md:314 (readings G12, G30).  Marks the potential stale. */
int wdm_set_deposit_mode(wdm_ctx *ctx, int deterministic);

/* Diagnostics of the current (time-level) state (Sect. 3.5-3.6), on demand: one reduction pass over
 * (psi, Phi) with the second-order central differences of Eq. 21 for K and Q, and three forward-only
 * axis sweeps (psi is read, nothing is written) for the spectral kinetic energy.  Synchronises the stream.
 * out_host must hold 12 doubles:
 *   [0] M = sum |psi|^2 dx^3       [1] max |psi|^2       [2] max |Phi_total|
 *   [3] V = sum |psi|^2 Phi dx^3 (as printed: no factor 1/2)
 *   [4] K = 1/2 sum |rho v|^2/rho dx^3, rho v = (hbar/m) Im(psi* grad psi)
 *   [5] Q = (hbar/m)^2/2 sum |grad sqrt(rho)|^2 dx^3   (Eq. 12 with its hbar^2/2m; reading G31)
 *   [6] dt_max of Eq. 26, without the safety factor
 *   [7] T = (hbar/m)^2/2 sum_k k^2 |psi~_k|^2 dx^3/N^3  (spectral kinetic energy; K + Q in the continuum limit)
 *   [8] W = V/2       [9] E = T + W, the energy the pure SPE conserves       [10], [11] reserved (0)
 * The potential is recomputed first if stale.  Particles do not enter (rho is the wave density). */
int wdm_get_diagnostics(wdm_ctx *ctx, double *out_host);

/* Diagnostics accumulated INSIDE the sweeps of a step, at no extra pass over the grid and no extra kernel launch
 * (SURVEY 8(f) rank 2): while switched on, wdm_step uses instantiations of its sweeps that also reduce what they have
 * in registers.  wdm_get_step_diagnostics returns, for the LAST step run,
 * the state between Eq. 18(c) and (d) -- psi_2 after the drift, before the closing half kick, the
 * Poisson source rho = |psi_2|^2 + particles and the potential just solved from it; synchronises the stream.
 * out_host must hold 8 doubles:
 *   [0] M = sum |psi_2|^2 dx^3, [1] max |psi_2|^2                      (density sweep; G > 0 only)
 *   [2] max |Phi_total|                                                 (complex-to-real sweep; G > 0 only)
 *   [3] T = T_x + T_y + T_z of psi_2, spectral: each axis sweep sums k_a^2 |F_a psi|^2 in its middle level (the other
 *       axes' drift factors have unit modulus, so T is the same before and after Eq. 18(b))
 *   [4] W = 1/2 sum rho Phi_grav dx^3 over the whole source, summed spectrally in the Green's-function sweep
 *   [5] T_x, [6] T_y, [7] T_z
 * E = T + W is the conserved energy of the pure SPE.  WDM_ESTATE until a step has run. */
int wdm_set_step_diagnostics(wdm_ctx *ctx, int on);
int wdm_get_step_diagnostics(wdm_ctx *ctx, double *out_host);

/* Instrumentation.  wdm_launch_count: kernels launched by this context so far.  With profiling on,
 * every kernel launch is bracketed by CUDA events on the context's stream;
 * wdm_kernel_stats synchronises and returns, for slot i < *n_inout, the kernel name, the number of
 * timed launches and their summed duration in ms, then resets the accumulators.
 * With WDM_NVTX=1 in the environment every launch is also wrapped in an NVTX range named like its slot
 * ("psi_sweep_z_kick", "poisson_z_green", "particle_cic_deposit", ...) for timeline tools. */
int wdm_launch_count(wdm_ctx *ctx, long long *count_out);
int wdm_set_profiling(wdm_ctx *ctx, int on);
int wdm_kernel_stats(wdm_ctx *ctx, int *n_inout, const char **names_out, long long *launches_out,
                     double *ms_out);

/* Text of the last error of this context (never NULL; valid until the next call on the context).
 * wdm_last_error(NULL) reports the last failure of wdm_create*. */
const char *wdm_last_error(const wdm_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* WDM_H */
