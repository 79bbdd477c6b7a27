/*
 * wdm_dist.h -- C ABI of the slab-decomposed (multi-GPU) form of the kick-drift-kick step of libwdm.so.
 *
 * NOT the path BASELINE.json's north_star names (that one is single-GPU, include/wdm.h): this is SURVEY.md 8(f) rank 4,
 * what the paper lists as future work ("distributed FFT requires MPI support, planned").  Pure SPE
 * (Eq. 18 PAPER.md:187-200 with the plain potential kick; no particles, no extra kick terms).
 *
 * One process per GPU, world ranks, N divisible by world; rank r owns the x-planes [r N/world, (r+1) N/world).  The
 * library runs every kernel of the path -- the single-GPU sweeps on slab-shaped arrays plus pack / unpack copies -- and
 * performs NO communication: a step is a fixed program of PHASES; after each phase the caller exchanges, all-to-all,
 * *exchange_bytes_per_peer bytes per peer from the send buffer (block d goes to rank d) into the recv buffer (block s
 * comes from rank s) -- e.g. torch.distributed.all_to_all_single over NCCL -- when that value is non-zero.  All ranks
 * run the same phases in the same order.  (The tests drive several contexts on ONE GPU and do the exchange with
 * device-to-device copies; no phase ever waits on another rank's kernel.)
 *
 *   after wdm_dist_set_psi:   s = wdm_dist_local_sum; all-reduce s; wdm_dist_set_mean(sum / N^3);
 *                             WDM_DIST_R1, R2, R3, R4                     (potential of the initial state; reading G8)
 *   wdm_step(nsteps, dt):     for each step: S1 (kick_dt = dt/2 in the first step of a call, dt afterwards: merged kicks,
 *                             reading G21), S2, S3, S4, S5; then WDM_DIST_KICK with kick_dt = dt/2 (closing half kick)
 *   reading psi:              G1, G2, then wdm_dist_get_psi
 *
 * Layouts (z contiguous, complex interleaved as in wdm.h): psi slabs are [N/world][N][N] = this rank's x-planes.  The
 * potential is returned in the library's transposed form Phi^T[y_l][x][z], y_l = this rank's y-rows [r N/world, ...).
 * Pointers are DEVICE pointers; every call returns a WDM_* code of wdm.h.
 */
#ifndef WDM_DIST_H
#define WDM_DIST_H

#include <stddef.h>

#include "wdm.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wdm_dist wdm_dist;

enum {
    WDM_DIST_R1 = 0, WDM_DIST_R2 = 1, WDM_DIST_R3 = 2, WDM_DIST_R4 = 3,   /* refresh: Phi from the current psi        */
    WDM_DIST_S1 = 4, WDM_DIST_S2 = 5, WDM_DIST_S3 = 6, WDM_DIST_S4 = 7, WDM_DIST_S5 = 8, /* one step                 */
    WDM_DIST_KICK = 9,                                                    /* psi *= exp(-i Phi kick_dt / mu)          */
    WDM_DIST_G1 = 10, WDM_DIST_G2 = 11                                    /* bring psi back to x-planes for a getter  */
};

/* N a power of two in [8, 1024], world dividing N (else WDM_EUNSUPPORTED); allocates with cudaMalloc on the current
 * device: about 5.5 N^3 / world complex elements. */
int wdm_dist_create(wdm_dist **out, int N, double L, double hbar_over_m, double G, int dtype, int rank, int world);
int wdm_dist_destroy(wdm_dist *d);
int wdm_dist_set_stream(wdm_dist *d, void *cuda_stream);

/* Size each of the two exchange buffers must have; the caller owns them (they must stay valid while set). */
int wdm_dist_exchange_bytes(wdm_dist *d, size_t *bytes_out);
int wdm_dist_set_buffers(wdm_dist *d, void *send_dev, void *recv_dev);

/* This rank's x-planes of psi, copied in; the potential becomes stale. */
int wdm_dist_set_psi(wdm_dist *d, const void *psi_xslab_dev);
/* sum |psi|^2 over this rank's slab (synchronises); global mean density = (sum over ranks) / N^3, subtracted from the
 * Poisson source (Eq. 23; reading G3). */
int wdm_dist_local_sum(wdm_dist *d, double *sum_out);
int wdm_dist_set_mean(wdm_dist *d, double mean_density);

/* Run the local kernels of one phase (asynchronous on the context's stream).  dt: the step (kinetic phase of Eq. 18(b));
 * kick_dt: the potential-kick interval of S1 / KICK.  *exchange_bytes_per_peer: see above. */
int wdm_dist_phase(wdm_dist *d, int phase, double dt, double kick_dt, size_t *exchange_bytes_per_peer);

int wdm_dist_get_psi(wdm_dist *d, void *psi_xslab_out_dev);
int wdm_dist_get_potential_t(wdm_dist *d, void *phi_t_out_dev);

/* Index map of a pack / unpack copy (host logic, no GPU needed; for tests): op 0..7 = psi T->x pack, unpack, psi x->T
 * pack, unpack, H T->kx pack, unpack, H kx->T pack, unpack.  out12 = n0, n1, n2, s0, s1, s2, d0, d1, d2, kmul, ksel, klim:
 * destination line i0 d0 + i1 d1 + i2 d2 <- source line i0 s0 + i1 s1 + i2 s2 (a line = N complex), skipped where
 * kmul > 0 and i0 kmul + i[ksel] >= klim. */
int wdm_dist_copy_plan(int N, int world, int op, long long *out12);

const char *wdm_dist_last_error(const wdm_dist *d);

#ifdef __cplusplus
}
#endif
#endif /* WDM_DIST_H */
