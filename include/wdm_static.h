/*
 * wdm_static.h -- one entry point of libwdm.so that ALLOCATES NOTHING: the particle mass deposit (cloud-in-cell, or
 * triangular-shaped cloud) onto the Poisson mesh, "N-body particles coupled through the shared
 * potential" / readings G12-G13 and G30 of DESIGN.md, in the bit-reproducible 64-bit fixed-point arithmetic of
 * wdm_set_deposit_mode(ctx, 1) (include/wdm.h).
 *
 * Why: a wdm_ctx takes its memory from cudaMalloc (or a caller workspace) and the deterministic deposit cudaMallocs its
 * accumulator mesh on first use.  Callers that cannot allocate -- code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc -- get this call instead: its only scratch, the fixed-point accumulator mesh, is a
 * file-scope `static __device__` array inside the library,
 *
 *     WDM_STATIC_MAX_CELLS = 64^3 cells x 8 bytes = 2 MiB,
 *
 * which every GPU that loads libwdm.so holds until the process exits.  The call performs no cudaMalloc, cudaFree or
 * allocating library call: a 2 MiB cudaMemsetAsync of the scratch (it keeps the last call's contents, so what must
 * start at zero is cleared every time), one deposit kernel, one conversion kernel, all on the caller's stream.
 *
 * ALL CALLS ON ONE GPU SHARE THE ARRAY.  Calls that overlap on the GPU (different streams, different threads or
 * contexts of one process) race on it and give wrong densities; calls on one stream, or ordered by events, are safe.
 * The CUDA device that owns the pointers and the stream must be current in the calling thread.
 */
#ifndef WDM_STATIC_H
#define WDM_STATIC_H

#include <stddef.h>

#include "wdm.h"

#ifdef __cplusplus
extern "C" {
#endif

#define WDM_STATIC_MAX_N 64                              /* largest mesh edge the static scratch holds */
#define WDM_STATIC_MAX_CELLS (64ull * 64ull * 64ull)     /* words of the accumulator mesh              */

/*
 * rho_out[x][y][z] (N^3 reals, z contiguous, OVERWRITTEN -- every cell is written, cells without mass get 0) = mass
 * density of n particles on the periodic mesh of the box [-L/2, L/2)^3, cell size L / N, assignment scheme `order`
 * (2: cloud-in-cell, 3: triangular-shaped cloud), exactly as the coupled step deposits it in deterministic mode.
 *
 *   pos_dev     (n, 3) reals, DEVICE, positions inside [-L/2, L/2) (positions outside are wrapped by the periodic mesh
 *               index only as far as the assignment stencil reaches: wrap them first)
 *   mass_dev    n reals, DEVICE, per-particle masses -- or NULL: every particle has mass mass_scalar
 *   total_mass  an upper bound of sum |m_i| (> 0, finite): fixes the fixed-point scale, a power of two such that the sum
 *               of everything fits in 62 bits.  The same bound gives the same bits; |mass_scalar| * n is what the coupled
 *               step uses for equal masses.
 *   dtype       WDM_C64: reals are float; WDM_C128: reals are double (the precision the matching wdm_ctx works in)
 *   rho_out_dev N^3 reals, DEVICE, owned by the caller
 *   cuda_stream a cudaStream_t (NULL: the default stream); the call is asynchronous on it
 *
 * Errors: WDM_EINVAL (null pointer, n < 0, L <= 0, bad dtype / order / total_mass), WDM_EUNSUPPORTED (N not a power of two
 * in [8, WDM_STATIC_MAX_N]: "N^3 cells exceed the static scratch"), WDM_ECUDA (a CUDA call failed).  The text is in
 * wdm_static_last_error() (per thread).  Nothing is launched when an error is returned before the first kernel.
 */
int wdm_deposit_static(const void *pos_dev, const void *mass_dev, double mass_scalar, long long n, int N, double L,
                       int dtype, int order, double total_mass, void *rho_out_dev, void *cuda_stream);

/* Bytes of the static scratch (WDM_STATIC_MAX_CELLS * 8); no GPU needed. */
size_t wdm_static_scratch_bytes(void);

const char *wdm_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* WDM_STATIC_H */
