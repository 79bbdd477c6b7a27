// wdm_internal.hpp -- interface between the host logic (wdm.cu) and the per-(dtype, N) sweep objects.
#pragma once
#include <cuda_runtime.h>

#include "wdm_plan.hpp"

namespace wdm {

// completion counters of a chained launch: (stages - 1) x planes words, zeroed once, monotone across launches;
// `target` is the value a finished plane's counter has reached in this launch (epoch x tiles per plane)
struct ChainCtl {
    unsigned int *done;
    unsigned int target;
    int lag;
};

// Launchers of one (dtype, N) instantiation; params is a SweepParams<T> of the matching T.
struct SweepTable {
    Fact fact;
    int dtype;
    cudaError_t (*init)();                                               // opt in to > 48 KB dynamic shared memory
    // diag: 0 plain; 1 the instantiation that also accumulates the per-step diagnostics into params->diag; 2 (psi sweeps,
    // no kick) forward transform only, sum k^2 |F psi|^2 into params->diag, nothing written
    cudaError_t (*psi_z)(const void *params, int kick, int diag, cudaStream_t);    // contiguous axis, optional kick on load
    cudaError_t (*psi_strided)(const void *params, int along_x, int diag, cudaStream_t);  // y axis (or x axis when G = 0)
    cudaError_t (*psi_x_rho)(const void *params, int drift, int diag, cudaStream_t);  // x axis + density + R2C -> H
    cudaError_t (*h_y_fwd)(const void *params, cudaStream_t);
    cudaError_t (*h_z_green)(const void *params, int diag, cudaStream_t);
    cudaError_t (*h_y_inv)(const void *params, cudaStream_t);
    cudaError_t (*c2r)(const void *params, int diag, cudaStream_t);
    // L2-chained forms (wdm_chain.cuh): z then y sweep of psi by x-planes; y forward, z Green, y inverse of H by
    // kx-planes.  chain_lag(stages, planes, requested) returns the lag to use (requested <= 0: automatic) or 0 when
    // no lag is both safe and meaningful for this size -- then the separate sweeps above must be used.
    int (*chain_lag)(int stages, int planes, int requested);
    cudaError_t (*psi_zy)(const void *params_z, const void *params_y, int kick, const ChainCtl *, cudaStream_t);
    cudaError_t (*h_yzy)(const void *params_y, const void *params_z, const ChainCtl *, cudaStream_t);
};

const SweepTable *sweep_table(int dtype, int N);

}  // namespace wdm
