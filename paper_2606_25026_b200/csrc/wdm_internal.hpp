// wdm_internal.hpp -- interface between the host logic (wdm.cu) and the per-(dtype, N) sweep objects.
#pragma once
#include <cuda_runtime.h>

#include "wdm_plan.hpp"

namespace wdm {

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
};

const SweepTable *sweep_table(int dtype, int N);

}  // namespace wdm
