// wdm_internal.hpp -- interface between the host logic (wdm.cu) and the per-(dtype, N) sweep objects.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "wdm_plan.hpp"

namespace wdm {

// Launchers of one (dtype, N) instantiation; params is a SweepParams<T> of the matching T.
struct SweepTable {
    Fact fact;
    int dtype;
    int c2r_w;
    int x2_w;                                                            // 0, or the lines per tile of the half-tile x sweeps (wdm_x2.cuh): the host then supplies their tables and boxes                                                           // lines per tile of the complex-to-real sweep (fact.W unless that sweep runs in place)
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
    // slab-decomposed runs (wdm_dist.cu): ntiles tiles of a slab-shaped array; x is the middle index of psi^T, H^T, Phi^T
    cudaError_t (*dist_init)();
    cudaError_t (*dist_psi_z)(const void *params, int kick, int ntiles, cudaStream_t);
    cudaError_t (*dist_psi_y)(const void *params, int ntiles, cudaStream_t);
    cudaError_t (*dist_psi_x_rho)(const void *params, int drift, int ntiles, cudaStream_t);
    cudaError_t (*dist_h_y)(const void *params, int inverse, int ntiles, cudaStream_t);
    cudaError_t (*dist_h_z_green)(const void *params, int ntiles, cudaStream_t);
    cudaError_t (*dist_c2r)(const void *params, int ntiles, cudaStream_t);
};

const SweepTable *sweep_table(int dtype, int N);

// TMA descriptor of a complex array [nx][ny][N] (z contiguous): boxes of W complex elements along z by `rows` points along
// axis 1 (the middle index) or 2 (the outer index).  Encoded in units of one real (float / double), no swizzle, no
// interleave: the box lands in shared memory as dense [row][W] -- the strided tile layout.  Returns 0, -1 when the
// driver entry point is missing, else the CUresult.
inline int encode_tmap(int dtype, int N, int W, void *base, int ny, int nx, int axis, int rows, CUtensorMap *out)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
        if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn) return -1;
        encode = (encode_fn)fn;
    }
    const size_t r = dtype == 0 ? 4 : 8;
    cuuint64_t dims[3] = {2 * (cuuint64_t)N, (cuuint64_t)ny, (cuuint64_t)nx};
    cuuint64_t strides[2] = {2 * (cuuint64_t)N * r, 2 * (cuuint64_t)N * (cuuint64_t)ny * r};
    cuuint32_t box[3] = {(cuuint32_t)(2 * W), axis == 1 ? (cuuint32_t)rows : 1u, axis == 2 ? (cuuint32_t)rows : 1u};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult res = encode(out, dtype == 0 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, dims,
                          strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                          CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return res == CUDA_SUCCESS ? 0 : (int)res;
}

}  // namespace wdm
