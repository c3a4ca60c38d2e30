// gdrr_denoise_scatter_static (include/gdrr.h): the denoiser with its scratch image in a file-scope __device__ array
// (denoise.cu).  A header of its own: gdrr_internal.h is part of every sampling kernel's source stamp
// (profiles/ncu_constants.json) and does not change for this.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace gdrr {

// = GDRR_DENOISE_STATIC_MAX_FLOATS of include/gdrr.h (gdrr_api.cu asserts it)
constexpr size_t kDenoiseStaticFloats = (size_t)4 << 20;

cudaError_t launch_denoise_static(const float* s_hat, float* s_dev, int nu, int nv, int n_images, double beta, double omega,
                                  int n_iter, double floor_value, cudaStream_t st, int* launches);

}  // namespace gdrr
