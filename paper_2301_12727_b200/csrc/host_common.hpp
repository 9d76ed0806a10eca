// host_common.hpp -- what the translation units of the C ABI share on the host side: the CUDA
// error record behind bvfdtd_last_cuda_error().
#pragma once
#include <cuda_runtime.h>

namespace bvfdtd {

// records "what: cuda error string" for bvfdtd_last_cuda_error(), clears the sticky error, returns BVFDTD_ECUDA
int cuda_fail(cudaError_t e, const char *what);

}  // namespace bvfdtd

#define CU(call)                                                      \
    do {                                                              \
        cudaError_t e__ = (call);                                     \
        if (e__ != cudaSuccess) return ::bvfdtd::cuda_fail(e__, #call); \
    } while (0)
