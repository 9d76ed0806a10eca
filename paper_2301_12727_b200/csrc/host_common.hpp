// host_common.hpp -- what the translation units of the C ABI share on the host side: the CUDA
// error record behind bvfdtd_last_cuda_error() and the device guard of the entry points.
#pragma once
#include <cuda_runtime.h>

namespace bvfdtd {

// records "what: cuda error string" for bvfdtd_last_cuda_error(), clears the sticky error, returns BVFDTD_ECUDA
int cuda_fail(cudaError_t e, const char *what);

// Makes `dev` the calling thread's current device for the lifetime of the object and restores the
// previous one afterwards: every entry point of a context runs on the device that owns the context's
// workspace, whatever device is current in the caller (a context created on cuda:1 is usable while
// cuda:0 is current).
struct DeviceScope {
    int prev = -1;
    bool switched = false;
    explicit DeviceScope(int dev) {
        if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceScope() {
        if (switched) cudaSetDevice(prev);
    }
    DeviceScope(const DeviceScope &) = delete;
    DeviceScope &operator=(const DeviceScope &) = delete;
};

// ordinal of the device that owns a device pointer (-1 when the query fails or the pointer is not device memory)
inline int device_of(const void *d_ptr) {
    cudaPointerAttributes a{};
    if (!d_ptr || cudaPointerGetAttributes(&a, d_ptr) != cudaSuccess) { (void)cudaGetLastError(); return -1; }
    return (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) ? a.device : -1;
}

}  // namespace bvfdtd

#define CU(call)                                                      \
    do {                                                              \
        cudaError_t e__ = (call);                                     \
        if (e__ != cudaSuccess) return ::bvfdtd::cuda_fail(e__, #call); \
    } while (0)
