// kernels_tiled.cuh -- placeholder while the boundary is brought up: forwards to the per-cell kernels.
#pragma once
#include <cuda_runtime.h>

#include "device_params.hpp"
#include "kernels_ref.cuh"

namespace bvfdtd {

struct TiledPlan {
    int dummy = 0;
};

inline const char *tiled_plan_error() { return ""; }
inline int tiled_plan_create(TiledPlan &, const Layout &, const Params &) { return 0; }
inline void tiled_plan_destroy(TiledPlan &) {}
inline int tiled_velocity(TiledPlan &, const Params &p, cudaStream_t st) {
    const dim3 b(32, 4, 2), g((p.nx + 31) / 32, (p.ny + 3) / 4, (p.nz + 1) / 2);
    k_velocity_ref<<<g, b, 0, st>>>(p);
    return 0;
}
inline int tiled_stress(TiledPlan &, const Params &p, cudaStream_t st) {
    const dim3 b(32, 4, 2), g((p.nx + 31) / 32, (p.ny + 3) / 4, (p.nz + 1) / 2);
    k_stress_ref<<<g, b, 0, st>>>(p);
    return 0;
}

}  // namespace bvfdtd
