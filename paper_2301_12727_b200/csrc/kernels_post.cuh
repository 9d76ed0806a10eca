// kernels_post.cuh -- reductions that follow the FDTD run.
//
// PAPER.md:L107-L110 (Eq. 2): E_L = sum_xy I_PA-brain(x,y,z_m) / sum_xy I_PA-water(x,y,z_m) on the plane
// z_m "where water conditions show the maximal intensity"; L164: T_S = sqrt(E_L).  Reading (DESIGN.md
// section 11): I_PA(cell) = rms_amp^2 / (2 rho c_L) = sumsq / (count rho c_L) with the cell's own
// table values; sums and maxima run over the cells outside the PML mask.
#pragma once
#include "device_params.hpp"

namespace bvfdtd {

// One CTA per z plane: fp32 intensity per cell, fp64 accumulation in a fixed order (deterministic).
// out[k] = plane sum, out[nz + k] = plane maximum; planes inside the z slabs give 0.
__global__ void __launch_bounds__(256) k_plane_intensity(const Params p, const float *__restrict__ inv_z, const float inv_count,
                                                         double *__restrict__ out) {
    __shared__ double ssum[256];
    __shared__ double smax[256];
    const int k = blockIdx.x, P = p.P;
    double acc = 0.0, mx = 0.0;
    if (k >= P && k < p.nz - P) {
        const int wx = p.nx - 2 * P, wy = p.ny - 2 * P;
        for (int q = threadIdx.x; q < wx * wy; q += blockDim.x) {
            const int i = P + q % wx, j = P + q / wx;
            const long long cm = i + (long long)p.px * j + p.sz * k;
            const float I = p.sumsq[p.org + cm] * inv_count * __ldg(inv_z + p.mat[cm]);
            acc += (double)I;
            mx = fmax(mx, (double)I);
        }
    }
    ssum[threadIdx.x] = acc; smax[threadIdx.x] = mx;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) {
            ssum[threadIdx.x] += ssum[threadIdx.x + s];
            smax[threadIdx.x] = fmax(smax[threadIdx.x], smax[threadIdx.x + s]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[k] = ssum[0]; out[p.nz + k] = smax[0]; }
}

// NEXT-4: heat deposition of the harmonic field, Q = coef[material] * sumsq with
// coef = scale a 2 alphaL / (count rho cL) folded on the host; dense x-fastest output.
__global__ void __launch_bounds__(128) k_heat_source(const Params p, const float *__restrict__ coef, float *__restrict__ Q) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= p.nx) return;
    const long long cm = i + (long long)p.px * j + p.sz * k;
    Q[i + (long long)p.nx * (j + (long long)p.ny * k)] = __ldg(coef + p.mat[cm]) * p.sumsq[p.org + cm];
}

}  // namespace bvfdtd
