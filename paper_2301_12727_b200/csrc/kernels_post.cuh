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

// NEXT-3, second half ("corrected phase programming of the transducer elements"): one CTA
// per element sums the back-propagated complex field over the element's surface points (fp64, fixed
// order) and writes E_m, the unit time-reversal weight conj(E_m)/|E_m| and the delay arg(E_m)/w in
// [0, 1/f).  An element that received nothing keeps the weight 1 and the delay 0.
__global__ void __launch_bounds__(128) k_element_phase(const int n_pts, const float *__restrict__ p_re, const float *__restrict__ p_im,
                                                       const int *__restrict__ element, const float inv_omega,
                                                       float2 *__restrict__ unit, float *__restrict__ delay, float2 *__restrict__ E) {
    __shared__ double sre[128], sim[128];
    const int m = blockIdx.x;
    double ar = 0.0, ai = 0.0;
    for (int q = threadIdx.x; q < n_pts; q += blockDim.x)
        if (element[q] == m) { ar += (double)p_re[q]; ai += (double)p_im[q]; }
    sre[threadIdx.x] = ar; sim[threadIdx.x] = ai;
    __syncthreads();
    for (int s = 64; s > 0; s >>= 1) {
        if (threadIdx.x < s) { sre[threadIdx.x] += sre[threadIdx.x + s]; sim[threadIdx.x] += sim[threadIdx.x + s]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double re = sre[0], im = sim[0], mag = sqrt(re * re + im * im);
        if (E) E[m] = make_float2((float)re, (float)im);
        if (mag > 0.0) {
            unit[m] = make_float2((float)(re / mag), (float)(-im / mag));
            const float two_pi = 6.283185307179586f;
            float phi = atan2f((float)im, (float)re);
            phi -= two_pi * floorf(phi / two_pi);
            delay[m] = phi * inv_omega;
        } else {
            unit[m] = make_float2(1.0f, 0.0f);
            delay[m] = 0.0f;
        }
    }
}

// weight of every surface point: u0 * area * conj(E_m)/|E_m| of its element
__global__ void __launch_bounds__(128) k_point_weights(const int n_pts, const int *__restrict__ element, const float *__restrict__ area,
                                                       const float2 *__restrict__ unit, const float u0, float2 *__restrict__ w_pts) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n_pts) return;
    const float2 u = unit[element[q]];
    const float a = u0 * area[q];
    w_pts[q] = make_float2(a * u.x, a * u.y);
}

}  // namespace bvfdtd
