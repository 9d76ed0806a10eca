// kernels_rs.cuh -- Rayleigh-Sommerfeld integral of a surface-decomposed transducer (SURVEY.md 8(f)
// NEXT-1).  PAPER.md:L95: "The selected transducer is modeled by numerical surface decomposition with
// surface elements of an area of lambda^2/16 ... The acoustic field is first calculated with a
// GPU-accelerated implementation of the Rayleigh-Sommerfeld equation [45] over the incident interface
// of the simulation domain, with the coupling medium modeled as water."
//
// Reading (the paper gives no formula): first Rayleigh integral of a baffled
// source with normal surface velocity u_s on elements of area A_s, e^{+j w t} convention,
//     P(r) = (j rho c k / 2 pi) sum_s u_s A_s exp(-j k R_s) / R_s,   R_s = |r - r_s|.
// One thread per receiver; the sources stream through shared memory in tiles.  SFU bound: per
// (source, receiver) pair one MUFU.RSQ and, after an explicit reduction of the phase to one turn
// (k R / 2 pi = R / lambda, minus its nearest integer: no slow path for large arguments), one
// MUFU.SIN and one MUFU.COS, plus ~20 FMA-class instructions; fp32; the sum is accumulated per
// receiver in a fixed order.
#pragma once
#include <cuda_runtime.h>

namespace bvfdtd {

constexpr int RS_TILE = 1024;

__device__ __forceinline__ float rs_rsqrt(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rs_sin(float x) { float r; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rs_cos(float x) { float r; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// src: n_src x (x, y, z, 0) and weight: n_src x (Re, Im) of u_s A_s;  rcv: n_rcv x (x, y, z)
__global__ void __launch_bounds__(128) k_rayleigh(const int n_src, const float4 *__restrict__ src, const float2 *__restrict__ wgt,
                                                  const int n_rcv, const float *__restrict__ rcv, const float k, const float pref,
                                                  const float omega, float *__restrict__ p_re, float *__restrict__ p_im,
                                                  float *__restrict__ amp, float *__restrict__ delay) {
    __shared__ float4 spos[RS_TILE];
    __shared__ float2 sw[RS_TILE];
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = r < n_rcv;
    float x = 0.0f, y = 0.0f, z = 0.0f;
    if (live) { x = rcv[3 * r]; y = rcv[3 * r + 1]; z = rcv[3 * r + 2]; }
    float ar = 0.0f, ai = 0.0f;
    const float inv_lambda = k * 0.15915494309189535f;
    for (int s0 = 0; s0 < n_src; s0 += RS_TILE) {
        const int n = min(RS_TILE, n_src - s0);
        __syncthreads();
        for (int q = threadIdx.x; q < n; q += blockDim.x) { spos[q] = src[s0 + q]; sw[q] = wgt[s0 + q]; }
        __syncthreads();
        if (live) {
#pragma unroll 4
            for (int q = 0; q < n; ++q) {
                const float4 s = spos[q];
                const float dx = x - s.x, dy = y - s.y, dz = z - s.z;
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                const float ir = r2 > 0.0f ? rs_rsqrt(r2) : 0.0f;   // a receiver ON a source point: that pair adds nothing
                const float turns = (r2 * ir) * inv_lambda;                 // k R / 2 pi
                const float ph = -6.283185307179586f * (turns - rintf(turns));   // -k R reduced to [-pi, pi]
                const float sn = rs_sin(ph), cs = rs_cos(ph);
                const float2 w = sw[q];
                ar = fmaf(fmaf(w.x, cs, -w.y * sn), ir, ar);
                ai = fmaf(fmaf(w.x, sn, w.y * cs), ir, ai);
            }
        }
    }
    if (!live) return;
    // multiply by j * pref
    const float re = -pref * ai, im = pref * ar;
    p_re[r] = re; p_im[r] = im;
    if (amp) {
        // P = |P| e^{j phi}: p(t) = |P| cos(w t + phi) = |P| sin(w (t - d)) with d = -(phi + pi/2) / w (mod one period)
        const float phi = atan2f(im, re);
        const float two_pi = 6.283185307179586f;
        float a = -(phi + 1.5707963267948966f);
        a -= two_pi * floorf(a / two_pi);
        amp[r] = sqrtf(re * re + im * im);
        delay[r] = a / omega;
    }
}

// MUFU throughput probe: the roofline denominator of k_rayleigh is measured, not assumed.  Every thread runs
// four independent chains of sin.approx (1024 threads x 2 blocks per SM hide the latency); ops = 4 * iters per thread.
__global__ void __launch_bounds__(1024) k_mufu_probe(float *__restrict__ out, const int iters) {
    float a0 = threadIdx.x * 1e-3f, a1 = a0 + 0.25f, a2 = a0 + 0.5f, a3 = a0 + 0.75f;
    for (int i = 0; i < iters; ++i) { a0 = rs_sin(a0); a1 = rs_sin(a1); a2 = rs_sin(a2); a3 = rs_sin(a3); }
    if (a0 + a1 + a2 + a3 == 12345.0f) out[0] = a0;     // keeps the chains alive
}

}  // namespace bvfdtd
