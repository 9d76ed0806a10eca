// kernels_ref.cuh -- one-thread-per-cell kernels (BVFDTD_FLAG_REFERENCE_KERNELS): the plain
// statement of S1-S4 on the device, used to cross-check the tiled kernels at sizes the CPU oracle
// cannot reach in reasonable time.  Same arithmetic as the tiled path, global loads only.
#pragma once
#include "device_params.hpp"

namespace bvfdtd {

#define BV_C1 1.125f
#define BV_C2 (-1.0f / 24.0f)

// D+ f(i) = [c1 (f(i+1)-f(i)) + c2 (f(i+2)-f(i-1))]/dx, lands on the half node i+1/2 (reading P1)
__device__ __forceinline__ float dplus(const float *__restrict__ f, long long c, long long s, float inv_dx) {
    return (BV_C1 * (f[c + s] - f[c]) + BV_C2 * (f[c + 2 * s] - f[c - s])) * inv_dx;
}
// D- f(i) = [c1 (f(i)-f(i-1)) + c2 (f(i+1)-f(i-2))]/dx, lands on the integer node i
__device__ __forceinline__ float dminus(const float *__restrict__ f, long long c, long long s, float inv_dx) {
    return (BV_C1 * (f[c] - f[c - s]) + BV_C2 * (f[c + s] - f[c - 2 * s])) * inv_dx;
}

// C-PML (reading P5): psi <- b psi + a D; D_eff = D + psi
__device__ __forceinline__ float cpml(float d, float *__restrict__ psi, long long q, float a, float b) {
    const float p = fmaf(b, psi[q], a * d);
    psi[q] = p;
    return d + p;
}

struct SlabIdx {
    bool in[3];
    long long q[3];
    int pos[3];
};

__device__ __forceinline__ SlabIdx slab_index(const Params &p, int i, int j, int k) {
    SlabIdx s;
    const int P = p.P;
    s.pos[0] = i; s.pos[1] = j; s.pos[2] = k;
    s.in[0] = (i < P) || (i >= p.nx - P);
    s.in[1] = (j < P) || (j >= p.ny - P);
    s.in[2] = (k < P) || (k >= p.nz - P);
    const int ix = i < P ? i : p.xp4 + (i - p.xhb);
    const int jy = j < P ? j : j - (p.ny - 2 * P);
    const int kz = k < P ? k : k - (p.nz - 2 * P);
    s.q[0] = ix + (long long)p.wx * (j + (long long)p.ny * k);
    s.q[1] = i + (long long)p.px * (jy + (long long)(2 * P) * k);
    s.q[2] = i + (long long)p.px * (j + (long long)p.ny * kz);
    return s;
}

// derivative along `axis` with its C-PML correction; term selects the psi array, half the profile
__device__ __forceinline__ float pml_term(const Params &p, const SlabIdx &s, int axis, int term, int half, float d) {
    if (!s.in[axis]) return d;
    const float a = __ldg(p.prof[axis][half ? 2 : 0] + s.pos[axis]);
    const float b = __ldg(p.prof[axis][half ? 3 : 1] + s.pos[axis]);
    return cpml(d, p.psi[axis * 6 + term], s.q[axis], a, b);
}

__device__ __forceinline__ void inject_cells(const Params &p, long long n_src, const long long *__restrict__ cell,
                                             const float *__restrict__ amp, const float *__restrict__ delay,
                                             int waveform, double f_src, int n_cycles, double t_n) {
    const long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (s >= n_src) return;
    const double t = t_n - (double)delay[s];
    if (t < 0.0) return;
    const double T = (double)n_cycles / f_src;
    double w;
    if (waveform == 0) {
        if (!(t < T)) return;
        w = sinpi(2.0 * f_src * t);
    } else {
        const double ramp = t < T ? 0.5 * (1.0 - cospi(t * f_src / (double)n_cycles)) : 1.0;
        w = ramp * sinpi(2.0 * f_src * t);
    }
    const float add = amp[s] * (float)w;
    const long long q = cell[s];
    const int i = (int)(q % p.nx), j = (int)((q / p.nx) % p.ny), k = (int)(q / ((long long)p.nx * p.ny));
    const long long c = p.org + i + (long long)p.px * j + p.sz * k;
    p.f[SXX][c] -= add;
    p.f[SYY][c] -= add;
    p.f[SZZ][c] -= add;
}

// S1 (reading P7): additive isotropic stress injection at t_n = n dt.
// The step index n is the host's `step`, or -- when the step is replayed from a CUDA graph, whose kernel
// arguments are frozen -- the device counter d_ctr[0], which the last block to finish advances by one
// (every block has read the counter before it can finish, so the update races with no reader).
__global__ void k_inject(Params p, long long n_src, const long long *__restrict__ cell,
                         const float *__restrict__ amp, const float *__restrict__ delay,
                         int waveform, double f_src, int n_cycles, double dt, long long step, long long *d_ctr) {
    if (d_ctr) {
        __shared__ long long s_step;
        if (threadIdx.x == 0) s_step = *reinterpret_cast<volatile long long *>(d_ctr);
        __syncthreads();
        step = s_step;
    }
    inject_cells(p, n_src, cell, amp, delay, waveform, f_src, n_cycles, (double)step * dt);
    if (d_ctr) {
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            unsigned int *done = reinterpret_cast<unsigned int *>(d_ctr + 1);
            if (atomicAdd(done, 1u) == gridDim.x - 1) {
                *done = 0u;
                *reinterpret_cast<volatile long long *>(d_ctr) = step + 1;
            }
        }
    }
}

// S2 (Eq. 1 rows 1-3; readings P1, P2, P4, P5)
__global__ void __launch_bounds__(256) k_velocity_ref(const Params p) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z * blockDim.z + threadIdx.z;
    if (i >= p.nx || j >= p.ny || k >= p.nz) return;
    const long long px = p.px, sz = p.sz;
    const long long cm = i + px * j + sz * k;
    const long long c = p.org + cm;
    const float idx = p.inv_dx;
    const SlabIdx s = slab_index(p, i, j, k);
    const float rho0 = p.rows[p.mat[cm]].rho;
    if (i < p.nx - 1) {
        const float d1 = pml_term(p, s, 0, 0, 1, dplus(p.f[SXX], c, 1, idx));
        const float d2 = pml_term(p, s, 1, 0, 0, dminus(p.f[SXY], c, px, idx));
        const float d3 = pml_term(p, s, 2, 0, 0, dminus(p.f[SXZ], c, sz, idx));
        const float rho = 0.5f * (rho0 + p.rows[p.mat[cm + 1]].rho);
        p.f[VX][c] += p.dt / rho * (d1 + d2 + d3);
    }
    if (j < p.ny - 1) {
        const float d1 = pml_term(p, s, 0, 1, 0, dminus(p.f[SXY], c, 1, idx));
        const float d2 = pml_term(p, s, 1, 1, 1, dplus(p.f[SYY], c, px, idx));
        const float d3 = pml_term(p, s, 2, 1, 0, dminus(p.f[SYZ], c, sz, idx));
        const float rho = 0.5f * (rho0 + p.rows[p.mat[cm + px]].rho);
        p.f[VY][c] += p.dt / rho * (d1 + d2 + d3);
    }
    if (k < p.nz - 1) {
        const float d1 = pml_term(p, s, 0, 2, 0, dminus(p.f[SXZ], c, 1, idx));
        const float d2 = pml_term(p, s, 1, 2, 0, dminus(p.f[SYZ], c, px, idx));
        const float d3 = pml_term(p, s, 2, 2, 1, dplus(p.f[SZZ], c, sz, idx));
        const float rho = 0.5f * (rho0 + p.rows[p.mat[cm + sz]].rho);
        p.f[VZ][c] += p.dt / rho * (d1 + d2 + d3);
    }
}

// shear node material (reading P2): harmonic mean of mu_R over the 4 cells (0 if any is fluid),
// arithmetic mean of tau_s
__device__ __forceinline__ void shear_node(const Params &p, int m0, int m1, int m2, int m3, float &mu_h, float &ts_h) {
    const KRow &a = p.rows[m0], &b = p.rows[m1], &c = p.rows[m2], &d = p.rows[m3];
    const float all_solid = a.solid * b.solid * c.solid * d.solid;
    const float sum_inv = (a.invMu + b.invMu) + (c.invMu + d.invMu);
    mu_h = all_solid != 0.0f ? 4.0f / sum_inv : 0.0f;
    ts_h = 0.25f * ((a.tauS + b.tauS) + (c.tauS + d.tauS));
}

// memory variable (Crank-Nicolson, reading P3 step 4) and stress: r' = A r - eR;
// s += eU + dt/2 (r' + r)   (eU already carries dt, eR already carries B = 2 beta/(1+beta))
__device__ __forceinline__ void sls(const Params &p, float *__restrict__ s, float *__restrict__ r, long long c, float eU, float eR) {
    const float r0 = r[c];
    const float rn = fmaf(p.A, r0, -eR);
    s[c] += eU + p.half_dt * (rn + r0);
    r[c] = rn;
}

// S3 + S4 (Eq. 1 rows 4-9; readings P1-P3, P5, P8)
__global__ void __launch_bounds__(256) k_stress_ref(const Params p) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z * blockDim.z + threadIdx.z;
    if (i >= p.nx || j >= p.ny || k >= p.nz) return;
    const long long px = p.px, sz = p.sz;
    const long long cm = i + px * j + sz * k;
    const long long c = p.org + cm;
    const float idx = p.inv_dx;
    const SlabIdx s = slab_index(p, i, j, k);
    const float *vx = p.f[VX], *vy = p.f[VY], *vz = p.f[VZ];

    const int m000 = p.mat[cm], m100 = p.mat[cm + 1], m010 = p.mat[cm + px], m110 = p.mat[cm + px + 1];
    const int m001 = p.mat[cm + sz], m101 = p.mat[cm + sz + 1], m011 = p.mat[cm + sz + px];

    const float vxx = pml_term(p, s, 0, 3, 0, dminus(vx, c, 1, idx));
    const float vyy = pml_term(p, s, 1, 4, 0, dminus(vy, c, px, idx));
    const float vzz = pml_term(p, s, 2, 5, 0, dminus(vz, c, sz, idx));
    const float th = vxx + vyy + vzz;
    const KRow row = p.rows[m000];
    const float vii[3] = {vxx, vyy, vzz};
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const float o = th - vii[q];
        sls(p, p.f[SXX + q], p.f[RXX + q], c, row.eP * th - row.eS * o, row.bP * th - row.bS * o);
    }
    float mu_h, ts_h, g;
    shear_node(p, m000, m100, m010, m110, mu_h, ts_h);
    g = pml_term(p, s, 1, 3, 1, dplus(vx, c, px, idx)) + pml_term(p, s, 0, 4, 1, dplus(vy, c, 1, idx));
    sls(p, p.f[SXY], p.f[RXY], c, p.dt * (mu_h * (1.0f + ts_h)) * g, p.B * (mu_h * ts_h) * g);
    shear_node(p, m000, m100, m001, m101, mu_h, ts_h);
    g = pml_term(p, s, 2, 3, 1, dplus(vx, c, sz, idx)) + pml_term(p, s, 0, 5, 1, dplus(vz, c, 1, idx));
    sls(p, p.f[SXZ], p.f[RXZ], c, p.dt * (mu_h * (1.0f + ts_h)) * g, p.B * (mu_h * ts_h) * g);
    shear_node(p, m000, m010, m001, m011, mu_h, ts_h);
    g = pml_term(p, s, 2, 4, 1, dplus(vy, c, sz, idx)) + pml_term(p, s, 1, 5, 1, dplus(vz, c, px, idx));
    sls(p, p.f[SYZ], p.f[RYZ], c, p.dt * (mu_h * (1.0f + ts_h)) * g, p.B * (mu_h * ts_h) * g);

    if (p.do_phasor) {
        const float pr = (p.f[SXX][c] + p.f[SYY][c] + p.f[SZZ][c]) * (-1.0f / 3.0f);
        p.phre[c] = fmaf(p.ph_cos, pr, p.phre[c]);
        p.phim[c] = fmaf(p.ph_sin, pr, p.phim[c]);
    } else if (p.do_peak | p.do_rms) {
        const float pr = (p.f[SXX][c] + p.f[SYY][c] + p.f[SZZ][c]) * (-1.0f / 3.0f);
        if (p.do_peak) p.peak[c] = fmaxf(p.peak[c], fabsf(pr));
        if (p.do_rms) p.sumsq[c] = fmaf(pr, pr, p.sumsq[c]);
    }
}

}  // namespace bvfdtd
