// kernels_bhte.cuh -- thermal step.
//
// Pennes bio-heat equation, forward Euler, conservative 7-point stencil on the cell grid, series
// (harmonic) face conductivity, cells on the six borders held at T_b, CEM43 dose and running maximum
// accumulated with the temperature reached at the end of the step (readings: DESIGN.md section 10).
//
// The state is the temperature RISE th = T - T_b in fp32 (an increment of 1e-3 K per step keeps 7
// digits instead of the 3 it would keep next to 37), ping-ponged between two buffers.
//
// HBM-bound: per cell-step th read + write, Q read, dose read + write, material byte, (+ maximum
// read + write) = 21 (29) B.  One CTA = a 64 x 16 column of cells marched along a z chunk: a thread
// owns 4 consecutive x cells (float4), keeps its own column's planes k-1, k, k+1 in registers, takes
// the x neighbours by shuffles inside its 16-lane row (edge lanes load one scalar) and the y
// neighbours as float4 loads that hit L1/L2 (the rows belong to the warps next door).  Where the
// whole neighbourhood of a warp's cells is one material (water, brain: most of a head) every face
// mean is k itself and the warp takes a path with no table look-ups or reciprocals per face.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace bvfdtd {

struct BhteParams {
    int nx, ny, nz, px;        // px = row pitch in cells (multiple of 64)
    int sz;                    // plane stride px * ny
    int zlen;                  // planes per z chunk
    int n_mat;
    const float *th_in;        // rise at step n
    float *th_out;             // rise at step n + 1
    const float *Q;            // W/m^3
    float *dose;               // CEM43, minutes
    float *tmax;               // running maximum of the rise (nullptr when not tracked)
    const uint8_t *mat;        // material index, same pitch
    const float4 *tab;         // per material: 1/k, dt/(rho C dx^2), dt w/(rho C), dt/(rho C)
    float hs;                  // heat scale of this step (duty cycle; 0 = ultrasound off)
    float d43;                 // T_b - 43
    float dose_dt;             // dt / 60
};

namespace bhte_detail {
constexpr int TX = 64, TY = 16, NT = 256;

__device__ __forceinline__ float4 ld4(const float *base, int idx) { return __ldg(reinterpret_cast<const float4 *>(base + idx)); }
__device__ __forceinline__ uint32_t ldm(const uint8_t *base, int idx) { return __ldg(reinterpret_cast<const uint32_t *>(base + idx)); }
__device__ __forceinline__ float rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float ex2(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
// series mean of two conductivities given their inverses: 2 / (1/ka + 1/kb)
__device__ __forceinline__ float kface(float ia, float ib) { return 2.0f * rcp(ia + ib); }
__device__ __forceinline__ float4 inv_k(const float4 *tab, uint32_t m4) {
    return make_float4(tab[m4 & 255u].x, tab[(m4 >> 8) & 255u].x, tab[(m4 >> 16) & 255u].x, tab[m4 >> 24].x);
}
}  // namespace bhte_detail

template <bool TMAX>
__global__ void __launch_bounds__(bhte_detail::NT, 4) k_bhte(const BhteParams p) {
    using namespace bhte_detail;
    __shared__ float4 tab[256];
    const int tid = threadIdx.x;
    tab[tid] = tid < p.n_mat ? p.tab[tid] : make_float4(1.0f, 0.0f, 0.0f, 0.0f);
    __syncthreads();

    const int l16 = tid & 15;
    const int i0 = blockIdx.x * TX + 4 * l16;
    const int jr = blockIdx.y * TY + (tid >> 4);
    const int j = min(jr, p.ny - 1);
    const bool store = jr < p.ny && i0 < p.nx;
    const int k0 = blockIdx.z * p.zlen, k1 = min(k0 + p.zlen, p.nz);
    if (k0 >= k1) return;
    const bool yborder = (j == 0) || (j == p.ny - 1);
    // neighbours outside the box are only ever used by border cells, whose result is discarded: clamp
    const int oc = i0 + p.px * j, oym = i0 + p.px * max(j - 1, 0), oyp = i0 + p.px * min(j + 1, p.ny - 1);
    const int oxl = max(i0 - 1, 0) + p.px * j, oxr = min(i0 + 4, p.nx - 1) + p.px * j;
    // bit c set: cell c of the quad is NOT held (strictly inside the box in x and y)
    uint32_t free_xy = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) free_xy |= ((i0 + c > 0) && (i0 + c < p.nx - 1) && !yborder) ? (1u << c) : 0u;

    const int km = max(k0 - 1, 0);
    float4 th_m = ld4(p.th_in, oc + p.sz * km);
    float4 th_c = ld4(p.th_in, oc + p.sz * k0);
    uint32_t mm = ldm(p.mat, oc + p.sz * km);
    uint32_t mc = ldm(p.mat, oc + p.sz * k0);

    for (int k = k0; k < k1; ++k) {
        const int kp = min(k + 1, p.nz - 1);
        const int zo = p.sz * k;
        // ---- every load of the plane, issued together ----
        const float4 th_p = ld4(p.th_in, oc + p.sz * kp);
        const uint32_t mp = ldm(p.mat, oc + p.sz * kp);
        const float4 t_ym = ld4(p.th_in, oym + zo), t_yp = ld4(p.th_in, oyp + zo);
        const uint32_t m_ym = ldm(p.mat, oym + zo), m_yp = ldm(p.mat, oyp + zo);
        const float4 q4 = ld4(p.Q, oc + zo);
        const float4 d4 = ld4(p.dose, oc + zo);
        float4 x4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (TMAX) x4 = ld4(p.tmax, oc + zo);
        float t_l = __shfl_up_sync(0xffffffffu, th_c.w, 1, 16);
        float t_r = __shfl_down_sync(0xffffffffu, th_c.x, 1, 16);
        uint32_t m_l = __shfl_up_sync(0xffffffffu, mc, 1, 16) >> 24;
        uint32_t m_r = __shfl_down_sync(0xffffffffu, mc, 1, 16) & 255u;
        if (l16 == 0) { t_l = __ldg(p.th_in + oxl + zo); m_l = __ldg(p.mat + oxl + zo); }
        if (l16 == 15) { t_r = __ldg(p.th_in + oxr + zo); m_r = __ldg(p.mat + oxr + zo); }

        const float T[6] = {t_l, th_c.x, th_c.y, th_c.z, th_c.w, t_r};
        const float Tym[4] = {t_ym.x, t_ym.y, t_ym.z, t_ym.w}, Typ[4] = {t_yp.x, t_yp.y, t_yp.z, t_yp.w};
        const float Tm[4] = {th_m.x, th_m.y, th_m.z, th_m.w}, Tp[4] = {th_p.x, th_p.y, th_p.z, th_p.w};
        float s[4];    // sum over the six faces of k_f (T_neighbour - T)

        // one material in the whole neighbourhood of the warp's cells: every face mean is k itself
        const uint32_t m0 = mc & 255u, rep = m0 * 0x01010101u;
        const bool same = (mc == rep) & (mm == rep) & (mp == rep) & (m_ym == rep) & (m_yp == rep) & (m_l == m0) & (m_r == m0);
        if (__all_sync(0xffffffffu, same)) {
            const float kc = rcp(tab[m0].x);
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const float th = T[c + 1];
                s[c] = kc * (((T[c] - th) + (T[c + 2] - th)) + ((Tym[c] - th) + (Typ[c] - th)) + ((Tm[c] - th) + (Tp[c] - th)));
            }
        } else {
            const float4 ik_c = inv_k(tab, mc), ik_m = inv_k(tab, mm), ik_p = inv_k(tab, mp);
            const float4 ik_ym = inv_k(tab, m_ym), ik_yp = inv_k(tab, m_yp);
            const float IK[6] = {tab[m_l].x, ik_c.x, ik_c.y, ik_c.z, ik_c.w, tab[m_r].x};
            const float Iym[4] = {ik_ym.x, ik_ym.y, ik_ym.z, ik_ym.w}, Iyp[4] = {ik_yp.x, ik_yp.y, ik_yp.z, ik_yp.w};
            const float Im[4] = {ik_m.x, ik_m.y, ik_m.z, ik_m.w}, Ip[4] = {ik_p.x, ik_p.y, ik_p.z, ik_p.w};
            float gx[5];   // flux through the x faces of the quad: gx[c] = k_f (T[c] - T[c+1])
#pragma unroll
            for (int c = 0; c < 5; ++c) gx[c] = kface(IK[c], IK[c + 1]) * (T[c] - T[c + 1]);
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const float th = T[c + 1], ik = IK[c + 1];
                float a = gx[c] - gx[c + 1];
                a += kface(ik, Iym[c]) * (Tym[c] - th) + kface(ik, Iyp[c]) * (Typ[c] - th);
                a += kface(ik, Im[c]) * (Tm[c] - th) + kface(ik, Ip[c]) * (Tp[c] - th);
                s[c] = a;
            }
        }

        const float Qs[4] = {q4.x, q4.y, q4.z, q4.w};
        float dose[4] = {d4.x, d4.y, d4.z, d4.w}, tmx[4] = {x4.x, x4.y, x4.z, x4.w};
        const uint32_t free_c = ((k == 0) || (k == p.nz - 1)) ? 0u : free_xy;
        float out[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const float th = T[c + 1];
            const float4 row = tab[(mc >> (8 * c)) & 255u];
            float tn = th + row.y * s[c] - row.z * th + row.w * (p.hs * Qs[c]);
            if (!((free_c >> c) & 1u)) tn = 0.0f;                         // Dirichlet border at T_b
            out[c] = tn;
            const float e = tn + p.d43;                                    // T - 43
            dose[c] += p.dose_dt * ex2(e >= 0.0f ? e : 2.0f * e);          // R^(43 - T), R = 0.5 / 0.25
            if (TMAX) tmx[c] = fmaxf(tmx[c], tn);
        }
        if (store) {
            *reinterpret_cast<float4 *>(p.th_out + oc + zo) = make_float4(out[0], out[1], out[2], out[3]);
            *reinterpret_cast<float4 *>(p.dose + oc + zo) = make_float4(dose[0], dose[1], dose[2], dose[3]);
            if (TMAX) *reinterpret_cast<float4 *>(p.tmax + oc + zo) = make_float4(tmx[0], tmx[1], tmx[2], tmx[3]);
        }
        th_m = th_c; th_c = th_p; mm = mc; mc = mp;
    }
}

// dense (nx, ny, nz) <-> pitched private layout
__global__ void k_bhte_pack(float *__restrict__ dst, float *__restrict__ tmax, const float *__restrict__ src, int nx, int ny, int nz, int px,
                            float T_b) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= nx) return;
    float v = src[i + (long long)nx * (j + (long long)ny * k)] - T_b;
    if (i == 0 || j == 0 || k == 0 || i == nx - 1 || j == ny - 1 || k == nz - 1) v = 0.0f;
    const long long o = i + (long long)px * (j + (long long)ny * k);
    dst[o] = v;
    if (tmax) tmax[o] = fmaxf(tmax[o], v);
}
__global__ void k_bhte_pack_raw(float *__restrict__ dst, const float *__restrict__ src, int nx, int ny, int px) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= nx) return;
    dst[i + (long long)px * (j + (long long)ny * k)] = src[i + (long long)nx * (j + (long long)ny * k)];
}
__global__ void k_bhte_unpack(float *__restrict__ dst, const float *__restrict__ src, int nx, int ny, int px, float offset) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= nx) return;
    dst[i + (long long)nx * (j + (long long)ny * k)] = offset + src[i + (long long)px * (j + (long long)ny * k)];
}
// dense uint8 map -> pitched map; max_index receives the largest index seen
__global__ void k_bhte_pack_map(uint8_t *__restrict__ dst, const uint8_t *__restrict__ src, int nx, int ny, int px, int *max_index) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    int v = 0;
    if (i < nx) {
        v = src[i + (long long)nx * (j + (long long)ny * k)];
        dst[i + (long long)px * (j + (long long)ny * k)] = (uint8_t)v;
    }
    v = __reduce_max_sync(0xffffffffu, v);
    if ((threadIdx.x & 31) == 0 && v > 0) atomicMax(max_index, v);
}

}  // namespace bvfdtd
