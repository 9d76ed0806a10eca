// kernels_tiled.cuh -- the sm_100a hot path: 2.5-D z-marching tiles staged in shared memory by TMA.
//
// One CTA owns a TX x TY tile of the x-y plane and marches a chunk of z-planes.  A producer warp
// (one elected lane) issues cp.async.bulk.tensor box loads for the planes of iteration m into a
// ring of NS shared-memory stages (mbarrier full/empty pairs); NC = (TX/4)*TY consumer threads
// each own 4 consecutive x-cells of one row (float4) and keep the z-direction stencil windows and
// the x-y partial sums of the not-yet-finished planes in registers (a sliding window), so every
// array plane is fetched from L2/HBM exactly once per CTA (plus the x-y halo of the box):
//
//   velocity pass  (S2, Eq. 1 rows 1-3): iteration m loads sxx,syy,sxy,sxz,syz,szz at plane m and
//       the old vx,vy (plane m-1), vz (plane m-2); it forms the x-y derivative sums of plane m,
//       then finishes vx,vy at plane m-1 (D-z needs sxz,syz up to plane m) and vz at plane m-2
//       (D+z needs szz up to plane m).
//   stress pass  (S3+S4, Eq. 1 rows 4-9, L148-L152): iteration m loads vx,vy,vz at plane m (with
//       halo) and the old sigma/r: normal components + sensor maps at plane m-1, sxy,rxy at plane
//       m, sxz,rxz,syz,ryz at plane m-2, and finishes exactly those.
//
// Out-of-grid reads: the private layout keeps zero gaps around every field (device_params.hpp)
// and TMA zero-fills boxes that leave the allocation, so the zero ghost of reading P4 needs no
// branch.  PML (reading P5): CTAs / planes that touch a slab take the psi branches (block- or
// iteration-uniform tests, per-cell predicates inside); psi itself is read-modify-written with
// plain global accesses because only slab cells touch it.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>

#include "device_params.hpp"

namespace bvfdtd {

// ------------------------------------------------------------------------------------------
// configuration
// ------------------------------------------------------------------------------------------
template <int TX_, int TY_, int NS_>
struct TileCfg {
    static constexpr int TX = TX_, TY = TY_, NS = NS_;
    static constexpr int NC = (TX / 4) * TY;            // consumer threads
    static constexpr int NT = NC + 32;                  // + producer warp
    static constexpr int AX = TX + 8, BY = TY + 4;      // halo box extents
    static constexpr int A_BYTES = AX * TY * 4;         // x-halo box
    static constexpr int B_BYTES = TX * BY * 4;         // y-halo box
    static constexpr int C_BYTES = AX * BY * 4;         // x-y-halo box
    static constexpr int D_BYTES = TX * TY * 4;         // plain tile
    static constexpr int MX = TX + 16, MY = TY + 1;     // material box (bytes)
    static constexpr int M_BYTES = (MX * MY + 127) / 128 * 128;
    static constexpr int MR = NS + 3;                   // material ring of the stress pass
    // velocity stage: sxx A, syy B, sxy C, sxz A, syz B, szz D, vx vy vz D, mat
    static constexpr int V_SXX = 0, V_SYY = V_SXX + A_BYTES, V_SXY = V_SYY + B_BYTES,
                         V_SXZ = V_SXY + C_BYTES, V_SYZ = V_SXZ + A_BYTES, V_SZZ = V_SYZ + B_BYTES,
                         V_VX = V_SZZ + D_BYTES, V_VY = V_VX + D_BYTES, V_VZ = V_VY + D_BYTES,
                         V_MAT = V_VZ + D_BYTES, V_STAGE = V_MAT + M_BYTES;
    // stress stage: vx vy vz C, 12 sigma/r D, peak, sumsq D
    static constexpr int S_V = 0, S_SR = 3 * C_BYTES, S_PEAK = S_SR + 12 * D_BYTES,
                         S_SUMSQ = S_PEAK + D_BYTES, S_STAGE = S_SUMSQ + D_BYTES;
    static constexpr int V_SMEM = NS * V_STAGE + 256 * 4 + 2 * NS * 8 + 128;
    static constexpr int S_SMEM = NS * S_STAGE + MR * M_BYTES + 256 * 32 + 2 * NS * 8 + 128;
    static_assert(A_BYTES % 128 == 0 && B_BYTES % 128 == 0 && C_BYTES % 128 == 0 && D_BYTES % 128 == 0, "TMA alignment");
};

using Cfg = TileCfg<64, 8, 2>;

struct TiledMaps {
    CUtensorMap boxA, boxB, boxC, boxD;   // 4-D (x, y, z+2, field) fp32 maps over the 17 grid arrays
    CUtensorMap mat;                      // 3-D uint8 map over the index map
};

struct TiledPlan {
    TiledMaps maps;
    int chunks = 1, nzc = 0;
    bool ready = false;
};

enum { F_PEAK = NSTATE, F_SUMSQ = NSTATE + 1 };

// ------------------------------------------------------------------------------------------
// PTX wrappers: mbarrier + TMA
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, uint64_t *bar, int x, int y, int z, int f) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(x), "r"(y), "r"(z), "r"(f), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, uint64_t *bar, int x, int y, int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap *m) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(m) : "memory");
}

// ------------------------------------------------------------------------------------------
// small device helpers
// ------------------------------------------------------------------------------------------
#define TC1 1.125f
#define TC2 (-1.0f / 24.0f)

__device__ __forceinline__ float4 lds4(const float *p) { return *reinterpret_cast<const float4 *>(p); }

// 12 consecutive x values around the thread's 4 cells: a[4..7] are its own cells i0..i0+3
struct Row12 {
    float a[12];
};
__device__ __forceinline__ Row12 load_row12(const float *row_own) {   // row_own -> own float4
    Row12 r;
    const float4 L = lds4(row_own - 4), O = lds4(row_own), R = lds4(row_own + 4);
    r.a[0] = L.x; r.a[1] = L.y; r.a[2] = L.z; r.a[3] = L.w;
    r.a[4] = O.x; r.a[5] = O.y; r.a[6] = O.z; r.a[7] = O.w;
    r.a[8] = R.x; r.a[9] = R.y; r.a[10] = R.z; r.a[11] = R.w;
    return r;
}
// D+x at cell c (result on the half node): c1 (f(i+1)-f(i)) + c2 (f(i+2)-f(i-1))
__device__ __forceinline__ float dpx(const Row12 &r, int c, float inv_dx) {
    return (TC1 * (r.a[5 + c] - r.a[4 + c]) + TC2 * (r.a[6 + c] - r.a[3 + c])) * inv_dx;
}
// D-x at cell c (result on the integer node): c1 (f(i)-f(i-1)) + c2 (f(i+1)-f(i-2))
__device__ __forceinline__ float dmx(const Row12 &r, int c, float inv_dx) {
    return (TC1 * (r.a[4 + c] - r.a[3 + c]) + TC2 * (r.a[5 + c] - r.a[2 + c])) * inv_dx;
}
__device__ __forceinline__ float comp(const float4 &v, int c) { return c == 0 ? v.x : c == 1 ? v.y : c == 2 ? v.z : v.w; }
// 4-point difference from four values ordered along the axis: c1 (b-a) + c2 (d-z)
__device__ __forceinline__ float d4(float z, float a, float b, float d, float inv_dx) {
    return (TC1 * (b - a) + TC2 * (d - z)) * inv_dx;
}

// per-thread PML bookkeeping for its 4 cells
struct PmlCtx {
    bool tile_x, row_y;     // this thread's cells can be in an x slab / its row is in a y slab
    bool in_x[4];
    int ix[4];              // slab-compact x index
    int jy;                 // slab-compact y index
};

__device__ __forceinline__ float psi_rmw(float *__restrict__ psi, long long q, float a, float b, float d) {
    const float p = fmaf(b, psi[q], a * d);
    psi[q] = p;
    return d + p;
}

// ------------------------------------------------------------------------------------------
// S2: velocity pass
// ------------------------------------------------------------------------------------------
template <class C>
__global__ void __launch_bounds__(C::NT, 2) k_velocity_tiled(const __grid_constant__ TiledMaps maps, const Params p, const int nzc) {
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char *stages = smem;
    float *rho_tab = reinterpret_cast<float *>(smem + C::NS * C::V_STAGE);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + C::NS * C::V_STAGE + 256 * 4);
    uint64_t *empty = full + C::NS;

    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * C::TX, y0 = blockIdx.y * C::TY;
    const int kz0 = blockIdx.z * nzc, kz1 = min(p.nz, kz0 + nzc);
    const int m_begin = kz0 - 2, m_end = kz1 + 2;   // iterations m in [m_begin, m_end)

    for (int q = tid; q < 256; q += C::NT) rho_tab[q] = p.rows[q].rho;
    if (tid == 0) {
        for (int s = 0; s < C::NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], C::NC / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (tid >= C::NC) {
        // ================= producer warp =================
        if (tid == C::NC) {
            prefetch_tmap(&maps.boxA); prefetch_tmap(&maps.boxB); prefetch_tmap(&maps.boxC);
            prefetch_tmap(&maps.boxD); prefetch_tmap(&maps.mat);
            int s = 0; uint32_t ph = 0;
            for (int m = m_begin; m < m_end; ++m) {
                mbar_wait(&empty[s], ph ^ 1);
                unsigned char *st = stages + s * C::V_STAGE;
                const bool ld_xy = (m - 1 >= kz0) && (m - 1 < kz1);
                const bool ld_z = (m - 2 >= kz0) && (m - 2 < kz1);
                uint32_t bytes = 2 * C::A_BYTES + 2 * C::B_BYTES + C::C_BYTES + C::D_BYTES + C::MX * C::MY;
                if (ld_xy) bytes += 2 * C::D_BYTES;
                if (ld_z) bytes += C::D_BYTES;
                mbar_expect_tx(&full[s], bytes);
                const int z = m + 2;
                tma_load_4d(st + C::V_SXX, &maps.boxA, &full[s], x0 - 4, y0, z, SXX);
                tma_load_4d(st + C::V_SYY, &maps.boxB, &full[s], x0, y0 - 1, z, SYY);
                tma_load_4d(st + C::V_SXY, &maps.boxC, &full[s], x0 - 4, y0 - 2, z, SXY);
                tma_load_4d(st + C::V_SXZ, &maps.boxA, &full[s], x0 - 4, y0, z, SXZ);
                tma_load_4d(st + C::V_SYZ, &maps.boxB, &full[s], x0, y0 - 2, z, SYZ);
                tma_load_4d(st + C::V_SZZ, &maps.boxD, &full[s], x0, y0, z, SZZ);
                if (ld_xy) {
                    tma_load_4d(st + C::V_VX, &maps.boxD, &full[s], x0, y0, z - 1, VX);
                    tma_load_4d(st + C::V_VY, &maps.boxD, &full[s], x0, y0, z - 1, VY);
                }
                if (ld_z) tma_load_4d(st + C::V_VZ, &maps.boxD, &full[s], x0, y0, z - 2, VZ);
                tma_load_3d(st + C::V_MAT, &maps.mat, &full[s], x0, y0, m - 1);
                if (++s == C::NS) { s = 0; ph ^= 1; }
            }
        }
        return;
    }

    // ================= consumers =================
    const int tx = tid % (C::TX / 4), ty = tid / (C::TX / 4);
    const int i0 = x0 + 4 * tx, j = y0 + ty;
    const bool row_ok = (j < p.ny) && (i0 < p.nx);   // the thread owns at least one cell
    const int P = p.P;
    const float inv_dx = p.inv_dx, dt = p.dt;
    bool ok[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) ok[c] = row_ok && (i0 + c < p.nx);

    PmlCtx pc;
    pc.tile_x = (P > 0) && (i0 < P || i0 + 3 >= p.nx - P);
    pc.row_y = (P > 0) && (j < P || j >= p.ny - P) && row_ok;
    pc.jy = j < P ? j : j - (p.ny - 2 * P);
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int i = i0 + c;
        pc.in_x[c] = pc.tile_x && ok[c] && (i < P || i >= p.nx - P);
        pc.ix[c] = i < P ? i : i - (p.nx - 2 * P);
    }

    float wxz[4][4], wyz[4][4], wzz[4][4];   // z windows: slot 3 = plane m ... slot 0 = plane m-3
    float pvx[4], pvy[4], pvz1[4], pvz2[4];  // x-y sums of planes m-1 (pvx, pvy, pvz1) and m-2 (pvz2)
    float rho_prev[4];                        // rho of the thread's cells at plane m-2
#pragma unroll
    for (int c = 0; c < 4; ++c) {
#pragma unroll
        for (int w = 0; w < 4; ++w) wxz[w][c] = wyz[w][c] = wzz[w][c] = 0.0f;
        pvx[c] = pvy[c] = pvz1[c] = pvz2[c] = 0.0f;
        rho_prev[c] = 1.0f;
    }

    int s = 0; uint32_t ph = 0;
    for (int m = m_begin; m < m_end; ++m) {
        mbar_wait(&full[s], ph);
        const unsigned char *st = stages + s * C::V_STAGE;
        const float *sA_xx = reinterpret_cast<const float *>(st + C::V_SXX) + ty * C::AX + 4 + 4 * tx;
        const float *sB_yy = reinterpret_cast<const float *>(st + C::V_SYY) + ty * C::TX + 4 * tx;
        const float *sC_xy = reinterpret_cast<const float *>(st + C::V_SXY) + ty * C::AX + 4 + 4 * tx;
        const float *sA_xz = reinterpret_cast<const float *>(st + C::V_SXZ) + ty * C::AX + 4 + 4 * tx;
        const float *sB_yz = reinterpret_cast<const float *>(st + C::V_SYZ) + ty * C::TX + 4 * tx;
        const float *sD = reinterpret_cast<const float *>(st + C::V_SZZ) + ty * C::TX + 4 * tx;

        float nvx[4], nvy[4], nvz[4];
        const bool plane_in = (m >= kz0) && (m < kz1);
        float4 xz_own, yz_own;
        {
            const Row12 rxz = load_row12(sA_xz);
            xz_own = make_float4(rxz.a[4], rxz.a[5], rxz.a[6], rxz.a[7]);
            const float4 y0v = lds4(sB_yz), y1v = lds4(sB_yz + C::TX), y2v = lds4(sB_yz + 2 * C::TX), y3v = lds4(sB_yz + 3 * C::TX);
            yz_own = y2v;
            if (plane_in) {
                const Row12 rxx = load_row12(sA_xx);
                const Row12 rxy = load_row12(sC_xy + 2 * C::AX);
                const float4 xy0 = lds4(sC_xy), xy1 = lds4(sC_xy + C::AX), xy3 = lds4(sC_xy + 3 * C::AX);
                const float4 yy0 = lds4(sB_yy), yy1 = lds4(sB_yy + C::TX), yy2 = lds4(sB_yy + 2 * C::TX), yy3 = lds4(sB_yy + 3 * C::TX);
                const bool zin = true;
                (void)zin;
                float ay_i = 0, by_i = 0, ay_h = 0, by_h = 0;
                if (pc.row_y) {
                    ay_i = __ldg(p.prof[1][0] + j); by_i = __ldg(p.prof[1][1] + j);
                    ay_h = __ldg(p.prof[1][2] + j); by_h = __ldg(p.prof[1][3] + j);
                }
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    float dxx = dpx(rxx, c, inv_dx);                                             // D+x sxx -> vx
                    float dxy_y = d4(comp(xy0, c), comp(xy1, c), rxy.a[4 + c], comp(xy3, c), inv_dx);   // D-y sxy -> vx
                    float dxy_x = dmx(rxy, c, inv_dx);                                           // D-x sxy -> vy
                    float dyy = d4(comp(yy0, c), comp(yy1, c), comp(yy2, c), comp(yy3, c), inv_dx);     // D+y syy -> vy
                    float dxz = dmx(rxz, c, inv_dx);                                             // D-x sxz -> vz
                    float dyz = d4(comp(y0v, c), comp(y1v, c), comp(y2v, c), comp(y3v, c), inv_dx);     // D-y syz -> vz
                    if (pc.in_x[c]) {
                        const int i = i0 + c;
                        const long long q = pc.ix[c] + (long long)p.wx * (j + (long long)p.ny * m);
                        dxx = psi_rmw(p.psi[0], q, __ldg(p.prof[0][2] + i), __ldg(p.prof[0][3] + i), dxx);
                        dxy_x = psi_rmw(p.psi[1], q, __ldg(p.prof[0][0] + i), __ldg(p.prof[0][1] + i), dxy_x);
                        dxz = psi_rmw(p.psi[2], q, __ldg(p.prof[0][0] + i), __ldg(p.prof[0][1] + i), dxz);
                    }
                    if (pc.row_y && ok[c]) {
                        const long long q = (i0 + c) + (long long)p.px * (pc.jy + (long long)(2 * P) * m);
                        dxy_y = psi_rmw(p.psi[6], q, ay_i, by_i, dxy_y);
                        dyy = psi_rmw(p.psi[7], q, ay_h, by_h, dyy);
                        dyz = psi_rmw(p.psi[8], q, ay_i, by_i, dyz);
                    }
                    nvx[c] = dxx + dxy_y;
                    nvy[c] = dxy_x + dyy;
                    nvz[c] = dxz + dyz;
                }
            } else {
#pragma unroll
                for (int c = 0; c < 4; ++c) nvx[c] = nvy[c] = nvz[c] = 0.0f;
            }
        }
        const float4 zz_own = lds4(sD);
        // slide the z windows and insert plane m
#pragma unroll
        for (int c = 0; c < 4; ++c) {
#pragma unroll
            for (int w = 0; w < 3; ++w) { wxz[w][c] = wxz[w + 1][c]; wyz[w][c] = wyz[w + 1][c]; wzz[w][c] = wzz[w + 1][c]; }
            wxz[3][c] = comp(xz_own, c); wyz[3][c] = comp(yz_own, c); wzz[3][c] = comp(zz_own, c);
        }

        // material of plane m-1: rho at i0..i0+4 of row j and i0..i0+3 of row j+1
        const unsigned char *mt = st + C::V_MAT + ty * C::MX + 4 * tx;
        float rho_j[5], rho_j1[4];
        {
            const uint32_t w0 = *reinterpret_cast<const uint32_t *>(mt);
            const uint32_t w1 = *reinterpret_cast<const uint32_t *>(mt + C::MX);
            rho_j[4] = rho_tab[mt[4]];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                rho_j[c] = rho_tab[(w0 >> (8 * c)) & 255u];
                rho_j1[c] = rho_tab[(w1 >> (8 * c)) & 255u];
            }
        }

        const int k1 = m - 1, k2 = m - 2;
        if (k1 >= kz0 && k1 < kz1 && row_ok) {
            // finish vx, vy at plane k1: D-z of sxz / syz over planes m-3..m
            const float4 vxo = lds4(reinterpret_cast<const float *>(st + C::V_VX) + ty * C::TX + 4 * tx);
            const float4 vyo = lds4(reinterpret_cast<const float *>(st + C::V_VY) + ty * C::TX + 4 * tx);
            const bool zs = (P > 0) && (k1 < P || k1 >= p.nz - P);
            float az = 0, bz = 0;
            int kz = 0;
            if (zs) { az = __ldg(p.prof[2][0] + k1); bz = __ldg(p.prof[2][1] + k1); kz = k1 < P ? k1 : k1 - (p.nz - 2 * P); }
            float ox[4], oy[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                float dzx = d4(wxz[0][c], wxz[1][c], wxz[2][c], wxz[3][c], inv_dx);
                float dzy = d4(wyz[0][c], wyz[1][c], wyz[2][c], wyz[3][c], inv_dx);
                if (zs && ok[c]) {
                    const long long q = (i0 + c) + (long long)p.px * (j + (long long)p.ny * kz);
                    dzx = psi_rmw(p.psi[12], q, az, bz, dzx);
                    dzy = psi_rmw(p.psi[13], q, az, bz, dzy);
                }
                const float rx = 0.5f * (rho_j[c] + rho_j[c + 1]);
                const float ry = 0.5f * (rho_j[c] + rho_j1[c]);
                const float nx_ = comp(vxo, c) + dt / rx * (pvx[c] + dzx);
                const float ny_ = comp(vyo, c) + dt / ry * (pvy[c] + dzy);
                ox[c] = (ok[c] && (i0 + c < p.nx - 1)) ? nx_ : 0.0f;
                oy[c] = (ok[c] && (j < p.ny - 1)) ? ny_ : 0.0f;
            }
            const long long g = p.org + i0 + (long long)p.px * j + p.sz * k1;
            *reinterpret_cast<float4 *>(p.f[VX] + g) = make_float4(ox[0], ox[1], ox[2], ox[3]);
            *reinterpret_cast<float4 *>(p.f[VY] + g) = make_float4(oy[0], oy[1], oy[2], oy[3]);
        }
        if (k2 >= kz0 && k2 < kz1 && row_ok) {
            // finish vz at plane k2: D+z of szz over planes m-3..m
            const float4 vzo = lds4(reinterpret_cast<const float *>(st + C::V_VZ) + ty * C::TX + 4 * tx);
            const bool zs = (P > 0) && (k2 < P || k2 >= p.nz - P);
            float az = 0, bz = 0;
            int kz = 0;
            if (zs) { az = __ldg(p.prof[2][2] + k2); bz = __ldg(p.prof[2][3] + k2); kz = k2 < P ? k2 : k2 - (p.nz - 2 * P); }
            float oz[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                float dzz = d4(wzz[0][c], wzz[1][c], wzz[2][c], wzz[3][c], inv_dx);
                if (zs && ok[c]) {
                    const long long q = (i0 + c) + (long long)p.px * (j + (long long)p.ny * kz);
                    dzz = psi_rmw(p.psi[14], q, az, bz, dzz);
                }
                const float rz = 0.5f * (rho_prev[c] + rho_j[c]);
                const float nz_ = comp(vzo, c) + dt / rz * (pvz2[c] + dzz);
                oz[c] = (ok[c] && (k2 < p.nz - 1)) ? nz_ : 0.0f;
            }
            const long long g = p.org + i0 + (long long)p.px * j + p.sz * k2;
            *reinterpret_cast<float4 *>(p.f[VZ] + g) = make_float4(oz[0], oz[1], oz[2], oz[3]);
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            pvz2[c] = pvz1[c]; pvz1[c] = nvz[c]; pvx[c] = nvx[c]; pvy[c] = nvy[c];
            rho_prev[c] = rho_j[c];
        }
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty[s]);
        if (++s == C::NS) { s = 0; ph ^= 1; }
    }
}

// ------------------------------------------------------------------------------------------
// S3 + S4: stress, memory variables, sensor
// ------------------------------------------------------------------------------------------
struct ShearMat {
    float inv, ts;   // 1/mu_R (+inf for a fluid) and tau_s of one cell
};

template <class C>
__global__ void __launch_bounds__(C::NT, 2) k_stress_tiled(const __grid_constant__ TiledMaps maps, const Params p, const int nzc) {
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char *stages = smem;
    unsigned char *mat_ring = smem + C::NS * C::S_STAGE;
    KRow *tab = reinterpret_cast<KRow *>(mat_ring + C::MR * C::M_BYTES);
    uint64_t *full = reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(tab) + 256 * 32);
    uint64_t *empty = full + C::NS;

    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * C::TX, y0 = blockIdx.y * C::TY;
    const int kz0 = blockIdx.z * nzc, kz1 = min(p.nz, kz0 + nzc);
    const int m_begin = kz0 - 2, m_end = kz1 + 2;
    const bool sens = p.do_peak | p.do_rms;

    for (int q = tid; q < 256; q += C::NT) {
        KRow r = p.rows[q];
        if (r.solid == 0.0f) r.invMu = __int_as_float(0x7f800000);   // +inf: harmonic mean -> 0 (P2)
        tab[q] = r;
    }
    if (tid == 0) {
        for (int s = 0; s < C::NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], C::NC / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (tid >= C::NC) {
        if (tid == C::NC) {
            prefetch_tmap(&maps.boxC); prefetch_tmap(&maps.boxD); prefetch_tmap(&maps.mat);
            int s = 0; uint32_t ph = 0;
            int mr = ((m_begin % C::MR) + C::MR) % C::MR;
            for (int m = m_begin; m < m_end; ++m) {
                mbar_wait(&empty[s], ph ^ 1);
                unsigned char *st = stages + s * C::S_STAGE;
                const bool in0 = (m >= kz0) && (m < kz1);
                const bool in1 = (m - 1 >= kz0) && (m - 1 < kz1);
                const bool in2 = (m - 2 >= kz0) && (m - 2 < kz1);
                uint32_t bytes = 3 * C::C_BYTES + C::MX * C::MY;
                if (in0) bytes += 2 * C::D_BYTES;
                if (in1) bytes += 6 * C::D_BYTES + (p.do_peak ? C::D_BYTES : 0) + (p.do_rms ? C::D_BYTES : 0);
                if (in2) bytes += 4 * C::D_BYTES;
                mbar_expect_tx(&full[s], bytes);
                const int z = m + 2;
                tma_load_4d(st + C::S_V, &maps.boxC, &full[s], x0 - 4, y0 - 2, z, VX);
                tma_load_4d(st + C::S_V + C::C_BYTES, &maps.boxC, &full[s], x0 - 4, y0 - 2, z, VY);
                tma_load_4d(st + C::S_V + 2 * C::C_BYTES, &maps.boxC, &full[s], x0 - 4, y0 - 2, z, VZ);
                unsigned char *sr = st + C::S_SR;
                if (in1) {
                    tma_load_4d(sr + 0 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z - 1, SXX);
                    tma_load_4d(sr + 1 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z - 1, SYY);
                    tma_load_4d(sr + 2 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z - 1, SZZ);
                    tma_load_4d(sr + 3 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z - 1, RXX);
                    tma_load_4d(sr + 4 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z - 1, RYY);
                    tma_load_4d(sr + 5 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z - 1, RZZ);
                    if (p.do_peak) tma_load_4d(st + C::S_PEAK, &maps.boxD, &full[s], x0, y0, z - 1, F_PEAK);
                    if (p.do_rms) tma_load_4d(st + C::S_SUMSQ, &maps.boxD, &full[s], x0, y0, z - 1, F_SUMSQ);
                }
                if (in0) {
                    tma_load_4d(sr + 6 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z, SXY);
                    tma_load_4d(sr + 7 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z, RXY);
                }
                if (in2) {
                    tma_load_4d(sr + 8 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z - 2, SXZ);
                    tma_load_4d(sr + 9 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z - 2, RXZ);
                    tma_load_4d(sr + 10 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z - 2, SYZ);
                    tma_load_4d(sr + 11 * C::D_BYTES, &maps.boxD, &full[s], x0, y0, z - 2, RYZ);
                }
                tma_load_3d(mat_ring + mr * C::M_BYTES, &maps.mat, &full[s], x0, y0, m);
                if (++mr == C::MR) mr = 0;
                if (++s == C::NS) { s = 0; ph ^= 1; }
            }
        }
        return;
    }

    // ================= consumers =================
    const int tx = tid % (C::TX / 4), ty = tid / (C::TX / 4);
    const int i0 = x0 + 4 * tx, j = y0 + ty;
    const bool row_ok = (j < p.ny) && (i0 < p.nx);   // the thread owns at least one cell
    const int P = p.P;
    const float inv_dx = p.inv_dx, dt = p.dt, hdt = p.half_dt, A = p.A, B = p.B;
    bool ok[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) ok[c] = row_ok && (i0 + c < p.nx);

    PmlCtx pc;
    pc.tile_x = (P > 0) && (i0 < P || i0 + 3 >= p.nx - P);
    pc.row_y = (P > 0) && (j < P || j >= p.ny - P) && row_ok;
    pc.jy = j < P ? j : j - (p.ny - 2 * P);
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int i = i0 + c;
        pc.in_x[c] = pc.tile_x && ok[c] && (i < P || i >= p.nx - P);
        pc.ix[c] = i < P ? i : i - (p.nx - 2 * P);
    }

    float wvx[4][4], wvy[4][4], wvz[4][4];     // z windows, slot 3 = plane m
    float nxx[4], nyy[4];                       // vxx, vyy of plane m-1
    float dxz1[4], dxz2[4], dyz1[4], dyz2[4];   // D+x vz, D+y vz of planes m-1 and m-2
#pragma unroll
    for (int c = 0; c < 4; ++c) {
#pragma unroll
        for (int w = 0; w < 4; ++w) wvx[w][c] = wvy[w][c] = wvz[w][c] = 0.0f;
        nxx[c] = nyy[c] = dxz1[c] = dxz2[c] = dyz1[c] = dyz2[c] = 0.0f;
    }

    int s = 0; uint32_t ph = 0;
    int mr0 = ((m_begin % C::MR) + C::MR) % C::MR;   // ring slot of plane m
    for (int m = m_begin; m < m_end; ++m) {
        mbar_wait(&full[s], ph);
        const unsigned char *st = stages + s * C::S_STAGE;
        const float *cvx = reinterpret_cast<const float *>(st + C::S_V) + (ty + 2) * C::AX + 4 + 4 * tx;
        const float *cvy = cvx + C::C_BYTES / 4;
        const float *cvz = cvy + C::C_BYTES / 4;
        const float *dbase = reinterpret_cast<const float *>(st + C::S_SR) + ty * C::TX + 4 * tx;
        const int mr1 = mr0 == 0 ? C::MR - 1 : mr0 - 1;          // plane m-1
        const int mr2 = mr1 == 0 ? C::MR - 1 : mr1 - 1;          // plane m-2
        const unsigned char *mat0 = mat_ring + mr0 * C::M_BYTES + ty * C::MX + 4 * tx;
        const unsigned char *mat1 = mat_ring + mr1 * C::M_BYTES + ty * C::MX + 4 * tx;
        const unsigned char *mat2 = mat_ring + mr2 * C::M_BYTES + ty * C::MX + 4 * tx;
        const bool in0 = (m >= kz0) && (m < kz1);
        const long long gcell = p.org + i0 + (long long)p.px * j;

        const Row12 rvx = load_row12(cvx), rvy = load_row12(cvy), rvz = load_row12(cvz);
        float nvxx[4], nvyy[4], ndxz[4], ndyz[4];
        if (in0) {
            const float4 vxm = lds4(cvx - C::AX), vxp = lds4(cvx + C::AX), vxpp = lds4(cvx + 2 * C::AX);
            const float4 vymm = lds4(cvy - 2 * C::AX), vym = lds4(cvy - C::AX), vyp = lds4(cvy + C::AX);
            const float4 vzm = lds4(cvz - C::AX), vzp = lds4(cvz + C::AX), vzpp = lds4(cvz + 2 * C::AX);
            const bool plane_ok = true;
            float ay_i = 0, by_i = 0, ay_h = 0, by_h = 0;
            if (pc.row_y) {
                ay_i = __ldg(p.prof[1][0] + j); by_i = __ldg(p.prof[1][1] + j);
                ay_h = __ldg(p.prof[1][2] + j); by_h = __ldg(p.prof[1][3] + j);
            }
            float gxy[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                float vxx = dmx(rvx, c, inv_dx);                                                    // D-x vx
                float vyy = d4(comp(vymm, c), comp(vym, c), rvy.a[4 + c], comp(vyp, c), inv_dx);    // D-y vy
                float vx_y = d4(comp(vxm, c), rvx.a[4 + c], comp(vxp, c), comp(vxpp, c), inv_dx);   // D+y vx
                float vy_x = dpx(rvy, c, inv_dx);                                                   // D+x vy
                float vz_x = dpx(rvz, c, inv_dx);                                                   // D+x vz
                float vz_y = d4(comp(vzm, c), rvz.a[4 + c], comp(vzp, c), comp(vzpp, c), inv_dx);   // D+y vz
                if (plane_ok) {
                    if (pc.in_x[c]) {
                        const int i = i0 + c;
                        const long long q = pc.ix[c] + (long long)p.wx * (j + (long long)p.ny * m);
                        const float ai = __ldg(p.prof[0][0] + i), bi = __ldg(p.prof[0][1] + i);
                        const float ah = __ldg(p.prof[0][2] + i), bh = __ldg(p.prof[0][3] + i);
                        vxx = psi_rmw(p.psi[3], q, ai, bi, vxx);
                        vy_x = psi_rmw(p.psi[4], q, ah, bh, vy_x);
                        vz_x = psi_rmw(p.psi[5], q, ah, bh, vz_x);
                    }
                    if (pc.row_y && ok[c]) {
                        const long long q = (i0 + c) + (long long)p.px * (pc.jy + (long long)(2 * P) * m);
                        vx_y = psi_rmw(p.psi[9], q, ay_h, by_h, vx_y);
                        vyy = psi_rmw(p.psi[10], q, ay_i, by_i, vyy);
                        vz_y = psi_rmw(p.psi[11], q, ay_h, by_h, vz_y);
                    }
                }
                nvxx[c] = vxx; nvyy[c] = vyy; ndxz[c] = vz_x; ndyz[c] = vz_y;
                gxy[c] = vx_y + vy_x;
            }
            if (in0 && row_ok) {
                // finish sxy, rxy at plane m: material of the 4 cells (i..i+1, j..j+1, m)
                const float4 so = lds4(dbase + 6 * (C::D_BYTES / 4)), ro = lds4(dbase + 7 * (C::D_BYTES / 4));
                float inv_a[5], ts_a[5], inv_b[5], ts_b[5];
#pragma unroll
                for (int c = 0; c < 5; ++c) {
                    const KRow &ra = tab[mat0[c]], &rb = tab[mat0[C::MX + c]];
                    inv_a[c] = ra.invMu; ts_a[c] = ra.tauS; inv_b[c] = rb.invMu; ts_b[c] = rb.tauS;
                }
                float os[4], orr[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float mu_h = 4.0f / ((inv_a[c] + inv_a[c + 1]) + (inv_b[c] + inv_b[c + 1]));
                    const float ts_h = 0.25f * ((ts_a[c] + ts_a[c + 1]) + (ts_b[c] + ts_b[c + 1]));
                    const float r0 = comp(ro, c);
                    const float rn = fmaf(A, r0, -(B * (mu_h * ts_h) * gxy[c]));
                    const float sn = comp(so, c) + (dt * (mu_h * (1.0f + ts_h)) * gxy[c] + hdt * (rn + r0));
                    os[c] = ok[c] ? sn : 0.0f;
                    orr[c] = ok[c] ? rn : 0.0f;
                }
                const long long g = gcell + p.sz * m;
                *reinterpret_cast<float4 *>(p.f[SXY] + g) = make_float4(os[0], os[1], os[2], os[3]);
                *reinterpret_cast<float4 *>(p.f[RXY] + g) = make_float4(orr[0], orr[1], orr[2], orr[3]);
            }
        } else {
#pragma unroll
            for (int c = 0; c < 4; ++c) nvxx[c] = nvyy[c] = ndxz[c] = ndyz[c] = 0.0f;
        }
        // slide the z windows and insert plane m
#pragma unroll
        for (int c = 0; c < 4; ++c) {
#pragma unroll
            for (int w = 0; w < 3; ++w) { wvx[w][c] = wvx[w + 1][c]; wvy[w][c] = wvy[w + 1][c]; wvz[w][c] = wvz[w + 1][c]; }
            wvx[3][c] = rvx.a[4 + c]; wvy[3][c] = rvy.a[4 + c]; wvz[3][c] = rvz.a[4 + c];
        }

        const int k1 = m - 1, k2 = m - 2;
        if (k1 >= kz0 && k1 < kz1 && row_ok) {
            // finish the normal stresses, their memory variables and the sensor at plane k1
            const bool zs = (P > 0) && (k1 < P || k1 >= p.nz - P);
            float az = 0, bz = 0;
            int kz = 0;
            if (zs) { az = __ldg(p.prof[2][0] + k1); bz = __ldg(p.prof[2][1] + k1); kz = k1 < P ? k1 : k1 - (p.nz - 2 * P); }
            const float4 s0 = lds4(dbase), s1 = lds4(dbase + (C::D_BYTES / 4)), s2 = lds4(dbase + 2 * (C::D_BYTES / 4));
            const float4 r0v = lds4(dbase + 3 * (C::D_BYTES / 4)), r1v = lds4(dbase + 4 * (C::D_BYTES / 4)), r2v = lds4(dbase + 5 * (C::D_BYTES / 4));
            float o[6][4], pr[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                float vzz = d4(wvz[0][c], wvz[1][c], wvz[2][c], wvz[3][c], inv_dx);   // D-z vz at k1
                if (zs && ok[c]) {
                    const long long q = (i0 + c) + (long long)p.px * (j + (long long)p.ny * kz);
                    vzz = psi_rmw(p.psi[17], q, az, bz, vzz);
                }
                const KRow row = tab[mat1[c]];
                const float th = nxx[c] + nyy[c] + vzz;
                const float vii[3] = {nxx[c], nyy[c], vzz};
                const float sold[3] = {comp(s0, c), comp(s1, c), comp(s2, c)};
                const float rold[3] = {comp(r0v, c), comp(r1v, c), comp(r2v, c)};
                float tr = 0.0f;
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    const float oth = th - vii[q];
                    const float eU = row.eP * th - row.eS * oth;
                    const float eR = row.bP * th - row.bS * oth;
                    const float rn = fmaf(A, rold[q], -eR);
                    const float sn = sold[q] + (eU + hdt * (rn + rold[q]));
                    o[q][c] = ok[c] ? sn : 0.0f;
                    o[3 + q][c] = ok[c] ? rn : 0.0f;
                    tr += o[q][c];
                }
                pr[c] = (o[0][c] + o[1][c] + o[2][c]) * (-1.0f / 3.0f);
                (void)tr;
            }
            const long long g = gcell + p.sz * k1;
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                *reinterpret_cast<float4 *>(p.f[SXX + q] + g) = make_float4(o[q][0], o[q][1], o[q][2], o[q][3]);
                *reinterpret_cast<float4 *>(p.f[RXX + q] + g) = make_float4(o[3 + q][0], o[3 + q][1], o[3 + q][2], o[3 + q][3]);
            }
            if (sens) {
                if (p.do_peak) {
                    const float4 pk = lds4(reinterpret_cast<const float *>(st + C::S_PEAK) + ty * C::TX + 4 * tx);
                    *reinterpret_cast<float4 *>(p.peak + g) = make_float4(fmaxf(pk.x, fabsf(pr[0])), fmaxf(pk.y, fabsf(pr[1])),
                                                                          fmaxf(pk.z, fabsf(pr[2])), fmaxf(pk.w, fabsf(pr[3])));
                }
                if (p.do_rms) {
                    const float4 sq = lds4(reinterpret_cast<const float *>(st + C::S_SUMSQ) + ty * C::TX + 4 * tx);
                    *reinterpret_cast<float4 *>(p.sumsq + g) = make_float4(fmaf(pr[0], pr[0], sq.x), fmaf(pr[1], pr[1], sq.y),
                                                                           fmaf(pr[2], pr[2], sq.z), fmaf(pr[3], pr[3], sq.w));
                }
            }
        }
        if (k2 >= kz0 && k2 < kz1 && row_ok) {
            // finish sxz, syz (+ r) at plane k2: D+z of vx, vy over planes m-3..m
            const bool zs = (P > 0) && (k2 < P || k2 >= p.nz - P);
            float az = 0, bz = 0;
            int kz = 0;
            if (zs) { az = __ldg(p.prof[2][2] + k2); bz = __ldg(p.prof[2][3] + k2); kz = k2 < P ? k2 : k2 - (p.nz - 2 * P); }
            const float4 sxz_o = lds4(dbase + 8 * (C::D_BYTES / 4)), rxz_o = lds4(dbase + 9 * (C::D_BYTES / 4));
            const float4 syz_o = lds4(dbase + 10 * (C::D_BYTES / 4)), ryz_o = lds4(dbase + 11 * (C::D_BYTES / 4));
            // materials: row j at planes k2 (mat2) and k2+1 (mat1), cells i0..i0+4; row j+1 cells i0..i0+3
            float inv_2[5], ts_2[5], inv_1[5], ts_1[5], inv_2b[4], ts_2b[4], inv_1b[4], ts_1b[4];
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                const KRow &ra = tab[mat2[c]], &rb = tab[mat1[c]];
                inv_2[c] = ra.invMu; ts_2[c] = ra.tauS; inv_1[c] = rb.invMu; ts_1[c] = rb.tauS;
            }
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const KRow &ra = tab[mat2[C::MX + c]], &rb = tab[mat1[C::MX + c]];
                inv_2b[c] = ra.invMu; ts_2b[c] = ra.tauS; inv_1b[c] = rb.invMu; ts_1b[c] = rb.tauS;
            }
            float oxz[4], orxz[4], oyz[4], oryz[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                float vx_z = d4(wvx[0][c], wvx[1][c], wvx[2][c], wvx[3][c], inv_dx);   // D+z vx at k2
                float vy_z = d4(wvy[0][c], wvy[1][c], wvy[2][c], wvy[3][c], inv_dx);   // D+z vy at k2
                if (zs && ok[c]) {
                    const long long q = (i0 + c) + (long long)p.px * (j + (long long)p.ny * kz);
                    vx_z = psi_rmw(p.psi[15], q, az, bz, vx_z);
                    vy_z = psi_rmw(p.psi[16], q, az, bz, vy_z);
                }
                {   // sxz: cells (i..i+1, j, k2..k2+1)
                    const float mu_h = 4.0f / ((inv_2[c] + inv_2[c + 1]) + (inv_1[c] + inv_1[c + 1]));
                    const float ts_h = 0.25f * ((ts_2[c] + ts_2[c + 1]) + (ts_1[c] + ts_1[c + 1]));
                    const float gg = vx_z + dxz2[c];
                    const float r0 = comp(rxz_o, c);
                    const float rn = fmaf(A, r0, -(B * (mu_h * ts_h) * gg));
                    const float sn = comp(sxz_o, c) + (dt * (mu_h * (1.0f + ts_h)) * gg + hdt * (rn + r0));
                    oxz[c] = ok[c] ? sn : 0.0f; orxz[c] = ok[c] ? rn : 0.0f;
                }
                {   // syz: cells (i, j..j+1, k2..k2+1)
                    const float mu_h = 4.0f / ((inv_2[c] + inv_2b[c]) + (inv_1[c] + inv_1b[c]));
                    const float ts_h = 0.25f * ((ts_2[c] + ts_2b[c]) + (ts_1[c] + ts_1b[c]));
                    const float gg = vy_z + dyz2[c];
                    const float r0 = comp(ryz_o, c);
                    const float rn = fmaf(A, r0, -(B * (mu_h * ts_h) * gg));
                    const float sn = comp(syz_o, c) + (dt * (mu_h * (1.0f + ts_h)) * gg + hdt * (rn + r0));
                    oyz[c] = ok[c] ? sn : 0.0f; oryz[c] = ok[c] ? rn : 0.0f;
                }
            }
            const long long g = gcell + p.sz * k2;
            *reinterpret_cast<float4 *>(p.f[SXZ] + g) = make_float4(oxz[0], oxz[1], oxz[2], oxz[3]);
            *reinterpret_cast<float4 *>(p.f[RXZ] + g) = make_float4(orxz[0], orxz[1], orxz[2], orxz[3]);
            *reinterpret_cast<float4 *>(p.f[SYZ] + g) = make_float4(oyz[0], oyz[1], oyz[2], oyz[3]);
            *reinterpret_cast<float4 *>(p.f[RYZ] + g) = make_float4(oryz[0], oryz[1], oryz[2], oryz[3]);
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            nxx[c] = nvxx[c]; nyy[c] = nvyy[c];
            dxz2[c] = dxz1[c]; dxz1[c] = ndxz[c];
            dyz2[c] = dyz1[c]; dyz1[c] = ndyz[c];
        }
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty[s]);
        if (++s == C::NS) { s = 0; ph ^= 1; }
        if (++mr0 == C::MR) mr0 = 0;
    }
}

// ------------------------------------------------------------------------------------------
// host side: tensor maps, launch plan
// ------------------------------------------------------------------------------------------
inline char *tiled_err_buf() {
    static thread_local char buf[256] = "";
    return buf;
}
inline const char *tiled_plan_error() { return tiled_err_buf(); }

typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline int tiled_plan_create(TiledPlan &plan, const Layout &L, const Params &p) {
    using C = Cfg;
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
        std::snprintf(tiled_err_buf(), 256, "cuTensorMapEncodeTiled entry point unavailable (%s)", cudaGetErrorString(e));
        (void)cudaGetLastError();
        return BVFDTD_ECUDA;
    }
    PFN_encodeTiled enc = (PFN_encodeTiled)fn;
    // the 17 grid arrays (15 state + peak + sumsq) are laid out back to back at a constant stride
    const long long fstride = (const char *)p.f[1] - (const char *)p.f[0];
    for (int q = 0; q < NSTATE; ++q)
        if ((const char *)p.f[q] - (const char *)p.f[0] != fstride * q) return BVFDTD_EINVAL;
    if ((const char *)p.peak - (const char *)p.f[0] != fstride * F_PEAK) return BVFDTD_EINVAL;
    if ((const char *)p.sumsq - (const char *)p.f[0] != fstride * F_SUMSQ) return BVFDTD_EINVAL;
    void *base = (void *)(p.f[0] + (L.org - 2 * L.sz));      // cell (0,0,-2)
    const cuuint64_t gdim[4] = {(cuuint64_t)L.px, (cuuint64_t)L.py, (cuuint64_t)(L.nz + 4), 17};
    const cuuint64_t gstr[3] = {(cuuint64_t)L.px * 4, (cuuint64_t)L.sz * 4, (cuuint64_t)fstride};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    struct { CUtensorMap *m; cuuint32_t bx, by; } boxes[4] = {
        {&plan.maps.boxA, (cuuint32_t)C::AX, (cuuint32_t)C::TY}, {&plan.maps.boxB, (cuuint32_t)C::TX, (cuuint32_t)C::BY},
        {&plan.maps.boxC, (cuuint32_t)C::AX, (cuuint32_t)C::BY}, {&plan.maps.boxD, (cuuint32_t)C::TX, (cuuint32_t)C::TY}};
    for (auto &b : boxes) {
        const cuuint32_t box[4] = {b.bx, b.by, 1, 1};
        CUresult r = enc(b.m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, base, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) {
            std::snprintf(tiled_err_buf(), 256, "cuTensorMapEncodeTiled(float box %ux%u) failed: %d", b.bx, b.by, (int)r);
            return BVFDTD_ECUDA;
        }
    }
    {
        const cuuint64_t mdim[3] = {(cuuint64_t)L.px, (cuuint64_t)L.py, (cuuint64_t)(L.nz + 1)};
        const cuuint64_t mstr[2] = {(cuuint64_t)L.px, (cuuint64_t)L.sz};
        const cuuint32_t mbox[3] = {(cuuint32_t)C::MX, (cuuint32_t)C::MY, 1};
        CUresult r = enc(&plan.maps.mat, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, (void *)p.mat, mdim, mstr, mbox, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) {
            std::snprintf(tiled_err_buf(), 256, "cuTensorMapEncodeTiled(material box) failed: %d", (int)r);
            return BVFDTD_ECUDA;
        }
    }
    e = cudaFuncSetAttribute(k_velocity_tiled<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::V_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_stress_tiled<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::S_SMEM);
    if (e != cudaSuccess) {
        std::snprintf(tiled_err_buf(), 256, "cudaFuncSetAttribute: %s", cudaGetErrorString(e));
        (void)cudaGetLastError();
        return BVFDTD_ECUDA;
    }
    // z chunks: fill the resident CTA slots (2 per SM) in as few waves as possible
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long tiles = (long long)((L.nx + C::TX - 1) / C::TX) * ((L.ny + C::TY - 1) / C::TY);
    const long long slots = 2LL * sms;
    int best = 1;
    double best_cost = 1e300;
    for (int ch = 1; ch <= (L.nz + 7) / 8; ++ch) {
        const int nzc = (L.nz + ch - 1) / ch;
        const long long blocks = tiles * ((L.nz + nzc - 1) / nzc);
        const double waves = (double)((blocks + slots - 1) / slots);
        const double cost = waves * (nzc + 4);
        if (cost < best_cost - 1e-9) { best_cost = cost; best = ch; }
    }
    plan.nzc = (L.nz + best - 1) / best;
    plan.chunks = (L.nz + plan.nzc - 1) / plan.nzc;
    plan.ready = true;
    return 0;
}

inline void tiled_plan_destroy(TiledPlan &plan) { plan.ready = false; }

inline dim3 tiled_grid(const TiledPlan &plan, const Params &p) {
    return dim3((p.nx + Cfg::TX - 1) / Cfg::TX, (p.ny + Cfg::TY - 1) / Cfg::TY, plan.chunks);
}
inline int tiled_velocity(TiledPlan &plan, const Params &p, cudaStream_t st) {
    k_velocity_tiled<Cfg><<<tiled_grid(plan, p), Cfg::NT, Cfg::V_SMEM, st>>>(plan.maps, p, plan.nzc);
    return 0;
}
inline int tiled_stress(TiledPlan &plan, const Params &p, cudaStream_t st) {
    k_stress_tiled<Cfg><<<tiled_grid(plan, p), Cfg::NT, Cfg::S_SMEM, st>>>(plan.maps, p, plan.nzc);
    return 0;
}

}  // namespace bvfdtd
