// kernels_tiled.cuh -- the sm_100a hot path: 2.5-D z-marching tiles staged in shared memory by TMA.
//
// One CTA owns a TX x TY tile of the x-y plane and marches a chunk of z-planes.  A producer warp
// (one elected lane) issues cp.async.bulk.tensor box loads for the planes of iteration m into a
// ring of shared-memory stages (mbarrier full/empty pairs); NC = (TX/4)*TY consumer threads each
// own 4 consecutive x-cells of one row (float4) and keep the z-direction stencil windows and the
// x-y partial sums of the not-yet-finished planes in registers (a sliding window), so every array
// plane is fetched from L2/HBM exactly once per CTA (plus the x-y halo of the box).  Consumers read
// shared memory only and write their results with 16-byte global stores: EVERY global read of the
// hot loop, including the C-PML memory variables psi and the material indices, is a TMA prefetch.
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
// branch.
//
// Tile-class flags: per (tile, plane) words say whether any shear node of
// kind xy / xz / yz has four solid cells and whether any cell is lossy.  Where a kind has no solid
// node its stress and memory variable are identically zero (mu_h = 0, reading P2; zero initial
// state, P9), so producer and consumers skip its loads, arithmetic and stores.  Both sides derive
// the same per-iteration load plan from the same flag words (vel_plan / str_plan below).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>

#include "device_params.hpp"

namespace bvfdtd {

// ------------------------------------------------------------------------------------------
// configuration
// ------------------------------------------------------------------------------------------
constexpr int MAX_STAGES = 4;

template <int TX_, int TY_>
struct TileCfg {
    static constexpr int TX = TX_, TY = TY_;
    static constexpr int NC = (TX / 4) * TY;            // consumer threads
    static constexpr int NT = NC + 32;                  // + producer warp
    static constexpr int AX = TX + 8, BY = TY + 4;      // halo box extents
    static constexpr int A_BYTES = AX * TY * 4;         // x-halo box
    static constexpr int B_BYTES = TX * BY * 4;         // y-halo box
    static constexpr int C_BYTES = AX * BY * 4;         // x-y-halo box
    static constexpr int D_BYTES = TX * TY * 4;         // plain tile
    static constexpr int MX = TX + 16, MY = TY + 1;     // material box (bytes)
    static constexpr int M_BYTES = (MX * MY + 127) / 128 * 128;
    static_assert(A_BYTES % 128 == 0 && B_BYTES % 128 == 0 && C_BYTES % 128 == 0 && D_BYTES % 128 == 0, "TMA alignment");
    static_assert(NC % 32 == 0, "whole consumer warps");
};

using CfgV = TileCfg<64, 8>;    // velocity pass: 4 consumer warps, 2 CTAs per SM
using CfgS = TileCfg<64, 16>;   // stress pass: 8 consumer warps, 1 CTA per SM
using CfgS8 = TileCfg<64, 8>;   // stress pass fallback when the 64 x 16 stages do not fit (very thick PML on a narrow grid)

struct TiledMaps {
    CUtensorMap boxA, boxB, boxC, boxD;   // 4-D (x, y, z+2, field) fp32 maps over the 17 grid arrays
    CUtensorMap mat;                      // 3-D uint8 map over the index map
    CUtensorMap psx, psy, psz;            // 4-D (x, y, z, array) maps over the slab-compact psi arrays
};

// What the producer tells the consumers about one stage (written before the stage's barrier is
// armed): the iteration's load/compute plan and the z-profile coefficients of the two planes the
// iteration finishes (a, b at the integer node of plane m-1 and at the half node of plane m-2).
struct StageHdr {
    uint32_t ctrl, pad[3];
    float az1, bz1, az2, bz2;
};

// Shared-memory plan of one pipeline stage (byte offsets inside the stage), fixed per context.
struct StagePlan {
    int hdr;               // per-stage header written by the producer (StageHdr)
    int psx, psy, psz;     // first psi slot of each axis (3 slots per axis)
    int yb;                // bytes of one y- or z-psi box (= the tile's D box)
    int xb;                // bytes of one x-psi box (low or high slab)
    int xhi, xt;           // byte offset of the high-slab box inside a term slot (0 when no tile touches both
                           // slabs), bytes of one term slot
    int wxb;               // x-psi box width in floats
    int bytes;             // stage size (multiple of 128)
    int ns;                // pipeline stages
    int smem;              // dynamic shared memory of the launch
    int spw;               // velocity pass: columns of the x-profile rows kept in shared memory (TX, or 32 when the
                           // slab part of a tile is at most 32 columns wide); 0 = TX
    int nrho;              // velocity pass: entries of the density table in shared memory (0 = 256)
};

// z chunks of a launch: chunk c covers planes [b[c], b[c+1]).  Blocks are dispatched in blockIdx.z
// order, so the long chunks come first and a few short ones last: they fill the gaps the last wave
// would otherwise leave (the passes run at the memory system's ceiling while all SMs are busy; the
// idle tail was 7-12 % of the kernel time with equal chunks).
constexpr int MAX_CHUNKS = 48;
struct ZChunks {
    int n;
    int b[MAX_CHUNKS + 1];
};

struct TiledPlan {
    TiledMaps mv, ms;      // velocity / stress pass (their tiles differ)
    StagePlan sv, ss;
    StagePlan svc{};       // compact velocity stage plan (ns = 0: unused), see k_velocity_tiled
    int occ_v = 2;         // register budget of the velocity instantiation in use (2 or 3 resident CTAs)
    int occ_v_res = 1, occ_s_res = 1;   // resident CTAs per SM the occupancy query reports for the two passes
    bool s16 = true;       // stress pass runs 64 x 16 tiles (else 64 x 8)
    ZChunks zv, zs;        // z chunks of the velocity / stress launch
    bool ready = false;
};

enum { F_PEAK = NSTATE, F_SUMSQ = NSTATE + 1, F_PHRE = NSTATE + 2, F_PHIM = NSTATE + 3, NGRID = NSTATE + 4,
       F_ALT = NGRID,            // alternates of VX..SZZ (ping-pong of the fused sweep, device_params.hpp)
       NGRID_ALL = NGRID + 6 };
enum { PSI7_ALT = 6 };          // array index of the alternate of psi[7] inside the y-psi block

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
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1, 0x989680;\n"
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
// One box load into the stage, counting its bytes for the stage barrier.
// (box4s marks the boxes only this CTA reads -- plain tiles of old values, psi.  Loading them with an L2
// evict-first policy, and storing the results with st.global.cs, was measured and made every pass 3-8 % slower
// (profiles/r2b_fused.md); both load the same way.)
struct Tma {
    unsigned char *st;
    uint64_t *bar;
    uint32_t bytes;
    __device__ __forceinline__ void box4(int off, uint32_t nbytes, const CUtensorMap *map, int x, int y, int z, int f) {
        tma_load_4d(st + off, map, bar, x, y, z, f); bytes += nbytes;
    }
    __device__ __forceinline__ void box4s(int off, uint32_t nbytes, const CUtensorMap *map, int x, int y, int z, int f) {
        tma_load_4d(st + off, map, bar, x, y, z, f); bytes += nbytes;
    }
    __device__ __forceinline__ void box3(int off, uint32_t nbytes, const CUtensorMap *map, int x, int y, int z) {
        tma_load_3d(st + off, map, bar, x, y, z); bytes += nbytes;
    }
};
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap *m) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(m) : "memory");
}

// ------------------------------------------------------------------------------------------
// packed arithmetic on a thread's four x-consecutive cells (FADD2 / FMUL2 / FFMA2 on sm_100)
// ------------------------------------------------------------------------------------------
struct Q4 {
    float2 a, b;   // cells (0,1) and (2,3)
};
__device__ __forceinline__ Q4 q_ld(const float *p) {
    const float4 v = *reinterpret_cast<const float4 *>(p);
    Q4 q; q.a = make_float2(v.x, v.y); q.b = make_float2(v.z, v.w); return q;
}
__device__ __forceinline__ Q4 q_set(float s) { Q4 q; q.a = make_float2(s, s); q.b = q.a; return q; }
__device__ __forceinline__ Q4 q_make(float x, float y, float z, float w) { Q4 q; q.a = make_float2(x, y); q.b = make_float2(z, w); return q; }
__device__ __forceinline__ float2 f2neg(float2 v) { return make_float2(-v.x, -v.y); }
__device__ __forceinline__ Q4 q_add(Q4 x, Q4 y) { Q4 q; q.a = __fadd2_rn(x.a, y.a); q.b = __fadd2_rn(x.b, y.b); return q; }
__device__ __forceinline__ Q4 q_sub(Q4 x, Q4 y) { Q4 q; q.a = __fadd2_rn(x.a, f2neg(y.a)); q.b = __fadd2_rn(x.b, f2neg(y.b)); return q; }
__device__ __forceinline__ Q4 q_mul(Q4 x, Q4 y) { Q4 q; q.a = __fmul2_rn(x.a, y.a); q.b = __fmul2_rn(x.b, y.b); return q; }
__device__ __forceinline__ Q4 q_muls(Q4 x, float s) { const float2 t = make_float2(s, s); Q4 q; q.a = __fmul2_rn(x.a, t); q.b = __fmul2_rn(x.b, t); return q; }
__device__ __forceinline__ Q4 q_fma(Q4 x, Q4 y, Q4 z) { Q4 q; q.a = __ffma2_rn(x.a, y.a, z.a); q.b = __ffma2_rn(x.b, y.b, z.b); return q; }
__device__ __forceinline__ Q4 q_fmas(float s, Q4 y, Q4 z) { const float2 t = make_float2(s, s); Q4 q; q.a = __ffma2_rn(t, y.a, z.a); q.b = __ffma2_rn(t, y.b, z.b); return q; }
// x - y*z
__device__ __forceinline__ Q4 q_fnma(Q4 y, Q4 z, Q4 x) { Q4 q; q.a = __ffma2_rn(f2neg(y.a), z.a, x.a); q.b = __ffma2_rn(f2neg(y.b), z.b, x.b); return q; }
__device__ __forceinline__ float q_get(const Q4 &q, int c) { return c == 0 ? q.a.x : c == 1 ? q.a.y : c == 2 ? q.b.x : q.b.y; }
__device__ __forceinline__ void q_st(float *g, const Q4 &q) { *reinterpret_cast<float4 *>(g) = make_float4(q.a.x, q.a.y, q.b.x, q.b.y); }
__device__ __forceinline__ void q_sts(float *g, const Q4 &q) { *reinterpret_cast<float4 *>(g) = make_float4(q.a.x, q.a.y, q.b.x, q.b.y); }
// store the first nv (1..4) cells only: partial quad at the ragged x edge
__device__ __forceinline__ void q_st_n(float *g, const Q4 &q, int nv) {
    if (nv >= 4) { q_st(g, q); return; }
    g[0] = q.a.x;
    if (nv > 1) g[1] = q.a.y;
    if (nv > 2) g[2] = q.b.x;
}

// 4-point staggered difference from four values ordered along the axis (weights carry 1/dx):
// c1 (b - a) + c2 (d - z)
__device__ __forceinline__ Q4 q_d4(const Q4 &z, const Q4 &a, const Q4 &b, const Q4 &d, float c1, float c2) {
    return q_fmas(c2, q_sub(d, z), q_muls(q_sub(b, a), c1));
}
// C-PML (reading P5): psi <- b psi + a D ; D <- D + psi.  psi_old comes from the TMA stage.
__device__ __forceinline__ Q4 q_cpml(Q4 &d, const Q4 &psi_old, const Q4 &a, const Q4 &b) {
    const Q4 pn = q_fma(b, psi_old, q_mul(a, d));
    d = q_add(d, pn);
    return pn;
}

// x-direction differences of a thread's four cells from f[-2..5] around its quad (scalar: the
// operand pairs are misaligned for the packed forms).  f points at the own quad in shared memory.
struct XRow { float f[8]; };   // f[0] = cell -2 ... f[7] = cell +5
// D- (lands on the integer node): c1 (f(i)-f(i-1)) + c2 (f(i+1)-f(i-2)); needs cells -2..4
__device__ __forceinline__ Q4 x_dminus(const float *own, float c1, float c2) {
    const float2 l = *reinterpret_cast<const float2 *>(own - 2);
    const float4 o = *reinterpret_cast<const float4 *>(own);
    const float r = own[4];
    return q_make(fmaf(c2, o.y - l.x, c1 * (o.x - l.y)), fmaf(c2, o.z - l.y, c1 * (o.y - o.x)),
                  fmaf(c2, o.w - o.x, c1 * (o.z - o.y)), fmaf(c2, r - o.y, c1 * (o.w - o.z)));
}
// D+ (lands on the half node): c1 (f(i+1)-f(i)) + c2 (f(i+2)-f(i-1)); needs cells -1..5
__device__ __forceinline__ Q4 x_dplus(const float *own, float c1, float c2) {
    const float l = own[-1];
    const float4 o = *reinterpret_cast<const float4 *>(own);
    const float2 r = *reinterpret_cast<const float2 *>(own + 4);
    return q_make(fmaf(c2, o.z - l, c1 * (o.y - o.x)), fmaf(c2, o.w - o.x, c1 * (o.z - o.y)),
                  fmaf(c2, r.x - o.y, c1 * (o.w - o.z)), fmaf(c2, r.y - o.z, c1 * (r.x - o.w)));
}

__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
// reciprocal with one Newton step (finite positive x)
__device__ __forceinline__ float rcp_newton(float x) {
    const float r = rcp_approx(x);
    return fmaf(r, fmaf(-x, r, 1.0f), r);
}

// z-direction 4-point difference as an accumulator chain: when plane m arrives it is the last (+c2)
// plane of one output, the +c1 plane of the next, the -c1 plane of the one after and the first
// (-c2) plane of a new one.  Three accumulators per array replace a four-plane register window and
// need no register moves.  The completed output is the D- difference at plane m-1 (array on half
// nodes in z) or, equally, the D+ difference at plane m-2 (array on integer nodes in z).
struct ZChain {
    Q4 a1, a2, a3;
};
__device__ __forceinline__ void zc_clear(ZChain &c) { c.a1 = c.a2 = c.a3 = q_set(0.0f); }
__device__ __forceinline__ Q4 zc_push(ZChain &c, const Q4 &f, float c1, float c2) {
    const Q4 out = q_fmas(c2, f, c.a1);
    c.a1 = q_fmas(c1, f, c.a2);
    c.a2 = q_fmas(-c1, f, c.a3);
    c.a3 = q_muls(f, -c2);
    return out;
}

// ------------------------------------------------------------------------------------------
// per-thread geometry shared by both passes
// ------------------------------------------------------------------------------------------
template <class C>
struct ThreadGeom {
    int tx, ty, i0, j, nv;       // nv = valid cells of the quad (0 = inactive thread)
    bool active;
    bool in_x;                   // quad touches an x slab
    bool row_y;                  // row in a y slab
    int psx_off;                 // float offset of the quad inside an x-psi slot (low or high box)
    uint32_t gx, gy, gz;         // float offset of the quad inside an x- / y- / z-psi array at (compact) plane 0
    uint32_t gcell;              // float offset of the quad inside a grid field at plane 0
    float ay_i, by_i, ay_h, by_h;
};

template <class C>
__device__ __forceinline__ ThreadGeom<C> make_geom(const Params &p, const StagePlan &sp, int tid, int x0, int y0) {
    ThreadGeom<C> g;
    g.tx = tid % (C::TX / 4); g.ty = tid / (C::TX / 4);
    g.i0 = x0 + 4 * g.tx; g.j = y0 + g.ty;
    g.active = (g.j < p.ny) && (g.i0 < p.nx);
    g.nv = g.active ? min(4, p.nx - g.i0) : 0;
    const int P = p.P;
    const bool in_lo = g.active && P > 0 && g.i0 < P;
    const bool in_hi = g.active && P > 0 && g.i0 >= p.xhb;
    g.in_x = in_lo || in_hi;
    // low box is loaded at compact x = x0, high box at compact x = xp4 + max(x0, xhb) - xhb
    const int hi0 = max(x0, p.xhb);
    g.psx_off = in_lo ? (g.ty * sp.wxb + (g.i0 - x0)) : (sp.xhi / 4 + g.ty * sp.wxb + (g.i0 - hi0));
    const int cx = in_lo ? g.i0 : p.xp4 + (g.i0 - p.xhb);
    g.gx = (uint32_t)(cx + p.wx * g.j);
    g.row_y = g.active && P > 0 && (g.j < P || g.j >= p.ny - P);
    const int jy = g.j < P ? g.j : g.j - (p.ny - 2 * P);
    g.gy = (uint32_t)(g.i0 + p.px * jy);
    g.gz = (uint32_t)(g.i0 + p.px * g.j);
    g.gcell = (uint32_t)(p.org + g.i0 + (long long)p.px * g.j);
    g.ay_i = g.by_i = g.ay_h = g.by_h = 0.0f;
    if (g.row_y) {
        g.ay_i = __ldg(p.prof[1][0] + g.j); g.by_i = __ldg(p.prof[1][1] + g.j);
        g.ay_h = __ldg(p.prof[1][2] + g.j); g.by_h = __ldg(p.prof[1][3] + g.j);
    }
    return g;
}

// x-slab profile coefficients of the tile columns, zero outside the slabs / the grid
// (w columns per row starting at tile column `base`: the whole tile by default)
template <class C>
__device__ __forceinline__ void fill_xprof(float *sprof, const Params &p, int x0, int tid, int w = C::TX, int base = 0) {
    for (int q = tid; q < 4 * w; q += C::NT) {
        const int a = q / w, c = q % w, i = x0 + base + c;
        const bool in = p.P > 0 && i < p.nx && (i < p.P || i >= p.nx - p.P);
        sprof[q] = in ? __ldg(p.prof[0][a] + i) : 0.0f;
    }
}

struct TileX {
    bool lo, hi;       // the tile touches the low / high x slab
    int cx_lo, cx_hi;  // compact x of the two boxes
};
template <class C>
__device__ __forceinline__ TileX make_tilex(const Params &p, int x0) {
    TileX t;
    t.lo = p.P > 0 && x0 < p.P;
    t.hi = p.P > 0 && x0 + C::TX > p.xhb && x0 < p.nx;
    t.cx_lo = x0;
    t.cx_hi = p.xp4 + max(x0, p.xhb) - p.xhb;
    return t;
}
template <class C>
__device__ __forceinline__ bool tile_in_y(const Params &p, int y0) { return p.P > 0 && (y0 < p.P || y0 + C::TY > p.ny - p.P); }
template <class C>
__device__ __forceinline__ int tile_jy0(const Params &p, int y0) { return y0 < p.P ? y0 : y0 - (p.ny - 2 * p.P); }
__device__ __forceinline__ bool z_in_slab(const Params &p, int k) { return p.P > 0 && k >= 0 && k < p.nz && (k < p.P || k >= p.nz - p.P); }
__device__ __forceinline__ int z_compact(const Params &p, int k) { return k < p.P ? k : k - (p.nz - 2 * p.P); }

// the store of a quad: EDGE CTAs may hold partial quads (nx % 4 != 0)
template <bool EDGE>
__device__ __forceinline__ void q_store(float *g, const Q4 &q, int nv) {
    if (EDGE) q_st_n(g, q, nv); else q_st(g, q);
}

// ------------------------------------------------------------------------------------------
// S2: velocity pass
// ------------------------------------------------------------------------------------------
// stage slots (bytes), fixed part
template <class C>
struct VStage {
    static constexpr int SXX = 0, SYY = SXX + C::A_BYTES, SZZ = SYY + C::B_BYTES, SXY = SZZ + C::D_BYTES,
                         SXZ = SXY + C::C_BYTES, SYZ = SXZ + C::A_BYTES, VXO = SYZ + C::B_BYTES,
                         VYO = VXO + C::D_BYTES, VZO = VYO + C::D_BYTES, MAT = VZO + C::D_BYTES,
                         FIXED = MAT + C::M_BYTES;
};

// control word of one velocity iteration (StageHdr::ctrl)
enum : uint32_t {
    VC_IN0 = 1u, VC_IN1 = 2u, VC_IN2 = 4u,   // plane m / m-1 / m-2 inside the chunk
    VC_XY = 8u, VC_XZ = 16u, VC_YZ = 32u,    // plane m carries non-zero sxy / sxz / syz (halo-extended tile)
    VC_WXZ = 64u, VC_WYZ = 128u,             // some plane of m-3..m carries non-zero sxz / syz
    VC_ZS1 = 256u, VC_ZS2 = 512u,            // plane m-1 / m-2 lies in a z slab (and inside the chunk)
    VC_FL = 1024u                            // plane m (inside the chunk): all-fluid extended tile, sigma_xx stands for the three
};

// The loads of one velocity iteration m, derived from the chunk range and the flag words of planes
// m-3..m (hist, 4 bits per plane, newest lowest).
template <class C>
struct VelIssue {
    const TiledMaps *maps; const Params *p; const StagePlan *sp;
    TileX tX; bool tY; int jy0, x0, y0, kz0, kz1;
    __device__ __forceinline__ uint32_t ctrl(int m, uint32_t hist) const {
        const bool in0 = m >= kz0 && m < kz1, in1 = m - 1 >= kz0 && m - 1 < kz1, in2 = m - 2 >= kz0 && m - 2 < kz1;
        const uint32_t fl = hist & 15u, any = (hist | (hist >> 4) | (hist >> 8) | (hist >> 12)) & 15u;
        uint32_t c = (in0 ? VC_IN0 : 0u) | (in1 ? VC_IN1 : 0u) | (in2 ? VC_IN2 : 0u);
        if (fl & TF_XY) c |= VC_XY;
        if (fl & TF_XZ) c |= VC_XZ;
        if (fl & TF_YZ) c |= VC_YZ;
        if (in0 && (fl & TF_VFLUID)) c |= VC_FL;
        if (any & TF_XZ) c |= VC_WXZ;
        if (any & TF_YZ) c |= VC_WYZ;
        if (in1 && z_in_slab(*p, m - 1)) c |= VC_ZS1;
        if (in2 && z_in_slab(*p, m - 2)) c |= VC_ZS2;
        return c;
    }
    __device__ __forceinline__ void run(Tma &t, int m, uint32_t hist) const {
        using VS = VStage<C>;
        const uint32_t c = ctrl(m, hist);
        const bool xy = c & VC_XY, xz = c & VC_XZ, yz = c & VC_YZ;
        const uint32_t xbox = (uint32_t)sp->wxb * C::TY * 4;
        const int z = m + 2;
        // all-fluid extended tile: sigma_xx = sigma_yy = sigma_zz bit for bit (eS = 0, isotropic source, zero
        // start), so ONE box of sigma_xx with both halos (rows j-1 .. j+9, in the idle sxy slot) serves D+x,
        // D+y and D+z instead of the three boxes
        if (c & VC_FL) t.box4(VS::SXY, C::C_BYTES, &maps->boxC, x0 - 4, y0 - 1, z, p->icur[SXX]);
        else t.box4s(VS::SZZ, C::D_BYTES, &maps->boxD, x0, y0, z, p->icur[SZZ]);
        if (xz) t.box4(VS::SXZ, C::A_BYTES, &maps->boxA, x0 - 4, y0, z, SXZ);
        if (yz) t.box4(VS::SYZ, C::B_BYTES, &maps->boxB, x0, y0 - 2, z, SYZ);
        if (c & VC_IN0) {
            if (!(c & VC_FL)) {
                t.box4(VS::SXX, C::A_BYTES, &maps->boxA, x0 - 4, y0, z, p->icur[SXX]);
                t.box4(VS::SYY, C::B_BYTES, &maps->boxB, x0, y0 - 1, z, p->icur[SYY]);
            }
            if (xy) t.box4(VS::SXY, C::C_BYTES, &maps->boxC, x0 - 4, y0 - 2, z, SXY);
            // psi of the x-y derivatives of plane m: x terms 0..2, y terms 0..2
            const bool use[3] = {true, xy, xz};
            const bool usey[3] = {xy, true, yz};
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                if (use[q]) {
                    const int d = sp->psx + q * sp->xt;
                    if (tX.lo) t.box4s(d, xbox, &maps->psx, tX.cx_lo, y0, m, q);
                    if (tX.hi) t.box4s(d + sp->xhi, xbox, &maps->psx, tX.cx_hi, y0, m, q);
                }
                if (tY && usey[q]) t.box4s(sp->psy + q * C::D_BYTES, C::D_BYTES, &maps->psy, x0, jy0, m, q == 1 ? p->ipsi7_cur : q);
            }
        }
        if (c & VC_IN1) {
            t.box4s(VS::VXO, C::D_BYTES, &maps->boxD, x0, y0, z - 1, p->icur[VX]);
            t.box4s(VS::VYO, C::D_BYTES, &maps->boxD, x0, y0, z - 1, p->icur[VY]);
        }
        if (c & VC_IN2) t.box4s(VS::VZO, C::D_BYTES, &maps->boxD, x0, y0, z - 2, p->icur[VZ]);
        if (c & VC_ZS1) {
            const int kc = z_compact(*p, m - 1);
            if (c & VC_WXZ) t.box4s(sp->psz, C::D_BYTES, &maps->psz, x0, y0, kc, 0);
            if (c & VC_WYZ) t.box4s(sp->psz + C::D_BYTES, C::D_BYTES, &maps->psz, x0, y0, kc, 1);
        }
        if (c & VC_ZS2) t.box4s(sp->psz + 2 * C::D_BYTES, C::D_BYTES, &maps->psz, x0, y0, z_compact(*p, m - 2), 2);
        t.box3(VS::MAT, C::MX * C::MY, &maps->mat, x0, y0, m - 1);
    }
};

template <class C, bool EDGE, bool TRIM>
__device__ __forceinline__ void velocity_consume(const Params &p, const StagePlan &sp, unsigned char *stages, const float *rho_tab,
                                                 const float *sprof, uint64_t *full, uint64_t *empty, int tid, int x0, int y0,
                                                 int m_begin, int m_end) {
    using VS = VStage<C>;
    constexpr int DQ = C::D_BYTES / 4;
    const ThreadGeom<C> g = make_geom<C>(p, sp, tid, x0, y0);
    const int tx = g.tx, ty = g.ty;
    const bool active = EDGE ? g.active : true;
    const float c1 = 1.125f * p.inv_dx, c2 = (-1.0f / 24.0f) * p.inv_dx;
    const float dt2 = 2.0f * p.dt;
    const bool wall_x = EDGE && g.active && (p.nx - 1 >= g.i0) && (p.nx - 1 <= g.i0 + 3);   // quad holds cell nx-1 (P4)
    const bool wall_y = EDGE && g.j == p.ny - 1;
    const Q4 zero = q_set(0.0f);
    const int qoff = ty * C::TX + 4 * tx;             // own quad inside a D / B(row 0) box
    const int aoff = ty * C::AX + 4 + 4 * tx;         // own quad inside an A / C(row 0) box
    const uint32_t zstride = (uint32_t)(p.px * p.ny);
    // x-profile rows: width and first tile column (TRIM: only the columns that can lie in a slab are kept)
    const int spw = (TRIM && sp.spw > 0) ? sp.spw : C::TX;
    const int xbase = (TRIM && sp.spw > 0 && x0 >= p.P) ? max(x0, p.xhb) - x0 : 0;

    ZChain zxz, zyz, zzz;                             // D-z sxz, D-z syz (finish at m-1), D+z szz (finish at m-2)
    zc_clear(zxz); zc_clear(zyz); zc_clear(zzz);
    Q4 pvx = zero, pvy = zero, pvz1 = zero, pvz2 = zero;   // x-y sums of planes m-1 (pvx, pvy, pvz1) and m-2 (pvz2)
    float rho_prev[4] = {1.0f, 1.0f, 1.0f, 1.0f};          // rho of the thread's cells at plane m-2

    uint32_t goff = g.gcell + (uint32_t)(p.sz * m_begin);              // field offset of the quad at plane m
    uint32_t gxo = g.gx + (uint32_t)(p.wx * p.ny) * (uint32_t)m_begin; // x-psi offset at plane m
    uint32_t gyo = g.gy + (uint32_t)(p.px * 2 * p.P) * (uint32_t)m_begin;
    int s = 0; uint32_t ph = 0;
    for (int m = m_begin; m < m_end; ++m) {
        mbar_wait(&full[s], ph);
        const unsigned char *st = stages + s * sp.bytes;
        const StageHdr *hdr = reinterpret_cast<const StageHdr *>(st + sp.hdr);
        const uint32_t ctrl = hdr->ctrl;
        if (active) {
            const float *sA_xz = reinterpret_cast<const float *>(st + VS::SXZ) + aoff;
            const float *sB_yz = reinterpret_cast<const float *>(st + VS::SYZ) + qoff;     // row j-2
            const float *psz = reinterpret_cast<const float *>(st + sp.psz) + qoff;
            // ---- z chains: push plane m ----
            const float *sF = reinterpret_cast<const float *>(st + VS::SXY) + aoff;      // VC_FL: sigma_xx box, row j-1
            Q4 dzz = zc_push(zzz, (ctrl & VC_FL) ? q_ld(sF + C::AX) : q_ld(reinterpret_cast<const float *>(st + VS::SZZ) + qoff), c1, c2);
            Q4 dzx = zero, dzy = zero;
            if (ctrl & VC_WXZ) dzx = zc_push(zxz, (ctrl & VC_XZ) ? q_ld(sA_xz) : zero, c1, c2);
            if (ctrl & VC_WYZ) dzy = zc_push(zyz, (ctrl & VC_YZ) ? q_ld(sB_yz + 2 * C::TX) : zero, c1, c2);

            // ---- material of plane m-1: rho at i0..i0+4 of row j and i0..i0+3 of row j+1 ----
            const unsigned char *mt = st + VS::MAT + ty * C::MX + 4 * tx;
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
            if (ctrl & VC_IN1) {
                // finish vx, vy at plane m-1
                if (ctrl & VC_ZS1) {
                    const uint32_t qz = g.gz + zstride * (uint32_t)z_compact(p, m - 1);
                    const Q4 az = q_set(hdr->az1), bz = q_set(hdr->bz1);
                    if (ctrl & VC_WXZ) q_store<EDGE>(p.psi[12] + qz, q_cpml(dzx, q_ld(psz), az, bz), g.nv);
                    if (ctrl & VC_WYZ) q_store<EDGE>(p.psi[13] + qz, q_cpml(dzy, q_ld(psz + DQ), az, bz), g.nv);
                }
                const Q4 cx = q_make(dt2 * rcp_newton(rho_j[0] + rho_j[1]), dt2 * rcp_newton(rho_j[1] + rho_j[2]),
                                     dt2 * rcp_newton(rho_j[2] + rho_j[3]), dt2 * rcp_newton(rho_j[3] + rho_j[4]));
                const Q4 cy = q_make(dt2 * rcp_newton(rho_j[0] + rho_j1[0]), dt2 * rcp_newton(rho_j[1] + rho_j1[1]),
                                     dt2 * rcp_newton(rho_j[2] + rho_j1[2]), dt2 * rcp_newton(rho_j[3] + rho_j1[3]));
                Q4 ox = q_fma(cx, q_add(pvx, dzx), q_ld(reinterpret_cast<const float *>(st + VS::VXO) + qoff));
                Q4 oy = q_fma(cy, q_add(pvy, dzy), q_ld(reinterpret_cast<const float *>(st + VS::VYO) + qoff));
                if (EDGE) {
                    if (wall_x) {
                        const int wc = p.nx - 1 - g.i0;
                        if (wc == 0) ox.a.x = 0.0f; else if (wc == 1) ox.a.y = 0.0f; else if (wc == 2) ox.b.x = 0.0f; else ox.b.y = 0.0f;
                    }
                    if (wall_y) oy = zero;
                }
                const uint32_t gq = goff - (uint32_t)p.sz;
                q_store<EDGE>(p.fnxt[VX] + gq, ox, g.nv);
                q_store<EDGE>(p.fnxt[VY] + gq, oy, g.nv);
            }
            if (ctrl & VC_IN2) {
                // finish vz at plane m-2
                if (ctrl & VC_ZS2) {
                    const uint32_t qz = g.gz + zstride * (uint32_t)z_compact(p, m - 2);
                    q_store<EDGE>(p.psi[14] + qz, q_cpml(dzz, q_ld(psz + 2 * DQ), q_set(hdr->az2), q_set(hdr->bz2)), g.nv);
                }
                const Q4 cz = q_make(dt2 * rcp_newton(rho_prev[0] + rho_j[0]), dt2 * rcp_newton(rho_prev[1] + rho_j[1]),
                                     dt2 * rcp_newton(rho_prev[2] + rho_j[2]), dt2 * rcp_newton(rho_prev[3] + rho_j[3]));
                Q4 oz = q_fma(cz, q_add(pvz2, dzz), q_ld(reinterpret_cast<const float *>(st + VS::VZO) + qoff));
                if (m - 2 == p.nz - 1) oz = zero;
                q_store<EDGE>(p.fnxt[VZ] + (goff - 2u * (uint32_t)p.sz), oz, g.nv);
            }
            pvz2 = pvz1;
#pragma unroll
            for (int c = 0; c < 4; ++c) rho_prev[c] = rho_j[c];

            // ---- x-y derivative sums of plane m ----
            if (ctrl & VC_IN0) {
                Q4 dxx, dyy;
                if (ctrl & VC_FL) {
                    dxx = x_dplus(sF + C::AX, c1, c2);                                       // D+x sxx -> vx
                    dyy = q_d4(q_ld(sF), q_ld(sF + C::AX), q_ld(sF + 2 * C::AX), q_ld(sF + 3 * C::AX), c1, c2);   // D+y (syy = sxx) -> vy
                } else {
                    const float *sA_xx = reinterpret_cast<const float *>(st + VS::SXX) + aoff;
                    const float *sB_yy = reinterpret_cast<const float *>(st + VS::SYY) + qoff;   // row j-1
                    dxx = x_dplus(sA_xx, c1, c2);                                            // D+x sxx -> vx
                    dyy = q_d4(q_ld(sB_yy), q_ld(sB_yy + C::TX), q_ld(sB_yy + 2 * C::TX), q_ld(sB_yy + 3 * C::TX), c1, c2);   // D+y syy -> vy
                }
                Q4 dxy_y = zero, dxy_x = zero, dxz = zero, dyz = zero;
                if (ctrl & VC_XY) {
                    const float *sC = reinterpret_cast<const float *>(st + VS::SXY) + aoff;  // row j-2
                    dxy_x = x_dminus(sC + 2 * C::AX, c1, c2);                                // D-x sxy -> vy
                    dxy_y = q_d4(q_ld(sC), q_ld(sC + C::AX), q_ld(sC + 2 * C::AX), q_ld(sC + 3 * C::AX), c1, c2);   // D-y sxy -> vx
                }
                if (ctrl & VC_XZ) dxz = x_dminus(sA_xz, c1, c2);                             // D-x sxz -> vz
                if (ctrl & VC_YZ) dyz = q_d4(q_ld(sB_yz), q_ld(sB_yz + C::TX), q_ld(sB_yz + 2 * C::TX), q_ld(sB_yz + 3 * C::TX), c1, c2);   // D-y syz -> vz
                if (g.in_x) {
                    const float *sp_x = sprof + (4 * tx - xbase);
                    const Q4 ai = q_ld(sp_x), bi = q_ld(sp_x + spw);
                    const float *ps = reinterpret_cast<const float *>(st + sp.psx) + g.psx_off;
                    q_st(p.psi[0] + gxo, q_cpml(dxx, q_ld(ps), q_ld(sp_x + 2 * spw), q_ld(sp_x + 3 * spw)));
                    if (ctrl & VC_XY) q_st(p.psi[1] + gxo, q_cpml(dxy_x, q_ld(ps + sp.xt / 4), ai, bi));
                    if (ctrl & VC_XZ) q_st(p.psi[2] + gxo, q_cpml(dxz, q_ld(ps + sp.xt / 2), ai, bi));
                }
                if (g.row_y) {
                    const float *ps = reinterpret_cast<const float *>(st + sp.psy) + qoff;
                    const Q4 ai = q_set(g.ay_i), bi = q_set(g.by_i);
                    if (ctrl & VC_XY) q_store<EDGE>(p.psi[6] + gyo, q_cpml(dxy_y, q_ld(ps), ai, bi), g.nv);
                    q_store<EDGE>(p.psi7_nxt + gyo, q_cpml(dyy, q_ld(ps + DQ), q_set(g.ay_h), q_set(g.by_h)), g.nv);
                    if (ctrl & VC_YZ) q_store<EDGE>(p.psi[8] + gyo, q_cpml(dyz, q_ld(ps + 2 * DQ), ai, bi), g.nv);
                }
                pvx = q_add(dxx, dxy_y);
                pvy = q_add(dxy_x, dyy);
                pvz1 = q_add(dxz, dyz);
            } else {
                pvx = pvy = pvz1 = zero;
            }
        }
        goff += (uint32_t)p.sz;
        gxo += (uint32_t)(p.wx * p.ny);
        gyo += (uint32_t)(p.px * 2 * p.P);
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty[s]);
        if (++s == sp.ns) { s = 0; ph ^= 1; }
    }
}

// OCC = resident CTAs per SM the registers are budgeted for.  `spf` is the stage plan with every psi
// slot; `spc` a compact one without the y- and z-psi slots (more stages in the same shared memory) that
// a CTA uses when its tile lies outside the y slabs and its chunk outside the z slabs (spc.ns = 0:
// every CTA uses spf).  The pass is bound by the latency of its consumer warps, not by issue slots or
// DRAM: three resident CTAs (12 consumer warps per SM) measured 8 % faster than two.
// TRIM: the density table and the x-profile rows are cut to what the context uses (sp.nrho, sp.spw), which
// frees the last bytes three CTAs need with thick PMLs; the untrimmed instantiation keeps compile-time
// strides (2 % faster on config 2).
template <class C, int OCC, bool TRIM>
__global__ void __launch_bounds__(C::NT, OCC) k_velocity_tiled(const __grid_constant__ TiledMaps maps, const Params p,
                                                               const ZChunks zc, const StagePlan spf, const StagePlan spc,
                                                               const int4 *__restrict__ items) {
    using VS = VStage<C>;
    extern __shared__ __align__(1024) unsigned char smem[];
    const int tid = threadIdx.x;
    // a block is (tile, z chunk) of the launch grid, or -- with a work list (the tile columns the fused sweep does
    // not take) -- item blockIdx.x = (tile x, tile y, first plane, one past the last plane)
    int bx = blockIdx.x, by = blockIdx.y, kz0, kz1;
    if (items) { const int4 it = __ldg(items + blockIdx.x); bx = it.x; by = it.y; kz0 = it.z; kz1 = it.w; }
    else { kz0 = zc.b[blockIdx.z]; kz1 = zc.b[blockIdx.z + 1]; }
    const int x0 = bx * C::TX, y0 = by * C::TY;
    const int m_begin = kz0 - 2, m_end = kz1 + 2;   // iterations m in [m_begin, m_end)
    // (a compact plan without x-psi slots, spc.xt == 0, also needs a tile outside the x slabs)
    const bool x_slab = p.P > 0 && (x0 < p.P || (x0 + C::TX > p.xhb && x0 < p.nx));
    const bool compact = spc.ns > 0 && !tile_in_y<C>(p, y0) && !(p.P > 0 && (kz0 < p.P || kz1 > p.nz - p.P)) &&
                         (spc.xt > 0 || !x_slab);
    const StagePlan sp = compact ? spc : spf;
    unsigned char *stages = smem;
    const int nrho = (TRIM && sp.nrho > 0) ? sp.nrho : 256, spw_k = (TRIM && sp.spw > 0) ? sp.spw : C::TX;
    float *rho_tab = reinterpret_cast<float *>(smem + sp.ns * sp.bytes);
    float *sprof = rho_tab + nrho;
    uint64_t *full = reinterpret_cast<uint64_t *>(sprof + 4 * spw_k);
    uint64_t *empty = full + MAX_STAGES;

    for (int q = tid; q < nrho; q += C::NT) rho_tab[q] = p.rows[q].rho;
    fill_xprof<C>(sprof, p, x0, tid, spw_k, (TRIM && sp.spw > 0 && x0 >= p.P) ? max(x0, p.xhb) - x0 : 0);
    if (tid == 0) {
        for (int s = 0; s < sp.ns; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], C::NC / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (tid >= C::NC) {
        // ================= producer warp =================
        if (tid == C::NC) {
            const uint32_t *flags = p.flagsV + (size_t)(bx + p.ntxV * by) * (p.nz + 4) + 2;
            VelIssue<C> iss;
            iss.maps = &maps; iss.p = &p; iss.sp = &sp;
            iss.tX = make_tilex<C>(p, x0); iss.tY = tile_in_y<C>(p, y0); iss.jy0 = tile_jy0<C>(p, y0);
            iss.x0 = x0; iss.y0 = y0; iss.kz0 = kz0; iss.kz1 = kz1;
            prefetch_tmap(&maps.boxA); prefetch_tmap(&maps.boxB); prefetch_tmap(&maps.boxC);
            prefetch_tmap(&maps.boxD); prefetch_tmap(&maps.mat);
            if (p.P > 0) { prefetch_tmap(&maps.psx); prefetch_tmap(&maps.psy); prefetch_tmap(&maps.psz); }
            int s = 0; uint32_t ph = 0;
            uint32_t hist = 0;       // flag words of the last planes, 4 bits each (newest in the low nibble)
            for (int m = m_begin; m < m_end; ++m) {
                hist = (hist << 4) | (__ldg(flags + m) & 15u);
                StageHdr h;
                h.ctrl = iss.ctrl(m, hist);
                h.az1 = h.bz1 = h.az2 = h.bz2 = 0.0f;
                if (h.ctrl & VC_ZS1) { h.az1 = __ldg(p.prof[2][0] + m - 1); h.bz1 = __ldg(p.prof[2][1] + m - 1); }
                if (h.ctrl & VC_ZS2) { h.az2 = __ldg(p.prof[2][2] + m - 2); h.bz2 = __ldg(p.prof[2][3] + m - 2); }
                mbar_wait(&empty[s], ph ^ 1);
                unsigned char *st = stages + s * sp.bytes;
                StageHdr *hd = reinterpret_cast<StageHdr *>(st + sp.hdr);
                hd->ctrl = h.ctrl; hd->az1 = h.az1; hd->bz1 = h.bz1; hd->az2 = h.az2; hd->bz2 = h.bz2;
                Tma t{st, &full[s], 0};
                iss.run(t, m, hist);
                mbar_expect_tx(&full[s], t.bytes);   // the arrival that lets the phase complete comes after the loads
                if (++s == sp.ns) { s = 0; ph ^= 1; }
            }
        }
        return;
    }

    // ================= consumers =================
    const bool edge = (x0 + C::TX >= p.nx) || (y0 + C::TY >= p.ny);
    if (edge) velocity_consume<C, true, TRIM>(p, sp, stages, rho_tab, sprof, full, empty, tid, x0, y0, m_begin, m_end);
    else velocity_consume<C, false, TRIM>(p, sp, stages, rho_tab, sprof, full, empty, tid, x0, y0, m_begin, m_end);
}

// ------------------------------------------------------------------------------------------
// S3 + S4: stress, memory variables, sensor
// ------------------------------------------------------------------------------------------
template <class C>
struct SStage {
    static constexpr int VXB = 0, VYB = C::C_BYTES, VZB = 2 * C::C_BYTES, SII = 3 * C::C_BYTES,
                         RII = SII + 3 * C::D_BYTES, PEAK = RII + 3 * C::D_BYTES, SUMSQ = PEAK + C::D_BYTES,
                         SXY = SUMSQ + C::D_BYTES, RXY = SXY + C::D_BYTES, SXZ = RXY + C::D_BYTES,
                         RXZ = SXZ + C::D_BYTES, SYZ = RXZ + C::D_BYTES, RYZ = SYZ + C::D_BYTES,
                         FIXED = RYZ + C::D_BYTES;
};

// control word of one stress iteration (StageHdr::ctrl)
enum : uint32_t {
    SC_IN0 = 1u, SC_IN1 = 2u, SC_IN2 = 4u,
    SC_XY0 = 8u, SC_XZ0 = 16u, SC_YZ0 = 32u,   // plane m: finish sxy / form the D+x vz, D+y vz partials
    SC_RII1 = 64u,                             // plane m-1 has lossy cells
    SC_XZ2 = 128u, SC_YZ2 = 256u,              // plane m-2: finish sxz / syz
    SC_ZS1 = 512u, SC_ZS2 = 1024u,             // plane m-1 / m-2 lies in a z slab (and inside the chunk)
    SC_PEAK = 2048u, SC_RMS = 4096u,
    SC_RFL1 = 8192u                            // plane m-1 is lossy but holds no solid cell: r_xx = r_yy = r_zz, only r_xx moves
};

struct ShearCoef { float cU, cR; };   // dt mu_U,h and B mu_h tau_h of one shear node (readings P2, P3)
__device__ __forceinline__ ShearCoef shear_coef(float2 a, float2 b, float2 c, float2 d, float dt, float B) {
    // .x = 1/mu_R (+inf for a fluid: the harmonic mean becomes 0), .y = tau_s
    const float mu_h = 4.0f * rcp_approx((a.x + b.x) + (c.x + d.x));
    const float ts_h = 0.25f * ((a.y + b.y) + (c.y + d.y));
    const float mt = mu_h * ts_h;
    ShearCoef r; r.cU = dt * (mu_h + mt); r.cR = B * mt;
    return r;
}
// one shear node: r' = A r - cR g ; s' = s + cU g + dt/2 (r' + r)
__device__ __forceinline__ void shear_update(const ShearCoef &k, float g, float s0, float r0, float A, float hdt, float &sn, float &rn) {
    rn = fmaf(A, r0, -(k.cR * g));
    sn = s0 + fmaf(k.cU, g, hdt * (rn + r0));
}

// The loads of one stress iteration m (flag words of planes m, m-1, m-2 in the low half of hist, 4 bits
// each, newest lowest; their TF_SOLID bits in the high half, 1 bit each, newest at bit 16).
template <class C>
struct StrIssue {
    const TiledMaps *maps; const Params *p; const StagePlan *sp;
    TileX tX; bool tY; int jy0, x0, y0, kz0, kz1;
    uint32_t sens;
    __device__ __forceinline__ uint32_t ctrl(int m, uint32_t hist) const {
        const bool in0 = m >= kz0 && m < kz1, in1 = m - 1 >= kz0 && m - 1 < kz1, in2 = m - 2 >= kz0 && m - 2 < kz1;
        const uint32_t f0 = hist & 15u, f1 = (hist >> 4) & 15u, f2 = (hist >> 8) & 15u;
        uint32_t c = sens;
        if (in0) c |= SC_IN0 | ((f0 & TF_XY) ? SC_XY0 : 0u) | ((f0 & TF_XZ) ? SC_XZ0 : 0u) | ((f0 & TF_YZ) ? SC_YZ0 : 0u);
        if (in1) c |= SC_IN1 | ((f1 & TF_RII) ? (SC_RII1 | (((hist >> 17) & 1u) ? 0u : SC_RFL1)) : 0u) | (z_in_slab(*p, m - 1) ? SC_ZS1 : 0u);
        if (in2) c |= SC_IN2 | ((f2 & TF_XZ) ? SC_XZ2 : 0u) | ((f2 & TF_YZ) ? SC_YZ2 : 0u) | (z_in_slab(*p, m - 2) ? SC_ZS2 : 0u);
        return c;
    }
    // mat_off: offset of the material ring slot of plane m relative to the stage base (loads only)
    __device__ __forceinline__ void run(Tma &t, int m, uint32_t hist, int mat_off) const {
        using SS = SStage<C>;
        const uint32_t c = ctrl(m, hist);
        const uint32_t xbox = (uint32_t)sp->wxb * C::TY * 4;
        const int z = m + 2;
        t.box4(SS::VXB, C::C_BYTES, &maps->boxC, x0 - 4, y0 - 2, z, p->inxt[VX]);
        t.box4(SS::VYB, C::C_BYTES, &maps->boxC, x0 - 4, y0 - 2, z, p->inxt[VY]);
        t.box4(SS::VZB, C::C_BYTES, &maps->boxC, x0 - 4, y0 - 2, z, p->inxt[VZ]);
        if (c & SC_IN0) {
            // psi of the x-y derivatives of plane m: x terms 3 (D-x vx), 4 (D+x vy), 5 (D+x vz);
            // y terms 3 (D+y vx), 4 (D-y vy), 5 (D+y vz)
            const bool use[3] = {true, (c & SC_XY0) != 0, (c & SC_XZ0) != 0};
            const bool usey[3] = {(c & SC_XY0) != 0, true, (c & SC_YZ0) != 0};
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                if (use[q]) {
                    const int d = sp->psx + q * sp->xt;
                    if (tX.lo) t.box4s(d, xbox, &maps->psx, tX.cx_lo, y0, m, 3 + q);
                    if (tX.hi) t.box4s(d + sp->xhi, xbox, &maps->psx, tX.cx_hi, y0, m, 3 + q);
                }
                if (tY && usey[q]) t.box4s(sp->psy + q * C::D_BYTES, C::D_BYTES, &maps->psy, x0, jy0, m, 3 + q);
            }
        }
        if (c & SC_XY0) {
            t.box4s(SS::SXY, C::D_BYTES, &maps->boxD, x0, y0, z, SXY);
            t.box4s(SS::RXY, C::D_BYTES, &maps->boxD, x0, y0, z, RXY);
        }
        if (c & SC_IN1) {
#pragma unroll
            for (int q = 0; q < 3; ++q) t.box4s(SS::SII + q * C::D_BYTES, C::D_BYTES, &maps->boxD, x0, y0, z - 1, p->icur[SXX + q]);
            if (c & SC_RII1) {
                t.box4s(SS::RII, C::D_BYTES, &maps->boxD, x0, y0, z - 1, RXX);
                if (!(c & SC_RFL1)) {
#pragma unroll
                    for (int q = 1; q < 3; ++q) t.box4s(SS::RII + q * C::D_BYTES, C::D_BYTES, &maps->boxD, x0, y0, z - 1, RXX + q);
                }
            }
            // phasor mode (NEXT-3) keeps its two accumulators in the peak / sumsq slots
            if (c & SC_PEAK) t.box4s(SS::PEAK, C::D_BYTES, &maps->boxD, x0, y0, z - 1, p->do_phasor ? F_PHRE : F_PEAK);
            if (c & SC_RMS) t.box4s(SS::SUMSQ, C::D_BYTES, &maps->boxD, x0, y0, z - 1, p->do_phasor ? F_PHIM : F_SUMSQ);
            if (c & SC_ZS1) t.box4s(sp->psz + 2 * C::D_BYTES, C::D_BYTES, &maps->psz, x0, y0, z_compact(*p, m - 1), 5);
        }
        if (c & SC_XZ2) {
            t.box4s(SS::SXZ, C::D_BYTES, &maps->boxD, x0, y0, z - 2, SXZ);
            t.box4s(SS::RXZ, C::D_BYTES, &maps->boxD, x0, y0, z - 2, RXZ);
            if (c & SC_ZS2) t.box4s(sp->psz, C::D_BYTES, &maps->psz, x0, y0, z_compact(*p, m - 2), 3);
        }
        if (c & SC_YZ2) {
            t.box4s(SS::SYZ, C::D_BYTES, &maps->boxD, x0, y0, z - 2, SYZ);
            t.box4s(SS::RYZ, C::D_BYTES, &maps->boxD, x0, y0, z - 2, RYZ);
            if (c & SC_ZS2) t.box4s(sp->psz + C::D_BYTES, C::D_BYTES, &maps->psz, x0, y0, z_compact(*p, m - 2), 4);
        }
        t.box3(mat_off, C::MX * C::MY, &maps->mat, x0, y0, m);
    }
};

template <class C, bool EDGE>
__device__ __forceinline__ void stress_consume(const Params &p, const StagePlan &sp, unsigned char *stages, unsigned char *mat_ring,
                                               const int MR, const float4 *tabN, const float2 *tabS, const float *sprof,
                                               uint64_t *full, uint64_t *empty, int tid, int x0, int y0, int m_begin, int m_end) {
    using SS = SStage<C>;
    constexpr int DQ = C::D_BYTES / 4;
    const ThreadGeom<C> g = make_geom<C>(p, sp, tid, x0, y0);
    const int tx = g.tx, ty = g.ty;
    const bool active = EDGE ? g.active : true;
    const float c1 = 1.125f * p.inv_dx, c2 = (-1.0f / 24.0f) * p.inv_dx;
    const float dt = p.dt, hdt = p.half_dt, A = p.A, B = p.B;
    const Q4 zero = q_set(0.0f);
    const int qoff = ty * C::TX + 4 * tx;
    const int coff = (ty + 2) * C::AX + 4 + 4 * tx;    // own quad inside a C box
    const int moff = ty * C::MX + 4 * tx;
    const uint32_t zstride = (uint32_t)(p.px * p.ny);

    ZChain zvx, zvy, zvz;          // D+z vx, D+z vy (finish at m-2), D-z vz (finish at m-1)
    zc_clear(zvx); zc_clear(zvy); zc_clear(zvz);
    Q4 nxx = zero, nyy = zero;     // vxx, vyy of plane m-1
    Q4 dxz1 = zero, dxz2 = zero, dyz1 = zero, dyz2 = zero;   // D+x vz, D+y vz of planes m-1 and m-2

    uint32_t goff = g.gcell + (uint32_t)(p.sz * m_begin);
    uint32_t gxo = g.gx + (uint32_t)(p.wx * p.ny) * (uint32_t)m_begin;
    uint32_t gyo = g.gy + (uint32_t)(p.px * 2 * p.P) * (uint32_t)m_begin;
    int s = 0; uint32_t ph = 0;
    int mr0 = ((m_begin % MR) + MR) % MR;   // ring slot of plane m
    for (int m = m_begin; m < m_end; ++m) {
        mbar_wait(&full[s], ph);
        const unsigned char *st = stages + s * sp.bytes;
        const StageHdr *hdr = reinterpret_cast<const StageHdr *>(st + sp.hdr);
        const uint32_t ctrl = hdr->ctrl;
        const int mr1 = mr0 == 0 ? MR - 1 : mr0 - 1;          // plane m-1
        const int mr2 = mr1 == 0 ? MR - 1 : mr1 - 1;          // plane m-2
        if (active) {
            const float *cvx = reinterpret_cast<const float *>(st + SS::VXB) + coff;
            const float *cvy = cvx + C::C_BYTES / 4;
            const float *cvz = cvy + C::C_BYTES / 4;
            const float *dbase = reinterpret_cast<const float *>(st) + qoff;
            const float *psz = reinterpret_cast<const float *>(st + sp.psz) + qoff;
            const unsigned char *mat0 = mat_ring + mr0 * C::M_BYTES + moff;
            const unsigned char *mat1 = mat_ring + mr1 * C::M_BYTES + moff;
            const unsigned char *mat2 = mat_ring + mr2 * C::M_BYTES + moff;

            // ---- z chains: push plane m ----
            const Q4 fvx = q_ld(cvx), fvy = q_ld(cvy), fvz = q_ld(cvz);
            Q4 vzz = zc_push(zvz, fvz, c1, c2);     // D-z vz at m-1
            Q4 vx_z = zc_push(zvx, fvx, c1, c2);    // D+z vx at m-2
            Q4 vy_z = zc_push(zvy, fvy, c1, c2);    // D+z vy at m-2

            if (ctrl & SC_IN1) {
                // finish the normal stresses, their memory variables and the sensor at plane m-1
                if (ctrl & SC_ZS1) {
                    const uint32_t qz = g.gz + zstride * (uint32_t)z_compact(p, m - 1);
                    q_store<EDGE>(p.psi[17] + qz, q_cpml(vzz, q_ld(psz + 2 * DQ), q_set(hdr->az1), q_set(hdr->bz1)), g.nv);
                }
                const uint32_t mw = *reinterpret_cast<const uint32_t *>(mat1);
                const float4 r0 = tabN[mw & 255u], r1 = tabN[(mw >> 8) & 255u], r2 = tabN[(mw >> 16) & 255u], r3 = tabN[mw >> 24];
                const Q4 eP = q_make(r0.x, r1.x, r2.x, r3.x), eS = q_make(r0.y, r1.y, r2.y, r3.y);
                const Q4 th = q_add(q_add(nxx, nyy), vzz);
                const Q4 ePth = q_mul(eP, th);
                const Q4 vii[3] = {nxx, nyy, vzz};
                const uint32_t gq = goff - (uint32_t)p.sz;
                Q4 tr = zero;
                if (ctrl & SC_RFL1) {
                    // no solid cell in the tile-plane: eS = bS = 0, so the three memory variables obey one and
                    // the same recursion from the same (zero) start and only r_xx is kept in memory; the
                    // arithmetic below is the general branch's with the terms that are exactly zero left out
                    // (x - 0 * y = x bit for bit), so both branches give the same bits
                    const Q4 bP = q_make(r0.z, r1.z, r2.z, r3.z);
                    const Q4 bPth = q_mul(bP, th);
                    const Q4 rold = q_ld(dbase + SS::RII / 4);
                    const Q4 rn = q_sub(q_muls(rold, A), bPth);
                    const Q4 inc = q_fmas(hdt, q_add(rn, rold), ePth);
                    q_store<EDGE>(p.f[RXX] + gq, rn, g.nv);
#pragma unroll
                    for (int q = 0; q < 3; ++q) {
                        const Q4 sn = q_add(q_ld(dbase + SS::SII / 4 + q * DQ), inc);
                        q_store<EDGE>(p.fnxt[SXX + q] + gq, sn, g.nv);
                        tr = q_add(tr, sn);
                    }
                } else if (ctrl & SC_RII1) {
                    const Q4 bP = q_make(r0.z, r1.z, r2.z, r3.z), bS = q_make(r0.w, r1.w, r2.w, r3.w);
                    const Q4 bPth = q_mul(bP, th);
#pragma unroll
                    for (int q = 0; q < 3; ++q) {
                        const Q4 oth = q_sub(th, vii[q]);
                        const Q4 eU = q_fnma(eS, oth, ePth);
                        const Q4 eR = q_fnma(bS, oth, bPth);
                        const Q4 rold = q_ld(dbase + SS::RII / 4 + q * DQ);
                        const Q4 rn = q_sub(q_muls(rold, A), eR);
                        const Q4 sn = q_add(q_ld(dbase + SS::SII / 4 + q * DQ), q_fmas(hdt, q_add(rn, rold), eU));
                        q_store<EDGE>(p.fnxt[SXX + q] + gq, sn, g.nv);
                        q_store<EDGE>(p.f[RXX + q] + gq, rn, g.nv);
                        tr = q_add(tr, sn);
                    }
                } else {
#pragma unroll
                    for (int q = 0; q < 3; ++q) {
                        const Q4 eU = q_fnma(eS, q_sub(th, vii[q]), ePth);
                        const Q4 sn = q_add(q_ld(dbase + SS::SII / 4 + q * DQ), eU);
                        q_store<EDGE>(p.fnxt[SXX + q] + gq, sn, g.nv);
                        tr = q_add(tr, sn);
                    }
                }
                if (ctrl & (SC_PEAK | SC_RMS)) {
                    const Q4 pr = q_muls(tr, -1.0f / 3.0f);
                    if (p.do_phasor) {
                        // single-frequency DFT of p: A += p cos(w t), B += p sin(w t)
                        q_store<EDGE>(p.phre + gq, q_fmas(p.ph_cos, pr, q_ld(dbase + SS::PEAK / 4)), g.nv);
                        q_store<EDGE>(p.phim + gq, q_fmas(p.ph_sin, pr, q_ld(dbase + SS::SUMSQ / 4)), g.nv);
                    } else if (ctrl & SC_PEAK) {
                        const Q4 pk = q_ld(dbase + SS::PEAK / 4);
                        q_store<EDGE>(p.peak + gq, q_make(fmaxf(pk.a.x, fabsf(pr.a.x)), fmaxf(pk.a.y, fabsf(pr.a.y)),
                                                          fmaxf(pk.b.x, fabsf(pr.b.x)), fmaxf(pk.b.y, fabsf(pr.b.y))), g.nv);
                    }
                    if (!p.do_phasor && (ctrl & SC_RMS)) q_store<EDGE>(p.sumsq + gq, q_fma(pr, pr, q_ld(dbase + SS::SUMSQ / 4)), g.nv);
                }
            }
            if (ctrl & (SC_XZ2 | SC_YZ2)) {
                // finish sxz, syz (+ r) at plane m-2
                const uint32_t qz = g.gz + zstride * (uint32_t)z_compact(p, m - 2);
                const Q4 az = q_set(hdr->az2), bz = q_set(hdr->bz2);
                const uint32_t gq = goff - 2u * (uint32_t)p.sz;
                // materials: row j at planes m-2 (mat2) and m-1 (mat1), cells i0..i0+4; row j+1 cells i0..i0+3
                float2 m2[5], m1[5];
#pragma unroll
                for (int c = 0; c < 5; ++c) { m2[c] = tabS[mat2[c]]; m1[c] = tabS[mat1[c]]; }
                if (ctrl & SC_XZ2) {
                    if (ctrl & SC_ZS2) q_store<EDGE>(p.psi[15] + qz, q_cpml(vx_z, q_ld(psz), az, bz), g.nv);
                    const Q4 gg4 = q_add(vx_z, dxz2);
                    const Q4 so = q_ld(dbase + SS::SXZ / 4), ro = q_ld(dbase + SS::RXZ / 4);
                    float os[4], orr[4];
#pragma unroll
                    for (int c = 0; c < 4; ++c)   // cells (i..i+1, j, k..k+1)
                        shear_update(shear_coef(m2[c], m2[c + 1], m1[c], m1[c + 1], dt, B), q_get(gg4, c), q_get(so, c), q_get(ro, c), A, hdt, os[c], orr[c]);
                    q_store<EDGE>(p.f[SXZ] + gq, q_make(os[0], os[1], os[2], os[3]), g.nv);
                    q_store<EDGE>(p.f[RXZ] + gq, q_make(orr[0], orr[1], orr[2], orr[3]), g.nv);
                }
                if (ctrl & SC_YZ2) {
                    if (ctrl & SC_ZS2) q_store<EDGE>(p.psi[16] + qz, q_cpml(vy_z, q_ld(psz + DQ), az, bz), g.nv);
                    const Q4 gg4 = q_add(vy_z, dyz2);
                    const Q4 so = q_ld(dbase + SS::SYZ / 4), ro = q_ld(dbase + SS::RYZ / 4);
                    float os[4], orr[4];
#pragma unroll
                    for (int c = 0; c < 4; ++c)   // cells (i, j..j+1, k..k+1)
                        shear_update(shear_coef(m2[c], tabS[mat2[C::MX + c]], m1[c], tabS[mat1[C::MX + c]], dt, B), q_get(gg4, c), q_get(so, c),
                                     q_get(ro, c), A, hdt, os[c], orr[c]);
                    q_store<EDGE>(p.f[SYZ] + gq, q_make(os[0], os[1], os[2], os[3]), g.nv);
                    q_store<EDGE>(p.f[RYZ] + gq, q_make(orr[0], orr[1], orr[2], orr[3]), g.nv);
                }
            }
            dxz2 = dxz1; dyz2 = dyz1;

            // ---- x-y derivatives of plane m ----
            if (ctrl & SC_IN0) {
                Q4 vxx = x_dminus(cvx, c1, c2);                                                       // D-x vx
                Q4 vyy = q_d4(q_ld(cvy - 2 * C::AX), q_ld(cvy - C::AX), fvy, q_ld(cvy + C::AX), c1, c2);  // D-y vy
                Q4 vx_y = zero, vy_x = zero, vz_x = zero, vz_y = zero;
                if (ctrl & SC_XY0) {
                    vx_y = q_d4(q_ld(cvx - C::AX), fvx, q_ld(cvx + C::AX), q_ld(cvx + 2 * C::AX), c1, c2);   // D+y vx
                    vy_x = x_dplus(cvy, c1, c2);                                                      // D+x vy
                }
                if (ctrl & SC_XZ0) vz_x = x_dplus(cvz, c1, c2);                                       // D+x vz
                if (ctrl & SC_YZ0) vz_y = q_d4(q_ld(cvz - C::AX), fvz, q_ld(cvz + C::AX), q_ld(cvz + 2 * C::AX), c1, c2);   // D+y vz
                if (g.in_x) {
                    const float *sp_x = sprof + 4 * tx;
                    const Q4 ah = q_ld(sp_x + 2 * C::TX), bh = q_ld(sp_x + 3 * C::TX);
                    const float *ps = reinterpret_cast<const float *>(st + sp.psx) + g.psx_off;
                    q_st(p.psi[3] + gxo, q_cpml(vxx, q_ld(ps), q_ld(sp_x), q_ld(sp_x + C::TX)));
                    if (ctrl & SC_XY0) q_st(p.psi[4] + gxo, q_cpml(vy_x, q_ld(ps + sp.xt / 4), ah, bh));
                    if (ctrl & SC_XZ0) q_st(p.psi[5] + gxo, q_cpml(vz_x, q_ld(ps + sp.xt / 2), ah, bh));
                }
                if (g.row_y) {
                    const float *ps = reinterpret_cast<const float *>(st + sp.psy) + qoff;
                    const Q4 ah = q_set(g.ay_h), bh = q_set(g.by_h);
                    if (ctrl & SC_XY0) q_store<EDGE>(p.psi[9] + gyo, q_cpml(vx_y, q_ld(ps), ah, bh), g.nv);
                    q_store<EDGE>(p.psi[10] + gyo, q_cpml(vyy, q_ld(ps + DQ), q_set(g.ay_i), q_set(g.by_i)), g.nv);
                    if (ctrl & SC_YZ0) q_store<EDGE>(p.psi[11] + gyo, q_cpml(vz_y, q_ld(ps + 2 * DQ), ah, bh), g.nv);
                }
                nxx = vxx; nyy = vyy; dxz1 = vz_x; dyz1 = vz_y;
                if (ctrl & SC_XY0) {
                    // finish sxy, rxy at plane m: material of the 4 cells (i..i+1, j..j+1, m)
                    const Q4 gxy = q_add(vx_y, vy_x);
                    const Q4 so = q_ld(dbase + SS::SXY / 4), ro = q_ld(dbase + SS::RXY / 4);
                    float2 ma[5], mb[5];
#pragma unroll
                    for (int c = 0; c < 5; ++c) { ma[c] = tabS[mat0[c]]; mb[c] = tabS[mat0[C::MX + c]]; }
                    float os[4], orr[4];
#pragma unroll
                    for (int c = 0; c < 4; ++c)
                        shear_update(shear_coef(ma[c], ma[c + 1], mb[c], mb[c + 1], dt, B), q_get(gxy, c), q_get(so, c), q_get(ro, c), A, hdt, os[c], orr[c]);
                    q_store<EDGE>(p.f[SXY] + goff, q_make(os[0], os[1], os[2], os[3]), g.nv);
                    q_store<EDGE>(p.f[RXY] + goff, q_make(orr[0], orr[1], orr[2], orr[3]), g.nv);
                }
            }
        }
        goff += (uint32_t)p.sz;
        gxo += (uint32_t)(p.wx * p.ny);
        gyo += (uint32_t)(p.px * 2 * p.P);
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty[s]);
        if (++s == sp.ns) { s = 0; ph ^= 1; }
        if (++mr0 == MR) mr0 = 0;
    }
}

template <class C>
__global__ void __launch_bounds__(C::NT, C::TY >= 16 ? 1 : 2) k_stress_tiled(const __grid_constant__ TiledMaps maps, const Params p,
                                                           const ZChunks zc, const StagePlan sp, const int4 *__restrict__ items) {
    using SS = SStage<C>;
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *stages = smem;
    const int MR = sp.ns + 2;                                   // material ring: planes m-2..m in use, ns-1 in flight
    const int NM = (p.n_mat + 31) & ~31;                        // table rows kept in shared memory
    unsigned char *mat_ring = smem + sp.ns * sp.bytes;
    float4 *tabN = reinterpret_cast<float4 *>(mat_ring + MR * C::M_BYTES);   // eP, eS, bP, bS
    float2 *tabS = reinterpret_cast<float2 *>(tabN + NM);                   // 1/mu_R (inf = fluid), tau_s
    float *sprof = reinterpret_cast<float *>(tabS + NM);
    uint64_t *full = reinterpret_cast<uint64_t *>(sprof + 4 * C::TX);
    uint64_t *empty = full + MAX_STAGES;

    const int tid = threadIdx.x;
    int bx = blockIdx.x, by = blockIdx.y, kz0, kz1;      // (tile, z chunk) of the grid, or an item of the work list
    if (items) { const int4 it = __ldg(items + blockIdx.x); bx = it.x; by = it.y; kz0 = it.z; kz1 = it.w; }
    else { kz0 = zc.b[blockIdx.z]; kz1 = zc.b[blockIdx.z + 1]; }
    const int x0 = bx * C::TX, y0 = by * C::TY;
    const int m_begin = kz0 - 2, m_end = kz1 + 2;

    for (int q = tid; q < NM; q += C::NT) {
        const KRow r = p.rows[q];
        tabN[q] = make_float4(r.eP, r.eS, r.bP, r.bS);
        tabS[q] = make_float2(r.solid == 0.0f ? __int_as_float(0x7f800000) : r.invMu, r.tauS);
    }
    fill_xprof<C>(sprof, p, x0, tid);
    if (tid == 0) {
        for (int s = 0; s < sp.ns; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], C::NC / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (tid >= C::NC) {
        // ================= producer warp =================
        if (tid == C::NC) {
            const uint32_t *flags = p.flagsS + (size_t)(bx + p.ntxS * by) * (p.nz + 4) + 2;
            StrIssue<C> iss;
            iss.maps = &maps; iss.p = &p; iss.sp = &sp;
            iss.tX = make_tilex<C>(p, x0); iss.tY = tile_in_y<C>(p, y0); iss.jy0 = tile_jy0<C>(p, y0);
            iss.x0 = x0; iss.y0 = y0; iss.kz0 = kz0; iss.kz1 = kz1;
            iss.sens = p.do_phasor ? (SC_PEAK | SC_RMS) : ((p.do_peak ? SC_PEAK : 0u) | (p.do_rms ? SC_RMS : 0u));
            prefetch_tmap(&maps.boxC); prefetch_tmap(&maps.boxD); prefetch_tmap(&maps.mat);
            if (p.P > 0) { prefetch_tmap(&maps.psx); prefetch_tmap(&maps.psy); prefetch_tmap(&maps.psz); }
            int s = 0; uint32_t ph = 0;
            int mr = ((m_begin % MR) + MR) % MR;
            uint32_t hist = 0;       // flag words of planes m, m-1, m-2 ..., 4 bits each
            for (int m = m_begin; m < m_end; ++m) {
                {
                    const uint32_t fw = __ldg(flags + m);
                    hist = ((hist << 4) & 0xffffu) | (fw & 15u) | (((((hist >> 16) << 1) | ((fw >> 4) & 1u)) & 0xffffu) << 16);
                }
                StageHdr h;
                h.ctrl = iss.ctrl(m, hist);
                h.az1 = h.bz1 = h.az2 = h.bz2 = 0.0f;
                if (h.ctrl & SC_ZS1) { h.az1 = __ldg(p.prof[2][0] + m - 1); h.bz1 = __ldg(p.prof[2][1] + m - 1); }
                if (h.ctrl & SC_ZS2) { h.az2 = __ldg(p.prof[2][2] + m - 2); h.bz2 = __ldg(p.prof[2][3] + m - 2); }
                mbar_wait(&empty[s], ph ^ 1);
                unsigned char *st = stages + s * sp.bytes;
                StageHdr *hd = reinterpret_cast<StageHdr *>(st + sp.hdr);
                hd->ctrl = h.ctrl; hd->az1 = h.az1; hd->bz1 = h.bz1; hd->az2 = h.az2; hd->bz2 = h.bz2;
                Tma t{st, &full[s], 0};
                iss.run(t, m, hist, (int)(mat_ring + mr * C::M_BYTES - st));
                mbar_expect_tx(&full[s], t.bytes);   // the arrival that lets the phase complete comes after the loads
                if (++mr == MR) mr = 0;
                if (++s == sp.ns) { s = 0; ph ^= 1; }
            }
        }
        return;
    }

    // ================= consumers =================
    const bool edge = (x0 + C::TX >= p.nx) || (y0 + C::TY >= p.ny);
    if (edge) stress_consume<C, true>(p, sp, stages, mat_ring, MR, tabN, tabS, sprof, full, empty, tid, x0, y0, m_begin, m_end);
    else stress_consume<C, false>(p, sp, stages, mat_ring, MR, tabN, tabS, sprof, full, empty, tid, x0, y0, m_begin, m_end);
}

// ------------------------------------------------------------------------------------------
// S0 on the device: tile-class flags from the index map
// ------------------------------------------------------------------------------------------
// One CTA per (tile, plane).  solid(m) = mu_R > 0; a shear node is "solid" when its four cells are
// (reading P2; out-of-grid neighbours are the replicated edge of the private index map).
// pass 0: velocity flags (taken over the halo-extended tile the pass reads), pass 1: stress flags.
// vfluid (pass 0 only): also set TF_VFLUID where the extended tile holds no solid cell (off once the caller
// has written a normal stress: sigma_xx = sigma_yy = sigma_zz is then no longer guaranteed)
template <class C>
__global__ void __launch_bounds__(128) k_tile_flags(const Params p, uint32_t *__restrict__ flags, const int ntx, const int pass, const int dense,
                                                    const int vfluid) {
    __shared__ uint32_t sf;
    const int x0 = blockIdx.x * C::TX, y0 = blockIdx.y * C::TY, k = blockIdx.z;
    if (threadIdx.x == 0) sf = 0;
    __syncthreads();
    uint32_t f = 0;
    if (dense) {
        f = pass == 0 ? (TF_XY | TF_XZ | TF_YZ) : (TF_XY | TF_XZ | TF_YZ | TF_RII | TF_SOLID);
    } else {
        const int h = pass == 0 ? 2 : 0;
        const int EX = C::TX + 2 * h, EY = C::TY + 2 * h;
        for (int q = threadIdx.x; q < EX * EY; q += blockDim.x) {
            const int i = x0 - h + q % EX, j = y0 - h + q / EX;
            if (i < 0 || j < 0 || i >= p.nx || j >= p.ny) continue;
            const uint8_t *mp = p.mat + i + (long long)p.px * j + p.sz * k;
            const KRow r000 = p.rows[mp[0]];
            const float s000 = r000.solid, s100 = p.rows[mp[1]].solid, s010 = p.rows[mp[p.px]].solid, s110 = p.rows[mp[p.px + 1]].solid;
            const float s001 = p.rows[mp[p.sz]].solid, s101 = p.rows[mp[p.sz + 1]].solid, s011 = p.rows[mp[p.sz + p.px]].solid;
            const bool nxy = s000 * s100 * s010 * s110 != 0.0f;
            const bool nxz = s000 * s100 * s001 * s101 != 0.0f;
            const bool nyz = s000 * s010 * s001 * s011 != 0.0f;
            const bool inx = i >= x0 && i < x0 + C::TX, iny = j >= y0 && j < y0 + C::TY;
            if (nxy) f |= TF_XY;
            if (nxz && iny) f |= TF_XZ;      // velocity reads sxz with an x halo only
            if (nyz && inx) f |= TF_YZ;      // ... syz with a y halo only
            if (pass == 1 && (r000.bP != 0.0f || r000.bS != 0.0f)) f |= TF_RII;
            if (s000 != 0.0f) f |= TF_SOLID;
        }
    }
    if (f) atomicOr(&sf, f);
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t w = sf;
        if (pass == 0) {
            w &= (TF_XY | TF_XZ | TF_YZ);
            if (vfluid && !dense && !(sf & TF_SOLID)) w |= TF_VFLUID;
        }
        flags[(size_t)(blockIdx.x + ntx * blockIdx.y) * (p.nz + 4) + 2 + k] = w;
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

inline int round128(int v) { return (v + 127) / 128 * 128; }
inline CUtensorMapL2promotion l2_promotion_of(int k) {
    return k == 1 ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B : k == 2 ? CU_TENSOR_MAP_L2_PROMOTION_NONE
         : k == 3 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B : CU_TENSOR_MAP_L2_PROMOTION_L2_128B;
}

// z chunks: a few long equal chunks (about 2.6 waves of resident CTAs; every chunk costs 4 priming
// planes) followed by a tail of chunks of halving length, not below 8 planes.  Measured on config 2:
// 90 90 90 90 45 25 12 8 planes -> 39.0 Gcell/s, nine equal chunks of 50 -> 36.6, three of 150 -> 33.6.
inline ZChunks plan_chunks(int nz, long long tiles, long long slots, double waves) {
    ZChunks z;
    // small grids (configs 0, 1): the whole launch fits the resident CTAs about once.  A CTA's time is its number
    // of iterations (planes + 4 priming planes; the data sits in L2), so the launch is cut into as many equal
    // chunks as fill ONE wave -- config 0: 8 tiles x 32 chunks of 2 planes (6 iterations instead of 12), config 1:
    // 32 tiles x 9 chunks instead of 16 chunks in two waves
    if (tiles * ((nz + 7) / 8) <= slots + slots / 3 && tiles <= slots) {
        int n = (int)std::min<long long>(slots / tiles, std::min(nz / 2, MAX_CHUNKS));
        n = std::max(1, n);
        for (int c = 0; c <= n; ++c) z.b[c] = (int)((long long)nz * c / n);
        z.n = n;
        return z;
    }
    int big = (int)std::floor(waves * (double)slots / (double)tiles + 0.5);
    big = std::max(1, std::min(big, std::min(nz / 8, MAX_CHUNKS - 8)));
    const int len = std::max(8, (nz + big) / (big + 1));
    int pos = 0, n = 0;
    z.b[0] = 0;
    while (n < big && nz - pos >= len + 8) { pos += len; z.b[++n] = pos; }
    while (nz - pos >= 16 && n < MAX_CHUNKS - 1) { pos += (nz - pos + 1) / 2; z.b[++n] = pos; }
    if (pos < nz) z.b[++n] = nz;
    z.n = n;
    return z;
}
inline bool parse_chunks(const char *env, int nz, ZChunks &z) {   // "56,56,...": explicit lengths (experiments)
    if (!env || !*env) return false;
    int pos = 0, n = 0;
    z.b[0] = 0;
    const char *c = env;
    while (*c && n < MAX_CHUNKS && pos < nz) {
        const int len = std::atoi(c);
        if (len <= 0) break;
        pos = std::min(nz, pos + len); z.b[++n] = pos;
        while (*c && *c != ',') ++c;
        if (*c == ',') ++c;
    }
    if (pos < nz && n < MAX_CHUNKS) z.b[++n] = nz;
    z.n = n;
    return n > 0 && z.b[n] == nz;
}

template <class C>
inline int encode_maps(PFN_encodeTiled enc, TiledMaps &maps, const Layout &L, const Params &p, char *const psi_base[3],
                       const long long psi_stride[3], int wxb, int l2_promotion = 0) {
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    auto encode = [&](CUtensorMap *m, CUtensorMapDataType ty, int rank, void *base, const cuuint64_t *gdim, const cuuint64_t *gstr,
                      const cuuint32_t *box, const char *what) -> int {
        CUresult r = enc(m, ty, rank, base, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                         l2_promotion_of(l2_promotion), CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) {
            std::snprintf(tiled_err_buf(), 256, "cuTensorMapEncodeTiled(%s) failed: %d", what, (int)r);
            return BVFDTD_ECUDA;
        }
        return 0;
    };
    const long long fstride = (const char *)p.f[1] - (const char *)p.f[0];
    {
        void *base = (void *)(p.f[0] + (L.org - 2 * L.sz));      // cell (0,0,-2)
        const cuuint64_t gdim[4] = {(cuuint64_t)L.px, (cuuint64_t)L.py, (cuuint64_t)(L.nz + 4), (cuuint64_t)NGRID_ALL};
        const cuuint64_t gstr[3] = {(cuuint64_t)L.px * 4, (cuuint64_t)L.sz * 4, (cuuint64_t)fstride};
        struct { CUtensorMap *m; cuuint32_t bx, by; } boxes[4] = {
            {&maps.boxA, (cuuint32_t)C::AX, (cuuint32_t)C::TY}, {&maps.boxB, (cuuint32_t)C::TX, (cuuint32_t)C::BY},
            {&maps.boxC, (cuuint32_t)C::AX, (cuuint32_t)C::BY}, {&maps.boxD, (cuuint32_t)C::TX, (cuuint32_t)C::TY}};
        for (auto &b : boxes) {
            const cuuint32_t box[4] = {b.bx, b.by, 1, 1};
            if (int rc = encode(b.m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, base, gdim, gstr, box, "field box")) return rc;
        }
    }
    {
        const cuuint64_t mdim[3] = {(cuuint64_t)L.px, (cuuint64_t)L.py, (cuuint64_t)(L.nz + 1)};
        const cuuint64_t mstr[2] = {(cuuint64_t)L.px, (cuuint64_t)L.sz};
        const cuuint32_t mbox[3] = {(cuuint32_t)C::MX, (cuuint32_t)C::MY, 1};
        if (int rc = encode(&maps.mat, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, (void *)p.mat, mdim, mstr, mbox, "material box")) return rc;
    }
    if (L.P > 0) {
        {   // x slabs: (wx, ny, nz, 6)
            const cuuint64_t d[4] = {(cuuint64_t)L.wx, (cuuint64_t)L.ny, (cuuint64_t)L.nz, 6};
            const cuuint64_t s[3] = {(cuuint64_t)L.wx * 4, (cuuint64_t)L.wx * L.ny * 4, (cuuint64_t)psi_stride[0]};
            const cuuint32_t b[4] = {(cuuint32_t)wxb, (cuuint32_t)C::TY, 1, 1};
            if (int rc = encode(&maps.psx, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, psi_base[0], d, s, b, "psi x box")) return rc;
        }
        {   // y slabs: (px, 2P, nz, 6)
            const cuuint64_t d[4] = {(cuuint64_t)L.px, (cuuint64_t)(2 * L.P), (cuuint64_t)L.nz, 7};   // 6 terms + the alternate of psi[7]
            const cuuint64_t s[3] = {(cuuint64_t)L.px * 4, (cuuint64_t)L.px * 2 * L.P * 4, (cuuint64_t)psi_stride[1]};
            const cuuint32_t b[4] = {(cuuint32_t)C::TX, (cuuint32_t)C::TY, 1, 1};
            if (int rc = encode(&maps.psy, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, psi_base[1], d, s, b, "psi y box")) return rc;
        }
        {   // z slabs: (px, ny, 2P, 6)
            const cuuint64_t d[4] = {(cuuint64_t)L.px, (cuuint64_t)L.ny, (cuuint64_t)(2 * L.P), 6};
            const cuuint64_t s[3] = {(cuuint64_t)L.px * 4, (cuuint64_t)L.px * L.ny * 4, (cuuint64_t)psi_stride[2]};
            const cuuint32_t b[4] = {(cuuint32_t)C::TX, (cuuint32_t)C::TY, 1, 1};
            if (int rc = encode(&maps.psz, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, psi_base[2], d, s, b, "psi z box")) return rc;
        }
    }
    return 0;
}

template <class C>
// yz_slots / x_slots: reserve the y- and z-psi (x-psi) slots (velocity pass: per-CTA compact plans)
inline StagePlan make_stage(const Layout &L, int fixed, int ns, int extra, int wxb, int hdr_at = -1, bool yz_slots = true,
                            bool x_slots = true) {
    StagePlan s{};
    s.wxb = wxb;
    s.xb = L.P > 0 ? round128(wxb * C::TY * 4) : 0;
    s.yb = C::D_BYTES;
    // header: its own 128 bytes, or (hdr_at >= 0) the unused tail of an existing slot
    s.hdr = hdr_at >= 0 ? hdr_at : fixed;
    s.psx = hdr_at >= 0 ? fixed : fixed + 128;
    // a tile touches both x slabs only on grids narrower than a tile + the slabs
    const bool both = L.P > 0 && (C::TX > L.xhb || L.P > C::TX);
    s.xhi = both ? s.xb : 0;
    s.xt = both ? 2 * s.xb : s.xb;
    if (!x_slots) s.xt = s.xhi = 0;
    s.psy = s.psx + 3 * s.xt;
    s.psz = s.psy + (L.P > 0 && yz_slots ? 3 * C::D_BYTES : 0);
    s.bytes = s.psz + (L.P > 0 && yz_slots ? 3 * C::D_BYTES : 0);
    s.ns = ns;
    s.smem = ns * s.bytes + extra;
    return s;
}

// launch-plan requests (bvfdtd_opts.tuning; 0 = the library's own choice).  The library reads no environment
// variable; a build with -DBVFDTD_DEV_KNOBS additionally honours BVFDTD_NS_V / _NS_S / _WAVES / _ZB_V / _ZB_S /
// _VERBOSE for experiments.
struct PlanTuning {
    int occ_v = 0;      // 0 auto, 2 or 3 resident CTAs of the velocity pass
    int stress_ty = 0;  // 0 auto, 8 or 16 rows per stress tile
    int l2_promotion = 0;   // experiments: 0 = 128 B (default), 1 = 64 B, 2 = none, 3 = 256 B (field tensor maps)
    int fused_chunk = 0;    // experiments: planes per chunk of the fused sweep (0 = the library's choice)
};

inline const char *dev_knob(const char *name) {
#ifdef BVFDTD_DEV_KNOBS
    return std::getenv(name);
#else
    (void)name;
    return nullptr;
#endif
}

inline int tiled_plan_create(TiledPlan &plan, Layout &L, Params &p, char *const psi_base[3], const long long psi_stride[3], bool dense,
                             const PlanTuning &tune = PlanTuning{}) {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
        std::snprintf(tiled_err_buf(), 256, "cuTensorMapEncodeTiled entry point unavailable (%s)", cudaGetErrorString(e));
        (void)cudaGetLastError();
        return BVFDTD_ECUDA;
    }
    PFN_encodeTiled enc = (PFN_encodeTiled)fn;
    // the grid arrays (15 state, peak, sumsq, the two phasor accumulators) are laid out back to back at a constant stride
    const long long fstride = (const char *)p.f[1] - (const char *)p.f[0];
    for (int q = 0; q < NSTATE; ++q)
        if ((const char *)p.f[q] - (const char *)p.f[0] != fstride * q) return BVFDTD_EINVAL;
    if ((const char *)p.peak - (const char *)p.f[0] != fstride * F_PEAK) return BVFDTD_EINVAL;
    if ((const char *)p.sumsq - (const char *)p.f[0] != fstride * F_SUMSQ) return BVFDTD_EINVAL;
    if ((const char *)p.phre - (const char *)p.f[0] != fstride * F_PHRE) return BVFDTD_EINVAL;
    if ((const char *)p.phim - (const char *)p.f[0] != fstride * F_PHIM) return BVFDTD_EINVAL;
    const int wxb = L.P > 0 ? std::min(L.xph, CfgV::TX) : 4;
    if (int rc = encode_maps<CfgV>(enc, plan.mv, L, p, psi_base, psi_stride, wxb, tune.l2_promotion)) return rc;

    const int bar_bytes = 2 * MAX_STAGES * 8;
    int dev = 0, sms = 148, smem_max = 227 * 1024;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const char *env_v = dev_knob("BVFDTD_NS_V"), *env_s = dev_knob("BVFDTD_NS_S");
    int ns_v = env_v ? std::atoi(env_v) : 3, ns_s = env_s ? std::atoi(env_s) : 0;
    ns_v = std::max(2, std::min(MAX_STAGES, ns_v));
    const int v_extra = 256 * 4 + 4 * CfgV::TX * 4 + bar_bytes;
    // the velocity stage header lives in the slack of the material slot (720 of 768 bytes used)
    static_assert(CfgV::M_BYTES - CfgV::MX * CfgV::MY >= (int)sizeof(StageHdr), "no room for the header behind the material box");
    const int v_hdr = VStage<CfgV>::MAT + CfgV::M_BYTES - (int)sizeof(StageHdr);
    const int smem_sm = 228 * 1024;
    // velocity pass, in order of preference (measured on config 2, PML 16: 0.320 / 0.337 / 0.344 ms):
    //   THREE resident CTAs per SM (124 registers): 3 stages where the CTA needs no y- / z-psi slots
    //   (compact plan), 2 stages elsewhere;  needs 3 (smem + 1 KB) <= 228 KB;
    //   two resident CTAs (141 registers), up to 3 stages (thick PMLs).
    const int occ_req = tune.occ_v;
    plan.svc = StagePlan{};
    plan.occ_v = 2;
    // (the dense sweep fills every stage and is bandwidth-bound: it measured better with 2 x 3 stages; small
    // grids are launch-latency bound and lose more to the extra chunks than they gain)
    if (occ_req != 2 && !env_v && (occ_req == 3 || (!dense && L.nz - 2 * L.P >= 128))) {
        // every byte counts against 3 (smem + 1 KB) <= 228 KB: the density table holds the materials in use,
        // and the x-profile rows only the (at most 32) columns of a tile that can lie in a slab
        const bool both = L.P > 0 && (CfgV::TX > L.xhb || L.P > CfgV::TX);
        int spw = CfgV::TX, nrho = 256;
        {
            // (only when the untrimmed plan does not fit)
            const StagePlan f0 = make_stage<CfgV>(L, VStage<CfgV>::FIXED, L.P > 0 ? 2 : 3, v_extra, wxb, v_hdr);
            if (3 * (f0.smem + 1024) > smem_sm) {
                if (L.P > 0 && !both && wxb <= 32 && ((L.P + 3) & ~3) <= 32) spw = 32;
                nrho = std::min(256, (p.n_mat + 31) & ~31);
            }
        }
        const int extra3 = nrho * 4 + 4 * spw * 4 + bar_bytes;
        StagePlan full2 = make_stage<CfgV>(L, VStage<CfgV>::FIXED, L.P > 0 ? 2 : 3, extra3, wxb, v_hdr);
        StagePlan comp3 = make_stage<CfgV>(L, VStage<CfgV>::FIXED, 3, extra3, wxb, v_hdr, false);            // x-psi slots only
        if (L.P > 0 && 3 * (comp3.smem + 1024) > smem_sm)
            comp3 = make_stage<CfgV>(L, VStage<CfgV>::FIXED, 3, extra3, wxb, v_hdr, false, false);           // no psi slot at all
        const int need = std::max(full2.smem, L.P > 0 ? comp3.smem : 0);
        if (3 * (need + 1024) <= smem_sm && need <= smem_max) {
            full2.spw = comp3.spw = spw == CfgV::TX ? 0 : spw;
            full2.nrho = comp3.nrho = nrho == 256 ? 0 : nrho;
            plan.sv = full2;
            if (L.P > 0) plan.svc = comp3;
            plan.sv.smem = need;
            plan.occ_v = 3;
        }
    }
    if (plan.occ_v == 2) {
        plan.sv = make_stage<CfgV>(L, VStage<CfgV>::FIXED, ns_v, v_extra, wxb, v_hdr);
        // two resident CTAs per SM matter more than a third stage
        while (plan.sv.ns > 2 && (plan.sv.smem > smem_max || 2 * (plan.sv.smem + 1024) > smem_sm))
            plan.sv = make_stage<CfgV>(L, VStage<CfgV>::FIXED, plan.sv.ns - 1, v_extra, wxb, v_hdr);
    }
    // stress pass, in order of preference (measured on config 2: 0.647 / 0.673 / 0.775 ms):
    //   64 x 8 tiles, 2 stages, TWO resident CTAs per SM (fits up to PML 16 with <= 128 materials);
    //   64 x 16 tiles, 2 stages, one CTA with 8 consumer warps;
    //   64 x 8 tiles, up to 3 stages, one CTA (very thick PML on a narrow grid).
    const int nm = (p.n_mat + 31) & ~31;
    auto s_extra16 = [&](int ns) { return (ns + 2) * CfgS::M_BYTES + nm * 24 + 4 * CfgS::TX * 4 + bar_bytes; };
    auto s_extra8 = [&](int ns) { return (ns + 2) * CfgS8::M_BYTES + nm * 24 + 4 * CfgS8::TX * 4 + bar_bytes; };
    const int ty_req = tune.stress_ty;
    bool chosen = false;
    // (the dense sweep, whose every iteration fills the whole stage, measured better on the 64 x 16 tile)
    if (ty_req != 16 && (!ns_s || ns_s == 2) && !(dense && ty_req != 8)) {
        plan.ss = make_stage<CfgS8>(L, SStage<CfgS8>::FIXED, 2, s_extra8(2), wxb);
        if (2 * (plan.ss.smem + 1024) <= smem_sm) { plan.s16 = false; chosen = true; }
    }
    if (!chosen && ty_req != 8) {
        const int ns = ns_s ? std::max(2, std::min(MAX_STAGES, ns_s)) : 2;
        plan.ss = make_stage<CfgS>(L, SStage<CfgS>::FIXED, ns, s_extra16(ns), wxb);
        while (plan.ss.smem > smem_max && plan.ss.ns > 2) plan.ss = make_stage<CfgS>(L, SStage<CfgS>::FIXED, plan.ss.ns - 1, s_extra16(plan.ss.ns - 1), wxb);
        if (plan.ss.smem <= smem_max) { plan.s16 = true; chosen = true; }
    }
    if (!chosen) {
        const int ns = ns_s ? std::max(2, std::min(MAX_STAGES, ns_s)) : 3;
        plan.s16 = false;
        plan.ss = make_stage<CfgS8>(L, SStage<CfgS8>::FIXED, ns, s_extra8(ns), wxb);
        while (plan.ss.smem > smem_max && plan.ss.ns > 2) plan.ss = make_stage<CfgS8>(L, SStage<CfgS8>::FIXED, plan.ss.ns - 1, s_extra8(plan.ss.ns - 1), wxb);
    }
    if (plan.ss.smem > smem_max || plan.sv.smem > smem_max) {
        std::snprintf(tiled_err_buf(), 256, "pml %d needs %d bytes of shared memory per CTA (max %d)", L.P, plan.ss.smem, smem_max);
        return BVFDTD_EINVAL;
    }
    const int sty = plan.s16 ? CfgS::TY : CfgS8::TY;
    L.ntxS = (L.nx + CfgS::TX - 1) / CfgS::TX;
    L.ntyS = (L.ny + sty - 1) / sty;
    p.ntxS = L.ntxS; p.ntyS = L.ntyS;
    if (int rc = plan.s16 ? encode_maps<CfgS>(enc, plan.ms, L, p, psi_base, psi_stride, wxb, tune.l2_promotion)
                          : encode_maps<CfgS8>(enc, plan.ms, L, p, psi_base, psi_stride, wxb, tune.l2_promotion)) return rc;
    int occ_v = 1, occ_s = 1;
    const bool trim_v = plan.sv.spw > 0 || plan.sv.nrho > 0;
    if (plan.occ_v == 3 && trim_v) {
        e = cudaFuncSetAttribute(k_velocity_tiled<CfgV, 3, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.sv.smem);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_v, k_velocity_tiled<CfgV, 3, true>, CfgV::NT, plan.sv.smem);
    } else if (plan.occ_v == 3) {
        e = cudaFuncSetAttribute(k_velocity_tiled<CfgV, 3, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.sv.smem);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_v, k_velocity_tiled<CfgV, 3, false>, CfgV::NT, plan.sv.smem);
    } else {
        e = cudaFuncSetAttribute(k_velocity_tiled<CfgV, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.sv.smem);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_v, k_velocity_tiled<CfgV, 2, false>, CfgV::NT, plan.sv.smem);
    }
    if (plan.s16) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_stress_tiled<CfgS>, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.ss.smem);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_s, k_stress_tiled<CfgS>, CfgS::NT, plan.ss.smem);
    } else {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_stress_tiled<CfgS8>, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.ss.smem);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_s, k_stress_tiled<CfgS8>, CfgS8::NT, plan.ss.smem);
    }
    if (e != cudaSuccess) {
        std::snprintf(tiled_err_buf(), 256, "kernel attribute/occupancy query: %s", cudaGetErrorString(e));
        (void)cudaGetLastError();
        return BVFDTD_ECUDA;
    }
    plan.occ_v_res = occ_v; plan.occ_s_res = occ_s;
    const char *env_w = dev_knob("BVFDTD_WAVES");
    const double waves = env_w ? std::atof(env_w) : 2.6;
    plan.zv = plan_chunks(L.nz, (long long)L.ntxV * L.ntyV, (long long)std::max(1, occ_v) * sms, waves);
    if (plan.svc.ns > 0 && L.P >= 8 && L.nz - 2 * L.P >= 16) {
        // the z slabs get chunks of their own, so that every other chunk can run the compact stage plan
        // (measured on config 2 with three resident CTAs: nine chunks of 42 planes + a short tail 0.318 ms,
        //  six of 60 0.327, four of 84 0.334, three of 105 0.357)
        const ZChunks in = plan_chunks(L.nz - 2 * L.P, (long long)L.ntxV * L.ntyV, (long long)std::max(1, occ_v) * sms, env_w ? waves : 3.9);
        if (in.n + 2 <= MAX_CHUNKS) {
            ZChunks z;
            z.n = in.n + 2;
            z.b[0] = 0;
            for (int c = 0; c <= in.n; ++c) z.b[c + 1] = L.P + in.b[c];
            z.b[z.n] = L.nz;
            plan.zv = z;
        }
    }
    plan.zs = plan_chunks(L.nz, (long long)L.ntxS * L.ntyS, (long long)std::max(1, occ_s) * sms, waves);
    parse_chunks(dev_knob("BVFDTD_ZB_V"), L.nz, plan.zv);
    parse_chunks(dev_knob("BVFDTD_ZB_S"), L.nz, plan.zs);
    if (dev_knob("BVFDTD_VERBOSE")) {
        std::fprintf(stderr, "[bvfdtd] velocity: ns %d (compact %d) stage %d smem %d occ %d; stress: tile 64x%d ns %d stage %d smem %d occ %d\n[bvfdtd] z chunks velocity:",
                     plan.sv.ns, plan.svc.ns, plan.sv.bytes, plan.sv.smem, occ_v, plan.s16 ? 16 : 8, plan.ss.ns, plan.ss.bytes, plan.ss.smem, occ_s);
        for (int c = 0; c < plan.zv.n; ++c) std::fprintf(stderr, " %d", plan.zv.b[c + 1] - plan.zv.b[c]);
        std::fprintf(stderr, "; stress:");
        for (int c = 0; c < plan.zs.n; ++c) std::fprintf(stderr, " %d", plan.zs.b[c + 1] - plan.zs.b[c]);
        std::fprintf(stderr, "\n");
    }
    plan.ready = true;
    return 0;
}

inline void tiled_plan_destroy(TiledPlan &plan) { plan.ready = false; }

// r_yy and r_zz of the tile-planes in which only r_xx is kept (SC_RFL1): fill them in from r_xx (before
// they are read back, and before the context switches to the dense sweep)
__global__ void __launch_bounds__(128) k_fill_rii(const Params p, const int ty_tile) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= p.nx) return;
    const uint32_t fw = p.flagsS[(size_t)(i / CfgS::TX + p.ntxS * (j / ty_tile)) * (p.nz + 4) + 2 + k];
    if (!(fw & TF_RII) || (fw & TF_SOLID)) return;
    const long long c = p.org + i + (long long)p.px * j + p.sz * k;
    const float r = p.f[RXX][c];
    p.f[RYY][c] = r;
    p.f[RZZ][c] = r;
}
inline void tiled_fill_rii(const TiledPlan &plan, const Params &p, cudaStream_t st) {
    k_fill_rii<<<dim3((p.nx + 127) / 128, p.ny, p.nz), 128, 0, st>>>(p, plan.s16 ? CfgS::TY : CfgS8::TY);
}

inline void tiled_flags(const TiledPlan &plan, const Params &p, uint32_t *flagsV, uint32_t *flagsS, bool dense, cudaStream_t st,
                        bool vfluid = true) {
    k_tile_flags<CfgV><<<dim3(p.ntxV, p.ntyV, p.nz), 128, 0, st>>>(p, flagsV, p.ntxV, 0, dense ? 1 : 0, vfluid ? 1 : 0);
    if (plan.s16) k_tile_flags<CfgS><<<dim3(p.ntxS, p.ntyS, p.nz), 128, 0, st>>>(p, flagsS, p.ntxS, 1, dense ? 1 : 0, 0);
    else k_tile_flags<CfgS8><<<dim3(p.ntxS, p.ntyS, p.nz), 128, 0, st>>>(p, flagsS, p.ntxS, 1, dense ? 1 : 0, 0);
}
// items != nullptr: a work list of n_items (tile, z range) entries replaces the (tiles) x (chunks) grid
inline int tiled_velocity(TiledPlan &plan, const Params &p, cudaStream_t st, const int4 *items = nullptr, int n_items = 0) {
    if (items && n_items == 0) return 0;
    const dim3 grid = items ? dim3(n_items) : dim3(p.ntxV, p.ntyV, plan.zv.n);
    if (plan.occ_v == 3 && (plan.sv.spw > 0 || plan.sv.nrho > 0))
        k_velocity_tiled<CfgV, 3, true><<<grid, CfgV::NT, plan.sv.smem, st>>>(plan.mv, p, plan.zv, plan.sv, plan.svc, items);
    else if (plan.occ_v == 3) k_velocity_tiled<CfgV, 3, false><<<grid, CfgV::NT, plan.sv.smem, st>>>(plan.mv, p, plan.zv, plan.sv, plan.svc, items);
    else k_velocity_tiled<CfgV, 2, false><<<grid, CfgV::NT, plan.sv.smem, st>>>(plan.mv, p, plan.zv, plan.sv, plan.svc, items);
    return 0;
}
inline int tiled_stress(TiledPlan &plan, const Params &p, cudaStream_t st, const int4 *items = nullptr, int n_items = 0) {
    if (items && n_items == 0) return 0;
    const dim3 grid = items ? dim3(n_items) : dim3(p.ntxS, p.ntyS, plan.zs.n);
    if (plan.s16) k_stress_tiled<CfgS><<<grid, CfgS::NT, plan.ss.smem, st>>>(plan.ms, p, plan.zs, plan.ss, items);
    else k_stress_tiled<CfgS8><<<grid, CfgS8::NT, plan.ss.smem, st>>>(plan.ms, p, plan.zs, plan.ss, items);
    return 0;
}

}  // namespace bvfdtd
