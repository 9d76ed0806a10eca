// kernels_fused.cuh -- the fused single-sweep step for all-fluid tile columns (SURVEY.md 8(d) "fused
// single-sweep").
//
// In a fluid the shear stresses are identically zero and sigma_xx = sigma_yy = sigma_zz (= -p), r_xx = r_yy =
// r_zz, so Eq. 1 reduces to one stress, one memory variable and the three velocities.  Where a
// 64 x 8 tile has no solid cell within reach of its stencils over a run of z planes, ONE CTA does the velocity
// update AND the stress update of the run in one z-march, instead of the two passes re-reading v and sigma:
//
//   iteration m (the plane of sigma_xx that arrives):
//     vx, vy at plane m      from the in-plane differences of sigma_xx(m); the CTA also forms vx on the two
//                            columns left / one column right of its tile and vy on the two rows below / one row
//                            above it (what D-x vx and D-y vy of its own cells reach), redundantly with the
//                            neighbouring CTAs and bit-identically to them; the new planes go through a
//                            double-buffered shared-memory exchange (one named barrier per plane);
//     vz at plane m-2        D+z sigma needs planes m-3..m (accumulator chain, kernels_tiled.cuh);
//     sigma, r_xx, sensor    at plane m-3: D-z vz needs vz up to plane m-2.
//   The chunk [kz0, kz1) also forms vz at planes kz0-2, kz0-1 and kz1 for its own D-z vz (not stored).
//
// Because CTAs of one launch read sigma_xx, v and the y-psi of D+y sigma of time level n in each other's tiles
// while the owners write level n+1, these arrays are ping-ponged (device_params.hpp: icur / inxt / fnxt).  The
// other tile columns run the two passes of kernels_tiled.cuh from work lists, against the same two copies.
//
// Per cell-step in a lossy fluid with the running peak on: read sigma 4 + v 12 + r 4 + peak 4 + index 1,
// write v 12 + sigma 4 + r 4 + peak 4 = 49 B (the two passes move 90 B there).
//
// The arithmetic is the two passes' (same operations in the same order on the same operands), so the results
// are bit-identical to theirs: tests/test_gpu_fused.py.
#pragma once
#include "kernels_tiled.cuh"

#include <algorithm>
#include <vector>

namespace bvfdtd {

using CfgF = TileCfg<64, 8>;

struct FusedMaps {
    CUtensorMap boxE;               // (TX + 8) x (TY + 6): sigma_xx with both halos, rows y0-3 .. y0+TY+2
    CUtensorMap boxA, boxB, boxD;   // as in TiledMaps (x halo / y halo rows y0-2 .. y0+TY+1 / plain tile)
    CUtensorMap mat;                // (TX + 32) x (TY + 4) bytes at (x0 - 16, y0 - 2)
    CUtensorMap psx, psy, psz;      // psi boxes of the tile (as in TiledMaps)
    CUtensorMap psyE;               // TX x (TY + 4) rows of a y-psi array: psi[7] under the rows y0-2 .. y0+TY+1
};

constexpr int round128c(int v) { return (v + 127) / 128 * 128; }

template <class C>
struct FStage {
    static constexpr int EX = C::TX + 8, EY = C::TY + 6;
    static constexpr int E_BYTES = round128c(EX * EY * 4);
    static constexpr int MXF = C::TX + 32, MYF = C::TY + 4;
    static constexpr int MF_BYTES = round128c(MXF * MYF);
    static constexpr int SIG = 0, VXO = SIG + E_BYTES, VYO = VXO + C::A_BYTES, VZO = VYO + C::B_BYTES,
                         RXX = VZO + C::D_BYTES, PEAK = RXX + C::D_BYTES, SUMSQ = PEAK + C::D_BYTES,
                         MAT = SUMSQ + C::D_BYTES, HDR = MAT + MF_BYTES, FIXED = HDR + 128;
    // the exchange planes of the new vx (A-box layout) and vy (B-box layout, rows y0-2 .. y0+TY), double-buffered
    static constexpr int XV_FLOATS = C::A_BYTES / 4, XY_FLOATS = C::B_BYTES / 4, XBUF_FLOATS = XV_FLOATS + XY_FLOATS;
};

// control word of one fused iteration (StageHdr::ctrl)
enum : uint32_t {
    FC_V0 = 1u,        // plane m inside the chunk: finish vx, vy
    FC_VZ2 = 2u,       // form vz at plane m-2 (a plane of the chunk, or one of the three recomputed around it)
    FC_VZ2S = 4u,      // ... and store it (plane inside the chunk)
    FC_S3 = 8u,        // plane m-3 inside the chunk: finish sigma, r_xx, the sensor
    FC_LOSSY3 = 16u,   // plane m-3 has lossy cells
    FC_ZS2 = 32u,      // plane m-2 (inside the chunk) lies in a z slab
    FC_ZS3 = 64u,      // plane m-3 (inside the chunk) lies in a z slab
    FC_WYY3 = 128u, FC_WZZ3 = 256u,   // plane m-3: also write sigma_yy / sigma_zz (a two-pass neighbour reads them)
    FC_PEAK = 512u, FC_RMS = 1024u
};

struct FusedPlan {
    FusedMaps maps;
    StagePlan full{}, compact{};   // with / without the y- and z-psi slots (per-CTA choice, as in the velocity pass)
    int smem = 0;
    int n_f = 0, n_v = 0, n_s = 0;             // work items of the fused sweep, the velocity pass, the stress pass
    const int4 *items_f = nullptr, *items_v = nullptr, *items_s = nullptr;   // device
    long long planes_f = 0, planes_all = 0;    // tile-planes the fused sweep takes / all (64 x 8 tiles)
    bool ready = false;
};

__device__ __forceinline__ void consumer_barrier(int n) { asm volatile("bar.sync 1, %0;" ::"r"(n) : "memory"); }

template <class C>
struct FusedIssue {
    const FusedMaps *maps; const Params *p; const StagePlan *sp;
    TileX tX; bool tY, tYe; int jy0, jy0e, x0, y0, kz0, kz1;
    uint32_t sens;
    // f3 = flag word of plane m-3
    __device__ __forceinline__ uint32_t ctrl(int m, uint32_t f3) const {
        uint32_t c = sens;
        if (m >= kz0 && m < kz1) c |= FC_V0;
        const int k2 = m - 2, k3 = m - 3;
        if (k2 >= kz0 - 2 && k2 <= kz1 && k2 >= 0 && k2 < p->nz - 1) {
            c |= FC_VZ2;
            if (k2 >= kz0 && k2 < kz1) c |= FC_VZ2S | (z_in_slab(*p, k2) ? FC_ZS2 : 0u);
        }
        if (k3 >= kz0 && k3 < kz1) {
            c |= FC_S3 | ((f3 & FF_LOSSY) ? FC_LOSSY3 : 0u) | ((f3 & FF_WYY) ? FC_WYY3 : 0u) | ((f3 & FF_WZZ) ? FC_WZZ3 : 0u) |
                 (z_in_slab(*p, k3) ? FC_ZS3 : 0u);
        }
        return c;
    }
    __device__ __forceinline__ void run(Tma &t, int m, uint32_t c) const {
        using FS = FStage<C>;
        const uint32_t xbox = (uint32_t)sp->wxb * C::TY * 4;
        const int z = m + 2;
        // sigma_xx(m) with both halos and the materials of plane m: every iteration (a plane outside the
        // allocation is zero-filled by the hardware: the zero ghost of reading P4)
        t.box4(FS::SIG, FS::EX * FS::EY * 4, &maps->boxE, x0 - 4, y0 - 3, z, p->icur[SXX]);
        t.box3(FS::MAT, FS::MXF * FS::MYF, &maps->mat, x0 - 16, y0 - 2, m);
        if (c & FC_V0) {
            t.box4(FS::VXO, C::A_BYTES, &maps->boxA, x0 - 4, y0, z, p->icur[VX]);
            t.box4(FS::VYO, C::B_BYTES, &maps->boxB, x0, y0 - 2, z, p->icur[VY]);
            // psi of plane m: x terms 0 (D+x sxx) and 3 (D-x vx); y terms 1 (D+y syy, with the halo rows) and 4 (D-y vy)
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const int d = sp->psx + q * sp->xt;
                if (tX.lo) t.box4s(d, xbox, &maps->psx, tX.cx_lo, y0, m, 3 * q);
                if (tX.hi) t.box4s(d + sp->xhi, xbox, &maps->psx, tX.cx_hi, y0, m, 3 * q);
            }
            if (tYe) t.box4(sp->psy, C::B_BYTES, &maps->psyE, x0, jy0e - 2, m, p->ipsi7_cur);
            if (tY) t.box4s(sp->psy + C::B_BYTES, C::D_BYTES, &maps->psy, x0, jy0, m, 4);
        }
        if (c & FC_VZ2) {
            t.box4s(FS::VZO, C::D_BYTES, &maps->boxD, x0, y0, z - 2, p->icur[VZ]);
            if (c & FC_ZS2) t.box4s(sp->psz, C::D_BYTES, &maps->psz, x0, y0, z_compact(*p, m - 2), 2);
        }
        if (c & FC_S3) {
            if (c & FC_LOSSY3) t.box4s(FS::RXX, C::D_BYTES, &maps->boxD, x0, y0, z - 3, RXX);
            if (c & FC_PEAK) t.box4s(FS::PEAK, C::D_BYTES, &maps->boxD, x0, y0, z - 3, F_PEAK);
            if (c & FC_RMS) t.box4s(FS::SUMSQ, C::D_BYTES, &maps->boxD, x0, y0, z - 3, F_SUMSQ);
            if (c & FC_ZS3) t.box4s(sp->psz + C::D_BYTES, C::D_BYTES, &maps->psz, x0, y0, z_compact(*p, m - 3), 5);
        }
    }
};

template <class C, bool EDGE>
__device__ __forceinline__ void fused_consume(const Params &p, const StagePlan &sp, unsigned char *stages, float *xbuf,
                                              const float *rho_tab, const float2 *tabP, const float *sprof, uint64_t *full,
                                              uint64_t *empty, int tid, int x0, int y0, int kz0, int kz1, bool tYe, int jrow0e) {
    using FS = FStage<C>;
    constexpr int DQ = C::D_BYTES / 4, EX = FS::EX, MXF = FS::MXF;
    const ThreadGeom<C> g = make_geom<C>(p, sp, tid, x0, y0);
    const int tx = g.tx, ty = g.ty;
    const bool active = EDGE ? g.active : true;
    const float c1 = 1.125f * p.inv_dx, c2 = (-1.0f / 24.0f) * p.inv_dx;
    const float dt2 = 2.0f * p.dt, hdt = p.half_dt, A = p.A;
    const Q4 zero = q_set(0.0f);
    const int eoff = (ty + 3) * EX + 4 + 4 * tx;        // own quad inside the sigma box
    const int aoff = ty * C::AX + 4 + 4 * tx;           // ... inside an A box (old vx, new-vx exchange plane)
    const int boff = (ty + 2) * C::TX + 4 * tx;         // ... inside a B box (old vy, new-vy exchange plane, psi[7] rows)
    const int qoff = ty * C::TX + 4 * tx;               // ... inside a D box
    const int moff = (ty + 2) * MXF + 16 + 4 * tx;      // ... inside the material box
    const uint32_t zstride = (uint32_t)(p.px * p.ny);
    // held wall layers (reading P4) and cells beyond the grid: a partial quad keeps zeros there
    const int nzero_x = EDGE ? max(0, min(4, g.i0 + 4 - (p.nx - 1))) : 0;   // trailing cells of the quad with i >= nx-1
    const bool wall_y = EDGE && g.j >= p.ny - 1;

    // the halo work of this thread: warp 0 forms vx on the columns x0-2, x0-1, x0+TX (3 cells x TY rows),
    // warps 1..3 form vy on the rows y0-2, y0-1, y0+TY (16 quads each)
    const int warp = tid >> 5, lane = tid & 31;
    const bool ex_vx = warp == 0 && lane < 3 * C::TY;
    const int exr = lane / 3, exc = (lane - 3 * exr) == 2 ? C::TX : (lane - 3 * exr) - 2;     // row, column of the vx cell
    const bool ex_vx_in = ex_vx && x0 + exc >= 0 && x0 + exc < p.nx - 1 && y0 + exr < p.ny;
    const bool ex_vy = warp >= 1 && warp <= 3 && lane < C::TX / 4;
    const int eyr = warp == 1 ? -2 : warp == 2 ? -1 : C::TY;                                  // row of the vy quad
    const bool ex_vy_in = ex_vy && y0 + eyr >= 0 && y0 + eyr < p.ny - 1 && x0 + 4 * lane < p.nx;
    float eay = 0.0f, eby = 0.0f;                                                             // half-node y profile of that row
    const bool ex_vy_slab = ex_vy_in && p.P > 0 && (y0 + eyr < p.P || y0 + eyr >= p.ny - p.P);
    if (ex_vy_slab) { eay = __ldg(p.prof[1][2] + y0 + eyr); eby = __ldg(p.prof[1][3] + y0 + eyr); }
    (void)jrow0e; (void)tYe;

    ZChain zs, zv;                 // D+z sigma (finishes at m-2), D-z vz (finishes at m-3)
    zc_clear(zs); zc_clear(zv);
    Q4 s1 = zero, s2 = zero, s3 = zero;        // sigma_xx of the own quad at planes m-1, m-2, m-3
    Q4 t1 = zero, t2 = zero, t3 = zero;        // D-x vx + D-y vy at planes m-1, m-2, m-3
    uint32_t w1 = 0, w2 = 0, w3 = 0;           // material bytes of the own quad at planes m-1, m-2, m-3

    const int m_begin = kz0 - 3, m_end = kz1 + 3;
    // offsets may run below zero for the priming planes: unsigned wrap-around, only used for planes inside the chunk
    uint32_t goff = g.gcell + (uint32_t)((long long)p.sz * m_begin);
    uint32_t gxo = g.gx + (uint32_t)((long long)(p.wx * p.ny) * m_begin);
    uint32_t gyo = g.gy + (uint32_t)((long long)(p.px * 2 * p.P) * m_begin);
    int s = 0; uint32_t ph = 0;
    for (int m = m_begin; m < m_end; ++m) {
        mbar_wait(&full[s], ph);
        const unsigned char *st = stages + s * sp.bytes;
        const StageHdr *hdr = reinterpret_cast<const StageHdr *>(st + FS::HDR);
        const uint32_t ctrl = hdr->ctrl;
        const float *sig = reinterpret_cast<const float *>(st + FS::SIG);
        const unsigned char *mat = st + FS::MAT;
        Q4 sig_own = zero, tnew = zero;
        uint32_t w0 = 0;
        if (active) {
            sig_own = q_ld(sig + eoff);
            w0 = *reinterpret_cast<const uint32_t *>(mat + moff);
            const float *psz = reinterpret_cast<const float *>(st + sp.psz) + qoff;
            // ---- vz at plane m-2 ----
            Q4 dzz = zc_push(zs, sig_own, c1, c2);
            Q4 vzn = zero;
            if (ctrl & FC_VZ2) {
                if (ctrl & FC_ZS2) {
                    const uint32_t qz = g.gz + zstride * (uint32_t)z_compact(p, m - 2);
                    q_store<EDGE>(p.psi[14] + qz, q_cpml(dzz, q_ld(psz), q_set(hdr->az2), q_set(hdr->bz2)), g.nv);
                }
                const Q4 cz = q_make(dt2 * rcp_newton(rho_tab[w2 & 255u] + rho_tab[w1 & 255u]),
                                     dt2 * rcp_newton(rho_tab[(w2 >> 8) & 255u] + rho_tab[(w1 >> 8) & 255u]),
                                     dt2 * rcp_newton(rho_tab[(w2 >> 16) & 255u] + rho_tab[(w1 >> 16) & 255u]),
                                     dt2 * rcp_newton(rho_tab[w2 >> 24] + rho_tab[w1 >> 24]));
                vzn = q_fma(cz, dzz, q_ld(reinterpret_cast<const float *>(st + FS::VZO) + qoff));
                if (ctrl & FC_VZ2S) q_store<EDGE>(p.fnxt[VZ] + (goff - 2u * (uint32_t)p.sz), vzn, g.nv);
            }
            // ---- sigma, r_xx, sensor at plane m-3 ----
            Q4 vzz = zc_push(zv, vzn, c1, c2);
            if (ctrl & FC_S3) {
                if (ctrl & FC_ZS3) {
                    const uint32_t qz = g.gz + zstride * (uint32_t)z_compact(p, m - 3);
                    q_store<EDGE>(p.psi[17] + qz, q_cpml(vzz, q_ld(psz + DQ), q_set(hdr->az1), q_set(hdr->bz1)), g.nv);
                }
                const float2 r0 = tabP[w3 & 255u], r1 = tabP[(w3 >> 8) & 255u], r2 = tabP[(w3 >> 16) & 255u], r3 = tabP[w3 >> 24];
                const Q4 th = q_add(t3, vzz);
                const Q4 ePth = q_mul(q_make(r0.x, r1.x, r2.x, r3.x), th);
                const uint32_t gq = goff - 3u * (uint32_t)p.sz;
                const float *dbase = reinterpret_cast<const float *>(st) + qoff;
                Q4 inc = ePth;
                if (ctrl & FC_LOSSY3) {
                    const Q4 bPth = q_mul(q_make(r0.y, r1.y, r2.y, r3.y), th);
                    const Q4 rold = q_ld(dbase + FS::RXX / 4);
                    const Q4 rn = q_sub(q_muls(rold, A), bPth);
                    inc = q_fmas(hdt, q_add(rn, rold), ePth);
                    q_store<EDGE>(p.f[RXX] + gq, rn, g.nv);
                }
                const Q4 sn = q_add(s3, inc);
                q_store<EDGE>(p.fnxt[SXX] + gq, sn, g.nv);
                if (ctrl & FC_WYY3) q_store<EDGE>(p.fnxt[SYY] + gq, sn, g.nv);
                if (ctrl & FC_WZZ3) q_store<EDGE>(p.fnxt[SZZ] + gq, sn, g.nv);
                if (ctrl & (FC_PEAK | FC_RMS)) {
                    const Q4 pr = q_muls(q_add(q_add(q_add(zero, sn), sn), sn), -1.0f / 3.0f);
                    if (ctrl & FC_PEAK) {
                        const Q4 pk = q_ld(dbase + FS::PEAK / 4);
                        q_store<EDGE>(p.peak + gq, q_make(fmaxf(pk.a.x, fabsf(pr.a.x)), fmaxf(pk.a.y, fabsf(pr.a.y)),
                                                          fmaxf(pk.b.x, fabsf(pr.b.x)), fmaxf(pk.b.y, fabsf(pr.b.y))), g.nv);
                    }
                    if (ctrl & FC_RMS) q_store<EDGE>(p.sumsq + gq, q_fma(pr, pr, q_ld(dbase + FS::SUMSQ / 4)), g.nv);
                }
            }
        }
        // ---- vx, vy at plane m; D-x vx + D-y vy of the own quad through the exchange planes ----
        if (ctrl & FC_V0) {
            float *xv = xbuf + (m & 1) * FS::XBUF_FLOATS, *xy = xv + FS::XV_FLOATS;
            const float *vxo = reinterpret_cast<const float *>(st + FS::VXO);
            const float *vyo = reinterpret_cast<const float *>(st + FS::VYO);
            Q4 ox = zero, oy = zero;
            if (active) {
                const unsigned char *mt = mat + moff;
                float rho_j[5], rho_j1[4];
                {
                    const uint32_t wr1 = *reinterpret_cast<const uint32_t *>(mt + MXF);
                    rho_j[4] = rho_tab[mt[4]];
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        rho_j[c] = rho_tab[(w0 >> (8 * c)) & 255u];
                        rho_j1[c] = rho_tab[(wr1 >> (8 * c)) & 255u];
                    }
                }
                Q4 dxx = x_dplus(sig + eoff, c1, c2);                                                               // D+x sxx -> vx
                Q4 dyy = q_d4(q_ld(sig + eoff - EX), sig_own, q_ld(sig + eoff + EX), q_ld(sig + eoff + 2 * EX), c1, c2);   // D+y syy -> vy
                if (g.in_x) {
                    const float *sp_x = sprof + 4 * tx;
                    const float *ps = reinterpret_cast<const float *>(st + sp.psx) + g.psx_off;
                    q_st(p.psi[0] + gxo, q_cpml(dxx, q_ld(ps), q_ld(sp_x + 2 * C::TX), q_ld(sp_x + 3 * C::TX)));
                }
                if (g.row_y) {
                    const float *ps = reinterpret_cast<const float *>(st + sp.psy) + boff;
                    q_store<EDGE>(p.psi7_nxt + gyo, q_cpml(dyy, q_ld(ps), q_set(g.ay_h), q_set(g.by_h)), g.nv);
                }
                const Q4 cx = q_make(dt2 * rcp_newton(rho_j[0] + rho_j[1]), dt2 * rcp_newton(rho_j[1] + rho_j[2]),
                                     dt2 * rcp_newton(rho_j[2] + rho_j[3]), dt2 * rcp_newton(rho_j[3] + rho_j[4]));
                const Q4 cy = q_make(dt2 * rcp_newton(rho_j[0] + rho_j1[0]), dt2 * rcp_newton(rho_j[1] + rho_j1[1]),
                                     dt2 * rcp_newton(rho_j[2] + rho_j1[2]), dt2 * rcp_newton(rho_j[3] + rho_j1[3]));
                ox = q_fma(cx, dxx, q_ld(vxo + aoff));
                oy = q_fma(cy, dyy, q_ld(vyo + boff));
                if (EDGE) {
                    if (nzero_x >= 1) ox.b.y = 0.0f;
                    if (nzero_x >= 2) ox.b.x = 0.0f;
                    if (nzero_x >= 3) ox.a.y = 0.0f;
                    if (nzero_x >= 4) ox.a.x = 0.0f;
                    if (wall_y) oy = zero;
                }
                q_store<EDGE>(p.fnxt[VX] + goff, ox, g.nv);
                q_store<EDGE>(p.fnxt[VY] + goff, oy, g.nv);
            }
            q_sts(xv + aoff, ox);
            q_sts(xy + boff, oy);
            if (ex_vx) {
                float val = 0.0f;
                if (ex_vx_in) {
                    const float *srow = sig + (exr + 3) * EX + 4 + exc;
                    const unsigned char *mr = mat + (exr + 2) * MXF + 16 + exc;
                    const float d = fmaf(c2, srow[2] - srow[-1], c1 * (srow[1] - srow[0]));
                    val = fmaf(dt2 * rcp_newton(rho_tab[mr[0]] + rho_tab[mr[1]]), d, vxo[exr * C::AX + 4 + exc]);
                }
                xv[exr * C::AX + 4 + exc] = val;
            }
            if (ex_vy) {
                Q4 val = zero;
                const int bo = (eyr + 2) * C::TX + 4 * lane;
                if (ex_vy_in) {
                    const float *srow = sig + (eyr + 3) * EX + 4 + 4 * lane;
                    Q4 dyy = q_d4(q_ld(srow - EX), q_ld(srow), q_ld(srow + EX), q_ld(srow + 2 * EX), c1, c2);
                    if (ex_vy_slab) (void)q_cpml(dyy, q_ld(reinterpret_cast<const float *>(st + sp.psy) + bo), q_set(eay), q_set(eby));
                    const unsigned char *mr = mat + (eyr + 2) * MXF + 16 + 4 * lane;
                    const uint32_t a = *reinterpret_cast<const uint32_t *>(mr), b = *reinterpret_cast<const uint32_t *>(mr + MXF);
                    const Q4 cy = q_make(dt2 * rcp_newton(rho_tab[a & 255u] + rho_tab[b & 255u]),
                                         dt2 * rcp_newton(rho_tab[(a >> 8) & 255u] + rho_tab[(b >> 8) & 255u]),
                                         dt2 * rcp_newton(rho_tab[(a >> 16) & 255u] + rho_tab[(b >> 16) & 255u]),
                                         dt2 * rcp_newton(rho_tab[a >> 24] + rho_tab[b >> 24]));
                    val = q_fma(cy, dyy, q_ld(vyo + bo));
                }
                q_sts(xy + bo, val);
            }
            consumer_barrier(C::NC);
            if (active) {
                Q4 vxx = x_dminus(xv + aoff, c1, c2);                                                                // D-x vx
                Q4 vyy = q_d4(q_ld(xy + boff - 2 * C::TX), q_ld(xy + boff - C::TX), oy, q_ld(xy + boff + C::TX), c1, c2);    // D-y vy
                if (g.in_x) {
                    const float *sp_x = sprof + 4 * tx;
                    const float *ps = reinterpret_cast<const float *>(st + sp.psx) + sp.xt / 4 + g.psx_off;
                    q_st(p.psi[3] + gxo, q_cpml(vxx, q_ld(ps), q_ld(sp_x), q_ld(sp_x + C::TX)));
                }
                if (g.row_y) {
                    const float *ps = reinterpret_cast<const float *>(st + sp.psy + C::B_BYTES) + qoff;
                    q_store<EDGE>(p.psi[10] + gyo, q_cpml(vyy, q_ld(ps), q_set(g.ay_i), q_set(g.by_i)), g.nv);
                }
                tnew = q_add(vxx, vyy);
            }
        }
        s3 = s2; s2 = s1; s1 = sig_own;
        t3 = t2; t2 = t1; t1 = tnew;
        w3 = w2; w2 = w1; w1 = w0;
        goff += (uint32_t)p.sz;
        gxo += (uint32_t)(p.wx * p.ny);
        gyo += (uint32_t)(p.px * 2 * p.P);
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty[s]);
        if (++s == sp.ns) { s = 0; ph ^= 1; }
    }
}

// One block per work item (tile x, tile y, first plane, one past the last plane).  Three resident CTAs per SM.
template <class C>
__global__ void __launch_bounds__(C::NT, 3) k_fluid_fused(const __grid_constant__ FusedMaps maps, const Params p, const StagePlan spf,
                                                          const StagePlan spc, const int4 *__restrict__ items) {
    using FS = FStage<C>;
    extern __shared__ __align__(1024) unsigned char smem[];
    const int tid = threadIdx.x;
    const int4 it = __ldg(items + blockIdx.x);
    const int bx = it.x, by = it.y, kz0 = it.z, kz1 = it.w;
    const int x0 = bx * C::TX, y0 = by * C::TY;
    // rows y0-2 .. y0+TY (the new vy the CTA forms) reach a y slab?  Which one decides the compact row of the box.
    const bool tYe = p.P > 0 && (y0 - 2 < p.P || y0 + C::TY >= p.ny - p.P);
    const int jy0e = (y0 - 2 < p.P) ? y0 : y0 - (p.ny - 2 * p.P);
    const bool compact = spc.ns > 0 && !tYe && !(p.P > 0 && (kz0 < p.P || kz1 > p.nz - p.P));
    const StagePlan sp = compact ? spc : spf;
    unsigned char *stages = smem;
    const int NM = (p.n_mat + 31) & ~31;
    float *xbuf = reinterpret_cast<float *>(smem + sp.ns * sp.bytes);
    float *rho_tab = xbuf + 2 * FS::XBUF_FLOATS;
    float2 *tabP = reinterpret_cast<float2 *>(rho_tab + NM);
    float *sprof = reinterpret_cast<float *>(tabP + NM);
    uint64_t *full = reinterpret_cast<uint64_t *>(sprof + 4 * C::TX);
    uint64_t *empty = full + MAX_STAGES;

    for (int q = tid; q < NM; q += C::NT) {
        const KRow r = p.rows[q];
        rho_tab[q] = r.rho;
        tabP[q] = make_float2(r.eP, r.bP);
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
            const uint32_t *flags = p.flagsF + (size_t)(bx + p.ntxV * by) * (p.nz + 4) + 2;
            FusedIssue<C> iss;
            iss.maps = &maps; iss.p = &p; iss.sp = &sp;
            iss.tX = make_tilex<C>(p, x0); iss.tY = tile_in_y<C>(p, y0); iss.tYe = tYe;
            iss.jy0 = tile_jy0<C>(p, y0); iss.jy0e = jy0e;
            iss.x0 = x0; iss.y0 = y0; iss.kz0 = kz0; iss.kz1 = kz1;
            iss.sens = (p.do_peak ? FC_PEAK : 0u) | (p.do_rms ? FC_RMS : 0u);
            prefetch_tmap(&maps.boxE); prefetch_tmap(&maps.boxA); prefetch_tmap(&maps.boxB); prefetch_tmap(&maps.boxD);
            prefetch_tmap(&maps.mat);
            if (p.P > 0) { prefetch_tmap(&maps.psx); prefetch_tmap(&maps.psy); prefetch_tmap(&maps.psyE); prefetch_tmap(&maps.psz); }
            int s = 0; uint32_t ph = 0;
            for (int m = kz0 - 3; m < kz1 + 3; ++m) {
                const uint32_t f3 = (m - 3 >= kz0 && m - 3 < kz1) ? __ldg(flags + m - 3) : 0u;
                StageHdr h;
                h.ctrl = iss.ctrl(m, f3);
                h.az1 = h.bz1 = h.az2 = h.bz2 = 0.0f;
                if (h.ctrl & FC_ZS3) { h.az1 = __ldg(p.prof[2][0] + m - 3); h.bz1 = __ldg(p.prof[2][1] + m - 3); }   // integer node: D-z vz
                if (h.ctrl & FC_ZS2) { h.az2 = __ldg(p.prof[2][2] + m - 2); h.bz2 = __ldg(p.prof[2][3] + m - 2); }   // half node: D+z szz
                mbar_wait(&empty[s], ph ^ 1);
                unsigned char *st = stages + s * sp.bytes;
                StageHdr *hd = reinterpret_cast<StageHdr *>(st + FS::HDR);
                hd->ctrl = h.ctrl; hd->az1 = h.az1; hd->bz1 = h.bz1; hd->az2 = h.az2; hd->bz2 = h.bz2;
                Tma t{st, &full[s], 0};
                iss.run(t, m, h.ctrl);
                mbar_expect_tx(&full[s], t.bytes);
                if (++s == sp.ns) { s = 0; ph ^= 1; }
            }
        }
        return;
    }

    // ================= consumers =================
    const bool edge = (x0 + C::TX >= p.nx) || (y0 + C::TY >= p.ny);
    if (edge) fused_consume<C, true>(p, sp, stages, xbuf, rho_tab, tabP, sprof, full, empty, tid, x0, y0, kz0, kz1, tYe, jy0e);
    else fused_consume<C, false>(p, sp, stages, xbuf, rho_tab, tabP, sprof, full, empty, tid, x0, y0, kz0, kz1, tYe, jy0e);
}

// ------------------------------------------------------------------------------------------
// S0 on the device: which tile-planes can run the fused sweep
// ------------------------------------------------------------------------------------------
// One CTA per (64 x 8 tile, plane): FF_FLUID4 when no cell within 4 cells (x, y) of the tile is a solid,
// FF_LOSSY when a cell of the tile itself is lossy.  The host combines the planes (kernels_fused.cuh: fused_lists).
__global__ void __launch_bounds__(128) k_fused_class(const Params p, uint8_t *__restrict__ cls) {
    __shared__ uint32_t solid, lossy;
    using C = CfgF;
    const int x0 = blockIdx.x * C::TX, y0 = blockIdx.y * C::TY, k = blockIdx.z;
    if (threadIdx.x == 0) { solid = 0; lossy = 0; }
    __syncthreads();
    constexpr int EXW = C::TX + 8, EYW = C::TY + 8;
    uint32_t so = 0, lo = 0;
    for (int q = threadIdx.x; q < EXW * EYW; q += blockDim.x) {
        const int i = x0 - 4 + q % EXW, j = y0 - 4 + q / EXW;
        if (i < 0 || j < 0 || i >= p.nx || j >= p.ny) continue;
        const KRow r = p.rows[p.mat[i + (long long)p.px * j + p.sz * k]];
        if (r.solid != 0.0f) so = 1;
        if (i >= x0 && i < x0 + C::TX && j >= y0 && j < y0 + C::TY && (r.bP != 0.0f || r.bS != 0.0f)) lo = 1;
    }
    if (so) atomicOr(&solid, 1u);
    if (lo) atomicOr(&lossy, 1u);
    __syncthreads();
    if (threadIdx.x == 0)
        cls[(size_t)(blockIdx.x + gridDim.x * blockIdx.y) * p.nz + k] = (uint8_t)((solid ? 0u : FF_FLUID4) | (lossy ? FF_LOSSY : 0u));
}

// sigma_yy, sigma_zz of the planes the fused sweep keeps as sigma_xx only: fill them in (before they are read back
// and before the context leaves the fused mode)
__global__ void __launch_bounds__(128) k_fill_sii(const Params p) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= p.nx) return;
    const uint32_t fw = p.flagsF[(size_t)(i / CfgF::TX + p.ntxV * (j / CfgF::TY)) * (p.nz + 4) + 2 + k];
    if (!(fw & FF_RUN)) return;
    const long long c = p.org + i + (long long)p.px * j + p.sz * k;
    const float s = p.f[SXX][c];
    p.f[SYY][c] = s;
    p.f[SZZ][c] = s;
}

// ------------------------------------------------------------------------------------------
// host side: runs, work lists, plan
// ------------------------------------------------------------------------------------------
struct FusedLists {
    std::vector<int4> f, v, s;          // work items (tile x, tile y, kz0, kz1): fused sweep, velocity pass, stress pass
    std::vector<uint32_t> flags;        // flagsF words, (tile, plane + 2)
    long long planes_f = 0;
};

// cls: one byte per (64 x 8 tile, plane) from k_fused_class.  sty = rows of a stress tile (8 or 16): a stress
// tile of 16 rows is fused only as a whole.  slots_* = resident CTAs of the device for each kernel.
inline FusedLists fused_lists(const Layout &L, const std::vector<uint8_t> &cls, int sty, int slots_f, int slots_v, int slots_s,
                              int fused_chunk = 0, int pass_chunk = 0) {
    FusedLists out;
    const int ntx = L.ntxV, nty = L.ntyV, nz = L.nz, P = L.P, TX = CfgF::TX, TY = CfgF::TY;
    const int LMIN = 16;
    out.flags.assign((size_t)ntx * nty * (nz + 4), 0u);
    std::vector<uint8_t> run((size_t)ntx * nty * nz, 0);
    auto C = [&](int bx, int by, int k) -> uint8_t { return cls[(size_t)(bx + ntx * by) * nz + k]; };
    // tiles whose halo columns would need the x-psi of a neighbouring tile stay with the two passes, and so does
    // everything on grids where one tile (or its halo rows) touches both slabs of an axis
    const bool grid_ok = P == 0 || (L.ny >= 2 * P + 3 * TY && !(TX > L.xhb || P > TX));
    auto in_xslab = [&](int i) { return P > 0 && i >= 0 && i < L.nx && (i < P || i >= L.nx - P); };
    const int group = sty / TY;         // velocity tiles per stress tile in y
    for (int bx = 0; bx < ntx && grid_ok; ++bx) {
        const int x0 = bx * TX;
        if (in_xslab(x0 - 2) || in_xslab(x0 - 1) || in_xslab(x0 + TX)) continue;
        for (int gy = 0; gy < nty; gy += group) {
            const int g1 = std::min(nty, gy + group);
            // planes in which every tile of the group is fluid within reach
            std::vector<uint8_t> e(nz, 1);
            for (int by = gy; by < g1; ++by)
                for (int k = 0; k < nz; ++k) e[k] &= (C(bx, by, k) & FF_FLUID4) ? 1 : 0;
            // plane k can be fused when planes k-3 .. k+3 are fluid within reach: its D-z vz takes vz at k-2 .. k+1,
            // which the sweep forms from sigma_xx (standing for sigma_zz) at planes k-3 .. k+3
            std::vector<uint8_t> ok(nz, 0);
            for (int k = 0; k < nz; ++k) {
                uint8_t a = 1;
                for (int q = std::max(0, k - 3); q <= std::min(nz - 1, k + 3); ++q) a &= e[q];
                ok[k] = a;
            }
            for (int a = 0; a < nz;) {
                if (!ok[a]) { ++a; continue; }
                int b = a;
                while (b < nz && ok[b]) ++b;
                // a chunk boundary inside (or within two planes of) a z slab would make the chunk recompute vz under
                // a psi it does not own: keep the boundaries at 0, nz or in [P + 2, nz - P - 1]
                int ra = a, rb = b;
                if (P > 0) {
                    if (ra > 0 && ra < P + 2) ra = P + 2;
                    if (rb < nz && rb > nz - P - 1) rb = nz - P - 1;
                    if ((ra > nz - P - 1 && ra < nz) || (rb > 0 && rb < P + 2)) rb = ra;   // the run lies inside a slab: dropped
                }
                if (rb - ra >= LMIN)
                    for (int by = gy; by < g1; ++by)
                        for (int k = ra; k < rb; ++k) run[(size_t)(bx + ntx * by) * nz + k] = 1;
                a = b;
            }
        }
    }
    auto R = [&](int bx, int by, int k) -> bool { return by >= 0 && by < nty && k >= 0 && k < nz && run[(size_t)(bx + ntx * by) * nz + k]; };
    long long planes_f = 0;
    for (int by = 0; by < nty; ++by)
        for (int bx = 0; bx < ntx; ++bx)
            for (int k = 0; k < nz; ++k) {
                uint32_t w = C(bx, by, k) & (FF_FLUID4 | FF_LOSSY);
                if (R(bx, by, k)) {
                    w |= FF_RUN;
                    ++planes_f;
                    if ((by > 0 && !R(bx, by - 1, k)) || (by + 1 < nty && !R(bx, by + 1, k))) w |= FF_WYY;
                    for (int q = k - 2; q <= k + 1; ++q)
                        if (q >= 0 && q < nz && !R(bx, by, q)) w |= FF_WZZ;
                }
                out.flags[(size_t)(bx + ntx * by) * (nz + 4) + 2 + k] = w;
            }
    out.planes_f = planes_f;
    // runs of each kind
    struct Run { int bx, by, a, b; };
    std::vector<Run> rf, rv, rs;
    for (int by = 0; by < nty; ++by)
        for (int bx = 0; bx < ntx; ++bx) {
            for (int a = 0; a < nz;) {
                const bool r = R(bx, by, a);
                int b = a;
                while (b < nz && R(bx, by, b) == r) ++b;
                if (r) rf.push_back({bx, by, a, b});
                else {
                    // velocity pass: the z slabs get chunks of their own (compact stage plan elsewhere)
                    // (a cut that would leave a piece under 8 planes is not made: a chunk costs 4 priming planes)
                    int cuts[4] = {a, std::min(b, std::max(a, P)), std::max(a, std::min(b, nz - P)), b};
                    if (cuts[1] - cuts[0] < 8 || cuts[2] - cuts[1] < 8) cuts[1] = cuts[0];
                    if (cuts[3] - cuts[2] < 8 || cuts[2] - cuts[1] < 8) cuts[2] = cuts[3];
                    if (cuts[2] < cuts[1]) cuts[1] = cuts[2] = cuts[0];
                    for (int c = 0; c < 3; ++c)
                        if (cuts[c + 1] > cuts[c]) rv.push_back({bx, by, cuts[c], cuts[c + 1]});
                    if (by % group == 0) rs.push_back({bx, by / group, a, b});
                }
                a = b;
            }
        }
    // Chunk lengths: SHORT chunks win, although a chunk costs 6 (fused) or 4 (two passes) priming planes: the CTAs of
    // one z range start together and stay within a few planes of each other, so the halo rows and columns a
    // neighbour needs are still in L2 (126 MB hold about 25 us of traffic), and many small items balance the last
    // round.  Measured (20-step bench, both sensors on; profiles/r2_fused.md): fused sweep on config 2 with chunks
    // of 50 / 24 / 16 / 12 planes 0.446 / 0.407 / 0.388 / 0.385 ms, on config 3 with 128 / 32 / 16: 1.65 / 1.50 / 1.29
    // ms; two-pass lists on config 4 with 66-96 / 32 / 16 / 12 planes: stress 0.84 / 0.75 / 0.70 / 0.70 ms.
    // (Choosing the length that minimises rounds x (planes + priming planes) in a model of equal items -- 2 rounds of
    // 90 planes on config 2 -- measured 2-8 % slower.)
    (void)slots_f; (void)slots_v; (void)slots_s;
    // [a, b) in about equal chunks of at most `len` planes; with `fused` no chunk boundary falls inside, or within
    // two planes of, a z slab (a fused chunk recomputes vz at kz0-2, kz0-1 and kz1 without their psi)
    auto split = [&](std::vector<int4> &dst, int bx, int by, int a, int b, int len, bool fused) {
        const int n = std::max(1, (b - a + len - 1) / len);
        const int lo = (fused && P > 0) ? P + 2 : a, hi = (fused && P > 0) ? nz - P - 1 : b;
        int k0 = a;
        for (int c = 1; c <= n; ++c) {
            int k1 = c == n ? b : a + (int)((long long)(b - a) * c / n);
            if (c < n) {
                k1 = std::max(lo, std::min(hi, k1));
                if (k1 <= k0 || k1 >= b) continue;
            }
            dst.push_back(make_int4(bx, by, k0, k1));
            k0 = k1;
        }
    };
    const int len_f = fused_chunk > 0 ? fused_chunk : 16, len_v = pass_chunk > 0 ? pass_chunk : 12, len_s = len_v;
    for (const Run &r : rf) split(out.f, r.bx, r.by, r.a, r.b, len_f, true);
    for (const Run &r : rv) split(out.v, r.bx, r.by, r.a, r.b, len_v, false);
    for (const Run &r : rs) split(out.s, r.bx, r.by, r.a, r.b, len_s, false);
    // launch order: the long items first (the short ones fill the last wave), and among items of about the same
    // length those of one z range together, tile rows in order: CTAs that run at the same time then share their
    // halo rows and columns in L2 (ordered by length alone, the halo reads of the fused sweep went to DRAM: L2
    // hit rate 21 %, DRAM reads twice the algorithmic bytes; profiles/r2b_fused.md)
    auto order = [](const int4 &x, const int4 &y) {
        const int bx_ = (x.w - x.z) / 32, by_ = (y.w - y.z) / 32;
        if (bx_ != by_) return bx_ > by_;
        if (x.z != y.z) return x.z < y.z;
        if (x.y != y.y) return x.y < y.y;
        return x.x < y.x;
    };
    std::sort(out.f.begin(), out.f.end(), order);
    std::sort(out.v.begin(), out.v.end(), order);
    std::sort(out.s.begin(), out.s.end(), order);
    return out;
}

inline size_t fused_items_capacity(const Layout &L) { return (size_t)L.ntxV * L.ntyV * (L.nz / 8 + 6); }

// tensor maps and stage plans of the fused sweep (after tiled_plan_create)
inline int fused_plan_create(FusedPlan &fp, const TiledPlan &tp, const Layout &L, const Params &p, char *psi_y_base,
                             long long psi_y_stride, int l2_promotion = 0) {
    using C = CfgF;
    using FS = FStage<C>;
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) { (void)cudaGetLastError(); return BVFDTD_ECUDA; }
    PFN_encodeTiled enc = (PFN_encodeTiled)fn;
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    fp.maps.boxA = tp.mv.boxA; fp.maps.boxB = tp.mv.boxB; fp.maps.boxD = tp.mv.boxD;
    fp.maps.psx = tp.mv.psx; fp.maps.psy = tp.mv.psy; fp.maps.psz = tp.mv.psz;
    fp.maps.psyE = tp.mv.psy;
    {
        const long long fstride = (const char *)p.f[1] - (const char *)p.f[0];
        void *base = (void *)(p.f[0] + (L.org - 2 * L.sz));
        const cuuint64_t gdim[4] = {(cuuint64_t)L.px, (cuuint64_t)L.py, (cuuint64_t)(L.nz + 4), (cuuint64_t)NGRID_ALL};
        const cuuint64_t gstr[3] = {(cuuint64_t)L.px * 4, (cuuint64_t)L.sz * 4, (cuuint64_t)fstride};
        const cuuint32_t box[4] = {(cuuint32_t)FS::EX, (cuuint32_t)FS::EY, 1, 1};
        if (enc(&fp.maps.boxE, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, base, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, l2_promotion_of(l2_promotion), CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return BVFDTD_ECUDA;
    }
    {
        const cuuint64_t mdim[3] = {(cuuint64_t)L.px, (cuuint64_t)L.py, (cuuint64_t)(L.nz + 1)};
        const cuuint64_t mstr[2] = {(cuuint64_t)L.px, (cuuint64_t)L.sz};
        const cuuint32_t mbox[3] = {(cuuint32_t)FS::MXF, (cuuint32_t)FS::MYF, 1};
        if (enc(&fp.maps.mat, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, (void *)p.mat, mdim, mstr, mbox, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, l2_promotion_of(l2_promotion), CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return BVFDTD_ECUDA;
    }
    if (L.P > 0) {
        const cuuint64_t d[4] = {(cuuint64_t)L.px, (cuuint64_t)(2 * L.P), (cuuint64_t)L.nz, 7};
        const cuuint64_t s[3] = {(cuuint64_t)L.px * 4, (cuuint64_t)L.px * 2 * L.P * 4, (cuuint64_t)psi_y_stride};
        const cuuint32_t b[4] = {(cuuint32_t)C::TX, (cuuint32_t)C::BY, 1, 1};
        if (enc(&fp.maps.psyE, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, psi_y_base, d, s, b, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, l2_promotion_of(l2_promotion), CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return BVFDTD_ECUDA;
    }
    // stage plans: fixed slots, then 2 x-psi slots, [psi[7] rows (B box) + psi[10] (D box)], [2 z-psi D boxes]
    const int wxb = tp.sv.wxb;
    auto stage = [&](int ns, bool yz) {
        StagePlan s{};
        s.wxb = wxb;
        s.xb = L.P > 0 ? round128(wxb * C::TY * 4) : 0;
        s.yb = C::D_BYTES;
        s.hdr = FS::HDR;
        s.psx = FS::FIXED;
        s.xhi = 0;                       // (grids on which a tile touches both x slabs do not run the fused sweep)
        s.xt = s.xb;
        s.psy = s.psx + 2 * s.xt;
        s.psz = s.psy + (L.P > 0 && yz ? C::B_BYTES + C::D_BYTES : 0);
        s.bytes = s.psz + (L.P > 0 && yz ? 2 * C::D_BYTES : 0);
        s.ns = ns;
        return s;
    };
    const int nm = (p.n_mat + 31) & ~31;
    const int extra = 2 * FS::XBUF_FLOATS * 4 + nm * 12 + 4 * C::TX * 4 + 2 * MAX_STAGES * 8;
    fp.full = stage(2, true);
    fp.compact = stage(3, false);
    if (L.P == 0) fp.compact.ns = 0;     // no psi slots anywhere: the full plan is already the compact one
    if (L.P == 0) fp.full.ns = 3;
    fp.smem = std::max(fp.full.ns * fp.full.bytes, fp.compact.ns * fp.compact.bytes) + extra;
    fp.full.smem = fp.compact.smem = fp.smem;
    int smem_max = 227 * 1024;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (fp.smem > smem_max) return BVFDTD_EINVAL;
    e = cudaFuncSetAttribute(k_fluid_fused<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, fp.smem);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return BVFDTD_ECUDA; }
    fp.ready = true;
    return 0;
}

inline void fused_launch(const FusedPlan &fp, const Params &p, cudaStream_t st) {
    if (fp.n_f > 0) k_fluid_fused<CfgF><<<fp.n_f, CfgF::NT, fp.smem, st>>>(fp.maps, p, fp.full, fp.compact, fp.items_f);
}

}  // namespace bvfdtd
