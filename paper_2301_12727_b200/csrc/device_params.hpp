// device_params.hpp -- the private device layout and the parameter block every kernel receives.
//
// Private layout of a grid field: x pitch px (multiple of 32
// floats, >= nx + 2), py = ny + 2 rows per plane, nz + 4 planes; cell (i,j,k) lives at
// org + i + px*j + sz*k with sz = px*py.  The gaps (x in [nx,px), rows ny..ny+1, planes -2,-1 and
// nz,nz+1, plus a lead of 2 rows) hold zeros that no kernel ever writes, so every 4-point stencil
// can read up to 2 cells outside the grid without a bounds test and gets the zero ghost value of
// reading P4 (cell (-1,j,k) is the tail of row j-1, etc.).  A TMA box that leaves the allocation
// is zero-filled by the hardware, which is the same value.
#pragma once
#include <cstdint>

#include "host_tables.hpp"

namespace bvfdtd {

enum { VX, VY, VZ, SXX, SYY, SZZ, SXY, SXZ, SYZ, RXX, RYY, RZZ, RXY, RXZ, RYZ, NSTATE };

struct Layout {
    int nx, ny, nz, P;
    int px, py;               // x pitch (floats), rows per plane
    long long sz;             // plane stride (floats)
    long long org;            // offset of cell (0,0,0) inside a field allocation (floats)
    long long field_floats;   // floats per field allocation (multiple of 64)
    long long mat_bytes;      // index map: px * py * (nz + 1) bytes, edges replicated (P2)
    int xp4, xhb, xph;        // x-slab psi: low slab at compact [0, xp4), xp4 = round_up(P, 4); high slab
                              // at xp4 + (i - xhb), xhb = floor4(nx - P), width xph = round_up(nx - xhb, 4)
    int wx;                   // x pitch of the x-slab psi arrays = xp4 + xph
    long long psi_floats[3];  // floats per psi array of axis x, y, z
    int ntxV, ntyV, ntxS, ntyS;   // x-y tiles of the velocity / stress kernels
    long long flag_wordsV, flag_wordsS;   // uint32 words per flag table: tiles * (nz + 4)
};

struct Params {
    int nx, ny, nz, P;
    int n_mat;             // rows of the material table in use
    int px, py, wx;
    int xp4, xhb, xph;     // x-slab compact index: i < P ? i : xp4 + (i - xhb)
    int ntxV, ntyV, ntxS, ntyS;
    long long sz, org;
    float *f[NSTATE];
    float *peak, *sumsq;
    float *phre, *phim;    // phasor accumulators sum p cos(w t), sum p sin(w t) (NEXT-3)
    const uint8_t *mat;
    float *psi[18];        // axis*6 + term; terms 0-2 velocity pass, 3-5 stress pass
    const KRow *rows;      // 256 rows
    const float *prof[3][4];  // per axis: a_int, b_int, a_half, b_half
    float inv_dx, dt, half_dt, A, B;
    int do_peak, do_rms;
    int do_phasor;         // this step accumulates the phasor (then do_peak = do_rms = 0)
    float ph_cos, ph_sin;  // cos / sin of w0 (n + 1) dt for this step
    // tile-class flags: one word per (tile, plane + 2), planes -2..nz+1
    const uint32_t *flagsV, *flagsS;
    // Ping-pong of the arrays the fused fluid sweep reads with a halo while other CTAs of the same launch write
    // them (vx, vy, vz, sigma_xx, sigma_yy, sigma_zz and the y-psi of D+y sigma_yy): every kernel of a step reads
    // the time level it starts from in the "cur" copy and writes its results to the "nxt" copy; the host swaps
    // the two after the step.  f[0..5] and psi[7] always name the cur copies.  Without the fused sweep
    // cur == nxt and the passes work in place, as before.
    int icur[6], inxt[6];     // array index of VX..SZZ inside the 4-D field tensor map
    float *fnxt[6];           // where the step writes VX..SZZ
    int ipsi7_cur;            // array index of psi[7] inside the y-psi tensor map (1, or 6 for the alternate)
    float *psi7_nxt;
    const uint32_t *flagsF;   // fused sweep: one word per (64 x 8 tile, plane + 2)
};

// tile-class flag bits
enum : uint32_t {
    TF_XY = 1u,    // stress: some xy shear node of the tile-plane has four solid cells
    TF_XZ = 2u,    //         ... xz ...
    TF_YZ = 4u,    //         ... yz ...
    TF_RII = 8u,   // stress: some cell of the tile-plane is lossy (r_ii can be non-zero)
    TF_VFLUID = 8u,  // velocity (shares the bit with TF_RII, which only the stress pass uses): every cell of the
                     // halo-extended tile-plane is a fluid, so sigma_xx = sigma_yy = sigma_zz there and one array serves
    TF_SOLID = 16u,  // stress: some cell of the tile-plane is a solid (else eS = bS = 0 and r_xx = r_yy = r_zz)
    // velocity: the same three bits, taken over the halo-extended region the pass reads
};

// fused-sweep flag bits (flagsF; kernels_fused.cuh)
enum : uint32_t {
    FF_FLUID4 = 1u,   // S0: no solid cell within 4 cells (x, y) of the 64 x 8 tile in this plane
    FF_LOSSY = 2u,    // S0: some cell of the tile-plane is lossy (r_xx moves)
    FF_RUN = 4u,      // host: the plane belongs to a run of the fused sweep
    FF_WYY = 8u,      // host: a y-neighbour tile runs the two passes here and reads sigma_yy: write it too
    FF_WZZ = 16u      // host: a plane within reach of the z stencil runs the two passes: write sigma_zz too
};

}  // namespace bvfdtd
