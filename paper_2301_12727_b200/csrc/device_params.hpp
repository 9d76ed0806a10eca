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
    int wx;                   // x pitch of the x-slab psi arrays = round_up(2P, 4)
    long long psi_floats[3];  // floats per psi array of axis x, y, z
};

struct Params {
    int nx, ny, nz, P;
    int px, py, wx;
    long long sz, org;
    float *f[NSTATE];
    float *peak, *sumsq;
    const uint8_t *mat;
    float *psi[18];        // axis*6 + term; terms 0-2 velocity pass, 3-5 stress pass
    const KRow *rows;      // 256 rows
    const float *prof[3][4];  // per axis: a_int, b_int, a_half, b_half
    float inv_dx, dt, half_dt, A, B;
    int do_peak, do_rms;
};

}  // namespace bvfdtd
