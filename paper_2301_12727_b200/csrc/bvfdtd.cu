// bvfdtd.cu -- the C ABI of include/bvfdtd.h: context, private layout, uploads, launches, readback.
// All arithmetic of the hot path runs in the kernels (kernels_ref.cuh, kernels_tiled.cuh); the
// host side only derives the S0 tables (host_tables.cpp) and enqueues work.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/bvfdtd.h"
#include "device_params.hpp"
#include "host_common.hpp"
#include "kernels_ref.cuh"
#include "kernels_tiled.cuh"
#include "kernels_fused.cuh"
#include "kernels_post.cuh"
#include "kernels_rs.cuh"

using namespace bvfdtd;

// ---------------------------------------------------------------------------------------------------
// Scratch of bvfdtd_rayleigh_noalloc (the entry point for callers that cannot call cudaMalloc): the
// sources packed as float4 (x, y, z, 0).  A file-scope device array: every GPU that loads the library holds
// these BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC * 16 bytes = 1 MiB until the process exits.  In HOST code the name
// below is only a stand-in for the symbol, not a device address: the address each device gives it is
// resolved once per device, with that device current, by cudaGetSymbolAddress (rs_noalloc_scratch()).
// ---------------------------------------------------------------------------------------------------
static __device__ __align__(256) float4 g_rs_noalloc_src[BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC];

// (x, y, z) triples -> float4 (x, y, z, 0) in the scratch: every entry the field kernel will read is written
// here, .w included, so nothing of an earlier call is seen; entries from n_src on keep old contents, unread
static __global__ void k_rs_noalloc_pack(const int n_src, const float *__restrict__ src_xyz, float4 *__restrict__ dst) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n_src) dst[q] = make_float4(src_xyz[3 * q], src_xyz[3 * q + 1], src_xyz[3 * q + 2], 0.0f);
}

// device address of g_rs_noalloc_src on the CURRENT device (resolved on first use per device, then cached)
static int rs_noalloc_scratch(float4 **out) {
    enum { MAX_DEVICES = 64 };
    static std::mutex mu;
    static float4 *addr[MAX_DEVICES] = {};
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return cuda_fail(cudaErrorInvalidDevice, "bvfdtd_rayleigh_noalloc: device ordinal out of range");
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void *p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_rs_noalloc_src));
        if (!p) return cuda_fail(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_rs_noalloc_src) returned null");
        addr[dev] = (float4 *)p;
    }
    *out = addr[dev];
    return BVFDTD_OK;
}

namespace {
thread_local char g_cuda_err[256] = "";
}

int bvfdtd::cuda_fail(cudaError_t e, const char *what) {
    std::snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
    (void)cudaGetLastError();
    return BVFDTD_ECUDA;
}

namespace {

long long round_up(long long v, long long m) { return (v + m - 1) / m * m; }

bool grid_ok(const bvfdtd_grid *g) {
    if (!g || g->pml < 0) return false;
    const long long lim = 2LL * g->pml + 8;
    if (g->nx < lim || g->ny < lim || g->nz < lim) return false;
    // the kernels address a field with 32-bit float offsets: keep a padded field under 2^31 floats
    if ((long long)(g->nx + 34) * (g->ny + 2) * (g->nz + 6) >= (1LL << 31)) return false;
    return g->nx <= 65535 * 16 && g->ny <= 65533 && g->nz <= 65534;
}

Layout make_layout(const bvfdtd_grid &g) {
    Layout L;
    L.nx = g.nx; L.ny = g.ny; L.nz = g.nz; L.P = g.pml;
    L.px = (int)round_up(g.nx + 2, 32);
    L.py = g.ny + 2;
    L.sz = (long long)L.px * L.py;
    L.org = 2 * L.sz + 2 * L.px + 32;
    L.field_floats = round_up(L.org + L.sz * (g.nz + 2) + 2 * L.px + 32, 64);
    L.mat_bytes = round_up(L.sz * (g.nz + 1), 256);
    L.xp4 = (int)round_up(g.pml, 4);
    L.xhb = (g.nx - g.pml) & ~3;
    L.xph = (int)round_up(g.nx - L.xhb, 4);
    L.wx = L.xp4 + L.xph;
    L.ntxV = (g.nx + CfgV::TX - 1) / CfgV::TX;
    L.ntyV = (g.ny + CfgV::TY - 1) / CfgV::TY;
    L.ntxS = (g.nx + CfgS::TX - 1) / CfgS::TX;
    L.ntyS = (g.ny + CfgS8::TY - 1) / CfgS8::TY;   // sized for the smaller stress tile; the plan fixes the real count
    L.flag_wordsV = round_up((long long)L.ntxV * L.ntyV * (g.nz + 4), 64);
    L.flag_wordsS = round_up((long long)L.ntxS * L.ntyS * (g.nz + 4), 64);
    L.psi_floats[0] = round_up((long long)L.wx * g.ny * g.nz, 64);
    L.psi_floats[1] = round_up((long long)L.px * (2 * g.pml) * g.nz, 64);
    L.psi_floats[2] = round_up((long long)L.px * g.ny * (2 * g.pml), 64);
    if (g.pml == 0) L.psi_floats[0] = L.psi_floats[1] = L.psi_floats[2] = 64;
    return L;
}

// Offsets (bytes) of every region of the caller's workspace.
struct WsMap {
    size_t field[NSTATE], peak, sumsq, phre, phim, alt[6], scratch, mat, psi[18], psi7_alt, rows, prof, flagsV, flagsS, flagsF,
        invz, ctr, src, items[3], cls, total;
    size_t zero0, zero1;      // [zero0, zero1): state, sensors, psi, flag words, counters -- what bvfdtd_create zeroes (reading P9)
    long long src_cap;        // source cells the workspace has room for (16 bytes each); more go to a library-owned allocation
};

WsMap make_wsmap(const Layout &L) {
    WsMap w;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += (bytes + 255) / 256 * 256; return o; };
    for (int q = 0; q < NSTATE; ++q) w.field[q] = take(L.field_floats * 4);
    w.peak = take(L.field_floats * 4);
    w.sumsq = take(L.field_floats * 4);
    w.phre = take(L.field_floats * 4);
    w.phim = take(L.field_floats * 4);
    for (int q = 0; q < 6; ++q) w.alt[q] = take(L.field_floats * 4);     // ping-pong copies of VX..SZZ (fused sweep)
    for (int a = 0; a < 3; ++a) {
        for (int t = 0; t < 6; ++t) w.psi[a * 6 + t] = take(L.psi_floats[a] * 4);
        if (a == 1) w.psi7_alt = take(L.psi_floats[1] * 4);              // ping-pong copy of psi[7], 7th array of the y block
    }
    w.flagsF = take((size_t)L.flag_wordsV * 4);
    w.flagsV = take((size_t)L.flag_wordsV * 4);          // (the words of planes -2, -1, nz, nz+1 stay zero)
    w.flagsS = take((size_t)L.flag_wordsS * 4);
    w.ctr = take(256);                                   // device step counter + block ticket of k_inject, index-map maximum
    w.zero0 = 0; w.zero1 = off;
    w.scratch = take((size_t)L.nx * L.ny * L.nz * 4);
    w.mat = take(L.mat_bytes);
    w.rows = take(256 * sizeof(KRow));
    w.prof = take((size_t)4 * (L.nx + L.ny + L.nz) * 4);
    w.invz = take(256 * 4);
    w.src_cap = 4LL * L.nx * L.ny;                       // a source plane or array fits; larger lists are library-owned
    w.src = take((size_t)w.src_cap * 16);
    for (int q = 0; q < 3; ++q) w.items[q] = take(fused_items_capacity(L) * sizeof(int4));   // work lists of the fused mode
    w.cls = take((size_t)L.ntxV * L.ntyV * L.nz);
    w.total = off;
    return w;
}

}  // namespace

struct bvfdtd_ctx {
    Layout L;
    WsMap W;
    char *ws = nullptr;
    cudaStream_t stream = nullptr;
    int device = -1;      // owner of the workspace: every entry point runs on it (DeviceScope)
    double dx = 0, dt = 0;
    bvfdtd_opts opts{};
    int n_materials = 0;
    std::vector<bvfdtd_material> table;   // the caller's rows (bvfdtd_heat_source needs alphaL)
    std::vector<Derived> derived;
    PmlAxis pml[3];
    Params prm{};
    int64_t step = 0;
    int phase_planes = 0; // planes of the pass in progress already run through bvfdtd_step_phase_planes
    int range_slot = 0;   // next slice of the work-list regions bvfdtd_step_phase_planes writes (round robin of 4)
    int phase_done = 0;   // passes of the current step already run through bvfdtd_step_phase (bit 0 inject, 1 velocity)
    int64_t rms_count = 0;
    // source
    int64_t n_src = 0;
    long long *d_cell = nullptr;
    float *d_amp = nullptr, *d_delay = nullptr;
    void *src_own = nullptr;     // library-owned copy of a source list too long for the workspace's source region
    int waveform = 0, n_cycles = 1;
    double f_src = 0;
    // tiled-kernel plan (tensor maps etc.)
    TiledPlan plan;
    // fused single sweep of the all-fluid tile columns (kernels_fused.cuh); sel = which copy of the ping-pong
    // arrays holds the current time level (0 = the primary arrays)
    FusedPlan fplan;
    bool ff_active = false;
    int sel = 0;
    bool sigma_written = false;   // a normal stress was written by the caller: no sigma_xx-for-all in the velocity pass
    bool dense = false;   // tile-class skipping off (BVFDTD_FLAG_DENSE, or a shear / memory field was written)
    // CUDA graphs of one step and of GRAPH_STEPS steps per sensor regime (peak on/off x rms on/off), built on first use
    enum { GRAPH_STEPS = 8 };
    cudaGraphExec_t graph[4][2][2] = {};
    cudaStream_t cap_stream2 = nullptr;    // second branch of a captured step: the velocity pass of the two-pass columns runs
    cudaEvent_t cap_fork = nullptr, cap_join = nullptr;   // beside the fused sweep (both read the cur copies, write the nxt ones)
    cudaStream_t cap_stream = nullptr;     // library-owned stream the graphs are captured on (the caller's may be the
                                           // legacy default stream, which cannot be captured); nothing ever runs on it   // [regime][one step | GRAPH_STEPS steps][sel at the first step]
    // kernel timing
    bool timing = false;
    std::vector<cudaEvent_t> ev;
    int64_t timed_steps = 0;
};

namespace {

__global__ void k_unpack(float *__restrict__ dst, const float *__restrict__ src, Params p) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= p.nx) return;
    dst[i + (long long)p.nx * (j + (long long)p.ny * k)] = src[p.org + i + (long long)p.px * j + p.sz * k];
}
__global__ void k_unpack_scaled(float *__restrict__ dst, const float *__restrict__ src, Params p, float scale) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= p.nx) return;
    dst[i + (long long)p.nx * (j + (long long)p.ny * k)] = scale * src[p.org + i + (long long)p.px * j + p.sz * k];
}
__global__ void k_pack(float *__restrict__ dst, const float *__restrict__ src, Params p, int hold_axis) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= p.nx) return;
    float v = src[i + (long long)p.nx * (j + (long long)p.ny * k)];
    if ((hold_axis == 0 && i == p.nx - 1) || (hold_axis == 1 && j == p.ny - 1) || (hold_axis == 2 && k == p.nz - 1)) v = 0.0f;
    dst[p.org + i + (long long)p.px * j + p.sz * k] = v;
}
__global__ void k_pressure(float *__restrict__ dst, Params p) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= p.nx) return;
    const long long c = p.org + i + (long long)p.px * j + p.sz * k;
    dst[i + (long long)p.nx * (j + (long long)p.ny * k)] = (p.f[SXX][c] + p.f[SYY][c] + p.f[SZZ][c]) * (-1.0f / 3.0f);
}
__global__ void k_rms_amp(float *__restrict__ dst, Params p, float two_over_count) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= p.nx) return;
    const long long c = p.org + i + (long long)p.px * j + p.sz * k;
    dst[i + (long long)p.nx * (j + (long long)p.ny * k)] = sqrtf(p.sumsq[c] * two_over_count);
}
// dense (nx, ny, nz) index map -> private layout (pitch px, py rows, nz + 1 planes) with the edges
// replicated by one cell in +x, +y, +z (reading P2); max_index receives the largest index seen
__global__ void k_pad_index_map(uint8_t *__restrict__ dst, const uint8_t *__restrict__ src, int nx, int ny, int nz, int px, int py,
                                long long sz, int *max_index) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    int v = 0;
    if (i < px) {
        const int is = min(i, nx - 1), js = min(j, ny - 1), ks = min(k, nz - 1);
        v = src[is + (long long)nx * (js + (long long)ny * ks)];
        dst[i + (long long)px * j + sz * k] = (uint8_t)v;
    }
    v = __reduce_max_sync(0xffffffffu, v);
    if ((threadIdx.x & 31) == 0 && v > 0) atomicMax(max_index, v);
}
__global__ void k_unpack_u8(uint8_t *__restrict__ dst, const uint8_t *__restrict__ src, Params p) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= p.nx) return;
    dst[i + (long long)p.nx * (j + (long long)p.ny * k)] = src[i + (long long)p.px * j + p.sz * k];
}
__global__ void k_mask(uint8_t *__restrict__ dst, Params p, int open_lo, int open_hi) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= p.nx) return;
    const int P = p.P;
    uint8_t m = 0;
    if (i < P || i >= p.nx - P) m |= 1;
    if (j < P || j >= p.ny - P) m |= 2;
    if ((k < P && !open_lo) || (k >= p.nz - P && !open_hi)) m |= 4;
    dst[i + (long long)p.nx * (j + (long long)p.ny * k)] = m;
}

// counts the non-zero floats of a field allocation that lie OUTSIDE the grid cells (the zero gaps of the private
// layout, device_params.hpp): no kernel may ever write there
__global__ void k_padding_nonzeros(const float *__restrict__ f, long long n_floats, Params p, unsigned long long *count) {
    const long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (q >= n_floats) return;
    const long long r = q - p.org;                 // offset from cell (0,0,0)
    bool cell = false;
    if (r >= 0) {
        const long long k = r / p.sz, rem = r - k * p.sz;
        const long long j = rem / p.px, i = rem - j * p.px;
        cell = k < p.nz && j < p.ny && i < p.nx;
    }
    if (!cell && f[q] != 0.0f) atomicAdd(count, 1ULL);
}

dim3 grid3(const Layout &L) { return dim3((L.nx + 127) / 128, L.ny, L.nz); }

size_t field_bytes(const bvfdtd_ctx *c, uint32_t id) {
    const size_t cells = (size_t)c->L.nx * c->L.ny * c->L.nz;
    if (id <= BVFDTD_F_PRESSURE || id == BVFDTD_F_SUMSQ) return cells * 4;
    if (id == BVFDTD_F_MATERIAL || id == BVFDTD_F_PML_MASK) return cells;
    if (id == BVFDTD_F_DERIVED) return (size_t)c->n_materials * 8 * 4;
    if (id == BVFDTD_F_PML_PROFILES) return (size_t)4 * (c->L.nx + c->L.ny + c->L.nz) * 4;
    return 0;
}

// dense device buffer `d_dense` -> caller's dst (host: via async copy + sync)
int deliver(bvfdtd_ctx *c, void *dst, const void *d_dense, size_t bytes, int dst_is_device) {
    if (dst_is_device) {
        if (dst != d_dense) CU(cudaMemcpyAsync(dst, d_dense, bytes, cudaMemcpyDeviceToDevice, c->stream));
        return BVFDTD_OK;
    }
    CU(cudaMemcpyAsync(dst, d_dense, bytes, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return BVFDTD_OK;
}

void drop_graphs(bvfdtd_ctx *c) {
    for (auto &a : c->graph)
        for (auto &b : a)
            for (cudaGraphExec_t &g : b)
                if (g) { cudaGraphExecDestroy(g); g = nullptr; }
}

// Decide which tile columns run the fused single sweep (kernels_fused.cuh) and build the three work lists.
// Not for the per-cell kernels, the dense sweep, the phasor sensor, z-slab contexts (their halo planes are
// refreshed between the passes) or on request (BVFDTD_TUNE_NO_FUSED).
int fused_setup(bvfdtd_ctx *c) {
    const uint32_t off = BVFDTD_FLAG_REFERENCE_KERNELS | BVFDTD_FLAG_DENSE | BVFDTD_FLAG_PHASOR | BVFDTD_FLAG_ZLO_OPEN | BVFDTD_FLAG_ZHI_OPEN;
    if ((c->opts.flags & off) || (c->opts.tuning & BVFDTD_TUNE_NO_FUSED)) return BVFDTD_OK;
    const Layout &L = c->L;
    // small grids are launch-bound and L2-resident: a third kernel per step costs more than the bytes it saves
    // (config 1, 128^3: 22 Gcell/s with the two passes, 17.7 fused); BVFDTD_TUNE_FUSED forces the fused mode
    if ((long long)L.nx * L.ny * L.nz < 6000000LL && !(c->opts.tuning & BVFDTD_TUNE_FUSED)) return BVFDTD_OK;
    int rc = fused_plan_create(c->fplan, c->plan, L, c->prm, c->ws + c->W.psi[6], (long long)(c->W.psi[7] - c->W.psi[6]),
                               (int)((c->opts.tuning >> 16) & 3u));
    if (rc == BVFDTD_EINVAL) return BVFDTD_OK;                 // the stages do not fit: stay with the two passes
    if (rc) return cuda_fail(cudaGetLastError(), "fused_plan_create");
    uint8_t *d_cls = (uint8_t *)(c->ws + c->W.cls);
    k_fused_class<<<dim3(L.ntxV, L.ntyV, L.nz), 128, 0, c->stream>>>(c->prm, d_cls);
    CU(cudaGetLastError());
    std::vector<uint8_t> cls((size_t)L.ntxV * L.ntyV * L.nz);
    CU(cudaMemcpyAsync(cls.data(), d_cls, cls.size(), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    int sms = 148, occ_f = 1;
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device));
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_f, k_fluid_fused<CfgF>, CfgF::NT, c->fplan.smem));
    const int sty = c->plan.s16 ? CfgS::TY : CfgS8::TY;
    const FusedLists lists = fused_lists(L, cls, sty, sms * std::max(1, occ_f), sms * std::max(1, c->plan.occ_v_res),
                                         sms * std::max(1, c->plan.occ_s_res), (int)((c->opts.tuning >> 8) & 0xffu),
                                         (int)((c->opts.tuning >> 18) & 0xffu));
    const long long planes_all = (long long)L.ntxV * L.ntyV * L.nz;
    c->fplan.planes_f = lists.planes_f;
    c->fplan.planes_all = planes_all;
    // worth it from a tenth of the tile-planes on (below that the extra launch costs more than it saves)
    if (lists.planes_f * 10 < planes_all && !(c->opts.tuning & BVFDTD_TUNE_FUSED)) return BVFDTD_OK;
    if (lists.planes_f == 0) return BVFDTD_OK;
    const size_t cap = fused_items_capacity(L);
    if (lists.f.size() > cap || lists.v.size() > cap || lists.s.size() > cap) return BVFDTD_OK;
    const std::vector<int4> *src[3] = {&lists.f, &lists.v, &lists.s};
    for (int q = 0; q < 3; ++q)
        if (!src[q]->empty())
            CU(cudaMemcpyAsync(c->ws + c->W.items[q], src[q]->data(), src[q]->size() * sizeof(int4), cudaMemcpyHostToDevice, c->stream));
    CU(cudaMemcpyAsync(c->ws + c->W.flagsF, lists.flags.data(), lists.flags.size() * 4, cudaMemcpyHostToDevice, c->stream));
    c->fplan.items_f = (const int4 *)(c->ws + c->W.items[0]); c->fplan.n_f = (int)lists.f.size();
    c->fplan.items_v = (const int4 *)(c->ws + c->W.items[1]); c->fplan.n_v = (int)lists.v.size();
    c->fplan.items_s = (const int4 *)(c->ws + c->W.items[2]); c->fplan.n_s = (int)lists.s.size();
    c->ff_active = true;
    return BVFDTD_OK;
}

// sigma_yy = sigma_zz = sigma_xx in the planes the fused sweep keeps as sigma_xx only
int fused_fill(bvfdtd_ctx *c) {
    if (!c->ff_active) return BVFDTD_OK;
    k_fill_sii<<<grid3(c->L), 128, 0, c->stream>>>(c->prm);
    CU(cudaGetLastError());
    return BVFDTD_OK;
}

// Leave the fused mode for good: every tile column runs the two passes again, in place on the current copies.
int fused_disable(bvfdtd_ctx *c) {
    if (!c->ff_active) return BVFDTD_OK;
    const int rc = fused_fill(c);
    if (rc) return rc;
    c->ff_active = false;
    drop_graphs(c);
    return BVFDTD_OK;
}

}  // namespace

extern "C" {

const char *bvfdtd_strerror(int code) {
    switch (code) {
        case BVFDTD_OK: return "ok";
        case BVFDTD_EINVAL: return "invalid argument";
        case BVFDTD_ENOMEM: return "workspace too small or out of host memory";
        case BVFDTD_ESTABILITY: return "time step violates the stability bound c_U dt/dx <= 0.494";
        case BVFDTD_ECUDA: return "CUDA error (see bvfdtd_last_cuda_error)";
        case BVFDTD_ESTATE: return "call not legal in the current state";
        default: return "unknown status";
    }
}

const char *bvfdtd_last_cuda_error(void) { return g_cuda_err; }

int bvfdtd_derive_materials(const bvfdtd_material *table, int32_t n, double f0, float *out) {
    if (!out) return BVFDTD_EINVAL;
    std::vector<Derived> d;
    const int rc = derive_materials(table, n, f0, d);
    if (rc) return rc;
    for (int m = 0; m < n; ++m) {
        const double v[8] = {d[m].rho, d[m].piR, d[m].muR, d[m].tauP, d[m].tauS, d[m].piU, d[m].muU, d[m].cU};
        for (int q = 0; q < 8; ++q) out[8 * m + q] = (float)v[q];
    }
    return BVFDTD_OK;
}

int bvfdtd_pml_profiles(int32_t n, int32_t pml, double dx, double dt, double f0, double pml_R,
                        double c_ref, float *a_int, float *b_int, float *a_half, float *b_half) {
    if (n < 1 || pml < 0 || 2 * pml > n || !(dx > 0) || !(dt > 0) || !(f0 > 0) || !(c_ref > 0) ||
        !a_int || !b_int || !a_half || !b_half)
        return BVFDTD_EINVAL;
    if (pml_R == 0.0) pml_R = 1e-4;
    if (!(pml_R > 0.0 && pml_R < 1.0)) return BVFDTD_EINVAL;
    PmlAxis p;
    pml_axis(n, pml, dx, dt, f0, pml_R, c_ref, p);
    std::memcpy(a_int, p.a_int.data(), n * 4);
    std::memcpy(b_int, p.b_int.data(), n * 4);
    std::memcpy(a_half, p.a_half.data(), n * 4);
    std::memcpy(b_half, p.b_half.data(), n * 4);
    return BVFDTD_OK;
}

int bvfdtd_pml_mask(const bvfdtd_grid *g, uint8_t *mask) {
    if (!grid_ok(g) || !mask) return BVFDTD_EINVAL;
    const int P = g->pml;
    size_t q = 0;
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                uint8_t m = 0;
                if (i < P || i >= g->nx - P) m |= 1;
                if (j < P || j >= g->ny - P) m |= 2;
                if (k < P || k >= g->nz - P) m |= 4;
                mask[q++] = m;
            }
    return BVFDTD_OK;
}

double bvfdtd_max_courant(const bvfdtd_material *table, int32_t n, double f0, double dt, double dx) {
    std::vector<Derived> d;
    const int rc = derive_materials(table, n, f0, d);
    if (rc) return (double)rc;
    if (!(dt > 0) || !(dx > 0)) return (double)BVFDTD_EINVAL;
    return max_courant(d, dt, dx);
}

int bvfdtd_workspace_bytes(const bvfdtd_grid *grid, size_t *out_bytes) {
    if (!grid_ok(grid) || !out_bytes) return BVFDTD_EINVAL;
    *out_bytes = make_wsmap(make_layout(*grid)).total;
    return BVFDTD_OK;
}

int bvfdtd_create(bvfdtd_ctx **out, const bvfdtd_grid *grid, double dx, double dt,
                  const bvfdtd_material *table, int32_t n_materials, const uint8_t *index_map,
                  const bvfdtd_opts *opts, void *d_workspace, size_t workspace_bytes,
                  void *cuda_stream) {
    if (!out) return BVFDTD_EINVAL;
    *out = nullptr;
    if (!grid_ok(grid) || !table || !index_map || !opts || !d_workspace) return BVFDTD_EINVAL;
    if (!(dx > 0.0) || !(dt > 0.0) || !std::isfinite(dx) || !std::isfinite(dt)) return BVFDTD_EINVAL;
    constexpr uint32_t TUNE_ALL = BVFDTD_TUNE_VEL_2CTA | BVFDTD_TUNE_VEL_3CTA | BVFDTD_TUNE_STRESS_8 | BVFDTD_TUNE_STRESS_16 |
                                  BVFDTD_TUNE_NO_GRAPH | BVFDTD_TUNE_NO_FUSED | BVFDTD_TUNE_FUSED | 0x3ffff00u;   // + the three experiment fields
    if (!(opts->f0 > 0.0) || (opts->tuning & ~TUNE_ALL) != 0) return BVFDTD_EINVAL;
    if ((opts->tuning & BVFDTD_TUNE_VEL_2CTA) && (opts->tuning & BVFDTD_TUNE_VEL_3CTA)) return BVFDTD_EINVAL;
    if ((opts->tuning & BVFDTD_TUNE_STRESS_8) && (opts->tuning & BVFDTD_TUNE_STRESS_16)) return BVFDTD_EINVAL;
    if ((opts->tuning & BVFDTD_TUNE_NO_FUSED) && (opts->tuning & BVFDTD_TUNE_FUSED)) return BVFDTD_EINVAL;
    double R = opts->pml_R == 0.0 ? 1e-4 : opts->pml_R;
    if (!(R > 0.0 && R < 1.0)) return BVFDTD_EINVAL;
    if (((uintptr_t)d_workspace & 255) != 0) return BVFDTD_EINVAL;

    bvfdtd_ctx *c = new (std::nothrow) bvfdtd_ctx;
    if (!c) return BVFDTD_ENOMEM;
    struct Guard { bvfdtd_ctx *c; ~Guard() { delete c; } } guard{c};

    int rc = derive_materials(table, n_materials, opts->f0, c->derived);
    if (rc) return rc;
    if (max_courant(c->derived, dt, dx) > 0.494) return BVFDTD_ESTABILITY;
    const size_t cells = (size_t)grid->nx * grid->ny * grid->nz;

    c->L = make_layout(*grid);
    c->W = make_wsmap(c->L);
    if (workspace_bytes < c->W.total) return BVFDTD_ENOMEM;
    // the context lives on the device that owns the workspace, whatever device is current in the caller
    c->device = device_of(d_workspace);
    if (c->device < 0) return cuda_fail(cudaErrorInvalidDevicePointer, "d_workspace is not device memory (or no CUDA device)");
    DeviceScope scope(c->device);
    c->ws = (char *)d_workspace;
    c->stream = (cudaStream_t)cuda_stream;
    c->dx = dx; c->dt = dt; c->opts = *opts; c->opts.pml_R = R; c->n_materials = n_materials;
    c->table.assign(table, table + n_materials);
    const Layout &L = c->L;

    // S0 tables
    std::vector<KRow> rows;
    kernel_rows(c->derived, dt, opts->f0, rows);
    rows.resize(256, rows[0]);
    double c_ref = 0.0;
    for (int m = 0; m < n_materials; ++m) c_ref = std::max(c_ref, table[m].cL);
    const int dims[3] = {L.nx, L.ny, L.nz};
    std::vector<float> prof;
    for (int a = 0; a < 3; ++a) {
        pml_axis(dims[a], L.P, dx, dt, opts->f0, R, c_ref, c->pml[a], a == 2 && (opts->flags & BVFDTD_FLAG_ZLO_OPEN),
                 a == 2 && (opts->flags & BVFDTD_FLAG_ZHI_OPEN));
        for (const std::vector<float> *v : {&c->pml[a].a_int, &c->pml[a].b_int, &c->pml[a].a_half, &c->pml[a].b_half})
            prof.insert(prof.end(), v->begin(), v->end());
    }
    // small tables first, while the stream is still empty (a pageable source is staged before cudaMemcpyAsync
    // returns, so the vectors may die at return; it also waits for the stream's earlier work)
    CU(cudaMemcpyAsync(c->ws + c->W.rows, rows.data(), 256 * sizeof(KRow), cudaMemcpyHostToDevice, c->stream));
    CU(cudaMemcpyAsync(c->ws + c->W.prof, prof.data(), prof.size() * 4, cudaMemcpyHostToDevice, c->stream));
    float invz[256];
    for (int m = 0; m < 256; ++m) invz[m] = m < n_materials ? (float)(1.0 / (table[m].rho * table[m].cL)) : 0.0f;
    CU(cudaMemcpyAsync(c->ws + c->W.invz, invz, sizeof(invz), cudaMemcpyHostToDevice, c->stream));
    // zero the state, the sensors, psi, the flag words and the counters (reading P9); the scratch plane, the
    // index map and the tables are fully written below
    CU(cudaMemsetAsync(c->ws + c->W.zero0, 0, c->W.zero1 - c->W.zero0, c->stream));
    // index map: dense upload into the scratch plane, then validated and padded into the private
    // layout on the device (edges replicated, reading P2)
    CU(cudaMemcpyAsync(c->ws + c->W.scratch, index_map, cells, cudaMemcpyHostToDevice, c->stream));
    int *d_max = (int *)(c->ws + c->W.ctr + 16);
    {
        const dim3 b(128), g((L.px + 127) / 128, L.py, L.nz + 1);
        k_pad_index_map<<<g, b, 0, c->stream>>>((uint8_t *)(c->ws + c->W.mat), (const uint8_t *)(c->ws + c->W.scratch), L.nx, L.ny, L.nz, L.px, L.py, L.sz, d_max);
        CU(cudaGetLastError());
    }
    Params &p = c->prm;
    p.nx = L.nx; p.ny = L.ny; p.nz = L.nz; p.P = L.P;
    p.n_mat = n_materials;
    p.px = L.px; p.py = L.py; p.wx = L.wx; p.sz = L.sz; p.org = L.org;
    p.xp4 = L.xp4; p.xhb = L.xhb; p.xph = L.xph;
    p.ntxV = L.ntxV; p.ntyV = L.ntyV; p.ntxS = L.ntxS; p.ntyS = L.ntyS;
    p.flagsV = (const uint32_t *)(c->ws + c->W.flagsV);
    p.flagsS = (const uint32_t *)(c->ws + c->W.flagsS);
    for (int q = 0; q < NSTATE; ++q) p.f[q] = (float *)(c->ws + c->W.field[q]);
    p.peak = (float *)(c->ws + c->W.peak);
    p.sumsq = (float *)(c->ws + c->W.sumsq);
    p.phre = (float *)(c->ws + c->W.phre);
    p.phim = (float *)(c->ws + c->W.phim);
    p.mat = (const uint8_t *)(c->ws + c->W.mat);
    for (int q = 0; q < 18; ++q) p.psi[q] = (float *)(c->ws + c->W.psi[q]);
    // no fused sweep (yet): the passes work in place, cur == nxt
    for (int q = 0; q < 6; ++q) { p.icur[q] = p.inxt[q] = q; p.fnxt[q] = p.f[q]; }
    p.ipsi7_cur = 1; p.psi7_nxt = p.psi[7];
    p.flagsF = (const uint32_t *)(c->ws + c->W.flagsF);
    p.rows = (const KRow *)(c->ws + c->W.rows);
    {
        const float *base = (const float *)(c->ws + c->W.prof);
        for (int a = 0; a < 3; ++a)
            for (int q = 0; q < 4; ++q) { p.prof[a][q] = base; base += dims[a]; }
    }
    const double tau_sigma = 1.0 / (2.0 * 3.14159265358979323846 * opts->f0);
    const double beta = dt / (2.0 * tau_sigma);
    p.inv_dx = (float)(1.0 / dx);
    p.dt = (float)dt;
    p.half_dt = (float)(0.5 * dt);
    p.A = (float)((1.0 - beta) / (1.0 + beta));
    p.B = (float)(2.0 * beta / (1.0 + beta));

    if (!(opts->flags & BVFDTD_FLAG_REFERENCE_KERNELS)) {
        char *psi_base[3];
        long long psi_stride[3];
        for (int a = 0; a < 3; ++a) {
            psi_base[a] = c->ws + c->W.psi[a * 6];
            psi_stride[a] = (long long)(c->W.psi[a * 6 + 1] - c->W.psi[a * 6]);
        }
        PlanTuning tune;
        tune.occ_v = (opts->tuning & BVFDTD_TUNE_VEL_2CTA) ? 2 : (opts->tuning & BVFDTD_TUNE_VEL_3CTA) ? 3 : 0;
        tune.stress_ty = (opts->tuning & BVFDTD_TUNE_STRESS_8) ? 8 : (opts->tuning & BVFDTD_TUNE_STRESS_16) ? 16 : 0;
        tune.fused_chunk = (int)((opts->tuning >> 8) & 0xffu);
        tune.l2_promotion = (int)((opts->tuning >> 16) & 3u);
        rc = tiled_plan_create(c->plan, c->L, c->prm, psi_base, psi_stride, (opts->flags & BVFDTD_FLAG_DENSE) != 0, tune);
        if (rc) return rc == BVFDTD_ECUDA ? cuda_fail(cudaErrorUnknown, tiled_plan_error()) : rc;
        {
            // z chunks of the two passes when they sweep a whole large grid (dense sweep, z-slab contexts, phasor runs,
            // BVFDTD_TUNE_NO_FUSED): short chunks, the z slabs in chunks of their own -- what the work lists of the
            // fused mode use and for the same reason (kernels_fused.cuh: CTAs of one z range share their halo rows in
            // L2).  Experiment field of opts.tuning: planes per chunk; 0 = the plan of tiled_plan_create.
            const int want = (int)((opts->tuning >> 18) & 0xffu);
            if (want > 0) {
                const int nz = c->L.nz, P = c->L.P;
                const int len = std::max(want, (nz + MAX_CHUNKS - 7) / (MAX_CHUNKS - 6));
                ZChunks z;
                int n = 0;
                z.b[0] = 0;
                auto add = [&](int a, int b) {
                    const int m = std::max(1, (b - a + len - 1) / len);
                    for (int q = 1; q <= m; ++q) z.b[++n] = a + (int)((long long)(b - a) * q / m);
                };
                if (P >= 8 && nz - 2 * P >= 16) { add(0, P); add(P, nz - P); add(nz - P, nz); }
                else add(0, nz);
                z.n = n;
                c->plan.zv = z;
                c->plan.zs = z;
            }
        }
        c->dense = (opts->flags & BVFDTD_FLAG_DENSE) != 0;
        tiled_flags(c->plan, c->prm, (uint32_t *)(c->ws + c->W.flagsV), (uint32_t *)(c->ws + c->W.flagsS), c->dense, c->stream);
        CU(cudaGetLastError());
    }
    // the one synchronisation of create: the largest material index of the map (validation)
    int h_max = 0;
    CU(cudaMemcpyAsync(&h_max, d_max, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (h_max >= n_materials) return BVFDTD_EINVAL;
    rc = fused_setup(c);
    if (rc) return rc;
    guard.c = nullptr;
    *out = c;
    return BVFDTD_OK;
}

int bvfdtd_set_source(bvfdtd_ctx *c, int64_t n_src, const int64_t *cell, const float *amp,
                      const float *delay_s, int32_t waveform, double f_src, int32_t n_cycles) {
    if (!c || n_src < 0) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    if (n_src > 0) {
        if (!cell || !amp || !delay_s || !(f_src > 0.0) || n_cycles < 1 || (waveform != 0 && waveform != 1))
            return BVFDTD_EINVAL;
        const Layout &L = c->L;
        const int64_t cells = (int64_t)L.nx * L.ny * L.nz;
        std::vector<int64_t> sorted(cell, cell + n_src);
        std::sort(sorted.begin(), sorted.end());
        for (int64_t s = 0; s < n_src; ++s) {
            const int64_t q = sorted[s];
            if (q < 0 || q >= cells) return BVFDTD_EINVAL;
            if (s && sorted[s - 1] == q) return BVFDTD_EINVAL;
            const int i = (int)(q % L.nx), j = (int)((q / L.nx) % L.ny), k = (int)(q / ((int64_t)L.nx * L.ny));
            const int P = L.P;
            const bool zlo = !(c->opts.flags & BVFDTD_FLAG_ZLO_OPEN), zhi = !(c->opts.flags & BVFDTD_FLAG_ZHI_OPEN);
            if (i < P || i >= L.nx - P || j < P || j >= L.ny - P || (zlo && k < P) || (zhi && k >= L.nz - P)) return BVFDTD_EINVAL;
            if (!std::isfinite(amp[s]) || !std::isfinite(delay_s[s])) return BVFDTD_EINVAL;
        }
    }
    // the device copy lives in the workspace's source region (room for four x-y planes of cells); only a longer
    // list gets a library-owned allocation.  The arrays are packed on the host first, so the caller's buffers
    // are free at return without a stream synchronisation (a pageable source is staged before
    // cudaMemcpyAsync returns).
    drop_graphs(c);
    c->n_src = 0;
    c->d_cell = nullptr; c->d_amp = c->d_delay = nullptr;
    if (c->src_own) {
        CU(cudaStreamSynchronize(c->stream));     // a step in flight may still read the old list
        cudaFree(c->src_own);
        c->src_own = nullptr;
    }
    if (n_src > 0) {
        char *d_base = c->ws + c->W.src;
        if (n_src > c->W.src_cap) {
            CU(cudaMalloc(&c->src_own, (size_t)n_src * 16));
            d_base = (char *)c->src_own;
        }
        std::vector<char> pack((size_t)n_src * 16);
        std::memcpy(pack.data(), cell, (size_t)n_src * 8);
        std::memcpy(pack.data() + (size_t)n_src * 8, amp, (size_t)n_src * 4);
        std::memcpy(pack.data() + (size_t)n_src * 12, delay_s, (size_t)n_src * 4);
        CU(cudaMemcpyAsync(d_base, pack.data(), pack.size(), cudaMemcpyHostToDevice, c->stream));
        c->d_cell = (long long *)d_base;
        c->d_amp = (float *)(d_base + (size_t)n_src * 8);
        c->d_delay = (float *)(d_base + (size_t)n_src * 12);
        c->n_src = n_src; c->waveform = waveform; c->f_src = f_src; c->n_cycles = n_cycles;
    }
    return BVFDTD_OK;
}

namespace {

enum { PH_INJECT = 1, PH_VELOCITY = 2, PH_STRESS = 4, PH_ALL = 7 };

__global__ void k_set_counter(long long *d_ctr, long long step) {
    d_ctr[0] = step;
    d_ctr[1] = 0;      // block ticket of k_inject
}

// sensor regime of step n: bit 0 running peak on, bit 1 sum of squares (or phasor) on (reading P8)
int regime_of(const bvfdtd_ctx *c, int64_t step) {
    const bool in_end = c->opts.sensor_end < 0 || step < c->opts.sensor_end;
    return (in_end && step >= c->opts.peak_begin ? 1 : 0) | (in_end && step >= c->opts.rms_begin ? 2 : 0);
}
// number of steps from `step` on (at most n) that share its regime
int64_t regime_run(const bvfdtd_ctx *c, int64_t step, int64_t n) {
    int64_t run = n;
    for (int64_t edge : {c->opts.peak_begin, c->opts.rms_begin, c->opts.sensor_end})
        if (edge > step) run = std::min(run, edge - step);
    return run;
}

// the cur / nxt copies of the ping-pong arrays for a step that starts with copy `sel` current
void select_copies(const bvfdtd_ctx *c, Params &p, int sel, bool pingpong) {
    for (int q = 0; q < 6; ++q) {
        float *prim = (float *)(c->ws + c->W.field[q]), *alt = (float *)(c->ws + c->W.alt[q]);
        p.f[q] = sel ? alt : prim;
        p.icur[q] = sel ? F_ALT + q : q;
        p.fnxt[q] = pingpong ? (sel ? prim : alt) : p.f[q];
        p.inxt[q] = pingpong ? (sel ? q : F_ALT + q) : p.icur[q];
    }
    float *p7 = (float *)(c->ws + c->W.psi[7]), *p7a = (float *)(c->ws + c->W.psi7_alt);
    p.psi[7] = sel ? p7a : p7;
    p.ipsi7_cur = sel ? PSI7_ALT : 1;
    p.psi7_nxt = pingpong ? (sel ? p7 : p7a) : p.psi[7];
}

// kernel parameters of step `step` when copy `sel` of the ping-pong arrays is current
Params step_params(const bvfdtd_ctx *c, int64_t step, int regime, int sel) {
    Params p = c->prm;
    select_copies(c, p, sel, c->ff_active);
    p.do_peak = regime & 1;
    p.do_rms = (regime >> 1) & 1;
    p.do_phasor = 0; p.ph_cos = p.ph_sin = 0.0f;
    if (c->opts.flags & BVFDTD_FLAG_PHASOR) {
        // NEXT-3: the window [rms_begin, sensor_end) accumulates the phasor at f0; no peak / rms
        p.do_phasor = p.do_rms;
        p.do_peak = p.do_rms = 0;
        if (p.do_phasor) {
            const double wt = 2.0 * 3.14159265358979323846 * c->opts.f0 * (double)(step + 1) * c->dt;
            p.ph_cos = (float)std::cos(wt); p.ph_sin = (float)std::sin(wt);
        }
    }
    return p;
}

// after a step of the fused mode the other copy is current
void flip_copies(bvfdtd_ctx *c, int64_t steps) {
    if (!c->ff_active || !(steps & 1)) return;
    c->sel ^= 1;
    select_copies(c, c->prm, c->sel, false);
}

// Enqueue the passes of one step selected by `phases`.  d_ctr != nullptr: the injection takes the step index
// from the device counter (graph replay); ev != nullptr: five events bracket the four kernels (inject, fused sweep,
// velocity pass, stress pass).
int enqueue_passes(bvfdtd_ctx *c, const Params &p, int phases, int64_t step, long long *d_ctr, cudaEvent_t *ev, cudaStream_t st) {
    const Layout &L = c->L;
    const bool ref = (c->opts.flags & BVFDTD_FLAG_REFERENCE_KERNELS) != 0;
    if (ev) CU(cudaEventRecord(ev[0], st));
    if ((phases & PH_INJECT) && c->n_src > 0) {
        const int tb = 128;
        k_inject<<<(unsigned)((c->n_src + tb - 1) / tb), tb, 0, st>>>(
            p, c->n_src, c->d_cell, c->d_amp, c->d_delay, c->waveform, c->f_src, c->n_cycles, c->dt, (long long)step, d_ctr);
    }
    if (ev) CU(cudaEventRecord(ev[1], st));
    const dim3 rb(32, 4, 2), rg((L.nx + 31) / 32, (L.ny + 3) / 4, (L.nz + 1) / 2);
    const bool ff = c->ff_active;       // (only whole steps run in the fused mode: bvfdtd_step_phase leaves it first)
    // in a captured step the fused sweep and the velocity pass of the other tile columns are two branches of the
    // graph: they are independent (both read the cur copies and write the nxt ones) and fill each other's last wave
    const bool fork = ff && d_ctr && c->cap_stream2 && c->fplan.n_f > 0 && c->fplan.n_v > 0 && (phases & PH_VELOCITY);
    cudaStream_t sv = st;
    if (fork) {
        CU(cudaEventRecord(c->cap_fork, st));
        CU(cudaStreamWaitEvent(c->cap_stream2, c->cap_fork, 0));
        sv = c->cap_stream2;
    }
    if (ff && (phases & PH_VELOCITY)) fused_launch(c->fplan, p, st);
    if (ev) CU(cudaEventRecord(ev[2], st));
    if (phases & PH_VELOCITY) {
        if (ref) k_velocity_ref<<<rg, rb, 0, st>>>(p);
        else if (tiled_velocity(c->plan, p, sv, ff ? c->fplan.items_v : nullptr, c->fplan.n_v)) return cuda_fail(cudaGetLastError(), "tiled_velocity");
    }
    if (fork) {
        CU(cudaEventRecord(c->cap_join, sv));
        CU(cudaStreamWaitEvent(st, c->cap_join, 0));
    }
    if (ev) CU(cudaEventRecord(ev[3], st));
    if (phases & PH_STRESS) {
        if (ref) k_stress_ref<<<rg, rb, 0, st>>>(p);
        else if (tiled_stress(c->plan, p, st, ff ? c->fplan.items_s : nullptr, c->fplan.n_s)) return cuda_fail(cudaGetLastError(), "tiled_stress");
    }
    if (ev) CU(cudaEventRecord(ev[4], st));
    return BVFDTD_OK;
}

// The passes of step c->step selected by `phases`; the step counter advances with the stress pass.
int run_phases(bvfdtd_ctx *c, int phases) {
    const int64_t step = c->step;
    const Params p = step_params(c, step, regime_of(c, step), c->sel);
    const bool timed = phases == PH_ALL && c->timing && c->timed_steps < BVFDTD_MAX_TIMED_STEPS;
    cudaEvent_t *ev = nullptr;
    if (timed) {
        if (c->ev.size() < (size_t)(c->timed_steps + 1) * 5) {
            for (int q = 0; q < 5; ++q) { cudaEvent_t e; CU(cudaEventCreate(&e)); c->ev.push_back(e); }
        }
        ev = &c->ev[c->timed_steps * 5];
    }
    const int rc = enqueue_passes(c, p, phases, step, nullptr, ev, c->stream);
    if (rc) return rc;
    if (timed) c->timed_steps++;
    if (phases & PH_STRESS) {
        if (p.do_rms || p.do_phasor) c->rms_count++;
        c->step++;
        c->phase_done = 0;
        flip_copies(c, 1);
    } else {
        c->phase_done |= phases;
    }
    return BVFDTD_OK;
}

// bvfdtd_step replays CUDA graphs unless the caller asked for per-kernel timing, the phasor sensor is on (its
// cos / sin change every step) or the context says no (BVFDTD_TUNE_NO_GRAPH)
bool graph_ok(const bvfdtd_ctx *c) {
    return !c->timing && !(c->opts.flags & BVFDTD_FLAG_PHASOR) && !(c->opts.tuning & BVFDTD_TUNE_NO_GRAPH);
}


// the graph of `len` (1 or GRAPH_STEPS) consecutive steps in sensor regime `regime`, captured on first use
int get_graph(bvfdtd_ctx *c, int regime, int len, cudaGraphExec_t *out) {
    cudaGraphExec_t &slot = c->graph[regime][len == 1 ? 0 : 1][c->sel];
    if (!slot) {
        long long *d_ctr = (long long *)(c->ws + c->W.ctr);
        if (!c->cap_stream) {
            CU(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
            CU(cudaStreamCreateWithFlags(&c->cap_stream2, cudaStreamNonBlocking));
            CU(cudaEventCreateWithFlags(&c->cap_fork, cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&c->cap_join, cudaEventDisableTiming));
        }
        CU(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeRelaxed));
        int rc = BVFDTD_OK;
        for (int s = 0; s < len && rc == BVFDTD_OK; ++s) {
            // (in the fused mode consecutive steps alternate between the two copies of the ping-pong arrays)
            const Params p = step_params(c, 0, regime, c->ff_active ? (c->sel ^ (s & 1)) : c->sel);
            rc = enqueue_passes(c, p, PH_ALL, 0, d_ctr, nullptr, c->cap_stream);
        }
        cudaGraph_t g = nullptr;
        const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
        if (rc) { if (g) cudaGraphDestroy(g); return rc; }
        if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture");
        const cudaError_t e2 = cudaGraphInstantiate(&slot, g, 0);
        cudaGraphDestroy(g);
        if (e2 != cudaSuccess) { slot = nullptr; return cuda_fail(e2, "cudaGraphInstantiate"); }
    }
    *out = slot;
    return BVFDTD_OK;
}

}  // namespace

int bvfdtd_step(bvfdtd_ctx *c, int64_t n) {
    if (!c || n < 0) return BVFDTD_EINVAL;
    if (c->phase_done != 0 || c->phase_planes != 0) return BVFDTD_ESTATE;   // a step begun with bvfdtd_step_phase must be finished first
    DeviceScope scope(c->device);
    if (n >= 2 && graph_ok(c)) {
        // one graph launch per GRAPH_STEPS steps (per step for the remainder) instead of three kernel launches
        // per step: the small grids are launch-bound
        if (c->n_src > 0) k_set_counter<<<1, 1, 0, c->stream>>>((long long *)(c->ws + c->W.ctr), (long long)c->step);
        int64_t left = n;
        while (left > 0) {
            const int regime = regime_of(c, c->step);
            int64_t run = regime_run(c, c->step, left);
            left -= run;
            while (run > 0) {
                const int len = run >= bvfdtd_ctx::GRAPH_STEPS ? (int)bvfdtd_ctx::GRAPH_STEPS : 1;
                cudaGraphExec_t g = nullptr;
                const int rc = get_graph(c, regime, len, &g);
                if (rc) return rc;
                CU(cudaGraphLaunch(g, c->stream));
                c->step += len;
                if (regime & 2) c->rms_count += len;
                flip_copies(c, len);
                run -= len;
            }
        }
        CU(cudaGetLastError());
        return BVFDTD_OK;
    }
    for (int64_t s = 0; s < n; ++s) {
        int rc = run_phases(c, PH_ALL);
        if (rc) return rc;
    }
    CU(cudaGetLastError());
    return BVFDTD_OK;
}

int bvfdtd_step_phase(bvfdtd_ctx *c, int32_t phase) {
    if (!c || phase < 0 || phase > 2) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    // the passes of one step run in order: inject (0), velocity (1), stress + sensor (2)
    const int bit = 1 << phase;
    const int before = bit - 1;                       // every earlier pass must have run, this one not
    if ((c->phase_done & before) != before || (c->phase_done & bit) || c->phase_planes != 0) return BVFDTD_ESTATE;
    int rc = fused_disable(c);          // single passes run on every tile column
    if (rc) return rc;
    rc = run_phases(c, bit);
    if (rc) return rc;
    CU(cudaGetLastError());
    return BVFDTD_OK;
}

int bvfdtd_step_phase_planes(bvfdtd_ctx *c, int32_t phase, int32_t k0, int32_t k1) {
    if (!c || (phase != 1 && phase != 2) || k0 < 0 || k1 <= k0 || k1 > c->L.nz) return BVFDTD_EINVAL;
    if (c->opts.flags & BVFDTD_FLAG_REFERENCE_KERNELS) return BVFDTD_ESTATE;      // the per-cell kernels sweep whole grids
    DeviceScope scope(c->device);
    const int bit = 1 << phase, before = bit - 1;
    if ((c->phase_done & before) != before || (c->phase_done & bit)) return BVFDTD_ESTATE;
    if (c->phase_planes + (k1 - k0) > c->L.nz) return BVFDTD_ESTATE;              // ranges of one pass must not overlap
    int rc = fused_disable(c);
    if (rc) return rc;
    // the pass over planes [k0, k1) of every tile column, as a work list in a slice of the list region
    const Layout &L = c->L;
    const bool vel = phase == 1;
    const int ntx = vel ? L.ntxV : L.ntxS, nty = vel ? L.ntyV : c->prm.ntyS;
    const int nchunk = (k1 - k0 + 47) / 48;
    std::vector<int4> items;
    items.reserve((size_t)ntx * nty * nchunk);
    for (int ch = 0; ch < nchunk; ++ch) {
        const int a = k0 + (int)((long long)(k1 - k0) * ch / nchunk), b = k0 + (int)((long long)(k1 - k0) * (ch + 1) / nchunk);
        for (int by = 0; by < nty; ++by)
            for (int bx = 0; bx < ntx; ++bx) items.push_back(make_int4(bx, by, a, b));
    }
    const size_t slice = fused_items_capacity(L) / 4;
    if (items.size() > slice) return BVFDTD_EINVAL;
    int4 *d_items = (int4 *)(c->ws + c->W.items[vel ? 1 : 2]) + slice * (size_t)(c->range_slot++ & 3);
    CU(cudaMemcpyAsync(d_items, items.data(), items.size() * sizeof(int4), cudaMemcpyHostToDevice, c->stream));
    const int64_t step = c->step;
    const Params p = step_params(c, step, regime_of(c, step), c->sel);
    if (vel) tiled_velocity(c->plan, p, c->stream, d_items, (int)items.size());
    else tiled_stress(c->plan, p, c->stream, d_items, (int)items.size());
    CU(cudaGetLastError());
    c->phase_planes += k1 - k0;
    if (c->phase_planes == L.nz) {
        c->phase_planes = 0;
        if (vel) c->phase_done |= bit;
        else {
            if (p.do_rms || p.do_phasor) c->rms_count++;
            c->step++;
            c->phase_done = 0;
        }
    }
    return BVFDTD_OK;
}

int bvfdtd_plane_span(const bvfdtd_grid *grid, uint32_t field_id, int32_t k, int32_t n_planes, size_t *offset_bytes, size_t *bytes) {
    if (!grid_ok(grid) || field_id >= NSTATE || !offset_bytes || !bytes || k < 0 || n_planes < 1 || k + n_planes > grid->nz)
        return BVFDTD_EINVAL;
    const Layout L = make_layout(*grid);
    const WsMap W = make_wsmap(L);
    *offset_bytes = W.field[field_id] + (size_t)(L.org + L.sz * k) * 4;
    *bytes = (size_t)L.sz * n_planes * 4;
    return BVFDTD_OK;
}

int64_t bvfdtd_step_index(const bvfdtd_ctx *c) { return c ? c->step : -1; }

int64_t bvfdtd_rms_count(const bvfdtd_ctx *c) { return c ? c->rms_count : -1; }

int bvfdtd_kernel_mode(const bvfdtd_ctx *c, uint32_t *mode) {
    if (!c || !mode) return BVFDTD_EINVAL;
    uint32_t m = 0;
    if (c->opts.flags & BVFDTD_FLAG_REFERENCE_KERNELS) m |= BVFDTD_MODE_REFERENCE;
    else if (c->dense) m |= BVFDTD_MODE_DENSE;
    if (c->sigma_written) m |= BVFDTD_MODE_SIGMA_WRITTEN;
    if (graph_ok(c)) m |= BVFDTD_MODE_GRAPH;
    if (c->ff_active) m |= BVFDTD_MODE_FUSED;
    *mode = m;
    return BVFDTD_OK;
}

int bvfdtd_read_fields(bvfdtd_ctx *c, uint32_t id, void *dst, size_t dst_bytes, int32_t dst_is_device) {
    if (!c || !dst) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    const size_t need = field_bytes(c, id);
    if (need == 0 || dst_bytes != need) return BVFDTD_EINVAL;
    const Layout &L = c->L;
    const dim3 b(128), g = grid3(L);
    float *scratch = (float *)(c->ws + c->W.scratch);
    if (id == BVFDTD_F_DERIVED || id == BVFDTD_F_PML_PROFILES) {
        if (dst_is_device) return BVFDTD_EINVAL;
        float *o = (float *)dst;
        if (id == BVFDTD_F_DERIVED) {
            for (int m = 0; m < c->n_materials; ++m) {
                const Derived &d = c->derived[m];
                const double v[8] = {d.rho, d.piR, d.muR, d.tauP, d.tauS, d.piU, d.muU, d.cU};
                for (int q = 0; q < 8; ++q) *o++ = (float)v[q];
            }
        } else {
            for (int a = 0; a < 3; ++a)
                for (const std::vector<float> *v : {&c->pml[a].a_int, &c->pml[a].b_int, &c->pml[a].a_half, &c->pml[a].b_half}) {
                    std::memcpy(o, v->data(), v->size() * 4);
                    o += v->size();
                }
        }
        return BVFDTD_OK;
    }
    void *target = dst_is_device ? dst : (void *)scratch;
    // r_yy / r_zz are not kept where they equal r_xx (all-fluid lossy tile-planes of the tiled path): fill them in
    if ((id == RYY || id == RZZ) && !c->dense && !(c->opts.flags & BVFDTD_FLAG_REFERENCE_KERNELS))
        tiled_fill_rii(c->plan, c->prm, c->stream);
    // ... and sigma_yy / sigma_zz where the fused sweep keeps sigma_xx only
    if (id == SYY || id == SZZ || id == BVFDTD_F_PRESSURE) {
        const int rcf = fused_fill(c);
        if (rcf) return rcf;
    }
    if (id < NSTATE) k_unpack<<<g, b, 0, c->stream>>>((float *)target, c->prm.f[id], c->prm);
    else if (id == BVFDTD_F_SUMSQ) k_unpack<<<g, b, 0, c->stream>>>((float *)target, c->prm.sumsq, c->prm);
    else if (id == BVFDTD_F_PRESSURE) k_pressure<<<g, b, 0, c->stream>>>((float *)target, c->prm);
    else if (id == BVFDTD_F_MATERIAL) k_unpack_u8<<<g, b, 0, c->stream>>>((uint8_t *)target, c->prm.mat, c->prm);
    else k_mask<<<g, b, 0, c->stream>>>((uint8_t *)target, c->prm, (c->opts.flags & BVFDTD_FLAG_ZLO_OPEN) != 0, (c->opts.flags & BVFDTD_FLAG_ZHI_OPEN) != 0);
    CU(cudaGetLastError());
    return deliver(c, dst, target, need, dst_is_device);
}

int bvfdtd_write_fields(bvfdtd_ctx *c, uint32_t id, const void *src, size_t src_bytes, int32_t src_is_device) {
    if (!c || !src || id >= NSTATE) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    if (src_bytes != field_bytes(c, id)) return BVFDTD_EINVAL;
    const float *d_src = (const float *)src;
    if (id >= SXX) {
        // a caller-supplied stress or memory variable ends the fused mode (it relies on sigma_xx = sigma_yy =
        // sigma_zz, r_xx = r_yy = r_zz and zero shear stresses in its tile columns)
        const int rcf = fused_disable(c);
        if (rcf) return rcf;
    }
    if (!src_is_device) {
        float *scratch = (float *)(c->ws + c->W.scratch);
        CU(cudaMemcpyAsync(scratch, src, src_bytes, cudaMemcpyHostToDevice, c->stream));
        d_src = scratch;
    }
    if (id >= SXY && !c->dense && !(c->opts.flags & BVFDTD_FLAG_REFERENCE_KERNELS)) {
        // a caller-supplied shear stress or memory variable may be non-zero where the tile-class
        // flags assume it is identically zero (or equal to r_xx): switch this context to the dense
        // sweep, after r_yy / r_zz have been filled in where only r_xx was kept
        tiled_fill_rii(c->plan, c->prm, c->stream);
        c->dense = true;
        tiled_flags(c->plan, c->prm, (uint32_t *)(c->ws + c->W.flagsV), (uint32_t *)(c->ws + c->W.flagsS), true, c->stream);
        CU(cudaGetLastError());
    }
    if (id >= SXX && id <= SZZ && !c->dense && !c->sigma_written && !(c->opts.flags & BVFDTD_FLAG_REFERENCE_KERNELS)) {
        // a caller-supplied normal stress need not satisfy sigma_xx = sigma_yy = sigma_zz in the fluid: the
        // velocity pass stops reading sigma_xx in place of the other two
        c->sigma_written = true;
        tiled_flags(c->plan, c->prm, (uint32_t *)(c->ws + c->W.flagsV), (uint32_t *)(c->ws + c->W.flagsS), false, c->stream, false);
        CU(cudaGetLastError());
    }
    k_pack<<<grid3(c->L), 128, 0, c->stream>>>(c->prm.f[id], d_src, c->prm, id <= VZ ? (int)id : -1);
    CU(cudaGetLastError());
    if (!src_is_device) CU(cudaStreamSynchronize(c->stream));
    return BVFDTD_OK;
}

int bvfdtd_read_peak_pressure(bvfdtd_ctx *c, float *peak, float *rms_amp, int32_t dst_is_device) {
    if (!c) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    const Layout &L = c->L;
    const size_t bytes = (size_t)L.nx * L.ny * L.nz * 4;
    float *scratch = (float *)(c->ws + c->W.scratch);
    if (peak) {
        float *target = dst_is_device ? peak : scratch;
        k_unpack<<<grid3(L), 128, 0, c->stream>>>(target, c->prm.peak, c->prm);
        CU(cudaGetLastError());
        const int rc = deliver(c, peak, target, bytes, dst_is_device);
        if (rc) return rc;
    }
    if (rms_amp) {
        float *target = dst_is_device ? rms_amp : scratch;
        const float toc = c->rms_count > 0 ? (float)(2.0 / (double)c->rms_count) : 0.0f;
        k_rms_amp<<<grid3(L), 128, 0, c->stream>>>(target, c->prm, toc);
        CU(cudaGetLastError());
        const int rc = deliver(c, rms_amp, target, bytes, dst_is_device);
        if (rc) return rc;
    }
    return BVFDTD_OK;
}

int bvfdtd_read_phasor(bvfdtd_ctx *c, float *re, float *im, int32_t dst_is_device) {
    if (!c || !re || !im) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    if (!(c->opts.flags & BVFDTD_FLAG_PHASOR)) return BVFDTD_ESTATE;
    const Layout &L = c->L;
    const size_t bytes = (size_t)L.nx * L.ny * L.nz * 4;
    float *scratch = (float *)(c->ws + c->W.scratch);
    const float sc = c->rms_count > 0 ? (float)(2.0 / (double)c->rms_count) : 0.0f;
    for (int part = 0; part < 2; ++part) {
        float *dst = part ? im : re;
        float *target = dst_is_device ? dst : scratch;
        k_unpack_scaled<<<grid3(L), 128, 0, c->stream>>>(target, part ? c->prm.phim : c->prm.phre, c->prm, part ? -sc : sc);
        CU(cudaGetLastError());
        const int rc = deliver(c, dst, target, bytes, dst_is_device);
        if (rc) return rc;
    }
    return BVFDTD_OK;
}

int bvfdtd_plane_intensity(bvfdtd_ctx *c, double *plane_sum, double *plane_max) {
    if (!c || !plane_sum || !plane_max) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    if (c->rms_count <= 0 || (c->opts.flags & BVFDTD_FLAG_PHASOR)) return BVFDTD_ESTATE;
    // a z-slab context holds interior planes where an undivided box has its z slabs: the reduction skips [0, P)
    // and [nz - P, nz), so it is refused there (reduce the owned planes of the slabs on the caller's side)
    if (c->opts.flags & (BVFDTD_FLAG_ZLO_OPEN | BVFDTD_FLAG_ZHI_OPEN)) return BVFDTD_ESTATE;
    const Layout &L = c->L;
    double *d_out = (double *)(c->ws + c->W.scratch);          // 2 nz doubles of the dense scratch plane
    k_plane_intensity<<<L.nz, 256, 0, c->stream>>>(c->prm, (const float *)(c->ws + c->W.invz), (float)(1.0 / (double)c->rms_count), d_out);
    CU(cudaGetLastError());
    std::vector<double> h(2 * (size_t)L.nz);
    CU(cudaMemcpyAsync(h.data(), d_out, h.size() * 8, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    std::memcpy(plane_sum, h.data(), (size_t)L.nz * 8);
    std::memcpy(plane_max, h.data() + L.nz, (size_t)L.nz * 8);
    return BVFDTD_OK;
}

int bvfdtd_heat_source(bvfdtd_ctx *c, const double *absorbed_fraction, double scale, float *Q) {
    if (!c || !absorbed_fraction || !Q || !(scale >= 0.0) || !std::isfinite(scale)) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    if (c->rms_count <= 0 || (c->opts.flags & BVFDTD_FLAG_PHASOR)) return BVFDTD_ESTATE;
    // Q = scale a 2 alphaL I,  I = p_amp^2 / (2 rho cL) = sumsq / (count rho cL): one fp32 factor per material
    float coef[256];
    for (int m = 0; m < 256; ++m) {
        coef[m] = 0.0f;
        if (m >= c->n_materials) continue;
        if (!(absorbed_fraction[m] >= 0.0) || !std::isfinite(absorbed_fraction[m])) return BVFDTD_EINVAL;
        const bvfdtd_material &t = c->table[m];
        coef[m] = (float)(scale * absorbed_fraction[m] * 2.0 * t.alphaL / ((double)c->rms_count * t.rho * t.cL));
    }
    const Layout &L = c->L;
    float *d_coef = (float *)(c->ws + c->W.scratch);           // 1 KB of the dense scratch plane
    CU(cudaMemcpyAsync(d_coef, coef, sizeof(coef), cudaMemcpyHostToDevice, c->stream));
    CU(cudaStreamSynchronize(c->stream));                       // coef lives on this stack frame
    dim3 b(128), g((L.nx + 127) / 128, L.ny, L.nz);
    k_heat_source<<<g, b, 0, c->stream>>>(c->prm, d_coef, Q);
    CU(cudaGetLastError());
    return BVFDTD_OK;
}

int bvfdtd_energy_loss(const double *sum_tissue, const double *sum_water, const double *max_water, int32_t nz, int32_t pml,
                       int32_t *z_m, double *E_L, double *T_S) {
    if (!sum_tissue || !sum_water || !max_water || !z_m || !E_L || !T_S || pml < 0 || nz <= 2 * pml) return BVFDTD_EINVAL;
    int k = pml;
    for (int q = pml; q < nz - pml; ++q)
        if (max_water[q] > max_water[k]) k = q;
    if (!(sum_water[k] > 0.0)) return BVFDTD_ESTATE;
    *z_m = k;
    *E_L = sum_tissue[k] / sum_water[k];
    *T_S = std::sqrt(*E_L);
    return BVFDTD_OK;
}

namespace {
__global__ void k_check_elements(const int n_pts, const int *__restrict__ element, const int n_elem, int *__restrict__ bad) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n_pts && (element[q] < 0 || element[q] >= n_elem)) atomicExch(bad, 1);
}
}  // namespace

int bvfdtd_refocus_weights(int64_t n_pts, const float *p_re, const float *p_im, const int32_t *element, const float *area,
                           int32_t n_elem, double f, double u0, float *w_pts, float *delay_s, float *E, void *cuda_stream) {
    if (n_pts <= 0 || n_pts > (1 << 30) || n_elem <= 0 || n_elem > 65535 || !p_re || !p_im || !element || !area || !w_pts || !delay_s)
        return BVFDTD_EINVAL;
    if (!(f > 0.0) || !std::isfinite(u0)) return BVFDTD_EINVAL;
    DeviceScope scope(device_of(p_re));      // the caller's arrays say which device the launch belongs to
    cudaStream_t st = (cudaStream_t)cuda_stream;
    float2 *d_unit = nullptr;
    int *d_bad = nullptr;
    CU(cudaMallocAsync(&d_unit, (size_t)n_elem * sizeof(float2), st));
    CU(cudaMallocAsync(&d_bad, sizeof(int), st));
    CU(cudaMemsetAsync(d_bad, 0, sizeof(int), st));
    k_check_elements<<<(unsigned)((n_pts + 127) / 128), 128, 0, st>>>((int)n_pts, element, n_elem, d_bad);
    int bad = 0;
    CU(cudaMemcpyAsync(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (!bad) {
        k_element_phase<<<n_elem, 128, 0, st>>>((int)n_pts, p_re, p_im, element, (float)(1.0 / (2.0 * 3.14159265358979323846 * f)), d_unit,
                                               delay_s, (float2 *)E);
        k_point_weights<<<(unsigned)((n_pts + 127) / 128), 128, 0, st>>>((int)n_pts, element, area, d_unit, (float)u0, (float2 *)w_pts);
    }
    CU(cudaGetLastError());
    CU(cudaFreeAsync(d_unit, st));
    CU(cudaFreeAsync(d_bad, st));
    return bad ? BVFDTD_EINVAL : BVFDTD_OK;
}

int bvfdtd_rayleigh(int64_t n_src, const float *src_xyz, const float *src_weight, int64_t n_rcv, const float *rcv_xyz,
                    double f, double c0, double rho0, float *p_re, float *p_im, float *amp, float *delay_s, void *cuda_stream) {
    if (n_src <= 0 || n_rcv <= 0 || n_src > (1 << 30) || n_rcv > (1 << 30) || !src_xyz || !src_weight || !rcv_xyz || !p_re || !p_im)
        return BVFDTD_EINVAL;
    if (!(f > 0.0) || !(c0 > 0.0) || !(rho0 > 0.0) || (amp == nullptr) != (delay_s == nullptr)) return BVFDTD_EINVAL;
    DeviceScope scope(device_of(p_re));      // the caller's arrays say which device the launch belongs to
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const double w = 2.0 * 3.14159265358979323846 * f, k = w / c0;
    // pack the sources as float4 (x, y, z, 0) on the device
    float4 *d_src = nullptr;
    CU(cudaMallocAsync(&d_src, (size_t)n_src * sizeof(float4), st));
    CU(cudaMemsetAsync(d_src, 0, (size_t)n_src * sizeof(float4), st));
    CU(cudaMemcpy2DAsync(d_src, sizeof(float4), src_xyz, 3 * sizeof(float), 3 * sizeof(float), (size_t)n_src, cudaMemcpyDeviceToDevice, st));
    k_rayleigh<<<(unsigned)((n_rcv + 127) / 128), 128, 0, st>>>((int)n_src, d_src, (const float2 *)src_weight, (int)n_rcv, rcv_xyz, (float)k,
                                                              (float)(rho0 * c0 * k / (2.0 * 3.14159265358979323846)), (float)w, p_re, p_im, amp, delay_s);
    CU(cudaGetLastError());
    CU(cudaFreeAsync(d_src, st));
    return BVFDTD_OK;
}

int bvfdtd_rayleigh_noalloc(int64_t n_src, const float *src_xyz, const float *src_weight, int64_t n_rcv, const float *rcv_xyz,
                            double f, double c0, double rho0, float *p_re, float *p_im, float *amp, float *delay_s, void *cuda_stream) {
    if (n_src <= 0 || n_rcv <= 0 || n_rcv > (1 << 30) || !src_xyz || !src_weight || !rcv_xyz || !p_re || !p_im) return BVFDTD_EINVAL;
    if (!(f > 0.0) || !(c0 > 0.0) || !(rho0 > 0.0) || (amp == nullptr) != (delay_s == nullptr)) return BVFDTD_EINVAL;
    if (n_src > BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC) {
        std::snprintf(g_cuda_err, sizeof(g_cuda_err), "bvfdtd_rayleigh_noalloc: n_src = %lld exceeds BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC = %d "
                      "(the static scratch); use bvfdtd_rayleigh", (long long)n_src, (int)BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC);
        return BVFDTD_ENOMEM;
    }
    DeviceScope scope(device_of(p_re));      // the caller's arrays say which device the launch belongs to
    cudaStream_t st = (cudaStream_t)cuda_stream;
    float4 *d_src = nullptr;                 // this device's address of the static scratch: no allocation anywhere
    if (int rc = rs_noalloc_scratch(&d_src)) return rc;
    const double w = 2.0 * 3.14159265358979323846 * f, k = w / c0;
    k_rs_noalloc_pack<<<(unsigned)((n_src + 255) / 256), 256, 0, st>>>((int)n_src, src_xyz, d_src);
    k_rayleigh<<<(unsigned)((n_rcv + 127) / 128), 128, 0, st>>>((int)n_src, d_src, (const float2 *)src_weight, (int)n_rcv, rcv_xyz, (float)k,
                                                              (float)(rho0 * c0 * k / (2.0 * 3.14159265358979323846)), (float)w, p_re, p_im, amp, delay_s);
    CU(cudaGetLastError());
    return BVFDTD_OK;
}

int bvfdtd_probe_mufu(double *ops_per_second, void *cuda_stream) {
    if (!ops_per_second) return BVFDTD_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float *d_out = nullptr;
    CU(cudaMalloc(&d_out, 4));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    const int iters = 1 << 14, blocks = 2 * sms;
    k_mufu_probe<<<blocks, 1024, 0, st>>>(d_out, 64);                  // warm-up
    CU(cudaEventRecord(e0, st));
    k_mufu_probe<<<blocks, 1024, 0, st>>>(d_out, iters);
    CU(cudaEventRecord(e1, st));
    CU(cudaEventSynchronize(e1));
    float ms = 0.0f;
    CU(cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
    CU(cudaGetLastError());
    *ops_per_second = 4.0 * iters * 1024.0 * blocks / (ms * 1e-3);
    return BVFDTD_OK;
}

int bvfdtd_enable_kernel_timing(bvfdtd_ctx *c, int32_t on) {
    if (!c) return BVFDTD_EINVAL;
    c->timing = on != 0;
    c->timed_steps = 0;
    return BVFDTD_OK;
}

int bvfdtd_kernel_times(bvfdtd_ctx *c, double ms[4], int64_t launches[4]) {
    if (!c || !ms || !launches) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    CU(cudaStreamSynchronize(c->stream));
    for (int q = 0; q < 4; ++q) { ms[q] = 0.0; launches[q] = 0; }
    for (int64_t s = 0; s < c->timed_steps; ++s) {
        cudaEvent_t *ev = &c->ev[s * 5];
        for (int q = 0; q < 4; ++q) {
            float t = 0.0f;
            CU(cudaEventElapsedTime(&t, ev[q], ev[q + 1]));
            ms[q] += t;
            launches[q] += 1;
        }
    }
    if (c->n_src == 0) { ms[0] = 0.0; launches[0] = 0; }
    if (!c->ff_active || c->fplan.n_f == 0) { ms[1] = 0.0; launches[1] = 0; }
    if (c->ff_active && c->fplan.n_v == 0) { ms[2] = 0.0; launches[2] = 0; }
    if (c->ff_active && c->fplan.n_s == 0) { ms[3] = 0.0; launches[3] = 0; }
    c->timed_steps = 0;
    return BVFDTD_OK;
}

int bvfdtd_padding_nonzeros(bvfdtd_ctx *c, int64_t *count) {
    if (!c || !count) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    unsigned long long *d_count = (unsigned long long *)(c->ws + c->W.ctr + 32);
    CU(cudaMemsetAsync(d_count, 0, 8, c->stream));
    const long long n = c->L.field_floats;
    for (int a = 0; a < NGRID_ALL; ++a) {
        const float *f = (const float *)(c->ws + c->W.field[0] + (size_t)a * (c->W.field[1] - c->W.field[0]));
        k_padding_nonzeros<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(f, n, c->prm, d_count);
    }
    CU(cudaGetLastError());
    unsigned long long h = 0;
    CU(cudaMemcpyAsync(&h, d_count, 8, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    *count = (int64_t)h;
    return BVFDTD_OK;
}

int bvfdtd_work_items(bvfdtd_ctx *c, int32_t which, int32_t *items, int64_t capacity, int64_t *n_items, int32_t tile_rows[1]) {
    if (!c || which < 0 || which > 2 || !n_items || capacity < 0 || (capacity > 0 && !items)) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    const int n = !c->ff_active ? 0 : which == 0 ? c->fplan.n_f : which == 1 ? c->fplan.n_v : c->fplan.n_s;
    *n_items = n;
    if (tile_rows) tile_rows[0] = which == 2 ? (c->plan.s16 ? CfgS::TY : CfgS8::TY) : CfgF::TY;
    const int64_t m = std::min<int64_t>(n, capacity);
    if (m > 0) {
        CU(cudaMemcpyAsync(items, c->ws + c->W.items[which], (size_t)m * sizeof(int4), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    return BVFDTD_OK;
}

int bvfdtd_fused_lists_host(const bvfdtd_grid *grid, const uint8_t *cls, int32_t stress_tile_rows, int32_t slots, int32_t which,
                            int32_t *items, int64_t capacity, int64_t *n_items, uint32_t *flags) {
    if (!grid_ok(grid) || !cls || (stress_tile_rows != 8 && stress_tile_rows != 16) || slots < 1 || which < 0 || which > 2 ||
        !n_items || capacity < 0 || (capacity > 0 && !items))
        return BVFDTD_EINVAL;
    const Layout L = make_layout(*grid);
    const std::vector<uint8_t> c(cls, cls + (size_t)L.ntxV * L.ntyV * L.nz);
    const FusedLists lists = fused_lists(L, c, stress_tile_rows, slots, slots, slots);
    const std::vector<int4> &v = which == 0 ? lists.f : which == 1 ? lists.v : lists.s;
    *n_items = (int64_t)v.size();
    const size_t m = (size_t)std::min<int64_t>((int64_t)v.size(), capacity);
    if (m) std::memcpy(items, v.data(), m * sizeof(int4));
    if (flags) std::memcpy(flags, lists.flags.data(), lists.flags.size() * 4);
    return BVFDTD_OK;
}

int bvfdtd_fused_coverage(const bvfdtd_ctx *c, int64_t *planes_fused, int64_t *planes_all) {
    if (!c || !planes_fused || !planes_all) return BVFDTD_EINVAL;
    *planes_fused = c->ff_active ? c->fplan.planes_f : 0;
    *planes_all = (int64_t)c->L.ntxV * c->L.ntyV * c->L.nz;
    return BVFDTD_OK;
}

int bvfdtd_destroy(bvfdtd_ctx *c) {
    if (!c) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    cudaStreamSynchronize(c->stream);
    drop_graphs(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->cap_stream2) cudaStreamDestroy(c->cap_stream2);
    if (c->cap_fork) cudaEventDestroy(c->cap_fork);
    if (c->cap_join) cudaEventDestroy(c->cap_join);
    if (c->src_own) cudaFree(c->src_own);
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    tiled_plan_destroy(c->plan);
    delete c;
    (void)cudaGetLastError();
    return BVFDTD_OK;
}

}  // extern "C"
