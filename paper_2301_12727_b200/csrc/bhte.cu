// bhte.cu -- C ABI of the thermal step (include/bvfdtd.h, NEXT-4 of SURVEY.md 8(f)).
// Host side only: validation, the per-material coefficient rows (fp64 -> fp32 once), uploads,
// launches and read-back.  All arithmetic of the step runs in kernels_bhte.cuh.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/bvfdtd.h"
#include "host_common.hpp"
#include "kernels_bhte.cuh"

using namespace bvfdtd;

namespace {

size_t up256(size_t v) { return (v + 255) / 256 * 256; }

struct BhteMap {
    size_t th[2], Q, dose, tmax, mat, tab, scratch, maxidx, total;
};

bool dims_ok(int nx, int ny, int nz) {
    if (nx < 3 || ny < 3 || nz < 3) return false;
    const long long px = ((long long)nx + 63) / 64 * 64;
    return px * ny * (long long)nz < (1LL << 31) && ny <= 65535 && nz <= 65535;
}

BhteMap make_map(int nx, int ny, int nz, uint32_t flags) {
    const size_t px = ((size_t)nx + 63) / 64 * 64;
    const size_t cells_p = px * ny * nz, cells = (size_t)nx * ny * nz;
    BhteMap m;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += up256(bytes); return o; };
    m.th[0] = take(cells_p * 4);
    m.th[1] = take(cells_p * 4);
    m.Q = take(cells_p * 4);
    m.dose = take(cells_p * 4);
    m.tmax = (flags & BVFDTD_BHTE_TRACK_MAX) ? take(cells_p * 4) : 0;
    m.mat = take(cells_p);
    m.tab = take(256 * sizeof(float4));
    m.scratch = take(cells * 4);      // dense staging plane for host <-> device transfers
    m.maxidx = take(256);
    m.total = off;
    return m;
}

}  // namespace

struct bvfdtd_bhte {
    int nx = 0, ny = 0, nz = 0, px = 0;
    uint32_t flags = 0;
    double dx = 0, dt = 0, T_b = 37.0;
    char *ws = nullptr;
    BhteMap W{};
    cudaStream_t stream = nullptr;
    int device = -1;        // owner of the workspace: every entry point runs on it (DeviceScope)
    int cur = 0;            // th[cur] holds the present state
    int zlen = 1, nchunk = 1;
    int n_mat = 0;
    int64_t step = 0;
};

extern "C" {

int bvfdtd_bhte_workspace_bytes(int32_t nx, int32_t ny, int32_t nz, uint32_t flags, size_t *out_bytes) {
    if (!out_bytes || !dims_ok(nx, ny, nz) || (flags & ~(uint32_t)BVFDTD_BHTE_TRACK_MAX)) return BVFDTD_EINVAL;
    *out_bytes = make_map(nx, ny, nz, flags).total;
    return BVFDTD_OK;
}

int bvfdtd_bhte_create(bvfdtd_bhte **out, int32_t nx, int32_t ny, int32_t nz, double dx, double dt, const bvfdtd_thermal *table,
                       int32_t n_materials, const uint8_t *index_map, double T_b, uint32_t flags, void *d_workspace,
                       size_t workspace_bytes, void *cuda_stream) {
    if (!out) return BVFDTD_EINVAL;
    *out = nullptr;
    if (!dims_ok(nx, ny, nz) || !table || !index_map || !d_workspace || n_materials < 1 || n_materials > 256) return BVFDTD_EINVAL;
    if (!(dx > 0.0) || !(dt > 0.0) || !std::isfinite(T_b) || (flags & ~(uint32_t)BVFDTD_BHTE_TRACK_MAX)) return BVFDTD_EINVAL;
    if (((uintptr_t)d_workspace & 255u) != 0) return BVFDTD_EINVAL;
    double kmax = 0.0;
    for (int m = 0; m < n_materials; ++m) {
        if (!(table[m].k > 0.0) || !(table[m].rho_c > 0.0) || !(table[m].perf >= 0.0)) return BVFDTD_EINVAL;
        if (!std::isfinite(table[m].k) || !std::isfinite(table[m].rho_c) || !std::isfinite(table[m].perf)) return BVFDTD_EINVAL;
        kmax = std::max(kmax, table[m].k);
    }
    // forward Euler keeps every update coefficient non-negative (no oscillation) iff, for every cell,
    // dt (sum of its six face conductivities / dx^2 + w) / (rho C) <= 1; a face mean never exceeds k_max
    for (int m = 0; m < n_materials; ++m)
        if (dt * (6.0 * kmax / (dx * dx) + table[m].perf) / table[m].rho_c > 1.0) return BVFDTD_ESTABILITY;
    const BhteMap W = make_map(nx, ny, nz, flags);
    if (workspace_bytes < W.total) return BVFDTD_ENOMEM;

    const int ws_dev = device_of(d_workspace);
    if (ws_dev < 0) return cuda_fail(cudaErrorInvalidDevicePointer, "d_workspace is not device memory (or no CUDA device)");
    DeviceScope scope(ws_dev);
    bvfdtd_bhte *c = new (std::nothrow) bvfdtd_bhte;
    if (!c) return BVFDTD_ENOMEM;
    struct Guard { bvfdtd_bhte *p; ~Guard() { delete p; } } guard{c};
    c->device = ws_dev;
    c->nx = nx; c->ny = ny; c->nz = nz; c->px = (nx + 63) / 64 * 64;
    c->flags = flags; c->dx = dx; c->dt = dt; c->T_b = T_b;
    c->ws = (char *)d_workspace; c->W = W; c->stream = (cudaStream_t)cuda_stream; c->n_mat = n_materials;

    // z chunks: the grid is (tiles) x (chunks); pick the chunk count (chunks of >= 8 planes, 3 to 8
    // waves of the resident slots: short chunks balance better than one long wave, measured) whose
    // CTA count fills whole waves best (a 2.1-wave grid idles a third of the kernel), fewer on ties
    int dev = 0, sms = 148, occ = 3;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (flags & BVFDTD_BHTE_TRACK_MAX) CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_bhte<true>, 256, 0));
    else CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_bhte<false>, 256, 0));
    const int slots = sms * std::max(occ, 1);
    const int tiles = ((nx + 63) / 64) * ((ny + 15) / 16);
    const int max_chunks = std::max(1, nz / 8);
    int best = max_chunks;                                     // small grids: as many chunks as allowed
    double best_eff = 0.0;
    for (int n = 1; n <= max_chunks; ++n) {
        const int zl = (nz + n - 1) / n;
        if ((nz + zl - 1) / zl != n) continue;                 // this count is not reachable with equal chunks
        const long long ctas = (long long)tiles * n;
        const long long waves = (ctas + slots - 1) / slots;
        if (waves < 3) continue;
        if (waves > 8) break;
        const double eff = (double)ctas / (double)(waves * slots);
        if (eff > best_eff + 0.02) { best_eff = eff; best = n; }
    }
#ifdef BVFDTD_DEV_KNOBS   // experiments only: the shipped library's launch plan does not depend on the environment
    if (const char *e = std::getenv("BVFDTD_BHTE_CHUNKS"); e && *e) best = std::max(1, std::min(max_chunks, std::atoi(e)));
#endif
    c->zlen = (nz + best - 1) / best;
    c->nchunk = (nz + c->zlen - 1) / c->zlen;
#ifdef BVFDTD_DEV_KNOBS
    if (std::getenv("BVFDTD_VERBOSE"))
        std::fprintf(stderr, "[bvfdtd] bhte: tiles %d chunks %d (zlen %d) occ %d slots %d\n", tiles, c->nchunk, c->zlen, occ, slots);
#endif

    const size_t cells = (size_t)nx * ny * nz;
    CU(cudaMemsetAsync(c->ws, 0, W.total, c->stream));
    std::vector<float4> rows(256, make_float4(1.0f, 0.0f, 0.0f, 0.0f));
    for (int m = 0; m < n_materials; ++m) {
        const bvfdtd_thermal &t = table[m];
        rows[m] = make_float4((float)(1.0 / t.k), (float)(dt / (t.rho_c * dx * dx)), (float)(dt * t.perf / t.rho_c), (float)(dt / t.rho_c));
    }
    CU(cudaMemcpyAsync(c->ws + W.tab, rows.data(), rows.size() * sizeof(float4), cudaMemcpyHostToDevice, c->stream));
    CU(cudaMemcpyAsync(c->ws + W.scratch, index_map, cells, cudaMemcpyHostToDevice, c->stream));
    int *d_max = (int *)(c->ws + W.maxidx);
    {
        dim3 b(128), g((nx + 127) / 128, ny, nz);
        k_bhte_pack_map<<<g, b, 0, c->stream>>>((uint8_t *)(c->ws + W.mat), (const uint8_t *)(c->ws + W.scratch), nx, ny, c->px, d_max);
        CU(cudaGetLastError());
    }
    int h_max = 0;
    CU(cudaMemcpyAsync(&h_max, d_max, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));   // host staging buffers die at return
    if (h_max >= n_materials) return BVFDTD_EINVAL;
    guard.p = nullptr;
    *out = c;
    return BVFDTD_OK;
}

namespace {

// dense fp32 source (host or device) -> device pointer (the scratch plane when it came from the host)
int stage_in(bvfdtd_bhte *c, const float *src, int32_t src_is_device, const float **d_src) {
    if (src_is_device) { *d_src = src; return BVFDTD_OK; }
    float *scratch = (float *)(c->ws + c->W.scratch);
    CU(cudaMemcpyAsync(scratch, src, (size_t)c->nx * c->ny * c->nz * 4, cudaMemcpyHostToDevice, c->stream));
    *d_src = scratch;
    return BVFDTD_OK;
}

}  // namespace

int bvfdtd_bhte_set_heat(bvfdtd_bhte *c, const float *Q, int32_t src_is_device) {
    if (!c || !Q) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    const float *d_src = nullptr;
    int rc = stage_in(c, Q, src_is_device, &d_src);
    if (rc) return rc;
    dim3 b(128), g((c->nx + 127) / 128, c->ny, c->nz);
    k_bhte_pack_raw<<<g, b, 0, c->stream>>>((float *)(c->ws + c->W.Q), d_src, c->nx, c->ny, c->px);
    CU(cudaGetLastError());
    if (!src_is_device) CU(cudaStreamSynchronize(c->stream));   // the caller may reuse its host buffer
    return BVFDTD_OK;
}

int bvfdtd_bhte_set_temperature(bvfdtd_bhte *c, const float *T, int32_t src_is_device) {
    if (!c || !T) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    const float *d_src = nullptr;
    int rc = stage_in(c, T, src_is_device, &d_src);
    if (rc) return rc;
    dim3 b(128), g((c->nx + 127) / 128, c->ny, c->nz);
    float *tmax = (c->flags & BVFDTD_BHTE_TRACK_MAX) ? (float *)(c->ws + c->W.tmax) : nullptr;
    k_bhte_pack<<<g, b, 0, c->stream>>>((float *)(c->ws + c->W.th[c->cur]), tmax, d_src, c->nx, c->ny, c->nz, c->px, (float)c->T_b);
    CU(cudaGetLastError());
    if (!src_is_device) CU(cudaStreamSynchronize(c->stream));
    return BVFDTD_OK;
}

int bvfdtd_bhte_step(bvfdtd_bhte *c, int64_t n, double heat_scale) {
    if (!c || n < 0 || !(heat_scale >= 0.0) || !std::isfinite(heat_scale)) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    BhteParams p;
    p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.px = c->px; p.sz = c->px * c->ny;
    p.zlen = c->zlen; p.n_mat = c->n_mat;
    p.Q = (const float *)(c->ws + c->W.Q);
    p.dose = (float *)(c->ws + c->W.dose);
    p.tmax = (c->flags & BVFDTD_BHTE_TRACK_MAX) ? (float *)(c->ws + c->W.tmax) : nullptr;
    p.mat = (const uint8_t *)(c->ws + c->W.mat);
    p.tab = (const float4 *)(c->ws + c->W.tab);
    p.hs = (float)heat_scale;
    p.d43 = (float)(c->T_b - 43.0);
    p.dose_dt = (float)(c->dt / 60.0);
    const dim3 grid((c->nx + 63) / 64, (c->ny + 15) / 16, c->nchunk), block(256);
    for (int64_t s = 0; s < n; ++s) {
        p.th_in = (const float *)(c->ws + c->W.th[c->cur]);
        p.th_out = (float *)(c->ws + c->W.th[c->cur ^ 1]);
        if (p.tmax) k_bhte<true><<<grid, block, 0, c->stream>>>(p);
        else k_bhte<false><<<grid, block, 0, c->stream>>>(p);
        c->cur ^= 1;
        ++c->step;
    }
    CU(cudaGetLastError());
    return BVFDTD_OK;
}

int bvfdtd_bhte_read(bvfdtd_bhte *c, uint32_t what, float *dst, size_t dst_bytes, int32_t dst_is_device) {
    if (!c || !dst || what > BVFDTD_BHTE_RISE) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    const size_t bytes = (size_t)c->nx * c->ny * c->nz * 4;
    if (dst_bytes < bytes) return BVFDTD_EINVAL;
    if (what == BVFDTD_BHTE_TMAX && !(c->flags & BVFDTD_BHTE_TRACK_MAX)) return BVFDTD_ESTATE;
    const float *src = nullptr;
    float offset = 0.0f;
    switch (what) {
        case BVFDTD_BHTE_T: src = (const float *)(c->ws + c->W.th[c->cur]); offset = (float)c->T_b; break;
        case BVFDTD_BHTE_RISE: src = (const float *)(c->ws + c->W.th[c->cur]); break;
        case BVFDTD_BHTE_DOSE: src = (const float *)(c->ws + c->W.dose); break;
        default: src = (const float *)(c->ws + c->W.tmax); offset = (float)c->T_b; break;
    }
    float *target = dst_is_device ? dst : (float *)(c->ws + c->W.scratch);
    dim3 b(128), g((c->nx + 127) / 128, c->ny, c->nz);
    k_bhte_unpack<<<g, b, 0, c->stream>>>(target, src, c->nx, c->ny, c->px, offset);
    CU(cudaGetLastError());
    if (!dst_is_device) {
        CU(cudaMemcpyAsync(dst, target, bytes, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    return BVFDTD_OK;
}

int bvfdtd_bhte_destroy(bvfdtd_bhte *c) {
    if (!c) return BVFDTD_EINVAL;
    DeviceScope scope(c->device);
    cudaStreamSynchronize(c->stream);
    delete c;
    return BVFDTD_OK;
}

}  // extern "C"
