/*
 * bvfdtd.h -- C ABI of the B200-native 3-D staggered-grid viscoelastic FDTD time step.
 *
 * What the library computes: the time iteration that arXiv 2301.12727 ("BabelBrain") runs through
 * its BabelViscoFDTD solver (PAPER.md = /root/reference/PAPER.md):
 *   - PAPER.md:L91 (Eq. 1)   velocity-stress viscoelastic system, rows 1-3 velocity, 4-9 stress;
 *   - PAPER.md:L93           "4th-order in space and 2nd-order in time ... staggered-grid";
 *   - PAPER.md:L148-L152     attenuation as a quality factor Q (Eq. 3) realised with relaxation
 *                            constants and memory variables;
 *   - PAPER.md:L95           the incident field enters "as a stress source perpendicular to the
 *                            acoustic axis";
 *   - PAPER.md:L65-L73       material rows (rho, cL, cS, alphaL, alphaS), Table 1;
 *   - PAPER.md:L107-L110, L158, L220-L229   outputs are pressure / peak / pulse-average maps.
 * Every discrete detail the paper defers to its reference [23] (L93) is fixed by the readings
 * P1-P9 in DESIGN.md; each call below names the readings it implements.
 *
 * Conventions
 *   - Grid nx x ny x nz INCLUDING the PML cells; cell (i,j,k) has linear index i + nx*(j + ny*k)
 *     (x fastest; z is the acoustic axis).  All grid arrays that cross this ABI are
 *     dense in that order, whatever the private device layout is.
 *   - SI units.  fp32 state and arithmetic on the device; coefficients are derived in fp64 on the
 *     host and rounded to fp32 once (reading P9).
 *   - "host" / "device" is stated for every pointer.  The caller owns every pointer it passes; the
 *     library copies host inputs during the call and never frees caller memory.
 *   - Every call returns 0 (BVFDTD_OK) or a negative bvfdtd_status; no exceptions, no aborts.
 *     A failed bvfdtd_create leaves *out = NULL.
 *   - One context = one CUDA stream = one simulation.  A context is not thread-safe; distinct
 *     contexts are independent.
 *   - There is no CPU fallback: every call that touches the device returns BVFDTD_ECUDA when no
 *     CUDA device / driver is present.
 */
#ifndef BVFDTD_H
#define BVFDTD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bvfdtd_ctx bvfdtd_ctx; /* opaque */

typedef enum {
    BVFDTD_OK = 0,
    BVFDTD_EINVAL = -1,     /* an argument violates a documented rule */
    BVFDTD_ENOMEM = -2,     /* the caller's device workspace is too small (or host malloc failed) */
    BVFDTD_ESTABILITY = -3, /* max unrelaxed speed * dt / dx > 0.494 (reading P6) */
    BVFDTD_ECUDA = -4,      /* a CUDA runtime / driver call failed (bvfdtd_last_cuda_error) */
    BVFDTD_ESTATE = -5      /* call not legal in the context's current state */
} bvfdtd_status;

/* Grid descriptor.  Dimensions INCLUDE the pml cells on every face. */
typedef struct {
    int32_t nx, ny, nz; /* each must be >= 2*pml + 8 */
    int32_t pml;        /* C-PML thickness in cells on all six faces, >= 0 (0 = rigid box, P4) */
} bvfdtd_grid;

/* One row of the material table = the columns of PAPER.md Table 1 (L65-L73).  alpha in Np/m AT
 * THE CENTRE FREQUENCY f0: the caller has already applied the frequency scaling and the paper's
 * Q correction factor q_c (alpha / q_c).  cS = 0 marks a fluid. */
typedef struct {
    double rho;    /* kg/m^3, > 0 */
    double cL;     /* m/s, > 0: longitudinal phase speed at f0 */
    double cS;     /* m/s, >= 0 and < (sqrt(3)/2) cL: shear phase speed at f0 */
    double alphaL; /* Np/m at f0, >= 0, alphaL*cL/(2 pi f0) < tan(pi/8) (Q > 1, reading P3) */
    double alphaS; /* Np/m at f0, >= 0, same bound with cS */
} bvfdtd_material;

enum { /* bvfdtd_opts.flags */
    BVFDTD_FLAG_REFERENCE_KERNELS = 1, /* debug: run the one-thread-per-cell kernels instead of
                                          the tiled TMA kernels (same arithmetic, same results up
                                          to fp32 rounding order) */
    BVFDTD_FLAG_DENSE = 2,             /* sweep every array everywhere: do not skip the shear
                                          stresses / memory variables of tile-planes in which they
                                          are identically zero (all-fluid or lossless regions,
                                          DESIGN.md section 6).  Results are the same either way;
                                          bvfdtd_write_fields of a shear stress or a memory variable
                                          selects this mode by itself. */
    BVFDTD_FLAG_PHASOR = 4,            /* NEXT-3 of SURVEY.md 8(f): over the window [rms_begin, sensor_end) the
                                          stress pass accumulates the single-frequency phasor of the
                                          pressure at f0 (in-kernel DFT) INSTEAD of the running peak and the
                                          sum of squares; read it with bvfdtd_read_phasor */
    BVFDTD_FLAG_ZLO_OPEN = 8,          /* NEXT-5 of SURVEY.md 8(f): the z = 0 face of this box is an interface
                                          with the neighbouring z slab of a larger domain, not an outer
                                          boundary: no absorber on that face (its C-PML profile is inert,
                                          the mask bit is clear, sources are allowed there); the two
                                          outermost planes are halo planes the caller refreshes */
    BVFDTD_FLAG_ZHI_OPEN = 16          /* the same for the z = nz - 1 face */
};

typedef struct {
    double f0;          /* Hz > 0: relaxation centre frequency, tau_sigma = 1/(2 pi f0) (P3), also
                           the frequency of the C-PML frequency shift (P5) */
    double pml_R;       /* theoretical PML reflection coefficient in (0,1); 0 selects 1e-4 (P5) */
    int64_t peak_begin; /* first step index n sampled into the running peak (P8) */
    int64_t rms_begin;  /* first step index n sampled into the sum of squares (P8) */
    int64_t sensor_end; /* one past the last sampled step for both windows; < 0 = unbounded */
    uint32_t flags;     /* BVFDTD_FLAG_* */
    uint32_t tuning;    /* BVFDTD_TUNE_*: launch-plan requests for tests and experiments; 0 = the library's
                           own choice.  Results never depend on it (every plan is bit-identical); any other
                           bit set is BVFDTD_EINVAL.  The library reads no environment variable. */
} bvfdtd_opts;

enum { /* bvfdtd_opts.tuning */
    BVFDTD_TUNE_VEL_2CTA = 1,   /* velocity pass: the two-resident-CTA plan (3 stages) */
    BVFDTD_TUNE_VEL_3CTA = 2,   /* velocity pass: the three-resident-CTA plan with per-CTA stage plans, if it fits */
    BVFDTD_TUNE_STRESS_8 = 4,   /* stress pass: 64 x 8 tiles */
    BVFDTD_TUNE_STRESS_16 = 8,  /* stress pass: 64 x 16 tiles */
    BVFDTD_TUNE_NO_GRAPH = 16,  /* bvfdtd_step launches kernel by kernel instead of replaying CUDA graphs */
    BVFDTD_TUNE_NO_FUSED = 32,  /* all-fluid tile columns run the two passes like every other tile (no fused sweep) */
    BVFDTD_TUNE_FUSED = 64      /* use the fused sweep wherever it applies, also on grids the library judges too small
                                   for it to pay (under 6 M cells) or with few all-fluid tile columns */
};

/* Field ids for bvfdtd_read_fields / bvfdtd_write_fields. */
enum {
    BVFDTD_F_VX = 0, BVFDTD_F_VY = 1, BVFDTD_F_VZ = 2,          /* particle velocity, fp32      */
    BVFDTD_F_SXX = 3, BVFDTD_F_SYY = 4, BVFDTD_F_SZZ = 5,       /* normal stresses, fp32        */
    BVFDTD_F_SXY = 6, BVFDTD_F_SXZ = 7, BVFDTD_F_SYZ = 8,       /* shear stresses, fp32         */
    BVFDTD_F_RXX = 9, BVFDTD_F_RYY = 10, BVFDTD_F_RZZ = 11,     /* memory variables, fp32       */
    BVFDTD_F_RXY = 12, BVFDTD_F_RXZ = 13, BVFDTD_F_RYZ = 14,
    BVFDTD_F_PRESSURE = 15,  /* p = -(sxx+syy+szz)/3, fp32, computed on read (reading P8)       */
    BVFDTD_F_MATERIAL = 16,  /* the uint8 index map, round trip (nx*ny*nz bytes)                */
    BVFDTD_F_PML_MASK = 17,  /* uint8: bit0 x-slab, bit1 y-slab, bit2 z-slab (reading P5)       */
    BVFDTD_F_DERIVED = 18,   /* n_materials x 8 fp32: rho, pi_R, mu_R, tau_p, tau_s, pi_U, mu_U,
                                c_U (reading P3); host destination only                         */
    BVFDTD_F_PML_PROFILES = 19, /* fp32, host destination only: for axis x then y then z, the four
                                arrays a_int, b_int, a_half, b_half, each of that axis' length:
                                4*(nx+ny+nz) floats (reading P5)                                */
    BVFDTD_F_SUMSQ = 20      /* running sum of p^2 over the rms window, fp32                    */
};

/* Bytes of caller-owned DEVICE workspace bvfdtd_create needs for this grid: 15 state arrays, the
 * peak and sum-of-squares maps, the index map, the slab-compact C-PML memory variables and the
 * coefficient tables, in the library's private padded layout.  Host-only computation. */
int bvfdtd_workspace_bytes(const bvfdtd_grid *grid, size_t *out_bytes);

/*
 * Create a simulation (step S0 of DESIGN.md: per-material constants, C-PML profiles and mask are
 * derived in fp64 and rounded to fp32 once; readings P2, P3, P5, P6).
 *   out            host; receives the context (NULL on failure)
 *   grid, dx, dt   grid descriptor, grid step (m), time step (s); the library does not choose dt
 *   table          host, n_materials rows, 1 <= n_materials <= 256
 *   index_map      host, nx*ny*nz uint8, each < n_materials
 *   opts           host
 *   d_workspace    DEVICE, caller-owned, >= bvfdtd_workspace_bytes(), 256-byte aligned; must
 *                  outlive the context.  The library zeroes all state in it (reading P9).
 *   cuda_stream    a cudaStream_t (NULL = the legacy default stream); all work of this context is
 *                  enqueued on it
 * Errors: EINVAL for any violated rule above / in the struct comments (dim < 2*pml + 8, index >=
 * n_materials, cS >= sqrt(3)/2 cL, Q <= 1, ...); ESTABILITY when max c_U*dt/dx > 0.494; ENOMEM
 * when workspace_bytes is too small; ECUDA.
 */
int bvfdtd_create(bvfdtd_ctx **out, const bvfdtd_grid *grid, double dx, double dt,
                  const bvfdtd_material *table, int32_t n_materials, const uint8_t *index_map,
                  const bvfdtd_opts *opts, void *d_workspace, size_t workspace_bytes,
                  void *cuda_stream);

/*
 * Additive isotropic stress source (step S1; reading P7): at step n (t_n = n*dt), for
 * every source cell s:  sxx, syy, szz -= amp[s] * w(t_n - delay_s[s]), injected before the
 * velocity update.  w: waveform 0 = burst  sin(2 pi f t) for 0 <= t < n_cycles/f, else 0;
 * waveform 1 = ramped CW  ramp(t) sin(2 pi f t), ramp = (1 - cos(pi t f / n_cycles))/2 for
 * t < n_cycles/f, 1 after; w = 0 for t < 0.
 *   cell, amp, delay_s   host arrays of n_src entries; cells are linear indices, unique, inside
 *                        the grid and outside the PML mask.  n_src = 0 removes the source.
 * The library keeps its own device copy in the workspace (room for 4 nx ny source cells; only a longer list gets a
 * library-owned allocation).  The call does not synchronise: the arrays are packed on the host before it returns.
 * Errors: EINVAL (cell outside the grid / inside the PML / duplicate, f_src <= 0, n_cycles < 1,
 * waveform not 0/1), ECUDA.
 */
int bvfdtd_set_source(bvfdtd_ctx *ctx, int64_t n_src, const int64_t *cell, const float *amp,
                      const float *delay_s, int32_t waveform, double f_src, int32_t n_cycles);

/*
 * Enqueue n full time steps on the context's stream, asynchronously: per step S1 inject -> S2
 * velocity update (Eq. 1 rows 1-3) -> S3 stress + memory-variable update (Eq. 1 rows 4-9, L148-L152)
 * with the S4 sensor (running peak of |p|, sum of p^2) fused into it.  No host<->device traffic.
 * Legal before bvfdtd_set_source (zero source).  n >= 0.
 * How the steps are launched is the library's choice and never changes a bit of the result (bvfdtd_kernel_mode
 * names it): for n >= 2 it replays CUDA graphs of 8 steps / 1 step per sensor regime (captured on a stream of its
 * own on first use; the injection then takes the step index from a device counter); on grids of 6 M cells or more
 * the tile columns without a solid cell within reach run a fused single sweep (v and sigma in one z-march over
 * ping-ponged copies of v and the normal stresses) and only the others the two passes.
 */
int bvfdtd_step(bvfdtd_ctx *ctx, int64_t n);

/* Number of steps enqueued so far (the index n of the next step). */
int64_t bvfdtd_step_index(const bvfdtd_ctx *ctx);

/* Number of steps sampled into the rms / phasor window so far (the `count` of reading P8). */
int64_t bvfdtd_rms_count(const bvfdtd_ctx *ctx);

/* Which kernels the next bvfdtd_step will run (a host-side query; tests and bench.py print it so that a
 * parity claim names the path it holds for).  Bits of *mode: */
enum {
    BVFDTD_MODE_REFERENCE = 1,   /* one-thread-per-cell kernels (BVFDTD_FLAG_REFERENCE_KERNELS) */
    BVFDTD_MODE_DENSE = 2,       /* tiled kernels, every array everywhere (BVFDTD_FLAG_DENSE, or a shear stress /
                                    memory variable was written through bvfdtd_write_fields) */
    BVFDTD_MODE_SIGMA_WRITTEN = 4, /* a normal stress was written by the caller: the fluid shortcuts that rely on
                                    sigma_xx = sigma_yy = sigma_zz are off */
    BVFDTD_MODE_FUSED = 8,       /* all-fluid tile columns run the fused single-sweep kernel */
    BVFDTD_MODE_GRAPH = 16       /* bvfdtd_step replays a captured CUDA graph of one step */
};
int bvfdtd_kernel_mode(const bvfdtd_ctx *ctx, uint32_t *mode);

/*
 * Copy one field out in the dense external layout.  dst_bytes must equal the field's size
 * (nx*ny*nz*4 for fp32 grid fields, nx*ny*nz for the uint8 fields, see the enum).  If
 * dst_is_device == 0, dst is host memory and the call synchronises the stream; otherwise dst is
 * device memory and the copy is enqueued on the stream.
 */
int bvfdtd_read_fields(bvfdtd_ctx *ctx, uint32_t field_id, void *dst, size_t dst_bytes,
                       int32_t dst_is_device);

/* Overwrite one of the 15 state fields (ids 0..14) from a dense fp32 array (restart, unit tests).
 * The outermost normal-velocity layer (reading P4) is forced to 0 whatever src holds. */
int bvfdtd_write_fields(bvfdtd_ctx *ctx, uint32_t field_id, const void *src, size_t src_bytes,
                        int32_t src_is_device);

/*
 * Sensor outputs (step S4; reading P8), dense fp32 nx*ny*nz each, either pointer may be NULL:
 *   peak     max |p| over steps n with peak_begin <= n < sensor_end
 *   rms_amp  sqrt(2 * sum p^2 / count) over steps n with rms_begin <= n < sensor_end (the amplitude
 *            of a sinusoid in steady state); 0 when count = 0
 */
int bvfdtd_read_peak_pressure(bvfdtd_ctx *ctx, float *peak, float *rms_amp, int32_t dst_is_device);

/* Release the context (host structs, the source copy, CUDA graphs).  Never touches the workspace. */
int bvfdtd_destroy(bvfdtd_ctx *ctx);

const char *bvfdtd_strerror(int code);
/* Text of the last CUDA error seen by this thread inside the library ("" if none). */
const char *bvfdtd_last_cuda_error(void);

/* Device-time accounting for benchmarks: when enabled the library brackets every kernel of
 * bvfdtd_step with CUDA events on the context's stream (and launches kernel by kernel instead of
 * replaying CUDA graphs); bvfdtd_kernel_times (which synchronises) returns the accumulated
 * milliseconds and launch counts per kernel (0 inject, 1 fused single sweep of the all-fluid tile
 * columns, 2 velocity pass, 3 stress + sensor pass) since the last call and resets them.  At most
 * `BVFDTD_MAX_TIMED_STEPS` steps are recorded between two reads. */
enum { BVFDTD_MAX_TIMED_STEPS = 4096 };
int bvfdtd_enable_kernel_timing(bvfdtd_ctx *ctx, int32_t on);
int bvfdtd_kernel_times(bvfdtd_ctx *ctx, double ms[4], int64_t launches[4]);
/* How much of the grid the fused single sweep takes: 64 x 8 tile-planes it runs / all tile-planes
 * (0 when the context is not in the fused mode, BVFDTD_MODE_FUSED).  Host-side query. */
int bvfdtd_fused_coverage(const bvfdtd_ctx *ctx, int64_t *planes_fused, int64_t *planes_all);
/* Host only (no CUDA device needed): the work lists the fused mode builds from the per-(64 x 8 tile, plane) class
 * bytes of S0 (bit 0: no solid cell within 4 cells of the tile in this plane, bit 1: a lossy cell in the tile;
 * cls[(tile_x + ntx * tile_y) * nz + k], ntx = ceil(nx / 64), nty = ceil(ny / 8)).  Same code path bvfdtd_create
 * uses; exposed so that the partition and the z-slab rules can be tested anywhere.  which / items / n_items as in
 * bvfdtd_work_items; slots = resident CTAs assumed for every kernel; flags (or NULL): ntx * nty * (nz + 4) words,
 * (tile, plane + 2), bit 2 = plane in a fused run, bit 3 / 4 = the run also writes sigma_yy / sigma_zz there. */
int bvfdtd_fused_lists_host(const bvfdtd_grid *grid, const uint8_t *cls, int32_t stress_tile_rows, int32_t slots,
                            int32_t which, int32_t *items, int64_t capacity, int64_t *n_items, uint32_t *flags);
/* Self-check (compute-sanitizer is not available everywhere): the number of non-zero floats in the zero gaps of
 * the private layout of all 25 grid arrays (x beyond nx, the two extra rows, the two planes before and after: the
 * zero ghost of reading P4, which no kernel may write).  0 on a healthy context.  Synchronises the stream. */
int bvfdtd_padding_nonzeros(bvfdtd_ctx *ctx, int64_t *count);
/* The work lists of the fused mode, for tests: which = 0 fused sweep, 1 velocity pass, 2 stress pass.  items
 * (HOST, capacity entries of 4 int32: tile x, tile y, first plane, one past the last plane) receives at most
 * `capacity` entries, *n_items the length of the list (0 outside the fused mode), tile_rows[0] the rows of the
 * tiles the list counts in (8, or 16 for the stress pass on 64 x 16 tiles; tiles are 64 cells wide).  Lists 0 and
 * 1, and lists 0 and 2, each cover every tile-plane of the grid exactly once. */
int bvfdtd_work_items(bvfdtd_ctx *ctx, int32_t which, int32_t *items, int64_t capacity, int64_t *n_items,
                      int32_t tile_rows[1]);

/* ---- host-only helpers (no CUDA device needed): the S0 constructions, exposed so that the
 * construction-parity tests can run anywhere.  Same code path bvfdtd_create uses. ---- */

/* Per-material derived constants (reading P3): out[8*m + 0..7] = rho, pi_R, mu_R, tau_p, tau_s,
 * pi_U, mu_U, c_U rounded to fp32.  Returns EINVAL on an invalid row. */
int bvfdtd_derive_materials(const bvfdtd_material *table, int32_t n_materials, double f0,
                            float *out);
/* C-PML profiles of one axis of n nodes (reading P5), each output of length n. */
int bvfdtd_pml_profiles(int32_t n, int32_t pml, double dx, double dt, double f0, double pml_R,
                        double c_ref, float *a_int, float *b_int, float *a_half, float *b_half);
/* PML mask (reading P5), nx*ny*nz uint8. */
int bvfdtd_pml_mask(const bvfdtd_grid *grid, uint8_t *mask);
/* Largest unrelaxed Courant number c_U*dt/dx of the table (reading P6), or a negative status. */
double bvfdtd_max_courant(const bvfdtd_material *table, int32_t n_materials, double f0, double dt,
                          double dx);

/*
 * NEXT-3 of SURVEY.md 8(f): complex pressure amplitude (for refocusing "a punctual source
 * is placed at the intended target, back-propagated to the domain interface", which needs amplitude and
 * phase there).  With BVFDTD_FLAG_PHASOR the sensor accumulates A = sum p cos(w t), B = sum p sin(w t),
 * w = 2 pi f0, t = (n + 1) dt (the time level after S3 of step n), over rms_begin <= n < sensor_end.
 * bvfdtd_read_phasor returns P = (2 / count)(A - j B), i.e. p(t) = Re{P e^{j w t}} in the steady state:
 *   re, im   nx*ny*nz fp32 each, host or device (dst_is_device); host destinations synchronise the
 *            stream.  BVFDTD_ESTATE without BVFDTD_FLAG_PHASOR.
 */
int bvfdtd_read_phasor(bvfdtd_ctx *ctx, float *re, float *im, int32_t dst_is_device);

/*
 * NEXT-2 of SURVEY.md 8(f): the reduction that turns the pressure maps of a tissue run and of the
 * water-only run on the same grid into the paper's energy-loss factor.
 *
 * bvfdtd_plane_intensity: pulse-average intensity I_PA = rms_amp^2 / (2 rho cL) = sumsq / (count rho cL)
 * of every cell (rho, cL = the table row of the cell's own material; rms_amp of reading P8) reduced
 * over the cells OUTSIDE the PML mask of every z plane, on the device (fp32 per cell, fp64 sums in a
 * fixed order).  plane_sum, plane_max: HOST arrays of nz doubles (W/m^2); planes inside the z slabs
 * give 0.  BVFDTD_ESTATE when no step has been sampled into the rms window yet, and on z-slab contexts
 * (BVFDTD_FLAG_ZLO_OPEN / _ZHI_OPEN: their outer planes are interior planes of the whole domain).  Synchronises the
 * context's stream.
 *
 * bvfdtd_energy_loss (host only): z_m = the interior plane on which max_water is largest (first on
 * ties), E_L = sum_tissue[z_m] / sum_water[z_m] (Eq. 2), T_S = sqrt(E_L)
 * (PAPER.md:L164).  BVFDTD_ESTATE when the water plane carries no intensity.
 */
int bvfdtd_plane_intensity(bvfdtd_ctx *ctx, double *plane_sum, double *plane_max);
int bvfdtd_energy_loss(const double *sum_tissue, const double *sum_water, const double *max_water,
                       int32_t nz, int32_t pml, int32_t *z_m, double *E_L, double *T_S);

/*
 * NEXT-1 of SURVEY.md 8(f): Rayleigh-Sommerfeld field of a surface-decomposed transducer over a set of
 * receiver points (the incident interface of the simulation domain), coupling medium water
 * (PAPER.md:L95).  First Rayleigh integral of a baffled source, e^{+j w t} convention:
 *     P(r) = (j rho0 c0 k / 2 pi) sum_s W_s exp(-j k |r - r_s|) / |r - r_s|,  k = 2 pi f / c0,
 * W_s = u_s A_s the complex normal velocity times the element area (m^3/s).
 *   src_xyz     DEVICE, n_src x 3 fp32 (m);   src_weight  DEVICE, n_src x 2 fp32 (Re, Im of W_s)
 *   rcv_xyz     DEVICE, n_rcv x 3 fp32 (m); a receiver that coincides with a source point gets the sum over the
 *               other source points (that pair has no finite value and is left out)
 *   p_re, p_im  DEVICE, n_rcv fp32 each (Pa)
 *   amp, delay_s  DEVICE, n_rcv fp32 each, or both NULL: the same field as the (amplitude, delay)
 *               pair bvfdtd_set_source takes for a CW source, p(t) = amp sin(2 pi f (t - delay)),
 *               delay in [0, 1/f)
 *   cuda_stream the launch is asynchronous on this stream
 * fp32 arithmetic, one thread per receiver; no context is needed.
 */
/*
 * The same field as bvfdtd_rayleigh for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it): this entry point allocates NOTHING -- no cudaMalloc / cudaMallocAsync,
 * no cudaFree, no allocating library routine.  bvfdtd_rayleigh packs the sources into a scratch array it allocates
 * per call; here that scratch is a static device array of the library, BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC float4
 * entries (1 MiB), which every GPU that loads the library holds until the process exits.
 *   - arguments, layouts and results as bvfdtd_rayleigh (same field kernel, same bits);
 *   - n_src > BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC returns BVFDTD_ENOMEM (bvfdtd_last_cuda_error names the limit): use
 *     bvfdtd_rayleigh for larger source sets;
 *   - all calls on one device SHARE the scratch, which keeps the last call's contents: every entry a call reads is
 *     rewritten by that call first (nothing needs to start at zero), but two calls that overlap on the GPU --
 *     different streams, or threads, without an ordering between them -- race on it.  Calls on one stream are safe;
 *   - the first call on each device resolves the scratch's device address (cudaGetSymbolAddress, cached per device;
 *     not an allocation): make that call once before starting a graph capture.
 * Asynchronous on cuda_stream.
 */
enum { BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC = 65536 };
int bvfdtd_rayleigh_noalloc(int64_t n_src, const float *src_xyz, const float *src_weight, int64_t n_rcv,
                            const float *rcv_xyz, double f, double c0, double rho0, float *p_re, float *p_im,
                            float *amp, float *delay_s, void *cuda_stream);
/* Measured MUFU (special-function unit) rate of the current device in operations per second: a short probe
 * kernel of independent sin.approx chains, timed with CUDA events.  bvfdtd_rayleigh spends three MUFU operations
 * per (source, receiver) pair, so its roofline is this rate / 3.  Synchronises. */
int bvfdtd_probe_mufu(double *ops_per_second, void *cuda_stream);
int bvfdtd_rayleigh(int64_t n_src, const float *src_xyz, const float *src_weight, int64_t n_rcv,
                    const float *rcv_xyz, double f, double c0, double rho0, float *p_re, float *p_im,
                    float *amp, float *delay_s, void *cuda_stream);

/*
 * NEXT-4 of SURVEY.md 8(f): thermal step ("solves the Bio Heat Transfer Equation (BHTE)
 * with a finite-difference time-difference solver in Cartesian coordinates [46].  Boundary conditions
 * are assumed conservatively with a temperature of 37 C at the domain's borders ... duration of
 * ultrasound, time off after ultrasound, and duty cycle ... fraction of attenuation in skull bone
 * transformed into heat was set to 0.16 ... maximal temperature, and thermal dose [48]").
 *
 * Readings (the paper prints neither the equation nor its discretisation):
 *   rho C dT/dt = div(k grad T) - w (T - T_b) + s Q     (Pennes; w = w_b rho_b C_b, arterial T = T_b)
 * forward Euler, conservative 7-point stencil on the cell grid of the acoustic run, face conductivity
 * = series mean 2 ka kb / (ka + kb), the cells on the six borders of the box held at T_b, s = the
 * `heat_scale` of the step (duty cycle while the ultrasound is on, 0 while it is off), and with the
 * temperature reached at the end of each step: CEM43 += (dt/60) R^(43 - T), R = 0.5 for T >= 43 else
 * 0.25, and the running maximum.  fp32 arithmetic; the state is kept as the rise T - T_b.
 */
typedef struct bvfdtd_bhte bvfdtd_bhte; /* opaque */

typedef struct {
    double k;     /* thermal conductivity, W/m/K, > 0 */
    double rho_c; /* density x specific heat, J/m^3/K, > 0 */
    double perf;  /* perfusion coefficient w_b rho_b C_b, W/m^3/K, >= 0 */
} bvfdtd_thermal;

enum { BVFDTD_BHTE_TRACK_MAX = 1u }; /* keep the running maximum temperature (8 more bytes per cell-step) */
enum { BVFDTD_BHTE_T = 0, BVFDTD_BHTE_DOSE = 1, BVFDTD_BHTE_TMAX = 2, BVFDTD_BHTE_RISE = 3 };

/* Bytes of device workspace a thermal context of this grid needs. */
int bvfdtd_bhte_workspace_bytes(int32_t nx, int32_t ny, int32_t nz, uint32_t flags, size_t *out_bytes);
/*
 * table        HOST, n_materials rows (1..256); index_map HOST, nx*ny*nz uint8, x fastest (same map
 *              as the acoustic run); copied during the call.
 * T_b          border = arterial = initial temperature (deg C; 37 in the paper)
 * d_workspace  DEVICE, caller-owned, >= bvfdtd_bhte_workspace_bytes, 256-byte aligned, must outlive
 *              the context; cuda_stream: every launch of the context goes to this stream.
 * Errors: EINVAL (dims < 3, a non-positive k or rho_c, negative perf, an index >= n_materials,
 * misaligned workspace), ENOMEM (workspace too small), ESTABILITY (dt (6 k_max/dx^2 + w) / (rho C) > 1
 * for some material: forward Euler would oscillate), ECUDA.  A failed create leaves *out = NULL.
 */
int bvfdtd_bhte_create(bvfdtd_bhte **out, int32_t nx, int32_t ny, int32_t nz, double dx, double dt,
                       const bvfdtd_thermal *table, int32_t n_materials, const uint8_t *index_map,
                       double T_b, uint32_t flags, void *d_workspace, size_t workspace_bytes,
                       void *cuda_stream);
/* Heat deposition Q (W/m^3), nx*ny*nz fp32 dense x-fastest, host or device; copied. */
int bvfdtd_bhte_set_heat(bvfdtd_bhte *ctx, const float *Q, int32_t src_is_device);
/* Initial temperature (deg C), same layout; border cells are set to T_b whatever is passed; the
 * running maximum takes it into account. */
int bvfdtd_bhte_set_temperature(bvfdtd_bhte *ctx, const float *T, int32_t src_is_device);
/* Enqueue n steps with the source scaled by heat_scale (>= 0); asynchronous. */
int bvfdtd_bhte_step(bvfdtd_bhte *ctx, int64_t n, double heat_scale);
/* what: BVFDTD_BHTE_T temperature, _DOSE CEM43 in minutes, _TMAX running maximum (ESTATE without
 * BVFDTD_BHTE_TRACK_MAX), _RISE T - T_b at full fp32 precision.  dst: nx*ny*nz fp32; a host
 * destination synchronises the stream. */
int bvfdtd_bhte_read(bvfdtd_bhte *ctx, uint32_t what, float *dst, size_t dst_bytes, int32_t dst_is_device);
int bvfdtd_bhte_destroy(bvfdtd_bhte *ctx);

/*
 * Heat deposition from the acoustic run: with the pressure amplitude of the rms window
 * (reading P8), I = p_amp^2 / (2 rho cL) and Q = scale * a_m * 2 alphaL_m * I per cell, a_m = the
 * fraction of the attenuation of material m turned into heat (0.16 in bone, 1 in soft tissue), scale =
 * the caller's intensity calibration factor.
 *   absorbed_fraction  HOST, one double per material of the context;  Q  DEVICE, nx*ny*nz fp32 dense.
 * BVFDTD_ESTATE when no step has been sampled into the rms window (or with BVFDTD_FLAG_PHASOR).
 * Asynchronous on the context's stream.
 */
int bvfdtd_heat_source(bvfdtd_ctx *ctx, const double *absorbed_fraction, double scale, float *Q);

/*
 * NEXT-5 of SURVEY.md 8(e)/(f): z-slab decomposition over several GPUs (PAPER.md:L41 footnote: the
 * large domains exceed one device).  A rank owns a contiguous range of z planes and holds them in a
 * context whose box is that range plus two halo planes on every face that is an interface
 * (BVFDTD_FLAG_ZLO_OPEN / _ZHI_OPEN; the 4th-order staggered differences reach two planes).  Per step:
 *     bvfdtd_step_phase(ctx, 0)   inject (S1)
 *     exchange the halo planes of the six stresses with the z neighbours
 *     bvfdtd_step_phase(ctx, 1)   velocity pass (S2)
 *     exchange the halo planes of the three velocities
 *     bvfdtd_step_phase(ctx, 2)   stress + sensor pass (S3 + S4); the step counter advances
 * Values the passes compute IN the halo planes are meaningless and are overwritten by the next
 * exchange; the owned planes are bit-identical to those of the undivided run.  Phases must be called in
 * order (BVFDTD_ESTATE otherwise; bvfdtd_step is refused in the middle of a step).
 *
 * bvfdtd_plane_span (host only, no context): byte offset inside the workspace, and byte count, of the
 * contiguous block that holds planes k .. k + n_planes - 1 of state field `field_id` (0-14) in the
 * private layout.  The block includes the layout's padding, which is identical on both sides of an
 * interface because x and y extents are: a halo exchange is a plain copy of this block between the
 * workspaces of two ranks (device-to-device, NCCL send/recv or a peer-to-peer put).  The block is where a z-slab
 * context (BVFDTD_FLAG_ZLO_OPEN / _ZHI_OPEN) keeps the field: such contexts never run the fused mode, whose steps
 * alternate between two copies of v and the normal stresses.
 */
int bvfdtd_step_phase(bvfdtd_ctx *ctx, int32_t phase);
/* The same pass (phase 1 velocity or 2 stress + sensor) over the z planes [k0, k1) only, so that a rank can run the
 * planes that read no halo plane while the halo exchange is in flight and the others after it:
 *     velocity / stress at plane k read planes k-2 .. k+2 of the exchanged arrays.
 * The ranges of one pass may come in any order, must not overlap and must add up to all nz planes; the pass (and, for
 * phase 2, the step) is complete when they do.  Results do not depend on the split (the kernels are bit-identical
 * under any z chunking).  BVFDTD_ESTATE out of order, on overlap, or with BVFDTD_FLAG_REFERENCE_KERNELS. */
int bvfdtd_step_phase_planes(bvfdtd_ctx *ctx, int32_t phase, int32_t k0, int32_t k1);
int bvfdtd_plane_span(const bvfdtd_grid *grid, uint32_t field_id, int32_t k, int32_t n_planes,
                      size_t *offset_bytes, size_t *bytes);

/*
 * NEXT-3, second half ("a punctual source is placed at the intended target,
 * back-propagated to the domain interface, and then propagated back with Rayleigh-Sommerfeld to the
 * transducer elements to calculate the corrected phase programming of the transducer elements").
 * The chain is: a run with BVFDTD_FLAG_PHASOR from a one-cell source at the target; the phasors of the
 * entry plane as the weights of bvfdtd_rayleigh towards the surface points of the array (the plane
 * radiates back as a baffled source with weight proportional to P); then this call:
 *   E_m = sum of the field over the surface points of element m,
 *   time reversal: element m emits Re{conj(E_m)/|E_m| e^{j w t}} = cos(w (t - tau_m)), tau_m = arg(E_m)/w
 *   taken in [0, 1/f); every surface point q of element m gets the weight u0 area_q conj(E_m)/|E_m|,
 * which is the src_weight of the forward bvfdtd_rayleigh call.
 *   p_re, p_im  DEVICE, n_pts fp32 each: the field at the surface points
 *   element     DEVICE, n_pts int32 in [0, n_elem) (EINVAL otherwise); area  DEVICE, n_pts fp32 (m^2)
 *   w_pts       DEVICE, n_pts x 2 fp32 (Re, Im);  delay_s  DEVICE, n_elem fp32
 *   E           DEVICE, n_elem x 2 fp32, or NULL
 * An element that received no field keeps weight u0 area and delay 0.  Synchronises the stream once
 * (index validation).  fp64 sums in a fixed order.
 */
int bvfdtd_refocus_weights(int64_t n_pts, const float *p_re, const float *p_im, const int32_t *element,
                           const float *area, int32_t n_elem, double f, double u0, float *w_pts,
                           float *delay_s, float *E, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* BVFDTD_H */
