/*
 * fdtd_oracle.c -- fp64 CPU ORACLE for the 3-D staggered-grid viscoelastic FDTD step.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no source, header,
 * table or constant generator with the CUDA library (paper_2301_12727_b200/csrc) and neither
 * imports the other.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md, arXiv 2301.12727):
 *   - Eq. 1: velocity-stress viscoelastic system, rows 1-3 velocity, rows 4-9
 *     stress (rows 8-9 are garbled in the extraction; repaired by symmetry, G1).
 *   - PAPER.md:L93: "4th-order in space and 2nd-order in time FDTD scheme ... staggered-grid".
 *   - Eq. 3 and L152: attenuation through a quality factor Q realised with
 *     relaxation constants and memory variables.
 *   - PAPER.md:L95: the incident field enters "as a stress source perpendicular to the
 *     acoustic axis".
 *   - PAPER.md:L65-L73 (Table 1): material rows are (rho, cL, cS, alphaL, alphaS).
 * The paper defers every discrete detail to its reference [23] (L93), which is not available;
 * the readings P1-P9 listed in DESIGN.md fix them.  Each function below names its reading.
 *
 * The method is a time iteration, so the oracle is the iteration itself, step by step, in
 * fp64, as plain loop nests: S1 inject -> S2 velocity pass -> S3 stress pass -> S4 sensor.
 * No blocking, fusion or reordering.  Zero ghost values (reading P4) are realised literally:
 * every field array carries a 2-cell ghost frame that is never written (except by the
 * test-only periodic wrap).
 *
 * Parity pins (tests/test_oracle_pins.py, -m "not gpu"): T1 discrete dispersion relation
 * (temporal form), T2 spatial phase speed / attenuation, T2b continuum Q and phase speed,
 * T3 plate transmission, T4 discrete energy, T5 reciprocity, T6 PML reflection, T7 order of
 * convergence, T8 elastic limit and axis symmetry; tests/test_oracle_source_pins.py: S1-S4 the
 * source (sign, amplitude, delay as a time shift, burst gate, raised-cosine ramp), A1 the staggered
 * material means on period-2 laminates (closed-form dispersion with rho arithmetic, mu harmonic,
 * tau_s arithmetic), A2 the C-PML of a solid at oblique incidence (which profile each shear psi
 * term takes).  Unpinned against the paper (the paper is
 * silent): the choice of ONE relaxation mechanism, the C-PML formulation, the averaging
 * rule -- "parity unpinned vs paper" for those choices; their implementation is pinned by
 * the closed forms above.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o liboracle.so fdtd_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#define GH 2                       /* ghost width: the 4-point stencils reach 2 cells */
#define C1 (9.0 / 8.0)             /* 4th-order staggered weights (reading P1) */
#define C2 (-1.0 / 24.0)

enum { VX, VY, VZ, SXX, SYY, SZZ, SXY, SXZ, SYZ, RXX, RYY, RZZ, RXY, RXZ, RYZ, NFIELD };
/* derived per-material constants (reading P3), 8 per material */
enum { D_RHO, D_PIR, D_MUR, D_TP, D_TS, D_PIU, D_MUU, D_CU, NDER };

typedef struct orc {
    int n[3];                      /* nx, ny, nz */
    int P;                         /* PML thickness requested */
    int per[3];                    /* test-only periodic axes */
    int Pa[3];                     /* PML thickness per axis (0 on periodic axes) */
    double dx, dt, f0, R;
    int nmat;
    double *der;                   /* nmat * NDER */
    uint8_t *idx;                  /* nx*ny*nz, dense */
    uint8_t *idp;                  /* (n+2)^3: idx with a 1-cell frame, replicated (P2) or wrapped */
    double *f[NFIELD];             /* padded (n+2GH)^3 arrays */
    double *psi[18];               /* slab-compact C-PML memory, index axis*6 + term */
    double *prof[3][4];            /* per axis: a_int, b_int, a_half, b_half */
    double *peak, *sumsq;          /* dense nx*ny*nz */
    double *phre, *phim;           /* phasor accumulators sum p cos(w t), sum p sin(w t) (NEXT-3), or NULL */
    int phasor;                    /* 1: the rms window accumulates the phasor instead of peak / sumsq */
    int64_t peak_begin, rms_begin, sensor_end, count;
    int64_t step;
    int64_t nsrc;
    int64_t *scell;
    double *samp, *sdelay;
    int waveform, ncyc;
    double fsrc;
    size_t sx, sy, sz;             /* padded strides */
} orc;

/* ------------------------------------------------------------------------------------ */
/* S0: per-material derived constants (reading P3 steps 1-2; Eq. 3).       */
/* row = (rho, cL, cS, alphaL, alphaS), alpha in Np/m at f0.  out = rho, pi_R, mu_R,     */
/* tau_p, tau_s, pi_U, mu_U, c_U.  Returns 0, or a negative code naming the violated     */
/* validity rule (same rules the C ABI states).                             */
/* ------------------------------------------------------------------------------------ */
static int tau_and_g(double alpha, double c, double w0, double *tau, double *g)
{
    /* tan(delta/2) = alpha c / w0 (exact inversion of alpha = (w0/c) tan(delta/2));      */
    /* Q = 1/tan(delta); tau = 2 tan(delta) / (1 - tan(delta)) = 2/(Q-1);                 */
    /* g = 2 cos^2(delta/2) / sqrt((2+tau)^2 + tau^2) makes c_p(w0) = c.                  */
    double t = alpha * c / w0;
    if (alpha == 0.0 || c == 0.0) { *tau = 0.0; *g = 1.0; return 0; }
    if (!(t < tan(M_PI / 8.0))) return -1;            /* Q <= 1: unrepresentable */
    double tand = 2.0 * t / (1.0 - t * t);
    *tau = 2.0 * tand / (1.0 - tand);
    double cos2 = 1.0 / (1.0 + t * t);
    *g = 2.0 * cos2 / sqrt((2.0 + *tau) * (2.0 + *tau) + (*tau) * (*tau));
    return 0;
}

int orc_derive_materials(int nmat, const double *table, double f0, double *out)
{
    double w0 = 2.0 * M_PI * f0;
    for (int m = 0; m < nmat; ++m) {
        const double *r = table + 5 * m;
        double rho = r[0], cL = r[1], cS = r[2], aL = r[3], aS = r[4];
        if (!(rho > 0.0) || !(cL > 0.0) || cS < 0.0 || aL < 0.0 || aS < 0.0) return -1;
        if (!(cS < 0.5 * sqrt(3.0) * cL)) return -1;   /* bulk modulus must stay positive */
        double tp, gp, ts, gs;
        if (tau_and_g(aL, cL, w0, &tp, &gp)) return -1;
        if (tau_and_g(aS, cS, w0, &ts, &gs)) return -1;
        double piR = rho * cL * cL * gp;
        double muR = rho * cS * cS * gs;
        double *o = out + NDER * m;
        o[D_RHO] = rho; o[D_PIR] = piR; o[D_MUR] = muR; o[D_TP] = tp; o[D_TS] = ts;
        o[D_PIU] = piR * (1.0 + tp);
        o[D_MUU] = muR * (1.0 + ts);
        o[D_CU] = sqrt(o[D_PIU] / rho);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* S0: C-PML profiles of one axis (reading P5).  n nodes, P layer cells, c_ref = max cL. */
/* Integer node i sits at i*dx, half node at (i+1/2)*dx; depth into the layer            */
/* xi = max(0, (P-1/2)dx - x, x - (n-P-1/2)dx); d = d0 (xi/L)^2, d0 = 3 c_ref ln(1/R)/(2L)*/
/* alpha = pi f0 (1 - xi/L); b = exp(-(d+alpha) dt); a = d (b-1)/(d+alpha), a=0 at d=0.   */
/* ------------------------------------------------------------------------------------ */
void orc_pml_profiles(int n, int P, double dx, double dt, double f0, double R, double c_ref,
                      double *a_int, double *b_int, double *a_half, double *b_half)
{
    for (int i = 0; i < n; ++i) {
        for (int h = 0; h < 2; ++h) {
            double a = 0.0, b = 1.0;
            if (P > 0) {
                double L = P * dx;
                double x = (i + 0.5 * h) * dx;
                double xi = 0.0;
                double lo = (P - 0.5) * dx - x, hi = x - (n - P - 0.5) * dx;
                if (lo > xi) xi = lo;
                if (hi > xi) xi = hi;
                double d0 = 3.0 * c_ref * log(1.0 / R) / (2.0 * L);
                double d = d0 * (xi / L) * (xi / L);
                double al = M_PI * f0 * (1.0 - xi / L);
                b = exp(-(d + al) * dt);
                a = (d > 0.0) ? d * (b - 1.0) / (d + al) : 0.0;
            }
            if (h) { a_half[i] = a; b_half[i] = b; } else { a_int[i] = a; b_int[i] = b; }
        }
    }
}

/* PML mask (reading P5): bit0 = i in an x slab, bit1 = j in a y slab, bit2 = k in a z slab */
void orc_pml_mask(int nx, int ny, int nz, int P, uint8_t *mask)
{
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                uint8_t m = 0;
                if (i < P || i >= nx - P) m |= 1;
                if (j < P || j >= ny - P) m |= 2;
                if (k < P || k >= nz - P) m |= 4;
                mask[(size_t)i + (size_t)nx * (j + (size_t)ny * k)] = m;
            }
}

/* largest unrelaxed Courant number c_U dt/dx over the table (reading P6) */
double orc_max_courant(int nmat, const double *der, double dt, double dx)
{
    double m = 0.0;
    for (int i = 0; i < nmat; ++i) {
        double c = der[NDER * i + D_CU] * dt / dx;
        if (c > m) m = c;
    }
    return m;
}

/* ------------------------------------------------------------------------------------ */
/* context                                                                               */
/* ------------------------------------------------------------------------------------ */
static size_t padded_cells(const orc *o)
{
    return (size_t)(o->n[0] + 2 * GH) * (o->n[1] + 2 * GH) * (o->n[2] + 2 * GH);
}
static inline size_t AT(const orc *o, int i, int j, int k)
{
    return (size_t)(i + GH) * o->sx + (size_t)(j + GH) * o->sy + (size_t)(k + GH) * o->sz;
}
static inline size_t DENSE(const orc *o, int i, int j, int k)
{
    return (size_t)i + (size_t)o->n[0] * (j + (size_t)o->n[1] * k);
}
static size_t psi_cells(const orc *o, int axis)
{
    size_t c = 2 * (size_t)o->Pa[axis];
    for (int a = 0; a < 3; ++a) if (a != axis) c *= (size_t)o->n[a];
    return c;
}

void orc_free(orc *o)
{
    if (!o) return;
    free(o->der); free(o->idx); free(o->idp);
    for (int q = 0; q < NFIELD; ++q) free(o->f[q]);
    for (int q = 0; q < 18; ++q) free(o->psi[q]);
    for (int a = 0; a < 3; ++a) for (int q = 0; q < 4; ++q) free(o->prof[a][q]);
    free(o->peak); free(o->sumsq); free(o->phre); free(o->phim); free(o->scell); free(o->samp); free(o->sdelay);
    free(o);
}

/* periodic[3]: TEST-ONLY periodic axes (no wall, no PML on those axes); production = 0,0,0 */
orc *orc_new(int nx, int ny, int nz, int P, double dx, double dt, int nmat, const double *table,
             const uint8_t *index_map, double f0, double pml_R, int64_t peak_begin,
             int64_t rms_begin, int64_t sensor_end, const int *periodic)
{
    orc *o = (orc *)calloc(1, sizeof(orc));
    if (!o) return NULL;
    o->n[0] = nx; o->n[1] = ny; o->n[2] = nz; o->P = P;
    o->dx = dx; o->dt = dt; o->f0 = f0; o->R = pml_R; o->nmat = nmat;
    o->peak_begin = peak_begin; o->rms_begin = rms_begin; o->sensor_end = sensor_end;
    for (int a = 0; a < 3; ++a) {
        o->per[a] = periodic ? periodic[a] : 0;
        o->Pa[a] = o->per[a] ? 0 : P;
    }
    o->sx = 1; o->sy = (size_t)(nx + 2 * GH); o->sz = o->sy * (size_t)(ny + 2 * GH);
    o->der = (double *)malloc(sizeof(double) * NDER * nmat);
    if (!o->der || orc_derive_materials(nmat, table, f0, o->der)) { orc_free(o); return NULL; }
    size_t nc = (size_t)nx * ny * nz;
    o->idx = (uint8_t *)malloc(nc);
    memcpy(o->idx, index_map, nc);
    for (size_t c = 0; c < nc; ++c) if (o->idx[c] >= nmat) { orc_free(o); return NULL; }
    /* material ids with a 1-cell frame: out-of-grid neighbours replicate the nearest in-grid
       cell (reading P2), or wrap on a test-only periodic axis */
    o->idp = (uint8_t *)malloc((size_t)(nx + 2) * (ny + 2) * (nz + 2));
    for (int k = -1; k <= nz; ++k)
        for (int j = -1; j <= ny; ++j)
            for (int i = -1; i <= nx; ++i) {
                int c[3] = { i, j, k };
                for (int a = 0; a < 3; ++a) {
                    if (o->per[a]) c[a] = ((c[a] % o->n[a]) + o->n[a]) % o->n[a];
                    else { if (c[a] < 0) c[a] = 0; if (c[a] >= o->n[a]) c[a] = o->n[a] - 1; }
                }
                o->idp[(size_t)(i + 1) + (size_t)(nx + 2) * ((j + 1) + (size_t)(ny + 2) * (k + 1))] =
                    o->idx[DENSE(o, c[0], c[1], c[2])];
            }
    for (int q = 0; q < NFIELD; ++q) o->f[q] = (double *)calloc(padded_cells(o), sizeof(double));
    double c_ref = 0.0;
    for (int m = 0; m < nmat; ++m) if (table[5 * m + 1] > c_ref) c_ref = table[5 * m + 1];
    for (int a = 0; a < 3; ++a) {
        for (int q = 0; q < 4; ++q) o->prof[a][q] = (double *)calloc(o->n[a], sizeof(double));
        orc_pml_profiles(o->n[a], o->Pa[a], dx, dt, f0, pml_R, c_ref, o->prof[a][0],
                         o->prof[a][1], o->prof[a][2], o->prof[a][3]);
        for (int t = 0; t < 6; ++t) {
            size_t pc = psi_cells(o, a);
            o->psi[a * 6 + t] = (double *)calloc(pc ? pc : 1, sizeof(double));
        }
    }
    o->peak = (double *)calloc(nc, sizeof(double));
    o->sumsq = (double *)calloc(nc, sizeof(double));
    return o;
}

int orc_set_source(orc *o, int64_t nsrc, const int64_t *cell, const double *amp,
                   const double *delay, int waveform, double fsrc, int ncyc)
{
    free(o->scell); free(o->samp); free(o->sdelay);
    o->nsrc = nsrc; o->waveform = waveform; o->fsrc = fsrc; o->ncyc = ncyc;
    o->scell = (int64_t *)malloc(sizeof(int64_t) * (nsrc ? nsrc : 1));
    o->samp = (double *)malloc(sizeof(double) * (nsrc ? nsrc : 1));
    o->sdelay = (double *)malloc(sizeof(double) * (nsrc ? nsrc : 1));
    int64_t nc = (int64_t)o->n[0] * o->n[1] * o->n[2];
    for (int64_t s = 0; s < nsrc; ++s) {
        if (cell[s] < 0 || cell[s] >= nc) return -1;
        o->scell[s] = cell[s]; o->samp[s] = amp[s]; o->sdelay[s] = delay[s];
    }
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* helpers used by the passes                                                            */
/* ------------------------------------------------------------------------------------ */

/* forward / backward 4-point staggered differences along a stride (reading P1):         */
/* D+ f(i) = [c1 (f(i+1)-f(i)) + c2 (f(i+2)-f(i-1))]/dx  lands on the half node i+1/2     */
/* D- f(i) = [c1 (f(i)-f(i-1)) + c2 (f(i+1)-f(i-2))]/dx  lands on the integer node i      */
static inline double Dp(const double *f, size_t c, size_t s, double dx)
{
    return (C1 * (f[c + s] - f[c]) + C2 * (f[c + 2 * s] - f[c - s])) / dx;
}
static inline double Dm(const double *f, size_t c, size_t s, double dx)
{
    return (C1 * (f[c] - f[c - s]) + C2 * (f[c + s] - f[c - 2 * s])) / dx;
}

/* material id of cell (i,j,k) with out-of-grid neighbours replicated (or wrapped on a    */
/* test-only periodic axis): reading P2                                                   */
static inline int mat_at(const orc *o, int i, int j, int k)   /* -1 <= i <= nx etc. */
{
    return o->idp[(size_t)(i + 1) + (size_t)(o->n[0] + 2) * ((j + 1) + (size_t)(o->n[1] + 2) * (k + 1))];
}

/* C-PML correction of one derivative (reading P5): in a slab of `axis`,                  */
/* psi <- b psi + a D, D_eff = D + psi, with the profile at the node where D lands        */
/* (half = 1: half node, 0: integer node).  term = 0..5 selects the psi array.            */
static inline double pml(orc *o, int axis, int term, int half, int i, int j, int k, double d)
{
    int P = o->Pa[axis];
    int c[3] = { i, j, k };
    int pos = c[axis], n = o->n[axis];
    if (!(pos < P || pos >= n - P)) return d;
    double a = o->prof[axis][half ? 2 : 0][pos];
    double b = o->prof[axis][half ? 3 : 1][pos];
    c[axis] = (pos < P) ? pos : pos - (n - 2 * P);          /* slab-compact coordinate */
    int dim[3] = { o->n[0], o->n[1], o->n[2] };
    dim[axis] = 2 * P;
    size_t q = (size_t)c[0] + (size_t)dim[0] * (c[1] + (size_t)dim[1] * c[2]);
    double *psi = &o->psi[axis * 6 + term][q];
    *psi = b * (*psi) + a * d;
    return d + *psi;
}

/* test-only: wrap the ghost frame of field q on periodic axes (ghosts stay 0 otherwise)  */
static void wrap_ghosts(orc *o, int q)
{
    double *f = o->f[q];
    int nx = o->n[0], ny = o->n[1], nz = o->n[2];
    if (o->per[0])
        for (int k = -GH; k < nz + GH; ++k) for (int j = -GH; j < ny + GH; ++j)
            for (int g = 1; g <= GH; ++g) {
                f[AT(o, -g, j, k)] = f[AT(o, nx - g, j, k)];
                f[AT(o, nx - 1 + g, j, k)] = f[AT(o, g - 1, j, k)];
            }
    if (o->per[1])
        for (int k = -GH; k < nz + GH; ++k) for (int i = -GH; i < nx + GH; ++i)
            for (int g = 1; g <= GH; ++g) {
                f[AT(o, i, -g, k)] = f[AT(o, i, ny - g, k)];
                f[AT(o, i, ny - 1 + g, k)] = f[AT(o, i, g - 1, k)];
            }
    if (o->per[2])
        for (int j = -GH; j < ny + GH; ++j) for (int i = -GH; i < nx + GH; ++i)
            for (int g = 1; g <= GH; ++g) {
                f[AT(o, i, j, -g)] = f[AT(o, i, j, nz - g)];
                f[AT(o, i, j, nz - 1 + g)] = f[AT(o, i, j, g - 1)];
            }
}

/* source time function (reading P7)                                                      */
static double waveform(int kind, double f, int ncyc, double t)
{
    if (t < 0.0) return 0.0;
    double T = ncyc / f;
    if (kind == 0) return (t < T) ? sin(2.0 * M_PI * f * t) : 0.0;          /* burst */
    double ramp = (t < T) ? 0.5 * (1.0 - cos(M_PI * t * f / ncyc)) : 1.0;   /* ramped CW */
    return ramp * sin(2.0 * M_PI * f * t);
}

/* ------------------------------------------------------------------------------------ */
/* S1: additive isotropic stress injection at step n, t_n = n dt (reading P7, L95)       */
/* ------------------------------------------------------------------------------------ */
void orc_inject(orc *o)
{
    double tn = (double)o->step * o->dt;
    for (int64_t s = 0; s < o->nsrc; ++s) {
        int64_t c = o->scell[s];
        int i = (int)(c % o->n[0]), j = (int)((c / o->n[0]) % o->n[1]);
        int k = (int)(c / ((int64_t)o->n[0] * o->n[1]));
        double w = o->samp[s] * waveform(o->waveform, o->fsrc, o->ncyc, tn - o->sdelay[s]);
        size_t p = AT(o, i, j, k);
        o->f[SXX][p] -= w; o->f[SYY][p] -= w; o->f[SZZ][p] -= w;
    }
}

/* ------------------------------------------------------------------------------------ */
/* S2: velocity pass (Eq. 1 rows 1-3, L91; readings P1, P2, P4, P5)                       */
/*   v_x(i+1/2,j,k) += dt/rho_x (D+x sxx + D-y sxy + D-z sxz)   rho_x = mean of 2 cells   */
/*   v_y(i,j+1/2,k) += dt/rho_y (D-x sxy + D+y syy + D-z syz)                             */
/*   v_z(i,j,k+1/2) += dt/rho_z (D-x sxz + D-y syz + D+z szz)                             */
/* the outermost normal-velocity layer (i = nx-1 for v_x, ...) is a rigid wall: held at 0 */
/* ------------------------------------------------------------------------------------ */
void orc_velocity_pass(orc *o)
{
    const int nx = o->n[0], ny = o->n[1], nz = o->n[2];
    const double dx = o->dx, dt = o->dt;
    const size_t sx = o->sx, sy = o->sy, sz = o->sz;
    for (int q = SXX; q <= SYZ; ++q) wrap_ghosts(o, q);
    const double *sxx = o->f[SXX], *syy = o->f[SYY], *szz = o->f[SZZ];
    const double *sxy = o->f[SXY], *sxz = o->f[SXZ], *syz = o->f[SYZ];
#pragma omp parallel for collapse(2) schedule(static) if ((size_t)nx * ny * nz > 32768)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = AT(o, i, j, k);
                double rho0 = o->der[NDER * mat_at(o, i, j, k) + D_RHO];
                if (o->per[0] || i < nx - 1) {
                    double d1 = pml(o, 0, 0, 1, i, j, k, Dp(sxx, c, sx, dx));
                    double d2 = pml(o, 1, 0, 0, i, j, k, Dm(sxy, c, sy, dx));
                    double d3 = pml(o, 2, 0, 0, i, j, k, Dm(sxz, c, sz, dx));
                    double rho = 0.5 * (rho0 + o->der[NDER * mat_at(o, i + 1, j, k) + D_RHO]);
                    o->f[VX][c] += dt / rho * (d1 + d2 + d3);
                }
                if (o->per[1] || j < ny - 1) {
                    double d1 = pml(o, 0, 1, 0, i, j, k, Dm(sxy, c, sx, dx));
                    double d2 = pml(o, 1, 1, 1, i, j, k, Dp(syy, c, sy, dx));
                    double d3 = pml(o, 2, 1, 0, i, j, k, Dm(syz, c, sz, dx));
                    double rho = 0.5 * (rho0 + o->der[NDER * mat_at(o, i, j + 1, k) + D_RHO]);
                    o->f[VY][c] += dt / rho * (d1 + d2 + d3);
                }
                if (o->per[2] || k < nz - 1) {
                    double d1 = pml(o, 0, 2, 0, i, j, k, Dm(sxz, c, sx, dx));
                    double d2 = pml(o, 1, 2, 0, i, j, k, Dm(syz, c, sy, dx));
                    double d3 = pml(o, 2, 2, 1, i, j, k, Dp(szz, c, sz, dx));
                    double rho = 0.5 * (rho0 + o->der[NDER * mat_at(o, i, j, k + 1) + D_RHO]);
                    o->f[VZ][c] += dt / rho * (d1 + d2 + d3);
                }
            }
}

/* shear-node material (reading P2): relaxed mu_h = harmonic mean of the 4 cells, 0 if    */
/* any of them is fluid; tau_s,h = arithmetic mean of the 4 cells                         */
static inline void shear_node(const orc *o, const int m[4], double *mu_h, double *ts_h)
{
    double inv = 0.0, ts = 0.0;
    int fluid = 0;
    for (int q = 0; q < 4; ++q) {
        double mu = o->der[NDER * m[q] + D_MUR];
        if (mu == 0.0) fluid = 1; else inv += 1.0 / mu;
        ts += o->der[NDER * m[q] + D_TS];
    }
    *mu_h = fluid ? 0.0 : 4.0 / inv;
    *ts_h = 0.25 * ts;
}

/* Crank-Nicolson memory-variable update + stress update (reading P3 step 4):             */
/*   r' = ((1-beta) r - 2 beta eR)/(1+beta);  s += dt eU + dt/2 (r' + r);  r = r'          */
static inline void sls_update(double *s, double *r, double eU, double eR, double beta, double dt)
{
    double rn = ((1.0 - beta) * (*r) - 2.0 * beta * eR) / (1.0 + beta);
    *s += dt * eU + 0.5 * dt * (rn + *r);
    *r = rn;
}

/* ------------------------------------------------------------------------------------ */
/* S3: stress + memory-variable pass (Eq. 1 rows 4-9, L91; L148-L152; P1, P2, P3, P5)     */
/* ------------------------------------------------------------------------------------ */
void orc_stress_pass(orc *o)
{
    const int nx = o->n[0], ny = o->n[1], nz = o->n[2];
    const double dx = o->dx, dt = o->dt;
    const double beta = dt / (2.0 * (1.0 / (2.0 * M_PI * o->f0)));   /* dt / (2 tau_sigma) */
    const size_t sx = o->sx, sy = o->sy, sz = o->sz;
    for (int q = VX; q <= VZ; ++q) wrap_ghosts(o, q);
    const double *vx = o->f[VX], *vy = o->f[VY], *vz = o->f[VZ];
#pragma omp parallel for collapse(2) schedule(static) if ((size_t)nx * ny * nz > 32768)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = AT(o, i, j, k);
                /* normal stresses at the integer node: the cell's own material */
                const double *d = o->der + NDER * mat_at(o, i, j, k);
                double vxx = pml(o, 0, 3, 0, i, j, k, Dm(vx, c, sx, dx));
                double vyy = pml(o, 1, 4, 0, i, j, k, Dm(vy, c, sy, dx));
                double vzz = pml(o, 2, 5, 0, i, j, k, Dm(vz, c, sz, dx));
                double th = vxx + vyy + vzz;
                double vii[3] = { vxx, vyy, vzz };
                for (int q = 0; q < 3; ++q) {
                    double eU = d[D_PIU] * th - 2.0 * d[D_MUU] * (th - vii[q]);
                    double eR = d[D_PIR] * d[D_TP] * th - 2.0 * d[D_MUR] * d[D_TS] * (th - vii[q]);
                    sls_update(&o->f[SXX + q][c], &o->f[RXX + q][c], eU, eR, beta, dt);
                }
                double mu_h, ts_h, g;
                /* sigma_xy at (i+1/2, j+1/2, k): cells (i..i+1, j..j+1, k) */
                {
                    int m[4] = { mat_at(o, i, j, k), mat_at(o, i + 1, j, k),
                                 mat_at(o, i, j + 1, k), mat_at(o, i + 1, j + 1, k) };
                    shear_node(o, m, &mu_h, &ts_h);
                    g = pml(o, 1, 3, 1, i, j, k, Dp(vx, c, sy, dx))
                      + pml(o, 0, 4, 1, i, j, k, Dp(vy, c, sx, dx));
                    sls_update(&o->f[SXY][c], &o->f[RXY][c], mu_h * (1.0 + ts_h) * g,
                               mu_h * ts_h * g, beta, dt);
                }
                /* sigma_xz at (i+1/2, j, k+1/2): cells (i..i+1, j, k..k+1) */
                {
                    int m[4] = { mat_at(o, i, j, k), mat_at(o, i + 1, j, k),
                                 mat_at(o, i, j, k + 1), mat_at(o, i + 1, j, k + 1) };
                    shear_node(o, m, &mu_h, &ts_h);
                    g = pml(o, 2, 3, 1, i, j, k, Dp(vx, c, sz, dx))
                      + pml(o, 0, 5, 1, i, j, k, Dp(vz, c, sx, dx));
                    sls_update(&o->f[SXZ][c], &o->f[RXZ][c], mu_h * (1.0 + ts_h) * g,
                               mu_h * ts_h * g, beta, dt);
                }
                /* sigma_yz at (i, j+1/2, k+1/2): cells (i, j..j+1, k..k+1) */
                {
                    int m[4] = { mat_at(o, i, j, k), mat_at(o, i, j + 1, k),
                                 mat_at(o, i, j, k + 1), mat_at(o, i, j + 1, k + 1) };
                    shear_node(o, m, &mu_h, &ts_h);
                    g = pml(o, 2, 4, 1, i, j, k, Dp(vy, c, sz, dx))
                      + pml(o, 1, 5, 1, i, j, k, Dp(vz, c, sy, dx));
                    sls_update(&o->f[SYZ][c], &o->f[RYZ][c], mu_h * (1.0 + ts_h) * g,
                               mu_h * ts_h * g, beta, dt);
                }
            }
}

/* ------------------------------------------------------------------------------------ */
/* S4: sensor after S3 of step n (reading P8): p = -(sxx+syy+szz)/3                       */
/* ------------------------------------------------------------------------------------ */
void orc_sensor(orc *o)
{
    const int nx = o->n[0], ny = o->n[1], nz = o->n[2];
    int64_t n = o->step;
    int in_end = (o->sensor_end < 0) || (n < o->sensor_end);
    int do_peak = in_end && n >= o->peak_begin;
    int do_rms = in_end && n >= o->rms_begin;
    if (o->phasor) {
        /* NEXT-3 (refocusing needs amplitude AND phase on the domain interface): single-
         * frequency DFT of p over the window [rms_begin, sensor_end) at f0; the state after S3 of step
         * n is time level (n + 1) dt.  A += p cos(w t), B += p sin(w t); P = (2 / count) (A - j B), so
         * that p(t) = Re{P e^{j w t}} in the steady state. */
        if (!do_rms) return;
        const double wt = 2.0 * 3.14159265358979323846 * o->f0 * (double)(n + 1) * o->dt;
        const double cs = cos(wt), sn = sin(wt);
#pragma omp parallel for collapse(2) schedule(static) if ((size_t)nx * ny * nz > 32768)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    size_t c = AT(o, i, j, k), q = DENSE(o, i, j, k);
                    double p = -(o->f[SXX][c] + o->f[SYY][c] + o->f[SZZ][c]) / 3.0;
                    o->phre[q] += p * cs;
                    o->phim[q] += p * sn;
                }
        o->count++;
        return;
    }
    if (!do_peak && !do_rms) return;
#pragma omp parallel for collapse(2) schedule(static) if ((size_t)nx * ny * nz > 32768)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = AT(o, i, j, k), q = DENSE(o, i, j, k);
                double p = -(o->f[SXX][c] + o->f[SYY][c] + o->f[SZZ][c]) / 3.0;
                if (do_peak && fabs(p) > o->peak[q]) o->peak[q] = fabs(p);
                if (do_rms) o->sumsq[q] += p * p;
            }
    if (do_rms) o->count++;
}

/* Subnormal numbers (reading P9): values below the smallest normal double, 2.2e-308, count as
 * the zero initial state while orc_step runs (x86 flush-to-zero + denormals-are-zero on the stepping threads, put
 * back afterwards).  Why: the 4-point stencils carry the discrete solution two cells per step, far ahead of the
 * physical wave front, where it decays super-exponentially; for most of a long run a large part of the domain holds
 * values between 5e-324 and 2e-308, every operation on which an x86 core executes in microcode.  Measured on
 * config 2: 1.1 s per step at step 50, 3.2 s at step 150 (0.9 M subnormal cells per field), 21 minutes for the
 * 3000 steps instead of 8; configs 3 / 4 up to 30x slower.  The change is below 1e-307 in absolute value, 300 orders
 * of magnitude under every tolerance, and no pin moves. */
#if defined(__x86_64__) || defined(__i386__)
#include <xmmintrin.h>
#define ORC_MXCSR_FTZ_DAZ 0x8040u
static void subnormals_as_zero(int on)
{
#pragma omp parallel
    { _mm_setcsr(on ? (_mm_getcsr() | ORC_MXCSR_FTZ_DAZ) : (_mm_getcsr() & ~ORC_MXCSR_FTZ_DAZ)); }
}
#else
static void subnormals_as_zero(int on) { (void)on; }
#endif

/* one full step: S1 -> S2 -> S3 -> S4 ("Per-step order is S1 -> S2 -> S3(+S4)") */
void orc_step(orc *o, int64_t nsteps)
{
    subnormals_as_zero(1);
    for (int64_t s = 0; s < nsteps; ++s) {
        orc_inject(o);
        orc_velocity_pass(o);
        orc_stress_pass(o);
        orc_sensor(o);
        o->step++;
    }
    subnormals_as_zero(0);
}

int64_t orc_step_index(const orc *o) { return o->step; }
void orc_set_step_index(orc *o, int64_t n) { o->step = n; }
int64_t orc_rms_count(const orc *o) { return o->count; }
/* switch the sensor to phasor mode (before stepping); returns 0 or -1 (out of memory) */
int orc_set_phasor(orc *o, int on)
{
    const size_t nc = (size_t)o->n[0] * o->n[1] * o->n[2];
    o->phasor = on != 0;
    if (o->phasor && !o->phre) {
        o->phre = (double *)calloc(nc, sizeof(double));
        o->phim = (double *)calloc(nc, sizeof(double));
        if (!o->phre || !o->phim) return -1;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* field access: dense x-fastest nx*ny*nz doubles.  field 0..14 state, 15 p = -tr/3,      */
/* 16 peak, 17 rms_amp = sqrt(2 sumsq / count) (0 if count = 0), 18 sumsq,                */
/* 19, 20 Re P, Im P of the phasor P = (2 / count)(A - j B) (phasor mode only)            */
/* ------------------------------------------------------------------------------------ */
int orc_get_field(const orc *o, int field, double *out)
{
    const int nx = o->n[0], ny = o->n[1], nz = o->n[2];
    if (field < 0 || field > 20) return -1;
    if (field >= 19 && !o->phre) return -1;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = AT(o, i, j, k), q = DENSE(o, i, j, k);
                if (field < NFIELD) out[q] = o->f[field][c];
                else if (field == 15) out[q] = -(o->f[SXX][c] + o->f[SYY][c] + o->f[SZZ][c]) / 3.0;
                else if (field == 16) out[q] = o->peak[q];
                else if (field == 17) out[q] = o->count ? sqrt(2.0 * o->sumsq[q] / (double)o->count) : 0.0;
                else if (field == 18) out[q] = o->sumsq[q];
                else if (field == 19) out[q] = o->count ? 2.0 * o->phre[q] / (double)o->count : 0.0;
                else out[q] = o->count ? -2.0 * o->phim[q] / (double)o->count : 0.0;
            }
    return 0;
}

int orc_set_field(orc *o, int field, const double *in)
{
    const int nx = o->n[0], ny = o->n[1], nz = o->n[2];
    if (field < 0 || field >= NFIELD) return -1;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i)
                o->f[field][AT(o, i, j, k)] = in[DENSE(o, i, j, k)];
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* Checkpoint of the time-dependent state (fields, psi, sensor maps, counters) to a file */
/* and back: test infrastructure for runs that outlast one job (the full-length runs of  */
/* configs 3 and 4 take hours).  No arithmetic: a resumed run is bit-identical to an      */
/* uninterrupted one (tests/test_oracle_pins.py::test_checkpoint_resume_is_bit_identical).*/
/* The context that loads must have been created with the same arguments.                */
/* ------------------------------------------------------------------------------------ */
static int io_block(FILE *fp, void *p, size_t bytes, int write)
{
    const size_t chunk = (size_t)1 << 28;
    char *c = (char *)p;
    while (bytes) {
        size_t n = bytes < chunk ? bytes : chunk;
        size_t done = write ? fwrite(c, 1, n, fp) : fread(c, 1, n, fp);
        if (done != n) return -1;
        c += n; bytes -= n;
    }
    return 0;
}
/* first touch of a freshly calloc'ed array by the threads that will sweep it (static schedule over contiguous
 * slabs, like the loop nests of the step): without it a resumed run has every page placed by the one thread
 * that reads the file */
static void touch_parallel(double *a, size_t n)
{
    const long long blocks = (long long)((n + 511) / 512);
#pragma omp parallel for schedule(static)
    for (long long b = 0; b < blocks; ++b) a[(size_t)b * 512] = 0.0;
}
static int state_io(orc *o, const char *path, int write)
{
    FILE *fp = fopen(path, write ? "wb" : "rb");
    if (!fp) return -1;
    if (!write) {
        const size_t ncell = (size_t)o->n[0] * o->n[1] * o->n[2];
        if (o->step == 0) {
            for (int q = 0; q < NFIELD; ++q) touch_parallel(o->f[q], padded_cells(o));
            touch_parallel(o->peak, ncell);
            touch_parallel(o->sumsq, ncell);
        }
    }
    int64_t hdr[8] = { 0x4f52434b50543031LL, o->n[0], o->n[1], o->n[2], o->P, o->nmat, o->step, o->count };
    int rc = 0;
    if (write) rc = io_block(fp, hdr, sizeof(hdr), 1);
    else {
        int64_t in[8];
        rc = io_block(fp, in, sizeof(in), 0);
        for (int q = 0; q < 6 && !rc; ++q) if (in[q] != hdr[q]) rc = -2;
        if (!rc) { o->step = in[6]; o->count = in[7]; }
    }
    const size_t nc = (size_t)o->n[0] * o->n[1] * o->n[2];
    for (int q = 0; q < NFIELD && !rc; ++q) rc = io_block(fp, o->f[q], sizeof(double) * padded_cells(o), write);
    for (int a = 0; a < 3 && !rc; ++a)
        for (int t = 0; t < 6 && !rc; ++t) {
            size_t pc = psi_cells(o, a);
            if (pc) rc = io_block(fp, o->psi[a * 6 + t], sizeof(double) * pc, write);
        }
    if (!rc) rc = io_block(fp, o->peak, sizeof(double) * nc, write);
    if (!rc) rc = io_block(fp, o->sumsq, sizeof(double) * nc, write);
    if (!rc && o->phre) rc = io_block(fp, o->phre, sizeof(double) * nc, write);
    if (!rc && o->phim) rc = io_block(fp, o->phim, sizeof(double) * nc, write);
    if (fclose(fp)) rc = rc ? rc : -3;
    return rc;
}
int orc_save_state(orc *o, const char *path) { return state_io(o, path, 1); }
int orc_load_state(orc *o, const char *path) { return state_io(o, path, 0); }

/* values of one field (0..15) at a list of dense cell indices (cheap probes for traces) */
int orc_probe(const orc *o, int field, int64_t ncell, const int64_t *cell, double *out)
{
    if (field < 0 || field > 15) return -1;
    for (int64_t s = 0; s < ncell; ++s) {
        int64_t q = cell[s];
        int i = (int)(q % o->n[0]), j = (int)((q / o->n[0]) % o->n[1]);
        int k = (int)(q / ((int64_t)o->n[0] * o->n[1]));
        size_t c = AT(o, i, j, k);
        out[s] = (field < NFIELD) ? o->f[field][c]
                                  : -(o->f[SXX][c] + o->f[SYY][c] + o->f[SZZ][c]) / 3.0;
    }
    return 0;
}

int orc_get_derived(const orc *o, double *out)      /* nmat * 8 */
{
    memcpy(out, o->der, sizeof(double) * NDER * o->nmat);
    return 0;
}
int orc_get_profile(const orc *o, int axis, int which, double *out)   /* which: a_int,b_int,a_half,b_half */
{
    if (axis < 0 || axis > 2 || which < 0 || which > 3) return -1;
    memcpy(out, o->prof[axis][which], sizeof(double) * o->n[axis]);
    return 0;
}
