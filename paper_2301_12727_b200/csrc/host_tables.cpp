// host_tables.cpp -- S0: per-material constants, kernel coefficient rows, C-PML profiles.
// Follows PAPER.md:L148-L152 (Eq. 3: Q = w/(2 c alpha), "relaxation constants and memory
// variables"), Table 1 (L65-L73) and, where the paper defers to its reference [23] (L93),
// DESIGN.md readings P3 (one standard-linear-solid mechanism, tau-method), P5 (C-PML), P6.
#include "host_tables.hpp"

#include <cmath>

namespace bvfdtd {

namespace {
const double kPi = 3.14159265358979323846;

// One wave type of one material: the loss angle delta follows from the table's attenuation by
// alpha = (w0/c) tan(delta/2) exactly; Q = 1/tan(delta); the SLS level is tau = 2/(Q-1); the
// relaxed modulus is scaled by g so that the phase speed at w0 is the table's c.
bool sls_level(double alpha, double c, double w0, double &tau, double &g) {
    tau = 0.0;
    g = 1.0;
    if (alpha == 0.0 || c == 0.0) return true;
    const double th = alpha * c / w0;              // tan(delta/2)
    if (!(th < std::tan(kPi / 8.0))) return false;  // delta >= 45 deg <=> Q <= 1
    const double td = 2.0 * th / (1.0 - th * th);  // tan(delta)
    const double Q = 1.0 / td;
    tau = 2.0 / (Q - 1.0);
    const double cos2_half = 1.0 / (1.0 + th * th);
    g = 2.0 * cos2_half / std::hypot(2.0 + tau, tau);
    return true;
}
}  // namespace

int derive_materials(const bvfdtd_material *table, int n, double f0, std::vector<Derived> &out) {
    if (!table || n < 1 || n > 256 || !(f0 > 0.0)) return BVFDTD_EINVAL;
    const double w0 = 2.0 * kPi * f0;
    out.resize(n);
    for (int m = 0; m < n; ++m) {
        const bvfdtd_material &t = table[m];
        if (!(t.rho > 0.0) || !(t.cL > 0.0) || !(t.cS >= 0.0) || !(t.alphaL >= 0.0) ||
            !(t.alphaS >= 0.0) || !std::isfinite(t.rho) || !std::isfinite(t.cL))
            return BVFDTD_EINVAL;
        // bulk modulus rho (cL^2 - 4/3 cS^2) must stay positive (PAPER.md:L142 validity remark)
        if (!(t.cS < 0.5 * std::sqrt(3.0) * t.cL)) return BVFDTD_EINVAL;
        Derived d;
        double gP, gS;
        if (!sls_level(t.alphaL, t.cL, w0, d.tauP, gP)) return BVFDTD_EINVAL;
        if (!sls_level(t.alphaS, t.cS, w0, d.tauS, gS)) return BVFDTD_EINVAL;
        d.rho = t.rho;
        d.piR = t.rho * t.cL * t.cL * gP;
        d.muR = t.rho * t.cS * t.cS * gS;
        d.piU = d.piR * (1.0 + d.tauP);
        d.muU = d.muR * (1.0 + d.tauS);
        d.cU = std::sqrt(d.piU / d.rho);
        out[m] = d;
    }
    return BVFDTD_OK;
}

void kernel_rows(const std::vector<Derived> &d, double dt, double f0, std::vector<KRow> &rows) {
    const double tau_sigma = 1.0 / (2.0 * kPi * f0);
    const double beta = dt / (2.0 * tau_sigma);
    const double B = 2.0 * beta / (1.0 + beta);
    rows.resize(d.size());
    for (size_t m = 0; m < d.size(); ++m) {
        KRow r;
        r.rho = (float)d[m].rho;
        r.eP = (float)(dt * d[m].piU);
        r.eS = (float)(2.0 * dt * d[m].muU);
        r.bP = (float)(B * d[m].piR * d[m].tauP);
        r.bS = (float)(2.0 * B * d[m].muR * d[m].tauS);
        r.invMu = d[m].muR > 0.0 ? (float)(1.0 / d[m].muR) : 0.0f;
        r.tauS = (float)d[m].tauS;
        r.solid = d[m].muR > 0.0 ? 1.0f : 0.0f;
        rows[m] = r;
    }
}

// C-PML, kappa = 1 (reading P5).  Node i sits at i dx (integer) or (i + 1/2) dx (half); the
// layer/interior interfaces are at (P - 1/2) dx and (n - P - 1/2) dx; xi = depth into the layer.
void pml_axis(int n, int pml, double dx, double dt, double f0, double R, double c_ref, PmlAxis &p, bool open_lo, bool open_hi) {
    p.a_int.assign(n, 0.0f);
    p.b_int.assign(n, 1.0f);
    p.a_half.assign(n, 0.0f);
    p.b_half.assign(n, 1.0f);
    if (pml <= 0) return;
    const double L = pml * dx;
    const double d0 = 3.0 * c_ref * std::log(1.0 / R) / (2.0 * L);
    const double lo_face = (pml - 0.5) * dx, hi_face = (n - pml - 0.5) * dx;
    for (int i = 0; i < n; ++i) {
        for (int half = 0; half < 2; ++half) {
            const double x = (i + (half ? 0.5 : 0.0)) * dx;
            double xi = 0.0;
            if (!open_lo && lo_face - x > xi) xi = lo_face - x;   // an open face is a slab interface (NEXT-5):
            if (!open_hi && x - hi_face > xi) xi = x - hi_face;   // no absorber there, the profile stays inert
            const double s = xi / L;
            const double d = d0 * s * s;
            const double al = kPi * f0 * (1.0 - s);
            const double b = std::exp(-(d + al) * dt);
            const double a = d > 0.0 ? d * (b - 1.0) / (d + al) : 0.0;
            (half ? p.a_half : p.a_int)[i] = (float)a;
            (half ? p.b_half : p.b_int)[i] = (float)b;
        }
    }
}

double max_courant(const std::vector<Derived> &d, double dt, double dx) {
    double m = 0.0;
    for (const Derived &e : d) m = std::fmax(m, e.cU * dt / dx);
    return m;
}

}  // namespace bvfdtd
