// ocn_ref.cpp — CPU ORACLE (test infrastructure only; see ocn_ref.h).
//
// Plain fp64 nested loops over dense arrays with 3-cell halos, 3-D byte masks found by brute
// force, every intermediate (zeta, K, D, fluxes) stored as a full 3-D array.  It follows
// DESIGN.md §3 step by step in that order and notation; it is deliberately NOT structured
// like the CUDA path (no tiles, no 2-D threshold maps, no fused passes, bottom-up Thomas).
// OpenMP, when enabled, only distributes independent rows: every cell's arithmetic and every
// sum's order is unchanged, so results are bit-identical to the serial run.
//
// Pins: tests/test_oracle_*.py (closed forms, invariants, brute force).
// Parity unpinned: nothing (but the SCHEMES are the readings listed in DESIGN.md §3, the
// paper prints no formulas or worked values to pin them to — PAPER.md:84-98).

#include "ocn_ref.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int HALO = 3;
thread_local std::string g_err;
int fail(const std::string& m) { g_err = m; return 1; }

// dense 3-D array with horizontal halos ------------------------------------------------------
struct A3 {
    int nx = 0, ny = 0, nl = 0, sx = 0, sy = 0;
    std::vector<double> a;
    void init(int nx_, int ny_, int nl_) {
        nx = nx_; ny = ny_; nl = nl_; sx = nx + 2 * HALO; sy = ny + 2 * HALO;
        a.assign((size_t)nl * sy * sx, 0.0);
    }
    inline double& operator()(int k, int j, int i) { return a[((size_t)k * sy + (j + HALO)) * sx + (i + HALO)]; }
    inline double operator()(int k, int j, int i) const { return a[((size_t)k * sy + (j + HALO)) * sx + (i + HALO)]; }
};
struct B3 {  // byte masks
    int nx = 0, ny = 0, nl = 0, sx = 0, sy = 0;
    std::vector<unsigned char> a;
    void init(int nx_, int ny_, int nl_) {
        nx = nx_; ny = ny_; nl = nl_; sx = nx + 2 * HALO; sy = ny + 2 * HALO;
        a.assign((size_t)nl * sy * sx, 0);
    }
    inline unsigned char& operator()(int k, int j, int i) { return a[((size_t)k * sy + (j + HALO)) * sx + (i + HALO)]; }
    inline unsigned char operator()(int k, int j, int i) const { return a[((size_t)k * sy + (j + HALO)) * sx + (i + HALO)]; }
};

template <class ARR>
void fill_halo(ARR& f, bool px, bool py) {
    // periodic directions wrap; bounded directions keep 0 (land halo) — DESIGN.md §3.3
    const int nx = f.nx, ny = f.ny;
    for (int k = 0; k < f.nl; ++k) {
        for (int j = 0; j < ny; ++j)
            for (int h = 1; h <= HALO; ++h) {
                f(k, j, -h) = px ? f(k, j, nx - h) : 0;
                f(k, j, nx - 1 + h) = px ? f(k, j, h - 1) : 0;
            }
        for (int h = 1; h <= HALO; ++h)
            for (int i = -HALO; i < nx + HALO; ++i) {
                f(k, -h, i) = py ? f(k, ny - h, i) : 0;
                f(k, ny - 1 + h, i) = py ? f(k, h - 1, i) : 0;
            }
    }
}

}  // namespace

struct ocn_ref_grid {
    ocn_ref_grid_desc d;
    int nx, ny, nz;
    bool px, py;
    std::vector<double> zf, dz, zc, dzc;          // dzc[k] = zc[k]-zc[k-1], k = 1..nz-1
    double dy;
    std::vector<double> dxC_, dxF_, AzC_, AzF_, fF_;   // rows j = -HALO .. ny+HALO
    double dxC(int j) const { return dxC_[j + HALO]; }
    double dxF(int j) const { return dxF_[j + HALO]; }
    double AzC(int j) const { return AzC_[j + HALO]; }
    double AzF(int j) const { return AzF_[j + HALO]; }
    double fF(int j) const { return fF_[j + HALO]; }
    B3 wet;                                       // nz levels, with halo
    // derived masks
    int mu(int k, int j, int i) const { return wet(k, j, i) && wet(k, j, i - 1); }
    int mv(int k, int j, int i) const { return wet(k, j, i) && wet(k, j - 1, i); }
    int mw(int k, int j, int i) const { return (k >= 1 && k <= nz - 1) ? (wet(k, j, i) && wet(k - 1, j, i)) : 0; }
    int zeta_valid(int k, int j, int i) const {
        return wet(k, j - 1, i - 1) && wet(k, j - 1, i) && wet(k, j, i - 1) && wet(k, j, i);
    }
    // tracer face orders: largest r such that the 2r cells n-r..n+r-1 along the axis are wet
    int order_x(int k, int j, int i) const {
        int o = 0;
        for (int r = 1; r <= 3; ++r) {
            bool ok = true;
            for (int m = i - r; m <= i + r - 1; ++m) ok = ok && wet(k, j, m);
            if (ok) o = r; else break;
        }
        return o;
    }
    int order_y(int k, int j, int i) const {
        int o = 0;
        for (int r = 1; r <= 3; ++r) {
            bool ok = true;
            for (int m = j - r; m <= j + r - 1; ++m) ok = ok && wet(k, m, i);
            if (ok) o = r; else break;
        }
        return o;
    }
    int order_z(int k, int j, int i) const {     // face below cell k, k = 0..nz
        int o = 0;
        for (int r = 1; r <= 3; ++r) {
            bool ok = true;
            for (int m = k - r; m <= k + r - 1; ++m) ok = ok && (m >= 0 && m < nz && wet(m, j, i));
            if (ok) o = r; else break;
        }
        return o;
    }
    // vorticity reconstruction orders: "cells" are zeta points; max(1, r) on open faces
    int order_zeta_u(int k, int j, int i) const {   // along y, interface between zeta[j], zeta[j+1]
        if (!mu(k, j, i)) return 0;
        int o = 0;
        for (int r = 1; r <= 3; ++r) {
            bool ok = true;
            for (int m = j + 1 - r; m <= j + r; ++m) ok = ok && zeta_valid(k, m, i);
            if (ok) o = r; else break;
        }
        return o < 1 ? 1 : o;
    }
    int order_zeta_v(int k, int j, int i) const {   // along x, interface between zeta[i], zeta[i+1]
        if (!mv(k, j, i)) return 0;
        int o = 0;
        for (int r = 1; r <= 3; ++r) {
            bool ok = true;
            for (int m = i + 1 - r; m <= i + r; ++m) ok = ok && zeta_valid(k, j, m);
            if (ok) o = r; else break;
        }
        return o < 1 ? 1 : o;
    }
};

struct ocn_ref_model {
    const ocn_ref_grid* g;
    ocn_ref_model_desc d;
    std::vector<double> a_w;        // filter weights a_m, m = 1..M  (index m-1)
    std::vector<double> b_w;        // filter weights of the transports U, V; = a_w unless given
    double dtau;
    A3 u, v, T, S, w, p;            // w has nz+1 levels
    A3 Gu, Gv, GT, GS;              // G^n
    A3 Gu1, Gv1, GT1, GS1;          // G^{n-1}
    A3 eta, U, V, taux, tauy, Hu, Hv;   // 2-D (nl = 1)
    A3 qT, qS, rT, rS;              // surface tracer fluxes and restoring targets (2-D)
    A3 nuc, kapc;                   // closure = 1: nu, kappa at the bottom face of tracer cell (k, j, i)
    bool have_history = false;
};

namespace {

// ---------------------------------------------------------------------------------------------
// WENO reconstruction (Jiang-Shu weights, uniform-grid coefficients)
// c[0..5] = cells n-3 .. n+2, interface between c[2] (n-1) and c[3] (n).
// ---------------------------------------------------------------------------------------------
// scheme 0: the classical Jiang-Shu weights alpha_s = d_s / (eps + beta_s)^2.
// scheme 1 (Borges et al. 2008 for r = 3, the same construction for r = 2): WENO-Z weights
//   alpha_s = d_s (1 + (tau / (eps + beta_s))^2),  tau = |beta_0 - beta_{r-1}|
// with the same candidate polynomials, smoothness indicators, linear weights and eps.
double weno(const double c[6], int order, double vel, int scheme = 0) {
    double qm2, qm1, q0, q1, q2;
    if (vel > 0.0) { qm2 = c[0]; qm1 = c[1]; q0 = c[2]; q1 = c[3]; q2 = c[4]; }
    else           { qm2 = c[5]; qm1 = c[4]; q0 = c[3]; q1 = c[2]; q2 = c[1]; }
    const double eps = 1e-6;
    if (order >= 3) {
        const double p0 = (2.0 * qm2 - 7.0 * qm1 + 11.0 * q0) / 6.0;
        const double p1 = (-qm1 + 5.0 * q0 + 2.0 * q1) / 6.0;
        const double p2 = (2.0 * q0 + 5.0 * q1 - q2) / 6.0;
        const double b0 = 13.0 / 12.0 * (qm2 - 2.0 * qm1 + q0) * (qm2 - 2.0 * qm1 + q0)
                        + 0.25 * (qm2 - 4.0 * qm1 + 3.0 * q0) * (qm2 - 4.0 * qm1 + 3.0 * q0);
        const double b1 = 13.0 / 12.0 * (qm1 - 2.0 * q0 + q1) * (qm1 - 2.0 * q0 + q1)
                        + 0.25 * (qm1 - q1) * (qm1 - q1);
        const double b2 = 13.0 / 12.0 * (q0 - 2.0 * q1 + q2) * (q0 - 2.0 * q1 + q2)
                        + 0.25 * (3.0 * q0 - 4.0 * q1 + q2) * (3.0 * q0 - 4.0 * q1 + q2);
        if (scheme == 1) {
            const double tau = std::fabs(b0 - b2);
            const double r0 = tau / (eps + b0), r1 = tau / (eps + b1), r2 = tau / (eps + b2);
            const double a0 = 0.1 * (1.0 + r0 * r0), a1 = 0.6 * (1.0 + r1 * r1), a2 = 0.3 * (1.0 + r2 * r2);
            return (a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2);
        }
        const double a0 = 0.1 / ((eps + b0) * (eps + b0));
        const double a1 = 0.6 / ((eps + b1) * (eps + b1));
        const double a2 = 0.3 / ((eps + b2) * (eps + b2));
        return (a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2);
    }
    if (order == 2) {
        const double p0 = (-qm1 + 3.0 * q0) / 2.0;
        const double p1 = (q0 + q1) / 2.0;
        const double b0 = (q0 - qm1) * (q0 - qm1);
        const double b1 = (q1 - q0) * (q1 - q0);
        if (scheme == 1) {
            const double tau = std::fabs(b0 - b1);
            const double r0 = tau / (eps + b0), r1 = tau / (eps + b1);
            const double a0 = (1.0 / 3.0) * (1.0 + r0 * r0), a1 = (2.0 / 3.0) * (1.0 + r1 * r1);
            return (a0 * p0 + a1 * p1) / (a0 + a1);
        }
        const double a0 = (1.0 / 3.0) / ((eps + b0) * (eps + b0));
        const double a1 = (2.0 / 3.0) / ((eps + b1) * (eps + b1));
        return (a0 * p0 + a1 * p1) / (a0 + a1);
    }
    if (order == 1) return q0;
    return 0.0;
}

// ---------------------------------------------------------------------------------------------
// DESIGN.md §3.8 step 4 — backward-Euler vertical diffusion of one column (Thomas, bottom-up)
//   (1 + s+_k + s-_k) phi_k - s+_k phi_{k+1} - s-_k phi_{k-1} = phi*_k
// ---------------------------------------------------------------------------------------------
//   dtk[k], k = 0..nz: dt * kappa at the face below cell k (a constant array for closure 0,
//   DESIGN.md §3.12 for closure 1); closed faces are not read
void implicit_column(int nz, const double* dz, const double* dzc, const unsigned char* open,
                     const double* dtk, double* phi, double* cp, double* dp) {
    for (int k = 0; k < nz; ++k) {
        const double sp = (k + 1 <= nz - 1 && open[k + 1]) ? dtk[k + 1] / (dz[k] * dzc[k + 1]) : 0.0;
        const double sm = (k >= 1 && open[k]) ? dtk[k] / (dz[k] * dzc[k]) : 0.0;
        const double b = 1.0 + sp + sm;
        const double lo = -sm, up = -sp;
        if (k == 0) {
            cp[k] = up / b;
            dp[k] = phi[k] / b;
        } else {
            const double m = b - lo * cp[k - 1];
            cp[k] = up / m;
            dp[k] = (phi[k] - lo * dp[k - 1]) / m;
        }
    }
    phi[nz - 1] = dp[nz - 1];
    for (int k = nz - 2; k >= 0; --k) phi[k] = dp[k] - cp[k] * phi[k + 1];
}

// power-law filter, p = 2, q = 4
void filter_weights(int M, std::vector<double>& a, double& dtau_over_dt) {
    a.assign(M, 0.0);
    double sum = 0.0;
    for (int m = 1; m <= M; ++m) {
        const double s = (double)m / (double)(M + 1);
        a[m - 1] = s * s * (1.0 - s * s * s * s);
        sum += a[m - 1];
    }
    double first = 0.0;
    for (int m = 1; m <= M; ++m) { a[m - 1] /= sum; first += m * a[m - 1]; }
    dtau_over_dt = 1.0 / first;
}

// ---------------------------------------------------------------------------------------------
// diagnostics
// ---------------------------------------------------------------------------------------------
void compute_w(ocn_ref_model& M) {
    const ocn_ref_grid& g = *M.g;
    fill_halo(M.u, g.px, g.py);
    fill_halo(M.v, g.px, g.py);
#pragma omp parallel for schedule(static)
    for (int j = 0; j < g.ny; ++j)
        for (int i = 0; i < g.nx; ++i) {
            M.w(0, j, i) = 0.0;
            for (int k = 0; k < g.nz; ++k) {
                const double D = (g.dy * (M.u(k, j, i + 1) - M.u(k, j, i))
                                  + g.dxF(j + 1) * M.v(k, j + 1, i) - g.dxF(j) * M.v(k, j, i)) / g.AzC(j);
                M.w(k + 1, j, i) = M.w(k, j, i) - g.dz[k] * D;
            }
        }
    fill_halo(M.w, g.px, g.py);
}

// eos 0, the linear equation of state b = g [alpha (T - T0) - beta_S (S - S0)].
// eos 1, a nonlinear equation of state with thermobaricity and cabbeling,
//   b = g [alpha (1 - gamma z_c) (T - T0) + (alpha2 / 2) (T - T0)^2 - beta_S (S - S0)],   z_c <= 0 the depth of the cell centre
inline double buoyancy(const ocn_ref_model& M, int k, int j, int i) {
    const double dT = M.T(k, j, i) - M.d.T0, dS = M.S(k, j, i) - M.d.S0;
    if (M.d.eos == 1)
        return M.d.g * (M.d.alpha * (1.0 - M.d.eos_gamma * M.g->zc[k]) * dT + 0.5 * M.d.eos_alpha2 * dT * dT - M.d.beta_s * dS);
    return M.d.g * (M.d.alpha * dT - M.d.beta_s * dS);
}

void compute_p(ocn_ref_model& M) {
    const ocn_ref_grid& g = *M.g;
    const int nz = g.nz;
#pragma omp parallel for schedule(static)
    for (int j = 0; j < g.ny; ++j)
        for (int i = 0; i < g.nx; ++i) {
            M.p(nz - 1, j, i) = -buoyancy(M, nz - 1, j, i) * (g.zf[nz] - g.zc[nz - 1]);
            for (int k = nz - 2; k >= 0; --k)
                M.p(k, j, i) = M.p(k + 1, j, i)
                             - 0.5 * (buoyancy(M, k + 1, j, i) + buoyancy(M, k, j, i)) * g.dzc[k + 1];
        }
    fill_halo(M.p, g.px, g.py);
}

// ---------------------------------------------------------------------------------------------
// Richardson-number-based vertical mixing with convective adjustment
// (PAPER.md:114 names it, PAPER.md:78 stores it; the formula is a reading).  At the face below
// tracer cell (k, j, i), k = 1..nz-1, open iff mw:
//   N2 = (b_k - b_{k-1}) / dzc_k
//   S2 = [ (du_w^2 + du_e^2)/2 + (dv_s^2 + dv_n^2)/2 ] / dzc_k^2,   du = u_k - u_{k-1} on the four faces of the column
//   Ri = max(N2, 0) / (S2 + S2min),  f = 1 / (1 + c Ri)
//   conv = kconv * min(1, max(-N2, 0) / N2c)          (continuous ramp instead of a switch)
//   nu = nu_z + nu0 f^2 + conv,   kappa = kappa_z + nu0 f^3 + conv
// Needs the halos of u, v of the current state.
// ---------------------------------------------------------------------------------------------
void compute_mixing(ocn_ref_model& M) {
    const ocn_ref_grid& g = *M.g;
    const ocn_ref_model_desc& d = M.d;
#pragma omp parallel for schedule(static)
    for (int j = 0; j < g.ny; ++j)
        for (int i = 0; i < g.nx; ++i) {
            M.nuc(0, j, i) = 0.0; M.kapc(0, j, i) = 0.0;
            for (int k = 1; k < g.nz; ++k) {
                if (!g.mw(k, j, i)) { M.nuc(k, j, i) = 0.0; M.kapc(k, j, i) = 0.0; continue; }
                const double N2 = (buoyancy(M, k, j, i) - buoyancy(M, k - 1, j, i)) / g.dzc[k];
                const double duw = M.u(k, j, i) - M.u(k - 1, j, i), due = M.u(k, j, i + 1) - M.u(k - 1, j, i + 1);
                const double dvs = M.v(k, j, i) - M.v(k - 1, j, i), dvn = M.v(k, j + 1, i) - M.v(k - 1, j + 1, i);
                const double S2 = (0.5 * (duw * duw + due * due) + 0.5 * (dvs * dvs + dvn * dvn)) / (g.dzc[k] * g.dzc[k]);
                const double Ri = std::max(N2, 0.0) / (S2 + d.ri_s2min);
                const double f = 1.0 / (1.0 + d.ri_c * Ri);
                const double conv = d.ri_kconv * std::min(1.0, std::max(-N2, 0.0) / d.ri_n2c);
                M.nuc(k, j, i) = d.nu_z + d.ri_nu0 * f * f + conv;
                M.kapc(k, j, i) = d.kappa_z + d.ri_nu0 * f * f * f + conv;
            }
        }
    fill_halo(M.nuc, g.px, g.py); fill_halo(M.kapc, g.px, g.py);
}

// ---------------------------------------------------------------------------------------------
// DESIGN.md §3.6 / §3.7 — tendencies G^n of the current state into (Gu, Gv, GT, GS)
// ---------------------------------------------------------------------------------------------
// surf / target / gamma: the surface forcing of the top cell: G += wet (surf + gamma (target - c)) / dz
void tracer_tendency(const ocn_ref_model& M, const A3& c, A3& G, A3& Fx, A3& Fy, A3& Fz,
                     const A3& surf, const A3& target, double gamma) {
    const ocn_ref_grid& g = *M.g;
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const double kh = M.d.kappa_h;
    // fluxes through the west (Fx), south (Fy) and bottom (Fz) faces
#pragma omp parallel for schedule(static)
    for (int j = 0; j <= ny; ++j)
        for (int k = 0; k < nz; ++k)
            for (int i = 0; i <= nx; ++i) {
                if (j < ny) {
                    const double cs[6] = {c(k, j, i - 3), c(k, j, i - 2), c(k, j, i - 1),
                                          c(k, j, i), c(k, j, i + 1), c(k, j, i + 2)};
                    const double uu = M.u(k, j, i);
                    const double cf = weno(cs, g.order_x(k, j, i), uu, M.d.advection);
                    Fx(k, j, i) = uu * g.dy * g.dz[k] * cf
                                - kh * g.dy * g.dz[k] * (c(k, j, i) - c(k, j, i - 1)) / g.dxC(j) * g.mu(k, j, i);
                }
                if (i < nx) {
                    const double cs[6] = {c(k, j - 3, i), c(k, j - 2, i), c(k, j - 1, i),
                                          c(k, j, i), c(k, j + 1, i), c(k, j + 2, i)};
                    const double vv = M.v(k, j, i);
                    const double cf = weno(cs, g.order_y(k, j, i), vv, M.d.advection);
                    Fy(k, j, i) = vv * g.dxF(j) * g.dz[k] * cf
                                - kh * g.dxF(j) * g.dz[k] * (c(k, j, i) - c(k, j - 1, i)) / g.dy * g.mv(k, j, i);
                }
            }
#pragma omp parallel for schedule(static)
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i)
            for (int k = 0; k <= nz; ++k) {
                if (k == 0 || k == nz) { Fz(k, j, i) = 0.0; continue; }
                double cs[6];
                for (int m = 0; m < 6; ++m) {
                    const int kk = k - 3 + m;
                    cs[m] = (kk >= 0 && kk < nz) ? c(kk, j, i) : 0.0;
                }
                const double ww = M.w(k, j, i);
                const double cf = weno(cs, g.order_z(k, j, i), ww, M.d.advection);
                Fz(k, j, i) = ww * g.AzC(j) * cf * g.mw(k, j, i);
            }
#pragma omp parallel for schedule(static)
    for (int j = 0; j < ny; ++j)
        for (int k = 0; k < nz; ++k)
            for (int i = 0; i < nx; ++i) {
                const double div = Fx(k, j, i + 1) - Fx(k, j, i) + Fy(k, j + 1, i) - Fy(k, j, i)
                                 + Fz(k + 1, j, i) - Fz(k, j, i);
                G(k, j, i) = -(double)g.wet(k, j, i) * div / (g.AzC(j) * g.dz[k]);
                if (k == nz - 1)
                    G(k, j, i) += (double)g.wet(k, j, i) * (surf(0, j, i) + gamma * (target(0, j, i) - c(k, j, i))) / g.dz[k];
            }
}

void momentum_tendency(const ocn_ref_model& M, A3& Gu, A3& Gv, A3& zeta, A3& Ke, A3& Dv) {
    const ocn_ref_grid& g = *M.g;
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const A3 &u = M.u, &v = M.v, &w = M.w, &p = M.p;
    // zeta at south-west corners, K and D at centres, on the interior plus 2 halo rings
    // (velocities are masked and halo-filled, so this is the same formula everywhere)
#pragma omp parallel for schedule(static)
    for (int j = -2; j < ny + HALO; ++j)
        for (int k = 0; k < nz; ++k)
            for (int i = -2; i < nx + HALO; ++i) {
                zeta(k, j, i) = (g.dy * (v(k, j, i) - v(k, j, i - 1))
                                 - (g.dxC(j) * u(k, j, i) - g.dxC(j - 1) * u(k, j - 1, i))) / g.AzF(j);
                if (j < ny + HALO - 1 && i < nx + HALO - 1) {
                    Ke(k, j, i) = 0.25 * (u(k, j, i) * u(k, j, i) + u(k, j, i + 1) * u(k, j, i + 1))
                                + 0.25 * (v(k, j, i) * v(k, j, i) + v(k, j + 1, i) * v(k, j + 1, i));
                    Dv(k, j, i) = (g.dy * (u(k, j, i + 1) - u(k, j, i))
                                   + g.dxF(j + 1) * v(k, j + 1, i) - g.dxF(j) * v(k, j, i)) / g.AzC(j);
                }
            }
    const double nu = M.d.nu_h;
#pragma omp parallel for schedule(static)
    for (int j = 0; j < ny; ++j)
        for (int k = 0; k < nz; ++k)
            for (int i = 0; i < nx; ++i) {
                // ---------------- u point ----------------
                {
                    const int m = g.mu(k, j, i);
                    const double vhat = 0.25 * (g.dxF(j) * (v(k, j, i - 1) + v(k, j, i))
                                              + g.dxF(j + 1) * (v(k, j + 1, i - 1) + v(k, j + 1, i))) / g.dxC(j);
                    const double zs[6] = {zeta(k, j - 2, i), zeta(k, j - 1, i), zeta(k, j, i),
                                          zeta(k, j + 1, i), zeta(k, j + 2, i), zeta(k, j + 3, i)};
                    const double zt = weno(zs, g.order_zeta_u(k, j, i), vhat, M.d.advection);
                    const double Cu = 0.5 * (g.fF(j) * 0.5 * g.dxF(j) * (v(k, j, i - 1) + v(k, j, i))
                                           + g.fF(j + 1) * 0.5 * g.dxF(j + 1) * (v(k, j + 1, i - 1) + v(k, j + 1, i))) / g.dxC(j);
                    const double dK = (Ke(k, j, i) - Ke(k, j, i - 1)) / g.dxC(j);
                    const double dP = (p(k, j, i) - p(k, j, i - 1)) / g.dxC(j);
                    // vertical advection, centred "w du/dz" form
                    const double Wlo = 0.5 * g.AzC(j) * (w(k, j, i - 1) + w(k, j, i));
                    const double Whi = 0.5 * g.AzC(j) * (w(k + 1, j, i - 1) + w(k + 1, j, i));
                    const double dlo = (k >= 1) ? (u(k, j, i) - u(k - 1, j, i)) * g.mu(k, j, i) * g.mu(k - 1, j, i) : 0.0;
                    const double dhi = (k + 1 <= nz - 1) ? (u(k + 1, j, i) - u(k, j, i)) * g.mu(k + 1, j, i) * g.mu(k, j, i) : 0.0;
                    const double Au = 0.5 * (Whi * dhi + Wlo * dlo) / (g.AzC(j) * g.dz[k]);
                    const double Vu = nu * ((Dv(k, j, i) - Dv(k, j, i - 1)) / g.dxC(j)
                                          - (zeta(k, j + 1, i) - zeta(k, j, i)) / g.dy);
                    const double tau = (k == nz - 1) ? M.taux(0, j, i) / (M.d.rho0 * g.dz[k]) : 0.0;
                    // bottom drag on the lowest open level of the u column
                    const bool bot = m && (k == 0 || !g.mu(k - 1, j, i));
                    const double drag = bot ? (M.d.drag_r + M.d.drag_cd * std::sqrt(u(k, j, i) * u(k, j, i) + vhat * vhat))
                                                  * u(k, j, i) / g.dz[k] : 0.0;
                    Gu(k, j, i) = m * (zt * vhat + Cu - dK - dP - Au + Vu + tau - drag);
                }
                // ---------------- v point ----------------
                {
                    const int m = g.mv(k, j, i);
                    const double uhat = 0.25 * (u(k, j - 1, i) + u(k, j, i) + u(k, j - 1, i + 1) + u(k, j, i + 1));
                    const double zs[6] = {zeta(k, j, i - 2), zeta(k, j, i - 1), zeta(k, j, i),
                                          zeta(k, j, i + 1), zeta(k, j, i + 2), zeta(k, j, i + 3)};
                    const double zt = weno(zs, g.order_zeta_v(k, j, i), uhat, M.d.advection);
                    const double Cv = g.fF(j) * uhat;
                    const double dK = (Ke(k, j, i) - Ke(k, j - 1, i)) / g.dy;
                    const double dP = (p(k, j, i) - p(k, j - 1, i)) / g.dy;
                    const double Wlo = 0.5 * (g.AzC(j - 1) * w(k, j - 1, i) + g.AzC(j) * w(k, j, i));
                    const double Whi = 0.5 * (g.AzC(j - 1) * w(k + 1, j - 1, i) + g.AzC(j) * w(k + 1, j, i));
                    const double dlo = (k >= 1) ? (v(k, j, i) - v(k - 1, j, i)) * g.mv(k, j, i) * g.mv(k - 1, j, i) : 0.0;
                    const double dhi = (k + 1 <= nz - 1) ? (v(k + 1, j, i) - v(k, j, i)) * g.mv(k + 1, j, i) * g.mv(k, j, i) : 0.0;
                    const double Av = 0.5 * (Whi * dhi + Wlo * dlo) / (g.AzF(j) * g.dz[k]);
                    const double Vv = nu * ((Dv(k, j, i) - Dv(k, j - 1, i)) / g.dy
                                          + (zeta(k, j, i + 1) - zeta(k, j, i)) / g.dxF(j));
                    const double tau = (k == nz - 1) ? M.tauy(0, j, i) / (M.d.rho0 * g.dz[k]) : 0.0;
                    const bool bot = m && (k == 0 || !g.mv(k - 1, j, i));
                    const double drag = bot ? (M.d.drag_r + M.d.drag_cd * std::sqrt(uhat * uhat + v(k, j, i) * v(k, j, i)))
                                                  * v(k, j, i) / g.dz[k] : 0.0;
                    Gv(k, j, i) = m * (-zt * uhat - Cv - dK - dP - Av + Vv + tau - drag);
                }
            }
}

// ---------------------------------------------------------------------------------------------
// biharmonic horizontal dissipation: the horizontal Laplacian applied twice.
//   vector Laplacian of a C-grid vector (a at u points, b at v points), in the vector-invariant form of §3.6:
//     Da = [dy (a[i+1] - a[i]) + dxF[j+1] b[j+1] - dxF[j] b[j]] / AzC[j]
//     Za = [dy (b[i] - b[i-1]) - (dxC[j] a[j] - dxC[j-1] a[j-1])] / AzF[j]
//     La = mu [(Da[i] - Da[i-1]) / dxC[j] - (Za[j+1] - Za[j]) / dy],  Lb = mv [(Da[j] - Da[j-1]) / dy + (Za[i+1] - Za[i]) / dxF[j]]
//   scalar Laplacian of a tracer with no flux through closed faces:
//     fx[i] = dy (c[i] - c[i-1]) / dxC[j] mu[i],  fy[j] = dxF[j] (c[j] - c[j-1]) / dy mv[j],
//     Lc = wet [(fx[i+1] - fx[i]) + (fy[j+1] - fy[j])] / AzC[j]
// Inputs must be halo-filled; outputs are halo-filled here.
// ---------------------------------------------------------------------------------------------
void vector_laplacian(const ocn_ref_grid& g, const A3& a, const A3& b, A3& La, A3& Lb) {
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    A3 Da, Za;
    Da.init(nx, ny, nz); Za.init(nx, ny, nz);
#pragma omp parallel for schedule(static)
    for (int j = -2; j < ny + HALO - 1; ++j)
        for (int k = 0; k < nz; ++k)
            for (int i = -2; i < nx + HALO - 1; ++i) {
                Da(k, j, i) = (g.dy * (a(k, j, i + 1) - a(k, j, i)) + g.dxF(j + 1) * b(k, j + 1, i) - g.dxF(j) * b(k, j, i)) / g.AzC(j);
                Za(k, j, i) = (g.dy * (b(k, j, i) - b(k, j, i - 1)) - (g.dxC(j) * a(k, j, i) - g.dxC(j - 1) * a(k, j - 1, i))) / g.AzF(j);
            }
#pragma omp parallel for schedule(static)
    for (int j = 0; j < ny; ++j)
        for (int k = 0; k < nz; ++k)
            for (int i = 0; i < nx; ++i) {
                La(k, j, i) = g.mu(k, j, i) * ((Da(k, j, i) - Da(k, j, i - 1)) / g.dxC(j) - (Za(k, j + 1, i) - Za(k, j, i)) / g.dy);
                Lb(k, j, i) = g.mv(k, j, i) * ((Da(k, j, i) - Da(k, j - 1, i)) / g.dy + (Za(k, j, i + 1) - Za(k, j, i)) / g.dxF(j));
            }
    fill_halo(La, g.px, g.py); fill_halo(Lb, g.px, g.py);
}

void scalar_laplacian(const ocn_ref_grid& g, const A3& c, A3& Lc) {
    const int nx = g.nx, ny = g.ny, nz = g.nz;
#pragma omp parallel for schedule(static)
    for (int j = 0; j < ny; ++j)
        for (int k = 0; k < nz; ++k)
            for (int i = 0; i < nx; ++i) {
                const double fxw = g.dy * (c(k, j, i) - c(k, j, i - 1)) / g.dxC(j) * g.mu(k, j, i);
                const double fxe = g.dy * (c(k, j, i + 1) - c(k, j, i)) / g.dxC(j) * g.mu(k, j, i + 1);
                const double fys = g.dxF(j) * (c(k, j, i) - c(k, j - 1, i)) / g.dy * g.mv(k, j, i);
                const double fyn = g.dxF(j + 1) * (c(k, j + 1, i) - c(k, j, i)) / g.dy * g.mv(k, j + 1, i);
                Lc(k, j, i) = g.wet(k, j, i) * ((fxe - fxw) + (fyn - fys)) / g.AzC(j);
            }
    fill_halo(Lc, g.px, g.py);
}

// G_u += -nu4 La(La(u, v)), G_v likewise, G_c += -kappa4 Lc(Lc(c))   (each evaluated on its own and added to the tendency)
void add_biharmonic(const ocn_ref_model& M, A3& Gu, A3& Gv, A3& GT, A3& GS) {
    const ocn_ref_grid& g = *M.g;
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    A3 l1, l2, m1, m2;
    l1.init(nx, ny, nz); l2.init(nx, ny, nz); m1.init(nx, ny, nz); m2.init(nx, ny, nz);
    if (M.d.nu4_h != 0.0) {
        vector_laplacian(g, M.u, M.v, l1, l2);
        vector_laplacian(g, l1, l2, m1, m2);
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    Gu(k, j, i) += -(M.d.nu4_h * m1(k, j, i));
                    Gv(k, j, i) += -(M.d.nu4_h * m2(k, j, i));
                }
    }
    if (M.d.kappa4_h != 0.0) {
        const A3* c[2] = {&M.T, &M.S};
        A3* G[2] = {&GT, &GS};
        for (int f = 0; f < 2; ++f) {
            scalar_laplacian(g, *c[f], l1);
            scalar_laplacian(g, l1, m1);
            for (int k = 0; k < nz; ++k)
                for (int j = 0; j < ny; ++j)
                    for (int i = 0; i < nx; ++i) (*G[f])(k, j, i) += -(M.d.kappa4_h * m1(k, j, i));
        }
    }
}

// state must be halo-filled and w, p consistent with it
void compute_tendencies(ocn_ref_model& M, A3& Gu, A3& Gv, A3& GT, A3& GS) {
    const ocn_ref_grid& g = *M.g;
    A3 t1, t2, t3;
    t1.init(g.nx, g.ny, g.nz); t2.init(g.nx, g.ny, g.nz); t3.init(g.nx, g.ny, g.nz + 1);
    momentum_tendency(M, Gu, Gv, t1, t2, t3);
    tracer_tendency(M, M.T, GT, t1, t2, t3, M.qT, M.rT, M.d.gamma_T);
    tracer_tendency(M, M.S, GS, t1, t2, t3, M.qS, M.rS, M.d.gamma_S);
    if (M.d.nu4_h != 0.0 || M.d.kappa4_h != 0.0) add_biharmonic(M, Gu, Gv, GT, GS);
}

void fill_state_halos(ocn_ref_model& M) {
    const ocn_ref_grid& g = *M.g;
    fill_halo(M.u, g.px, g.py); fill_halo(M.v, g.px, g.py);
    fill_halo(M.T, g.px, g.py); fill_halo(M.S, g.px, g.py);
    fill_halo(M.eta, g.px, g.py); fill_halo(M.U, g.px, g.py); fill_halo(M.V, g.px, g.py);
}

// ---------------------------------------------------------------------------------------------
// DESIGN.md §3.8 step 6 — one forward-backward barotropic sub-step (eta first, then U, V)
// ---------------------------------------------------------------------------------------------
void barotropic_substep(ocn_ref_model& M, double dtau, const A3* GU, const A3* GV) {
    const ocn_ref_grid& g = *M.g;
    const int nx = g.nx, ny = g.ny, top = g.nz - 1;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i)
            if (g.wet(top, j, i))
                M.eta(0, j, i) -= dtau * (g.dy * (M.U(0, j, i + 1) - M.U(0, j, i))
                                          + g.dxF(j + 1) * M.V(0, j + 1, i) - g.dxF(j) * M.V(0, j, i)) / g.AzC(j);
    fill_halo(M.eta, g.px, g.py);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const double gu = GU ? (*GU)(0, j, i) : 0.0, gv = GV ? (*GV)(0, j, i) : 0.0;
            M.U(0, j, i) = (M.U(0, j, i) + dtau * (-M.d.g * M.Hu(0, j, i) * (M.eta(0, j, i) - M.eta(0, j, i - 1)) / g.dxC(j) + gu))
                         * g.mu(top, j, i);
            M.V(0, j, i) = (M.V(0, j, i) + dtau * (-M.d.g * M.Hv(0, j, i) * (M.eta(0, j, i) - M.eta(0, j - 1, i)) / g.dy + gv))
                         * g.mv(top, j, i);
        }
    fill_halo(M.U, g.px, g.py);
    fill_halo(M.V, g.px, g.py);
}

// ---------------------------------------------------------------------------------------------
// one baroclinic time step
// ---------------------------------------------------------------------------------------------
void time_step(ocn_ref_model& M) {
    const ocn_ref_grid& g = *M.g;
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const double dt = M.d.dt;
    // 0. vertical mixing coefficients of state n (closure 1)
    if (M.d.closure == 1) compute_mixing(M);
    // 1. G^n from state n
    compute_tendencies(M, M.Gu, M.Gv, M.GT, M.GS);
    // 2. AB2 combination (Euler on the first step after set_fields)
    const double c0 = M.have_history ? 1.5 + M.d.chi : 1.0;
    const double c1 = M.have_history ? 0.5 + M.d.chi : 0.0;
    A3 Ghu, Ghv;
    Ghu.init(nx, ny, nz); Ghv.init(nx, ny, nz);
    A3* fld[4] = {&M.u, &M.v, &M.T, &M.S};
    A3* Gn[4] = {&M.Gu, &M.Gv, &M.GT, &M.GS};
    A3* Gm[4] = {&M.Gu1, &M.Gv1, &M.GT1, &M.GS1};
    for (int f = 0; f < 4; ++f) {
#pragma omp parallel for schedule(static)
        for (int j = 0; j < ny; ++j) {
            std::vector<double> col(nz), cp(nz), dp(nz), dtk(nz + 1);
            std::vector<unsigned char> open(nz + 1);
            for (int i = 0; i < nx; ++i) {
                for (int k = 0; k < nz; ++k) {
                    const double Gh = c0 * (*Gn[f])(k, j, i) - c1 * (*Gm[f])(k, j, i);
                    if (f == 0) Ghu(k, j, i) = Gh;
                    if (f == 1) Ghv(k, j, i) = Gh;
                    const int m = f == 0 ? g.mu(k, j, i) : f == 1 ? g.mv(k, j, i) : g.wet(k, j, i);
                    // 3. explicit predictor
                    col[k] = ((*fld[f])(k, j, i) + dt * Gh) * m;
                }
                for (int k = 0; k <= nz; ++k) {
                    if (k == 0 || k == nz) { open[k] = 0; continue; }
                    open[k] = f == 0 ? (g.mu(k, j, i) && g.mu(k - 1, j, i))
                            : f == 1 ? (g.mv(k, j, i) && g.mv(k - 1, j, i))
                                     : g.mw(k, j, i);
                }
                // 4. implicit corrector; dt * kappa per face: constant, or the closure's value at the
                //    field's own vertical face (nu averaged from the two tracer columns that share the u / v face)
                for (int k = 0; k <= nz; ++k) {
                    if (M.d.closure != 1) { dtk[k] = dt * (f < 2 ? M.d.nu_z : M.d.kappa_z); continue; }
                    if (!open[k]) { dtk[k] = 0.0; continue; }
                    dtk[k] = f == 0 ? dt * (0.5 * (M.nuc(k, j, i - 1) + M.nuc(k, j, i)))
                           : f == 1 ? dt * (0.5 * (M.nuc(k, j - 1, i) + M.nuc(k, j, i)))
                                    : dt * M.kapc(k, j, i);
                }
                implicit_column(nz, g.dz.data(), g.dzc.data(), open.data(), dtk.data(), col.data(), cp.data(), dp.data());
                for (int k = 0; k < nz; ++k) (*fld[f])(k, j, i) = col[k];
            }
        }
    }
    // 5. barotropic forcing
    A3 GU, GV, etab, Ub, Vb;
    GU.init(nx, ny, 1); GV.init(nx, ny, 1); etab.init(nx, ny, 1); Ub.init(nx, ny, 1); Vb.init(nx, ny, 1);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            double su = 0.0, sv = 0.0;
            for (int k = 0; k < nz; ++k) {
                su += g.dz[k] * g.mu(k, j, i) * Ghu(k, j, i);
                sv += g.dz[k] * g.mv(k, j, i) * Ghv(k, j, i);
            }
            GU(0, j, i) = su; GV(0, j, i) = sv;
        }
    // 6. sub-cycle from (eta^n, U^n, V^n) with running weighted averages
    fill_halo(M.eta, g.px, g.py); fill_halo(M.U, g.px, g.py); fill_halo(M.V, g.px, g.py);
    for (int m = 1; m <= M.d.substeps; ++m) {
        barotropic_substep(M, M.dtau, &GU, &GV);
        const double a = M.a_w[m - 1], b = M.b_w[m - 1];
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                etab(0, j, i) += a * M.eta(0, j, i);
                Ub(0, j, i) += b * M.U(0, j, i);
                Vb(0, j, i) += b * M.V(0, j, i);
            }
    }
    // 7. the filtered values become the new barotropic state
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            M.eta(0, j, i) = etab(0, j, i); M.U(0, j, i) = Ub(0, j, i); M.V(0, j, i) = Vb(0, j, i);
        }
    // 8. barotropic correction of the baroclinic velocities
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            double su = 0.0, sv = 0.0;
            for (int k = 0; k < nz; ++k) { su += g.dz[k] * M.u(k, j, i); sv += g.dz[k] * M.v(k, j, i); }
            const double cu = M.Hu(0, j, i) > 0.0 ? (M.U(0, j, i) - su) / M.Hu(0, j, i) : 0.0;
            const double cv = M.Hv(0, j, i) > 0.0 ? (M.V(0, j, i) - sv) / M.Hv(0, j, i) : 0.0;
            for (int k = 0; k < nz; ++k) {
                M.u(k, j, i) = g.mu(k, j, i) * (M.u(k, j, i) + cu);
                M.v(k, j, i) = g.mv(k, j, i) * (M.v(k, j, i) + cv);
            }
        }
    // 9. G^- <- G^n
    M.Gu1.a = M.Gu.a; M.Gv1.a = M.Gv.a; M.GT1.a = M.GT.a; M.GS1.a = M.GS.a;
    M.have_history = true;
    // 10. diagnostics of the new state
    fill_state_halos(M);
    compute_w(M);
    compute_p(M);
}

template <class T>
void copy_in(A3& f, const T* src, int nl) {
    for (int k = 0; k < nl; ++k)
        for (int j = 0; j < f.ny; ++j)
            for (int i = 0; i < f.nx; ++i) f(k, j, i) = src[((size_t)k * f.ny + j) * f.nx + i];
}
void copy_out(const A3& f, double* dst, int nl) {
    for (int k = 0; k < nl; ++k)
        for (int j = 0; j < f.ny; ++j)
            for (int i = 0; i < f.nx; ++i) dst[((size_t)k * f.ny + j) * f.nx + i] = f(k, j, i);
}

}  // namespace

// ===============================================================================================
extern "C" {

const char* ocn_ref_last_error(void) { return g_err.c_str(); }

int ocn_ref_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void ocn_ref_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int ocn_ref_grid_create(const ocn_ref_grid_desc* d, const double* z_faces, const double* depth,
                        ocn_ref_grid** out) {
    if (!d || !z_faces || !depth || !out) return fail("null argument");
    if (d->nx < HALO || d->ny < HALO || d->nz < 2) return fail("grid too small (nx, ny >= 3, nz >= 2)");
    if (d->kind != 0 && d->kind != 1) return fail("kind must be 0 or 1");
    if (d->kind == 1 && d->periodic_y) return fail("lat-lon grid cannot be periodic in y");
    ocn_ref_grid* g = new ocn_ref_grid();
    g->d = *d; g->nx = d->nx; g->ny = d->ny; g->nz = d->nz; g->px = d->periodic_x != 0; g->py = d->periodic_y != 0;
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    // §3.1 vertical grid
    g->zf.assign(z_faces, z_faces + nz + 1);
    for (int k = 0; k < nz; ++k)
        if (!(g->zf[k + 1] > g->zf[k])) { delete g; return fail("z_faces must increase"); }
    g->dz.resize(nz); g->zc.resize(nz); g->dzc.assign(nz, 0.0);
    for (int k = 0; k < nz; ++k) { g->dz[k] = g->zf[k + 1] - g->zf[k]; g->zc[k] = 0.5 * (g->zf[k] + g->zf[k + 1]); }
    for (int k = 1; k < nz; ++k) g->dzc[k] = g->zc[k] - g->zc[k - 1];
    // §3.2 horizontal metrics, rows j = -HALO .. ny+HALO
    const int nr = ny + 2 * HALO + 1;
    g->dxC_.resize(nr); g->dxF_.resize(nr); g->AzC_.resize(nr); g->AzF_.resize(nr); g->fF_.resize(nr);
    if (d->kind == 1) {
        const double rad = M_PI / 180.0, a = d->radius;
        const double dlam = d->dx * rad, dphi = d->dy * rad;
        g->dy = a * dphi;
        for (int r = 0; r < nr; ++r) {
            const int j = r - HALO;
            const double pf = (d->y0 + j * d->dy) * rad, pc = pf + 0.5 * dphi;
            g->dxC_[r] = a * std::cos(pc) * dlam;
            g->dxF_[r] = a * std::cos(pf) * dlam;
            g->AzC_[r] = a * a * dlam * (std::sin(pf + dphi) - std::sin(pf));
            g->AzF_[r] = a * a * dlam * (std::sin(pc) - std::sin(pc - dphi));
            g->fF_[r] = 2.0 * d->rotation_rate * std::sin(pf);
        }
    } else {
        g->dy = d->dy;
        const double ymid = d->y0 + 0.5 * ny * d->dy;
        for (int r = 0; r < nr; ++r) {
            const int j = r - HALO;
            g->dxC_[r] = d->dx; g->dxF_[r] = d->dx;
            g->AzC_[r] = d->dx * d->dy; g->AzF_[r] = d->dx * d->dy;
            g->fF_[r] = d->f0 + d->beta * ((d->y0 + j * d->dy) - ymid);
        }
    }
    // §3.3 wet mask by brute force: full cells, centre test, columns with < 2 wet cells are land
    g->wet.init(nx, ny, nz);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const double h = depth[(size_t)j * nx + i];
            int cnt = 0;
            for (int k = 0; k < nz; ++k) cnt += (h > 0.0 && g->zc[k] > -h) ? 1 : 0;
            for (int k = 0; k < nz; ++k) g->wet(k, j, i) = (cnt >= 2 && h > 0.0 && g->zc[k] > -h) ? 1 : 0;
        }
    fill_halo(g->wet, g->px, g->py);
    *out = g;
    return 0;
}
int ocn_ref_grid_destroy(ocn_ref_grid* g) { delete g; return 0; }

int ocn_ref_model_create(const ocn_ref_grid* g, const ocn_ref_model_desc* d, ocn_ref_model** out) {
    if (!g || !d || !out) return fail("null argument");
    if (d->substeps < 1 || !(d->dt > 0)) return fail("bad dt / substeps");
    if (d->closure != 0 && d->closure != 1) return fail("closure must be 0 or 1");
    if (!(d->nu4_h >= 0 && d->kappa4_h >= 0)) return fail("nu4_h, kappa4_h must be >= 0");
    if (d->eos != 0 && d->eos != 1) return fail("eos must be 0 (linear) or 1 (nonlinear)");
    if (d->advection != 0 && d->advection != 1) return fail("advection must be 0 (WENO-JS) or 1 (WENO-Z)");
    if (d->closure == 1 && !(d->ri_n2c > 0 && d->ri_s2min > 0 && d->ri_c >= 0 && d->ri_nu0 >= 0 && d->ri_kconv >= 0))
        return fail("bad Ri closure parameters");
    ocn_ref_model* M = new ocn_ref_model();
    M->g = g; M->d = *d; M->d.filter_weights = nullptr; M->d.filter_weights_uv = nullptr;
    double ratio;
    if (d->filter_weights) {
        M->a_w.assign(d->filter_weights, d->filter_weights + d->substeps);
        double first = 0.0;
        for (int m = 1; m <= d->substeps; ++m) first += m * M->a_w[m - 1];
        ratio = 1.0 / first;
    } else {
        filter_weights(d->substeps, M->a_w, ratio);
    }
    M->dtau = d->dt * ratio;
    M->b_w = M->a_w;
    if (d->filter_weights_uv) M->b_w.assign(d->filter_weights_uv, d->filter_weights_uv + d->substeps);
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    for (A3* f : {&M->u, &M->v, &M->T, &M->S, &M->p, &M->Gu, &M->Gv, &M->GT, &M->GS,
                  &M->Gu1, &M->Gv1, &M->GT1, &M->GS1}) f->init(nx, ny, nz);
    M->w.init(nx, ny, nz + 1);
    if (d->closure == 1) { M->nuc.init(nx, ny, nz); M->kapc.init(nx, ny, nz); }
    for (A3* f : {&M->eta, &M->U, &M->V, &M->taux, &M->tauy, &M->Hu, &M->Hv, &M->qT, &M->qS, &M->rT, &M->rS}) f->init(nx, ny, 1);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            double hu = 0.0, hv = 0.0;
            for (int k = 0; k < nz; ++k) { hu += g->dz[k] * g->mu(k, j, i); hv += g->dz[k] * g->mv(k, j, i); }
            M->Hu(0, j, i) = hu; M->Hv(0, j, i) = hv;
        }
    fill_halo(M->Hu, g->px, g->py); fill_halo(M->Hv, g->px, g->py);
    compute_w(*M); compute_p(*M);
    *out = M;
    return 0;
}
int ocn_ref_model_destroy(ocn_ref_model* M) { delete M; return 0; }

int ocn_ref_set_fields(ocn_ref_model* M, const ocn_ref_fields* f) {
    if (!M || !f) return fail("null argument");
    const ocn_ref_grid& g = *M->g;
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    if (f->u) copy_in(M->u, f->u, nz);
    if (f->v) copy_in(M->v, f->v, nz);
    if (f->T) copy_in(M->T, f->T, nz);
    if (f->S) copy_in(M->S, f->S, nz);
    if (f->eta) copy_in(M->eta, f->eta, 1);
    if (f->tau_x) copy_in(M->taux, f->tau_x, 1);
    if (f->tau_y) copy_in(M->tauy, f->tau_y, 1);
    if (f->flux_T) copy_in(M->qT, f->flux_T, 1);
    if (f->flux_S) copy_in(M->qS, f->flux_S, 1);
    if (f->restore_T) copy_in(M->rT, f->restore_T, 1);
    if (f->restore_S) copy_in(M->rS, f->restore_S, 1);
    // forcing-only update (tau, fluxes, restoring targets): the state and the AB2 history stay (per-step forcing, as
    // include/ocn.h states for ocn_set_fields)
    if (!(f->u || f->v || f->T || f->S || f->eta)) return 0;
    // masks: closed faces carry no flow, land cells hold 0 (§3.3)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                M->u(k, j, i) *= g.mu(k, j, i); M->v(k, j, i) *= g.mv(k, j, i);
                M->T(k, j, i) *= g.wet(k, j, i); M->S(k, j, i) *= g.wet(k, j, i);
            }
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            M->eta(0, j, i) *= g.wet(nz - 1, j, i);
            double su = 0.0, sv = 0.0;
            for (int k = 0; k < nz; ++k) { su += g.dz[k] * M->u(k, j, i); sv += g.dz[k] * M->v(k, j, i); }
            M->U(0, j, i) = su; M->V(0, j, i) = sv;
        }
    M->have_history = false;
    fill_state_halos(*M);
    compute_w(*M); compute_p(*M);
    return 0;
}

int ocn_ref_time_step(ocn_ref_model* M, int n) {
    if (!M || n < 0) return fail("bad argument");
    for (int s = 0; s < n; ++s) time_step(*M);
    return 0;
}

int ocn_ref_get_fields(ocn_ref_model* M, ocn_ref_fields* f) {
    if (!M || !f) return fail("null argument");
    const int nz = M->g->nz;
    if (f->u) copy_out(M->u, f->u, nz);
    if (f->v) copy_out(M->v, f->v, nz);
    if (f->T) copy_out(M->T, f->T, nz);
    if (f->S) copy_out(M->S, f->S, nz);
    if (f->w) copy_out(M->w, f->w, nz + 1);
    if (f->eta) copy_out(M->eta, f->eta, 1);
    if (f->tau_x) copy_out(M->taux, f->tau_x, 1);
    if (f->tau_y) copy_out(M->tauy, f->tau_y, 1);
    return 0;
}

int ocn_ref_get_masks(const ocn_ref_grid* g, unsigned char* wet, unsigned char* ox, unsigned char* oy,
                      unsigned char* oz, unsigned char* ozu, unsigned char* ozv) {
    if (!g) return fail("null argument");
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    for (int k = 0; k <= nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const size_t n = ((size_t)k * ny + j) * nx + i;
                if (oz) oz[n] = (unsigned char)g->order_z(k, j, i);
                if (k == nz) continue;
                if (wet) wet[n] = g->wet(k, j, i);
                if (ox) ox[n] = (unsigned char)g->order_x(k, j, i);
                if (oy) oy[n] = (unsigned char)g->order_y(k, j, i);
                if (ozu) ozu[n] = (unsigned char)g->order_zeta_u(k, j, i);
                if (ozv) ozv[n] = (unsigned char)g->order_zeta_v(k, j, i);
            }
    return 0;
}

int ocn_ref_get_metrics(const ocn_ref_grid* g, double* dxC, double* dxF, double* AzC, double* AzF,
                        double* fF, double* dy) {
    if (!g) return fail("null argument");
    for (int j = 0; j < g->ny; ++j) {
        if (dxC) dxC[j] = g->dxC(j);
        if (dxF) dxF[j] = g->dxF(j);
        if (AzC) AzC[j] = g->AzC(j);
        if (AzF) AzF[j] = g->AzF(j);
        if (fF) fF[j] = g->fF(j);
    }
    if (dy) *dy = g->dy;
    return 0;
}

double ocn_ref_weno(const double c[6], int order, double vel) { return weno(c, order, vel); }
double ocn_ref_weno_scheme(const double c[6], int order, double vel, int scheme) { return weno(c, order, vel, scheme); }

int ocn_ref_implicit_column(int nz, const double* z_faces, const unsigned char* open, double dtk, double* phi) {
    if (nz < 2 || !z_faces || !open || !phi) return fail("bad argument");
    std::vector<double> dz(nz), zc(nz), dzc(nz, 0.0), cp(nz), dp(nz);
    for (int k = 0; k < nz; ++k) { dz[k] = z_faces[k + 1] - z_faces[k]; zc[k] = 0.5 * (z_faces[k] + z_faces[k + 1]); }
    for (int k = 1; k < nz; ++k) dzc[k] = zc[k] - zc[k - 1];
    const std::vector<double> dtkv(nz + 1, dtk);
    implicit_column(nz, dz.data(), dzc.data(), open, dtkv.data(), phi, cp.data(), dp.data());
    return 0;
}

int ocn_ref_implicit_column_var(int nz, const double* z_faces, const unsigned char* open, const double* dtk, double* phi) {
    if (nz < 2 || !z_faces || !open || !dtk || !phi) return fail("bad argument");
    std::vector<double> dz(nz), zc(nz), dzc(nz, 0.0), cp(nz), dp(nz);
    for (int k = 0; k < nz; ++k) { dz[k] = z_faces[k + 1] - z_faces[k]; zc[k] = 0.5 * (z_faces[k] + z_faces[k + 1]); }
    for (int k = 1; k < nz; ++k) dzc[k] = zc[k] - zc[k - 1];
    implicit_column(nz, dz.data(), dzc.data(), open, dtk, phi, cp.data(), dp.data());
    return 0;
}

int ocn_ref_get_mixing(ocn_ref_model* M, double* nu, double* kappa) {
    if (!M) return fail("null argument");
    if (M->d.closure != 1) return fail("model has no Ri closure (closure = 0)");
    compute_mixing(*M);
    if (nu) copy_out(M->nuc, nu, M->g->nz);
    if (kappa) copy_out(M->kapc, kappa, M->g->nz);
    return 0;
}

int ocn_ref_filter_weights(int M, double* a, double* ratio) {
    if (M < 1 || !a || !ratio) return fail("bad argument");
    std::vector<double> w;
    filter_weights(M, w, *ratio);
    std::memcpy(a, w.data(), sizeof(double) * M);
    return 0;
}

int ocn_ref_get_tendencies(ocn_ref_model* M, double* Gu, double* Gv, double* GT, double* GS) {
    if (!M) return fail("null argument");
    const ocn_ref_grid& g = *M->g;
    A3 a, b, c, d;
    a.init(g.nx, g.ny, g.nz); b.init(g.nx, g.ny, g.nz); c.init(g.nx, g.ny, g.nz); d.init(g.nx, g.ny, g.nz);
    compute_tendencies(*M, a, b, c, d);
    if (Gu) copy_out(a, Gu, g.nz);
    if (Gv) copy_out(b, Gv, g.nz);
    if (GT) copy_out(c, GT, g.nz);
    if (GS) copy_out(d, GS, g.nz);
    return 0;
}

int ocn_ref_get_diagnostics(ocn_ref_model* M, double* p, double* U, double* V) {
    if (!M) return fail("null argument");
    if (p) copy_out(M->p, p, M->g->nz);
    if (U) copy_out(M->U, U, 1);
    if (V) copy_out(M->V, V, 1);
    return 0;
}

int ocn_ref_get_momentum_diagnostics(ocn_ref_model* M, double* zeta, double* K, double* D) {
    if (!M) return fail("null argument");
    const ocn_ref_grid& g = *M->g;
    A3 gu, gv, z, ke, dv;
    gu.init(g.nx, g.ny, g.nz); gv.init(g.nx, g.ny, g.nz); z.init(g.nx, g.ny, g.nz); ke.init(g.nx, g.ny, g.nz); dv.init(g.nx, g.ny, g.nz);
    momentum_tendency(*M, gu, gv, z, ke, dv);
    if (zeta) copy_out(z, zeta, g.nz);
    if (K) copy_out(ke, K, g.nz);
    if (D) copy_out(dv, D, g.nz);
    return 0;
}

int ocn_ref_barotropic_raw(ocn_ref_model* M, int m, double dtau) {
    if (!M || m < 0) return fail("bad argument");
    const ocn_ref_grid& g = *M->g;
    fill_halo(M->eta, g.px, g.py); fill_halo(M->U, g.px, g.py); fill_halo(M->V, g.px, g.py);
    for (int s = 0; s < m; ++s) barotropic_substep(*M, dtau, nullptr, nullptr);
    return 0;
}

}  // extern "C"
