"""Mutation check of the oracle's pins: every one-token mistake below — a metric factor of the wrong row or kind, a dropped
mask, a wrong sign — is applied to a scratch copy of oracle/ocn_ref.cpp, built on its own, and the pin tests are run
against it in a subprocess (oracle/__init__.py loads the copy when OCN_REF_MUTANT_SRC is set).  Each mutant must make
at least one pin FAIL; the unmodified source must pass.  This is what "pinned" means in DESIGN.md §5: a plausible mistake
anywhere in the lat-lon metric factors or bathymetry masks of momentum_tendency, tracer_tendency, compute_w and
barotropic_substep — and of the biharmonic operators (B1-B7) — does not survive `-m "not gpu"`.  (The list is the one the round-1 review injected, plus a few more.
Not listed because they are EQUIVALENT mutants: dropping the open-face masks of U, V in barotropic_substep — a closed
face has H = 0, G^U = 0 and starts from U = 0, so it stays 0 with or without the mask.)
"""
import os

import pytest
import shutil
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "ocn_ref.cpp")
# pins that the mutants are run against (fast ones first; -x stops at the first failure)
PINS = ["tests/test_oracle_latlon.py", "tests/test_oracle_handcalc.py", "tests/test_oracle_variants.py"]

# (name, exact text in ocn_ref.cpp (must occur once), replacement)
MUTANTS = [
    ("M1 zeta: dxC(j-1) u[j-1] -> dxC(j) u[j-1]",
     "- (g.dxC(j) * u(k, j, i) - g.dxC(j - 1) * u(k, j - 1, i))) / g.AzF(j);",
     "- (g.dxC(j) * u(k, j, i) - g.dxC(j) * u(k, j - 1, i))) / g.AzF(j);"),
    ("M2 F_y: v dxF(j) -> v dxC(j)",
     "Fy(k, j, i) = vv * g.dxF(j) * g.dz[k] * cf",
     "Fy(k, j, i) = vv * g.dxC(j) * g.dz[k] * cf"),
    ("M3 W_v: AzC(j-1) w[j-1] -> AzC(j) w[j-1]",
     "const double Wlo = 0.5 * (g.AzC(j - 1) * w(k, j - 1, i) + g.AzC(j) * w(k, j, i));",
     "const double Wlo = 0.5 * (g.AzC(j) * w(k, j - 1, i) + g.AzC(j) * w(k, j, i));"),
    ("M4 C_u: fF(j+1) -> fF(j) in the northern half",
     "+ g.fF(j + 1) * 0.5 * g.dxF(j + 1) * (v(k, j + 1, i - 1) + v(k, j + 1, i))) / g.dxC(j);",
     "+ g.fF(j) * 0.5 * g.dxF(j + 1) * (v(k, j + 1, i - 1) + v(k, j + 1, i))) / g.dxC(j);"),
    ("M5 vhat: dxF(j+1) -> dxF(j)",
     "+ g.dxF(j + 1) * (v(k, j + 1, i - 1) + v(k, j + 1, i))) / g.dxC(j);\n                    const double zs[6] = {zeta(k, j - 2, i)",
     "+ g.dxF(j) * (v(k, j + 1, i - 1) + v(k, j + 1, i))) / g.dxC(j);\n                    const double zs[6] = {zeta(k, j - 2, i)"),
    ("M6 compute_w: dxF(j+1) v[j+1] -> dxF(j) v[j+1]",
     "+ g.dxF(j + 1) * M.v(k, j + 1, i) - g.dxF(j) * M.v(k, j, i)) / g.AzC(j);\n                M.w(k + 1, j, i)",
     "+ g.dxF(j) * M.v(k, j + 1, i) - g.dxF(j) * M.v(k, j, i)) / g.AzC(j);\n                M.w(k + 1, j, i)"),
    ("M7 V_v: (zeta[i+1]-zeta[i]) / dxF(j) -> / dxC(j)",
     "+ (zeta(k, j, i + 1) - zeta(k, j, i)) / g.dxF(j));",
     "+ (zeta(k, j, i + 1) - zeta(k, j, i)) / g.dxC(j));"),
    ("M8 A_v: / (AzF(j) dz) -> / (AzC(j) dz)",
     "const double Av = 0.5 * (Whi * dhi + Wlo * dlo) / (g.AzF(j) * g.dz[k]);",
     "const double Av = 0.5 * (Whi * dhi + Wlo * dlo) / (g.AzC(j) * g.dz[k]);"),
    ("M9 vertical advection of u: mask mu[k-1] dropped below",
     "const double dlo = (k >= 1) ? (u(k, j, i) - u(k - 1, j, i)) * g.mu(k, j, i) * g.mu(k - 1, j, i) : 0.0;",
     "const double dlo = (k >= 1) ? (u(k, j, i) - u(k - 1, j, i)) * g.mu(k, j, i) : 0.0;"),
    ("M10 vertical advection of v: mask mv[k-1] dropped below",
     "const double dlo = (k >= 1) ? (v(k, j, i) - v(k - 1, j, i)) * g.mv(k, j, i) * g.mv(k - 1, j, i) : 0.0;",
     "const double dlo = (k >= 1) ? (v(k, j, i) - v(k - 1, j, i)) * g.mv(k, j, i) : 0.0;"),
    ("M13 barotropic eta: dxF(j+1) V[j+1] -> dxF(j) V[j+1]",
     "+ g.dxF(j + 1) * M.V(0, j + 1, i) - g.dxF(j) * M.V(0, j, i)) / g.AzC(j);",
     "+ g.dxF(j) * M.V(0, j + 1, i) - g.dxF(j) * M.V(0, j, i)) / g.AzC(j);"),
    ("M14 barotropic U: d(eta) / dxC(j) -> / dxF(j)",
     "(M.eta(0, j, i) - M.eta(0, j, i - 1)) / g.dxC(j) + gu))",
     "(M.eta(0, j, i) - M.eta(0, j, i - 1)) / g.dxF(j) + gu))"),
    ("M15 grad p in G_u: / dxC(j) -> / dxF(j)",
     "const double dP = (p(k, j, i) - p(k, j, i - 1)) / g.dxC(j);",
     "const double dP = (p(k, j, i) - p(k, j, i - 1)) / g.dxF(j);"),
    ("M16 tracer G: / (AzC(j) dz) -> / (AzF(j) dz)",
     "G(k, j, i) = -(double)g.wet(k, j, i) * div / (g.AzC(j) * g.dz[k]);",
     "G(k, j, i) = -(double)g.wet(k, j, i) * div / (g.AzF(j) * g.dz[k]);"),
    ("M17 zeta: / AzF(j) -> / AzC(j)",
     "g.dxC(j - 1) * u(k, j - 1, i))) / g.AzF(j);",
     "g.dxC(j - 1) * u(k, j - 1, i))) / g.AzC(j);"),
    ("M18 D in the momentum tendency: dxF(j) v[j] -> dxF(j+1) v[j]",
     "+ g.dxF(j + 1) * v(k, j + 1, i) - g.dxF(j) * v(k, j, i)) / g.AzC(j);",
     "+ g.dxF(j + 1) * v(k, j + 1, i) - g.dxF(j + 1) * v(k, j, i)) / g.AzC(j);"),
    ("M19 dK/dx in G_u: / dxC(j) -> / dxF(j)",
     "const double dK = (Ke(k, j, i) - Ke(k, j, i - 1)) / g.dxC(j);",
     "const double dK = (Ke(k, j, i) - Ke(k, j, i - 1)) / g.dxF(j);"),
    ("M20 C_v: fF(j) -> fF(j+1)",
     "const double Cv = g.fF(j) * uhat;",
     "const double Cv = g.fF(j + 1) * uhat;"),
    ("M21 F_x diffusion: / dxC(j) -> / dxF(j)",
     "- kh * g.dy * g.dz[k] * (c(k, j, i) - c(k, j, i - 1)) / g.dxC(j) * g.mu(k, j, i);",
     "- kh * g.dy * g.dz[k] * (c(k, j, i) - c(k, j, i - 1)) / g.dxF(j) * g.mu(k, j, i);"),
    ("M22 F_z: AzC(j) -> AzF(j)",
     "Fz(k, j, i) = ww * g.AzC(j) * cf * g.mw(k, j, i);",
     "Fz(k, j, i) = ww * g.AzF(j) * cf * g.mw(k, j, i);"),
    ("M23 V_u: (D[i]-D[i-1]) / dxC(j) -> / dxF(j)",
     "const double Vu = nu * ((Dv(k, j, i) - Dv(k, j, i - 1)) / g.dxC(j)",
     "const double Vu = nu * ((Dv(k, j, i) - Dv(k, j, i - 1)) / g.dxF(j)"),
    ("M25 metric: AzF from phi_c +- wrong row",
     "g->AzF_[r] = a * a * dlam * (std::sin(pc) - std::sin(pc - dphi));",
     "g->AzF_[r] = a * a * dlam * (std::sin(pc + dphi) - std::sin(pc));"),
    ("M26 metric: fF at the cell centre instead of the corner",
     "g->fF_[r] = 2.0 * d->rotation_rate * std::sin(pf);",
     "g->fF_[r] = 2.0 * d->rotation_rate * std::sin(pc);"),
    ("B1 biharmonic La: (Da[i]-Da[i-1]) / dxC(j) -> / dxF(j)",
     "La(k, j, i) = g.mu(k, j, i) * ((Da(k, j, i) - Da(k, j, i - 1)) / g.dxC(j)",
     "La(k, j, i) = g.mu(k, j, i) * ((Da(k, j, i) - Da(k, j, i - 1)) / g.dxF(j)"),
    ("B2 biharmonic Za: dxC(j-1) a[j-1] -> dxC(j) a[j-1]",
     "- (g.dxC(j) * a(k, j, i) - g.dxC(j - 1) * a(k, j - 1, i))) / g.AzF(j);",
     "- (g.dxC(j) * a(k, j, i) - g.dxC(j) * a(k, j - 1, i))) / g.AzF(j);"),
    ("B3 biharmonic Lb: (Za[i+1]-Za[i]) / dxF(j) -> / dxC(j)",
     "+ (Za(k, j, i + 1) - Za(k, j, i)) / g.dxF(j));",
     "+ (Za(k, j, i + 1) - Za(k, j, i)) / g.dxC(j));"),
    ("B4 biharmonic Da: / AzC(j) -> / AzF(j)",
     "g.dxF(j + 1) * b(k, j + 1, i) - g.dxF(j) * b(k, j, i)) / g.AzC(j);",
     "g.dxF(j + 1) * b(k, j + 1, i) - g.dxF(j) * b(k, j, i)) / g.AzF(j);"),
    ("B5 scalar Laplacian: northern flux with dxF(j) instead of dxF(j+1)",
     "const double fyn = g.dxF(j + 1) * (c(k, j + 1, i) - c(k, j, i)) / g.dy * g.mv(k, j + 1, i);",
     "const double fyn = g.dxF(j) * (c(k, j + 1, i) - c(k, j, i)) / g.dy * g.mv(k, j + 1, i);"),
    ("B6 scalar Laplacian: eastern flux not masked",
     "const double fxe = g.dy * (c(k, j, i + 1) - c(k, j, i)) / g.dxC(j) * g.mu(k, j, i + 1);",
     "const double fxe = g.dy * (c(k, j, i + 1) - c(k, j, i)) / g.dxC(j);"),
    ("B7 biharmonic: sign of the tracer term",
     "(*G[f])(k, j, i) += -(M.d.kappa4_h * m1(k, j, i));",
     "(*G[f])(k, j, i) += (M.d.kappa4_h * m1(k, j, i));"),
    ("control: 1/4 -> 1/2 in K",
     "Ke(k, j, i) = 0.25 * (u(k, j, i) * u(k, j, i) + u(k, j, i + 1) * u(k, j, i + 1))",
     "Ke(k, j, i) = 0.5 * (u(k, j, i) * u(k, j, i) + u(k, j, i + 1) * u(k, j, i + 1))"),
]


# the same check for the options beyond the north_star path: vertical mixing closure, nonlinear equation of
# state (§3.16), bottom drag (§3.14), surface tracer forcing (§3.13), the implicit vertical solve (§3.8 step 4)
PINS_OPTIONS = ["tests/test_oracle_closure.py", "tests/test_oracle_forcing.py", "tests/test_oracle_variants.py",
                "tests/test_oracle_handcalc.py", "tests/test_oracle_physics.py"]
MUTANTS_OPTIONS = [
    ("C1 closure: nu with f^3 instead of f^2",
     "M.nuc(k, j, i) = d.nu_z + d.ri_nu0 * f * f + conv;",
     "M.nuc(k, j, i) = d.nu_z + d.ri_nu0 * f * f * f + conv;"),
    ("C2 closure: Ri from N2 without the clip at 0",
     "const double Ri = std::max(N2, 0.0) / (S2 + d.ri_s2min);",
     "const double Ri = N2 / (S2 + d.ri_s2min);"),
    ("C3 closure: convective ramp on +N2",
     "const double conv = d.ri_kconv * std::min(1.0, std::max(-N2, 0.0) / d.ri_n2c);",
     "const double conv = d.ri_kconv * std::min(1.0, std::max(N2, 0.0) / d.ri_n2c);"),
    ("C4 closure: kappa without the convective term",
     "M.kapc(k, j, i) = d.kappa_z + d.ri_nu0 * f * f * f + conv;",
     "M.kapc(k, j, i) = d.kappa_z + d.ri_nu0 * f * f * f;"),
    ("C5 closure: shear of the east face taken at i instead of i + 1",
     "due = M.u(k, j, i + 1) - M.u(k - 1, j, i + 1);",
     "due = M.u(k, j, i) - M.u(k - 1, j, i + 1);"),
    ("C6 closure: S2 divided by dzc once",
     "+ 0.5 * (dvs * dvs + dvn * dvn)) / (g.dzc[k] * g.dzc[k]);",
     "+ 0.5 * (dvs * dvs + dvn * dvn)) / (g.dzc[k]);"),
    ("E1 equation of state: thermobaric factor 1 + gamma z",
     "(1.0 - M.d.eos_gamma * M.g->zc[k]) * dT",
     "(1.0 + M.d.eos_gamma * M.g->zc[k]) * dT"),
    ("E2 equation of state: cabbeling without the 1/2",
     "+ 0.5 * M.d.eos_alpha2 * dT * dT",
     "+ M.d.eos_alpha2 * dT * dT"),
    ("D1 bottom drag on u: speed without the transverse velocity",
     "std::sqrt(u(k, j, i) * u(k, j, i) + vhat * vhat))",
     "std::sqrt(u(k, j, i) * u(k, j, i)))"),
    ("D2 bottom drag on u: every level instead of the lowest open one",
     "const bool bot = m && (k == 0 || !g.mu(k - 1, j, i));",
     "const bool bot = m;"),
    ("F1 surface forcing: restoring with the wrong sign",
     "(surf(0, j, i) + gamma * (target(0, j, i) - c(k, j, i))) / g.dz[k];",
     "(surf(0, j, i) - gamma * (target(0, j, i) - c(k, j, i))) / g.dz[k];"),
    ("T1 implicit solve: upper coefficient with dzc[k] instead of dzc[k + 1]",
     "const double sp = (k + 1 <= nz - 1 && open[k + 1]) ? dtk[k + 1] / (dz[k] * dzc[k + 1]) : 0.0;",
     "const double sp = (k + 1 <= nz - 1 && open[k + 1]) ? dtk[k + 1] / (dz[k] * dzc[k]) : 0.0;"),
    ("T2 implicit solve: back-substitution with the wrong sign",
     "phi[k] = dp[k] - cp[k] * phi[k + 1];",
     "phi[k] = dp[k] + cp[k] * phi[k + 1];"),
]


# and for the time stepping itself: quasi-AB2, predictor, barotropic forcing and filter, correction, history
PINS_STEP = ["tests/test_oracle_handcalc.py", "tests/test_oracle_physics.py", "tests/test_oracle_units.py",
             "tests/test_oracle_variants.py", "tests/test_oracle_closure.py", "tests/test_oracle_forcing.py"]
MUTANTS_STEP = [
    ("S1 quasi-AB2: c0 = 3/2 - chi",
     "const double c0 = M.have_history ? 1.5 + M.d.chi : 1.0;",
     "const double c0 = M.have_history ? 1.5 - M.d.chi : 1.0;"),
    ("S2 quasi-AB2: c1 without chi",
     "const double c1 = M.have_history ? 0.5 + M.d.chi : 0.0;",
     "const double c1 = M.have_history ? 0.5 : 0.0;"),
    ("S3 Euler start with c0 = 3/2",
     "const double c0 = M.have_history ? 1.5 + M.d.chi : 1.0;",
     "const double c0 = M.have_history ? 1.5 + M.d.chi : 1.5;"),
    ("S4 predictor from G^n instead of the AB2 combination",
     "col[k] = ((*fld[f])(k, j, i) + dt * Gh) * m;",
     "col[k] = ((*fld[f])(k, j, i) + dt * (*Gn[f])(k, j, i)) * m;"),
    ("S5 barotropic forcing: sum of G without the layer thickness",
     "su += g.dz[k] * g.mu(k, j, i) * Ghu(k, j, i);",
     "su += g.mu(k, j, i) * Ghu(k, j, i);"),
    ("S6 filter: transports averaged with the eta weights",
     "Ub(0, j, i) += b * M.U(0, j, i);",
     "Ub(0, j, i) += a * M.U(0, j, i);"),
    ("S7 filter: eta averaged with the transport weights",
     "etab(0, j, i) += a * M.eta(0, j, i);",
     "etab(0, j, i) += b * M.eta(0, j, i);"),
    ("S8 correction of u divided by Hv",
     "const double cu = M.Hu(0, j, i) > 0.0 ? (M.U(0, j, i) - su) / M.Hu(0, j, i) : 0.0;",
     "const double cu = M.Hu(0, j, i) > 0.0 ? (M.U(0, j, i) - su) / M.Hv(0, j, i) : 0.0;"),
    ("S9 closure: nu at the u face from columns i, i + 1",
     "dtk[k] = f == 0 ? dt * (0.5 * (M.nuc(k, j, i - 1) + M.nuc(k, j, i)))",
     "dtk[k] = f == 0 ? dt * (0.5 * (M.nuc(k, j, i) + M.nuc(k, j, i + 1)))"),
    ("S10 closure: nu at the v face from the column to the west",
     ": f == 1 ? dt * (0.5 * (M.nuc(k, j - 1, i) + M.nuc(k, j, i)))",
     ": f == 1 ? dt * (0.5 * (M.nuc(k, j, i - 1) + M.nuc(k, j, i)))"),
    ("S11 closure: tracers diffused with nu",
     ": dt * M.kapc(k, j, i);",
     ": dt * M.nuc(k, j, i);"),
    ("S12 history of S takes the tendency of T",
     "M.GS1.a = M.GS.a;",
     "M.GS1.a = M.GT.a;"),
    ("S13 barotropic eta with the wrong sign",
     "M.eta(0, j, i) -= dtau * (g.dy * (M.U(0, j, i + 1) - M.U(0, j, i))",
     "M.eta(0, j, i) += dtau * (g.dy * (M.U(0, j, i + 1) - M.U(0, j, i))"),
    ("S14 implicit solve of u: face open if the upper cell is",
     "open[k] = f == 0 ? (g.mu(k, j, i) && g.mu(k - 1, j, i))",
     "open[k] = f == 0 ? (g.mu(k, j, i))"),
    ("S15 sub-step length from the zeroth instead of the first moment of the weights",
     "for (int m = 1; m <= d->substeps; ++m) first += m * M->a_w[m - 1];",
     "for (int m = 1; m <= d->substeps; ++m) first += M->a_w[m - 1];"),
    ("S16 pressure: top half cell with the full thickness",
     "M.p(nz - 1, j, i) = -buoyancy(M, nz - 1, j, i) * (g.zf[nz] - g.zc[nz - 1]);",
     "M.p(nz - 1, j, i) = -buoyancy(M, nz - 1, j, i) * (g.zf[nz] - g.zf[nz - 1]);"),
    ("S17 pressure: trapezoid with the spacing of the wrong face",
     "- 0.5 * (buoyancy(M, k + 1, j, i) + buoyancy(M, k, j, i)) * g.dzc[k + 1];",
     "- 0.5 * (buoyancy(M, k + 1, j, i) + buoyancy(M, k, j, i)) * g.dzc[k];"),
    ("S18 vertical velocity integrated with the wrong sign",
     "M.w(k + 1, j, i) = M.w(k, j, i) - g.dz[k] * D;",
     "M.w(k + 1, j, i) = M.w(k, j, i) + g.dz[k] * D;"),
]


# signs, factors and stencil directions of the tendencies that are not metric rows (those are in MUTANTS)
PINS_TERMS = ["tests/test_oracle_handcalc.py", "tests/test_oracle_latlon.py", "tests/test_oracle_physics.py",
              "tests/test_oracle_units.py", "tests/test_oracle_forcing.py"]
MUTANTS_TERMS = [
    ("G1 u: vorticity flux with the wrong sign",
     "Gu(k, j, i) = m * (zt * vhat + Cu - dK - dP - Au + Vu + tau - drag);",
     "Gu(k, j, i) = m * (-zt * vhat + Cu - dK - dP - Au + Vu + tau - drag);"),
    ("G2 v: Coriolis with the wrong sign",
     "Gv(k, j, i) = m * (-zt * uhat - Cv - dK - dP - Av + Vv + tau - drag);",
     "Gv(k, j, i) = m * (-zt * uhat + Cv - dK - dP - Av + Vv + tau - drag);"),
    ("G3 u: viscous term with the wrong sign",
     "Gu(k, j, i) = m * (zt * vhat + Cu - dK - dP - Au + Vu + tau - drag);",
     "Gu(k, j, i) = m * (zt * vhat + Cu - dK - dP - Au - Vu + tau - drag);"),
    ("G4 v: vertical advection with the wrong sign",
     "Gv(k, j, i) = m * (-zt * uhat - Cv - dK - dP - Av + Vv + tau - drag);",
     "Gv(k, j, i) = m * (-zt * uhat - Cv - dK - dP + Av + Vv + tau - drag);"),
    ("G5 u: vorticity upwinded against the flow",
     "const double zt = weno(zs, g.order_zeta_u(k, j, i), vhat, M.d.advection);",
     "const double zt = weno(zs, g.order_zeta_u(k, j, i), -vhat, M.d.advection);"),
    ("G6 v: vorticity stencil shifted by one column",
     "const double zs[6] = {zeta(k, j, i - 2), zeta(k, j, i - 1), zeta(k, j, i),\n                                          zeta(k, j, i + 1), zeta(k, j, i + 2), zeta(k, j, i + 3)};",
     "const double zs[6] = {zeta(k, j, i - 3), zeta(k, j, i - 2), zeta(k, j, i - 1),\n                                          zeta(k, j, i), zeta(k, j, i + 1), zeta(k, j, i + 2)};"),
    ("G7 u: viscous vorticity term with the wrong sign inside V_u",
     "- (zeta(k, j + 1, i) - zeta(k, j, i)) / g.dy);\n                    const double tau = (k == nz - 1) ? M.taux",
     "+ (zeta(k, j + 1, i) - zeta(k, j, i)) / g.dy);\n                    const double tau = (k == nz - 1) ? M.taux"),
    ("G8 wind stress without the reference density",
     "const double tau = (k == nz - 1) ? M.taux(0, j, i) / (M.d.rho0 * g.dz[k]) : 0.0;",
     "const double tau = (k == nz - 1) ? M.taux(0, j, i) / (g.dz[k]) : 0.0;"),
    ("G9 u: upper half of the vertical advection uses the lower velocity difference",
     "const double Au = 0.5 * (Whi * dhi + Wlo * dlo) / (g.AzC(j) * g.dz[k]);",
     "const double Au = 0.5 * (Whi * dlo + Wlo * dlo) / (g.AzC(j) * g.dz[k]);"),
    ("G10 uhat from three of its four neighbours twice",
     "const double uhat = 0.25 * (u(k, j - 1, i) + u(k, j, i) + u(k, j - 1, i + 1) + u(k, j, i + 1));",
     "const double uhat = 0.25 * (u(k, j - 1, i) + u(k, j, i) + u(k, j, i + 1) + u(k, j, i + 1));"),
    ("R1 tracers: zonal flux upwinded against the flow",
     "const double cf = weno(cs, g.order_x(k, j, i), uu, M.d.advection);",
     "const double cf = weno(cs, g.order_x(k, j, i), -uu, M.d.advection);"),
    ("R2 tracers: horizontal diffusion with the wrong sign",
     "- kh * g.dxF(j) * g.dz[k] * (c(k, j, i) - c(k, j - 1, i)) / g.dy * g.mv(k, j, i);",
     "+ kh * g.dxF(j) * g.dz[k] * (c(k, j, i) - c(k, j - 1, i)) / g.dy * g.mv(k, j, i);"),
    ("R3 tracers: vertical stencil shifted by one level",
     "const int kk = k - 3 + m;",
     "const int kk = k - 2 + m;"),
    ("R4 tracers: divergence without the vertical flux below",
     "+ Fz(k + 1, j, i) - Fz(k, j, i);",
     "+ Fz(k + 1, j, i);"),
    ("R5 surface flux spread over the wrong thickness",
     "(surf(0, j, i) + gamma * (target(0, j, i) - c(k, j, i))) / g.dz[k];",
     "(surf(0, j, i) + gamma * (target(0, j, i) - c(k, j, i))) / g.dz[0];"),
    ("K1 divergence: zonal difference taken one cell to the west",
     "Dv(k, j, i) = (g.dy * (u(k, j, i + 1) - u(k, j, i))",
     "Dv(k, j, i) = (g.dy * (u(k, j, i) - u(k, j, i - 1))"),
    ("K2 kinetic energy without the meridional half",
     "+ 0.25 * (v(k, j, i) * v(k, j, i) + v(k, j + 1, i) * v(k, j + 1, i));",
     "+ 0.25 * (v(k, j, i) * v(k, j, i) + v(k, j, i) * v(k, j, i));"),
]


# the reconstruction itself, the default filter and the initial transports
PINS_WENO = ["tests/test_oracle_units.py", "tests/test_oracle_variants.py", "tests/test_oracle_handcalc.py", "tests/test_oracle_physics.py"]
MUTANTS_WENO = [
    ("W1 WENO5: first candidate with -5 instead of -7",
     "const double p0 = (2.0 * qm2 - 7.0 * qm1 + 11.0 * q0) / 6.0;",
     "const double p0 = (2.0 * qm2 - 5.0 * qm1 + 11.0 * q0) / 6.0;"),
    ("W2 WENO5: smoothness indicator with 13/10",
     "const double b1 = 13.0 / 12.0 * (qm1 - 2.0 * q0 + q1) * (qm1 - 2.0 * q0 + q1)",
     "const double b1 = 13.0 / 10.0 * (qm1 - 2.0 * q0 + q1) * (qm1 - 2.0 * q0 + q1)"),
    ("W3 WENO5: first-difference part of beta_2 with the wrong stencil",
     "+ 0.25 * (3.0 * q0 - 4.0 * q1 + q2) * (3.0 * q0 - 4.0 * q1 + q2);",
     "+ 0.25 * (q0 - 4.0 * q1 + 3.0 * q2) * (q0 - 4.0 * q1 + 3.0 * q2);"),
    ("W4 WENO5: linear weights 0.1 and 0.3 swapped",
     "const double a0 = 0.1 / ((eps + b0) * (eps + b0));",
     "const double a0 = 0.3 / ((eps + b0) * (eps + b0));"),
    ("W5 WENO5: weights with the first power of the indicator",
     "const double a1 = 0.6 / ((eps + b1) * (eps + b1));",
     "const double a1 = 0.6 / ((eps + b1));"),
    ("W6 WENO3: linear weights 1/3 and 2/3 swapped",
     "const double a1 = (2.0 / 3.0) / ((eps + b1) * (eps + b1));",
     "const double a1 = (1.0 / 3.0) / ((eps + b1) * (eps + b1));"),
    ("W7 WENO3: extrapolating candidate with 2 instead of 3",
     "const double p0 = (-qm1 + 3.0 * q0) / 2.0;",
     "const double p0 = (-qm1 + 2.0 * q0) / 2.0;"),
    ("W8 downwind stencil not mirrored",
     "else           { qm2 = c[5]; qm1 = c[4]; q0 = c[3]; q1 = c[2]; q2 = c[1]; }",
     "else           { qm2 = c[5]; qm1 = c[4]; q0 = c[3]; q1 = c[2]; q2 = c[0]; }"),
    ("W9 WENO-Z: tau from beta_0 and beta_1",
     "const double tau = std::fabs(b0 - b2);",
     "const double tau = std::fabs(b0 - b1);"),
    ("W10 eps of the weights",
     "const double eps = 1e-6;",
     "const double eps = 1e-2;"),
    ("P1 default filter: exponent q = 2",
     "a[m - 1] = s * s * (1.0 - s * s * s * s);",
     "a[m - 1] = s * s * (1.0 - s * s);"),
    ("P2 default filter: s = m / M",
     "const double s = (double)m / (double)(M + 1);",
     "const double s = (double)m / (double)(M);"),
    ("I1 initial transports without the layer thickness",
     "su += g.dz[k] * M->u(k, j, i); sv += g.dz[k] * M->v(k, j, i);",
     "su += M->u(k, j, i); sv += g.dz[k] * M->v(k, j, i);"),
]


def _run_pins(src_path, pins=None):
    env = dict(os.environ, OCN_REF_MUTANT_SRC=src_path, OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider"] + (pins or PINS), cwd=ROOT, env=env,
                       stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    return r.returncode, r.stdout[-3000:]


@pytest.mark.parametrize("group", ["options", "step", "terms", "weno"])
def test_every_mutant_of_the_options_and_of_the_time_stepping_is_caught(group):
    mutants, pins = {"options": (MUTANTS_OPTIONS, PINS_OPTIONS), "step": (MUTANTS_STEP, PINS_STEP), "terms": (MUTANTS_TERMS, PINS_TERMS),
                     "weno": (MUTANTS_WENO, PINS_WENO)}[group]
    text = open(SRC).read()
    tmp = tempfile.mkdtemp(prefix="ocn_mut_")
    try:
        jobs = []
        for n, (name, old, new) in enumerate(mutants):
            assert text.count(old) == 1, "mutation target not found exactly once (oracle source changed?): " + name
            path = os.path.join(tmp, "option_%02d.cpp" % n)
            with open(path, "w") as f:
                f.write(text.replace(old, new))
            jobs.append((name, path))
        with ThreadPoolExecutor(max_workers=max(2, (os.cpu_count() or 4) // 2)) as ex:
            res = list(ex.map(lambda j: _run_pins(j[1], pins), jobs))
        survivors = [name for (name, _), (rc, _) in zip(jobs, res) if rc == 0]
        assert not survivors, "mutants that survive every pin: %s" % survivors
        for (name, _), (rc, out) in zip(jobs, res):
            assert rc == 1 and "AssertionError" in out, (name, rc, out)
    finally:
        shutil.rmtree(tmp, ignore_errors=True)


def test_every_mutant_of_the_latlon_metrics_and_masks_is_caught():
    text = open(SRC).read()
    tmp = tempfile.mkdtemp(prefix="ocn_mut_")
    try:
        jobs = []
        for n, (name, old, new) in enumerate(MUTANTS):
            assert text.count(old) == 1, "mutation target not found exactly once (oracle source changed?): " + name
            path = os.path.join(tmp, "mutant_%02d.cpp" % n)
            with open(path, "w") as f:
                f.write(text.replace(old, new))
            jobs.append((name, path))
        clean = os.path.join(tmp, "clean.cpp")
        shutil.copy(SRC, clean)
        with ThreadPoolExecutor(max_workers=max(2, (os.cpu_count() or 4) // 2)) as ex:
            res = list(ex.map(lambda j: _run_pins(j[1]), jobs + [("clean", clean)]))
        rc, out = res[-1]
        assert rc == 0, "the unmodified oracle fails its pins through the mutant loader:\n" + out
        survivors = [name for (name, _), (rc, _) in zip(jobs, res[:-1]) if rc == 0]
        assert not survivors, "mutants that survive every pin: %s" % survivors
        # the harness must have run the pins and seen an assertion fail (pytest exit code 1), not crashed on build / import
        for (name, _), (rc, out) in zip(jobs, res[:-1]):
            assert rc == 1 and "AssertionError" in out, (name, rc, out)
    finally:
        shutil.rmtree(tmp, ignore_errors=True)


if __name__ == "__main__":          # python tests/test_oracle_mutations.py: prints which pin catches which mutant
    text = open(SRC).read()
    tmp = tempfile.mkdtemp(prefix="ocn_mut_")
    for n, (name, old, new) in enumerate(MUTANTS + MUTANTS_OPTIONS + MUTANTS_STEP):
        path = os.path.join(tmp, "m%02d.cpp" % n)
        open(path, "w").write(text.replace(old, new))
        rc, out = _run_pins(path, PINS if n < len(MUTANTS) else PINS_OPTIONS if n < len(MUTANTS) + len(MUTANTS_OPTIONS) else PINS_STEP)
        first = [ln for ln in out.splitlines() if ln.startswith("FAILED")]
        print("%-70s %s" % (name, first[0] if first else ("SURVIVES" if rc == 0 else "rc=%d" % rc)))
    shutil.rmtree(tmp, ignore_errors=True)
