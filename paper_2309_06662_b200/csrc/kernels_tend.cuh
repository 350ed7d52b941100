// kernels_tend.cuh — K1: fused tendency kernel (S1 + S2 + S3 + forward half of S4 + S5).
//
// One thread owns one (j, i) column and marches k from the bottom up.  Per level it
//   * evaluates G_u, G_v, G_T, G_S from the halo'd state n and the stored
//     hydrostatic pressure p (written by K3 of the previous step),
//   * forms the quasi-AB2 combination and the explicit predictor phi* (S3),
//   * does the elimination sweep (bottom-up, as the equations are written in DESIGN.md §3.8)
//     of the backward-Euler tridiagonal system with table pivots (S4) and
//     writes the eliminated right-hand side d',
//   * accumulates the barotropic forcing sum_k dz G^_u and sum_k dz u* (S5).
// Loads are coalesced along i; horizontal neighbours come through L1/L2 (no shared-memory
// staging in this version).
#pragma once
#include "common.cuh"

namespace ocn {

template <class T>
__global__ void __launch_bounds__(128) k_tendency(const DevP<T> P, const T c0, const T c1) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const int sx = P.sx, nz = P.nz;
    const long long sz = P.sz;
    const long long c = (long long)(j + OCN_HALO) * sx + i;

    // ---- compact masks: level thresholds of this column and its east / north faces ----------
    const uint2 m = P.m8[c], me = P.m8[c + 1], mn = P.m8[c + sx];
    const uchar4 mzt = P.mz[c];
    const int kb = m.x & 255, tx1 = (m.x >> 8) & 255, tx2 = (m.x >> 16) & 255, tx3 = m.x >> 24;
    const int ty1 = m.y & 255, ty2 = (m.y >> 8) & 255, ty3 = (m.y >> 16) & 255;
    const int ex1 = (me.x >> 8) & 255, ex2 = (me.x >> 16) & 255, ex3 = me.x >> 24;
    const int ny1 = mn.y & 255, ny2 = (mn.y >> 8) & 255, ny3 = (mn.y >> 16) & 255;
    if (kb >= nz) {                       // land column: nothing to do, forcing sums are zero
        P.GU[c] = T(0); P.GV[c] = T(0); P.SU[c] = T(0); P.SV[c] = T(0);
        return;
    }

    // ---- row metrics ---------------------------------------------------------------------------
    const int r = j + OCN_HALO;
    const T dy = P.dy, rdy = P.rdy;
    const T dxCj = P.dxC[r], rdxCj = P.rdxC[r];
    const T dxFj = P.dxF[r], dxFn = P.dxF[r + 1], rdxFj = P.rdxF[r];
    const T AzCj = P.AzC[r], AzCs = P.AzC[r - 1], rAzCj = P.rAzC[r], rAzFj = P.rAzF[r];
    const T fFj = P.fF[r], fFn = P.fF[r + 1];

    // ---- running state up the column -------------------------------------------------------
    T tw[7], sw[7];                       // vertical windows c[k-3 .. k+3]
#pragma unroll
    for (int q = 0; q < 7; ++q) {
        const int kk = kb - 3 + q;
        const bool in = kk >= 0 && kk < nz;
        tw[q] = in ? P.t[kk * sz + c] : T(0);
        sw[q] = in ? P.s[kk * sz + c] : T(0);
    }
    T fzT_bot = 0, fzS_bot = 0;           // vertical tracer flux through the face below (0 at the bottom)
    T w_c0 = P.w[kb * sz + c], w_w0 = P.w[kb * sz + c - 1], w_s0 = P.w[kb * sz + c - sx];   // w[k]
    const T w_surf = P.w[nz * sz + c];
    T u_dn = 0, v_dn = 0;                 // u, v at k-1 (masked differences never use the initial value)
    T u_c = P.u[kb * sz + c], v_c = P.v[kb * sz + c];
    T ddu = 0, ddv = 0, ddt = 0, dds = 0; // eliminated right-hand side of the level below
    double aGU = 0, aGV = 0, aSU = 0, aSV = 0;
    const T* __restrict__ cpt = P.cp_t + kb * nz;  const T* __restrict__ mt = P.m_t + kb * nz;  const T* __restrict__ rmt = P.rm_t + kb * nz;
    const T* __restrict__ mmu = P.m_m + tx1 * nz;  const T* __restrict__ rmu = P.rm_m + tx1 * nz;
    const T* __restrict__ mmv = P.m_m + ty1 * nz;  const T* __restrict__ rmv = P.rm_m + ty1 * nz;
    (void)cpt;

    for (int k = kb; k < nz; ++k) {
        const long long o = k * sz + c;
        const T* __restrict__ pu = P.u + o;
        const T* __restrict__ pv = P.v + o;
        const T* __restrict__ pt = P.t + o;
        const T* __restrict__ pS = P.s + o;
        const bool mu = k >= tx1, mv = k >= ty1, mue = k >= ex1, mvn = k >= ny1;
        const T dzk = P.dz[k], rdzk = P.rdz[k];
        const T u_up = k + 1 < nz ? pu[sz] : T(0), v_up = k + 1 < nz ? pv[sz] : T(0);
        const T w_c1 = P.w[o + sz], w_w1 = P.w[o + sz - 1], w_s1 = P.w[o + sz - sx];
        const T tc = tw[3], sc = sw[3];

        // ---------------- tracers ----------------
        const T uw = u_c, ue = pu[1], vs = v_c, vn = pv[sx];
        const int oxw = order3(k, tx1, tx2, tx3), oxe = order3(k, ex1, ex2, ex3);
        const int oys = order3(k, ty1, ty2, ty3), oyn = order3(k, ny1, ny2, ny3);
        const int ozt = (k + 1 < nz) ? min(3, min(k + 1 - kb, nz - k - 1)) : 0;   // face above cell k
        const T ax = dy * dzk, ays = dxFj * dzk, ayn = dxFn * dzk;
        T GT, GS;
        {
            const T q0 = pt[-3], q1 = pt[-2], q2 = pt[-1], q4 = pt[1], q5 = pt[2], q6 = pt[3];
            const T r0 = pt[-3 * sx], r1 = pt[-2 * sx], r2 = pt[-sx], r4 = pt[sx], r5 = pt[2 * sx], r6 = pt[3 * sx];
            const T fw = uw * ax * weno_face(q0, q1, q2, tc, q4, q5, uw, oxw) - (mu ? P.kappa_h * ax * (tc - q2) * rdxCj : T(0));
            const T fe = ue * ax * weno_face(q1, q2, tc, q4, q5, q6, ue, oxe) - (mue ? P.kappa_h * ax * (q4 - tc) * rdxCj : T(0));
            const T fs = vs * ays * weno_face(r0, r1, r2, tc, r4, r5, vs, oys) - (mv ? P.kappa_h * ays * (tc - r2) * rdy : T(0));
            const T fn = vn * ayn * weno_face(r1, r2, tc, r4, r5, r6, vn, oyn) - (mvn ? P.kappa_h * ayn * (r4 - tc) * rdy : T(0));
            const T ft = ozt > 0 ? w_c1 * AzCj * weno_face(tw[1], tw[2], tw[3], tw[4], tw[5], tw[6], w_c1, ozt) : T(0);
            GT = -((fe - fw) + (fn - fs) + (ft - fzT_bot)) * rAzCj * rdzk;
            fzT_bot = ft;
        }
        {
            const T q0 = pS[-3], q1 = pS[-2], q2 = pS[-1], q4 = pS[1], q5 = pS[2], q6 = pS[3];
            const T r0 = pS[-3 * sx], r1 = pS[-2 * sx], r2 = pS[-sx], r4 = pS[sx], r5 = pS[2 * sx], r6 = pS[3 * sx];
            const T fw = uw * ax * weno_face(q0, q1, q2, sc, q4, q5, uw, oxw) - (mu ? P.kappa_h * ax * (sc - q2) * rdxCj : T(0));
            const T fe = ue * ax * weno_face(q1, q2, sc, q4, q5, q6, ue, oxe) - (mue ? P.kappa_h * ax * (q4 - sc) * rdxCj : T(0));
            const T fs = vs * ays * weno_face(r0, r1, r2, sc, r4, r5, vs, oys) - (mv ? P.kappa_h * ays * (sc - r2) * rdy : T(0));
            const T fn = vn * ayn * weno_face(r1, r2, sc, r4, r5, r6, vn, oyn) - (mvn ? P.kappa_h * ayn * (r4 - sc) * rdy : T(0));
            const T ft = ozt > 0 ? w_c1 * AzCj * weno_face(sw[1], sw[2], sw[3], sw[4], sw[5], sw[6], w_c1, ozt) : T(0);
            GS = -((fe - fw) + (fn - fs) + (ft - fzS_bot)) * rAzCj * rdzk;
            fzS_bot = ft;
        }
        if (k == nz - 1) {                // tracers are stored as offsets from (Toff, Soff): exact source of
            const T src = w_surf * rdzk;  // the constant under the zero-top-flux linear free surface
            GT += P.Toff * src; GS += P.Soff * src;
        }

        // ---------------- momentum ----------------
        T Gu = 0, Gv = 0;
        if (mu | mv) {
            auto zeta = [&](int dj, int di) -> T {
                const T* a = pu + dj * sx + di;
                const T* b = pv + dj * sx + di;
                return (dy * (b[0] - b[-1]) - (P.dxC[r + dj] * a[0] - P.dxC[r + dj - 1] * a[-sx])) * P.rAzF[r + dj];
            };
            auto kin = [&](int dj, int di) -> T {
                const T* a = pu + dj * sx + di;
                const T* b = pv + dj * sx + di;
                return T(0.25) * (a[0] * a[0] + a[1] * a[1]) + T(0.25) * (b[0] * b[0] + b[sx] * b[sx]);
            };
            auto divh = [&](int dj, int di) -> T {
                const T* a = pu + dj * sx + di;
                const T* b = pv + dj * sx + di;
                return (dy * (a[1] - a[0]) + P.dxF[r + dj + 1] * b[sx] - P.dxF[r + dj] * b[0]) * P.rAzC[r + dj];
            };
            const T z00 = zeta(0, 0), Kc = kin(0, 0), Dc = divh(0, 0);
            if (mu) {
                const T vsum_s = pv[-1] + pv[0], vsum_n = pv[sx - 1] + pv[sx];
                const T vhat = T(0.25) * (dxFj * vsum_s + dxFn * vsum_n) * rdxCj;
                const int ozu = 1 + (k >= mzt.x) + (k >= mzt.y);
                const T z01 = zeta(1, 0);
                const T zt = ozu == 1 ? (vhat > T(0) ? z00 : z01)
                                      : weno_face(zeta(-2, 0), zeta(-1, 0), z00, z01, zeta(2, 0), zeta(3, 0), vhat, ozu);
                const T Cu = T(0.5) * (fFj * T(0.5) * dxFj * vsum_s + fFn * T(0.5) * dxFn * vsum_n) * rdxCj;
                const T dK = (Kc - kin(0, -1)) * rdxCj;
                const T dP = (P.p[o] - P.p[o - 1]) * rdxCj;
                const T dlo = (k >= 1 && k - 1 >= tx1) ? u_c - u_dn : T(0);
                const T dhi = (k + 1 <= nz - 1) ? u_up - u_c : T(0);
                const T Au = T(0.5) * (T(0.5) * (w_w1 + w_c1) * dhi + T(0.5) * (w_w0 + w_c0) * dlo) * rdzk;
                const T Vu = P.nu_h * ((Dc - divh(0, -1)) * rdxCj - (z01 - z00) * rdy);
                const T tau = (k == nz - 1) ? P.taux[c] * P.rrho0 * rdzk : T(0);
                Gu = zt * vhat + Cu - dK - dP - Au + Vu + tau;
            }
            if (mv) {
                const T uhat = T(0.25) * (pu[-sx] + pu[0] + pu[-sx + 1] + pu[1]);
                const int ozv = 1 + (k >= mzt.z) + (k >= mzt.w);
                const T z10 = zeta(0, 1);
                const T zt = ozv == 1 ? (uhat > T(0) ? z00 : z10)
                                      : weno_face(zeta(0, -2), zeta(0, -1), z00, z10, zeta(0, 2), zeta(0, 3), uhat, ozv);
                const T Cv = fFj * uhat;
                const T dK = (Kc - kin(-1, 0)) * rdy;
                const T dP = (P.p[o] - P.p[o - sx]) * rdy;
                const T dlo = (k >= 1 && k - 1 >= ty1) ? v_c - v_dn : T(0);
                const T dhi = (k + 1 <= nz - 1) ? v_up - v_c : T(0);
                const T Av = T(0.5) * (T(0.5) * (AzCs * w_s1 + AzCj * w_c1) * dhi
                                     + T(0.5) * (AzCs * w_s0 + AzCj * w_c0) * dlo) * rAzFj * rdzk;
                const T Vv = P.nu_h * ((Dc - divh(-1, 0)) * rdy + (z10 - z00) * rdxFj);
                const T tau = (k == nz - 1) ? P.tauy[c] * P.rrho0 * rdzk : T(0);
                Gv = -zt * uhat - Cv - dK - dP - Av + Vv + tau;
            }
        }

        // ---------------- quasi-AB2, predictor, elimination sweep (S3, S4) ----------------
        const T Ghu = c0 * Gu - c1 * P.Gu[o], Ghv = c0 * Gv - c1 * P.Gv[o];
        const T Ght = c0 * GT - c1 * P.Gt[o], Ghs = c0 * GS - c1 * P.Gs[o];
        P.Gu[o] = Gu; P.Gv[o] = Gv; P.Gt[o] = GT; P.Gs[o] = GS;
        typedef Ex<T> E;
        if (mu) {
            const T us = E::add(u_c, E::mul(P.dt, Ghu));
            aGU += (double)dzk * (double)Ghu; aSU += (double)dzk * (double)us;
            const T smk = k > tx1 ? P.sm_m[k] : T(0);
            ddu = E::div(E::add(us, E::mul(smk, ddu)), mmu[k], rmu[k]);
            P.du[o] = ddu;
        }
        if (mv) {
            const T vs2 = E::add(v_c, E::mul(P.dt, Ghv));
            aGV += (double)dzk * (double)Ghv; aSV += (double)dzk * (double)vs2;
            const T smk = k > ty1 ? P.sm_m[k] : T(0);
            ddv = E::div(E::add(vs2, E::mul(smk, ddv)), mmv[k], rmv[k]);
            P.dv[o] = ddv;
        }
        {
            const T smk = k > kb ? P.sm_t[k] : T(0);
            const T mk = mt[k], rmk = rmt[k];
            ddt = E::div(E::add(E::add(tc, E::mul(P.dt, Ght)), E::mul(smk, ddt)), mk, rmk);
            dds = E::div(E::add(E::add(sc, E::mul(P.dt, Ghs)), E::mul(smk, dds)), mk, rmk);
            P.dt_[o] = ddt; P.ds[o] = dds;
        }

        // ---------------- shift the vertical windows ----------------
        w_c0 = w_c1; w_w0 = w_w1; w_s0 = w_s1;
        u_dn = u_c; u_c = u_up; v_dn = v_c; v_c = v_up;
#pragma unroll
        for (int q = 0; q < 6; ++q) { tw[q] = tw[q + 1]; sw[q] = sw[q + 1]; }
        const int kn = k + 4;
        tw[6] = kn < nz ? P.t[kn * sz + c] : T(0);
        sw[6] = kn < nz ? P.s[kn * sz + c] : T(0);
    }
    P.GU[c] = (T)aGU; P.GV[c] = (T)aGV; P.SU[c] = (T)aSU; P.SV[c] = (T)aSV;
}

}  // namespace ocn
