// kernels_mixing.cuh — the Richardson-number-based vertical mixing closure (the stored
// vertical-diffusivity diagnostic of PAPER.md:78; formulas in DESIGN.md §3.12) and the per-column
// Thomas elimination with the resulting face diffusivities.  Launched only when closure = 1; K1 then
// runs with identity pivot tables (its d arrays hold the explicit predictor phi*) and K3 reads the
// modified super-diagonals written here.
#pragma once
#include "common.cuh"
#include "kernels_column.cuh"

namespace ocn {

// ---------------------------------------------------------------------------------------------
// K4: (nu, kappa) of state n at the open vertical faces of every tracer column, bottom-up, one thread
// per column.  All arithmetic in fp64 with the association of DESIGN.md §3.12 (the stored pair is
// rounded to the model precision); closed faces are never written and stay 0.
// ---------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(128) k_ri_mixing(const DevP<T> P) {
    typedef typename Pair<T>::type T2;
    typedef Xv<double> V;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const int sx = P.sx, nz = P.nz;
    const long long sz = P.sz, c = (long long)(j + OCN_HALO) * sx + i;
    const int kb = P.m8[c].x & 255;
    if (kb >= nz - 1) return;
    const bool edge = (P.px && (i < OCN_HALO || i >= P.nx - OCN_HALO)) || (P.py && (j < OCN_HALO || j >= P.ny - OCN_HALO));
    T2 q = P.ts[kb * sz + c];
    double b0 = buoyancy(P, q.x, q.y);
    T2 w0 = P.uv[kb * sz + c];
    double ue0 = (double)P.uv[kb * sz + c + 1].x, vn0 = (double)P.uv[kb * sz + c + sx].y;
    for (int k = kb + 1; k < nz; ++k) {
        const long long o = k * sz + c;
        q = P.ts[o];
        const double b1 = buoyancy(P, q.x, q.y);
        const T2 w1 = P.uv[o];
        const double ue1 = (double)P.uv[o + 1].x, vn1 = (double)P.uv[o + sx].y;
        const V dzc(P.dzc_d[k]);
        const V N2 = (V(b1) - V(b0)) / dzc;
        const V duw = V((double)w1.x) - V((double)w0.x), due = V(ue1) - V(ue0);
        const V dvs = V((double)w1.y) - V((double)w0.y), dvn = V(vn1) - V(vn0);
        const V S2 = (V(0.5) * (duw * duw + due * due) + V(0.5) * (dvs * dvs + dvn * dvn)) / (dzc * dzc);
        const V Ri = V(fmax(N2.v, 0.0)) / (S2 + V(P.ri_s2min));
        const V f = V(1.0) / (V(1.0) + V(P.ri_c) * Ri);
        const V conv = V(P.ri_kconv) * V(fmin(1.0, (V(fmax(-N2.v, 0.0)) / V(P.ri_n2c)).v));
        const V nu = V(P.nu_z_d) + V(P.ri_nu0) * f * f + conv;
        const V kap = V(P.kappa_z_d) + V(P.ri_nu0) * f * f * f + conv;
        const T2 out = mk2((T)nu.v, (T)kap.v);
        if (edge) store_halo(P.nk + k * sz, sx, P.nx, P.ny, P.px, P.py, j, i, out);
        else P.nk[o] = out;
        b0 = b1; w0 = w1; ue0 = ue1; vn0 = vn1;
    }
}

// ---------------------------------------------------------------------------------------------
// K5: Thomas elimination of the four fields of a column with per-face diffusivities (DESIGN.md §3.8
// step 4 with dt*kappa per face, §3.12), bottom-up in the order the equations are written:
//   s+ = dtk[k+1] / (dz_k dzc_{k+1}),  s- = dtk[k] / (dz_k dzc_k),  b = 1 + s+ + s-,
//   m = b - (-s-) cp_{k-1},  cp_k = (-s+) / m,  d_k = (phi*_k - (-s-) d_{k-1}) / m.
// dtk = dt * kappa for T, S; dt * (nu_{i-1} + nu_i)/2 for u; dt * (nu_{j-1} + nu_j)/2 for v.
// Reads phi* from the d arrays (K1 with identity tables), writes d in place and cp to cpt / cpuv.
// ---------------------------------------------------------------------------------------------
template <class T>
struct ThomasRow {
    T cp, d0, d1;                                // modified super-diagonal and two right-hand sides that share it
    __device__ __forceinline__ void step(bool first, T dtk_lo, T dtk_hi, bool has_hi, T dzk, T dzc_lo, T dzc_hi, T phi0, T phi1) {
        typedef Xv<T> V;
        const V sp = has_hi ? V(dtk_hi) / (V(dzk) * V(dzc_hi)) : V(T(0));
        const V sm = first ? V(T(0)) : V(dtk_lo) / (V(dzk) * V(dzc_lo));
        const V b = V(T(1)) + sp + sm;
        const V lo = -sm, up = -sp;
        const V m = first ? b : b - lo * V(cp);
        d0 = first ? (V(phi0) / m).v : ((V(phi0) - lo * V(d0)) / m).v;
        d1 = first ? (V(phi1) / m).v : ((V(phi1) - lo * V(d1)) / m).v;
        cp = (up / m).v;
    }
};

template <class T>
__global__ void __launch_bounds__(128) k_ri_eliminate(const DevP<T> P) {
    typedef typename Pair<T>::type T2;
    typedef Xv<T> V;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const int sx = P.sx, nz = P.nz;
    const long long sz = P.sz, c = (long long)(j + OCN_HALO) * sx + i;
    const uint2 m8 = P.m8[c];
    const int kb = (int)(m8.x & 255), tx1 = (int)((m8.x >> 8) & 255), ty1 = (int)(m8.y & 255);
    if (kb >= nz) return;
    ThomasRow<T> rt{T(0), T(0), T(0)}, ru{T(0), T(0), T(0)}, rv{T(0), T(0), T(0)};
    // dt * kappa at the face below level k for the three kinds of column (valid where that face is open)
    T2 here = kb + 1 < nz ? P.nk[(kb + 1) * sz + c] : mk2(T(0), T(0));
    T kt_lo = 0, ku_lo = 0, kv_lo = 0;
    for (int k = kb; k < nz; ++k) {
        const long long o = k * sz + c;
        const bool has_hi = k + 1 < nz;
        // face k+1: own pair was fetched last iteration (`here`), neighbours now
        T kt_hi = 0, ku_hi = 0, kv_hi = 0;
        if (has_hi) {
            kt_hi = (V(P.dt) * V(here.y)).v;
            if (k >= tx1) ku_hi = (V(P.dt) * (V(T(0.5)) * (V(P.nk[o + sz - 1].x) + V(here.x)))).v;
            if (k >= ty1) kv_hi = (V(P.dt) * (V(T(0.5)) * (V(P.nk[o + sz - sx].x) + V(here.x)))).v;
        }
        const T dzk = P.dz[k], dzc_lo = k > 0 ? P.dzc[k] : T(1), dzc_hi = has_hi ? P.dzc[k + 1] : T(1);
        const T2 pt = P.dts[o];
        rt.step(k == kb, kt_lo, kt_hi, has_hi, dzk, dzc_lo, dzc_hi, pt.x, pt.y);
        P.dts[o] = mk2(rt.d0, rt.d1);
        P.cpt[o] = rt.cp;
        if (k >= tx1 || k >= ty1) {
            const T2 pm = P.duv[o];
            T2 dout = mk2(T(0), T(0)), cout = mk2(T(0), T(0));
            if (k >= tx1) { ru.step(k == tx1, ku_lo, ku_hi, has_hi, dzk, dzc_lo, dzc_hi, pm.x, T(0)); dout.x = ru.d0; cout.x = ru.cp; }
            if (k >= ty1) { rv.step(k == ty1, kv_lo, kv_hi, has_hi, dzk, dzc_lo, dzc_hi, pm.y, T(0)); dout.y = rv.d0; cout.y = rv.cp; }
            P.duv[o] = dout;
            P.cpuv[o] = cout;
        }
        kt_lo = kt_hi; ku_lo = ku_hi; kv_lo = kv_hi;
        if (k + 2 < nz) here = P.nk[o + 2 * sz];
    }
}

}  // namespace ocn
