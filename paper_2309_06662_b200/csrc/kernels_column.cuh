// kernels_column.cuh — column and 2-D kernels: barotropic sub-step (S6), back-substitution +
// barotropic correction (second half of S4, S7), vertical velocity scan (S8), halo-aware
// scatter / gather for ocn_set_fields / ocn_get_fields (S10 is folded into store_halo).
#pragma once
#include "common.cuh"

namespace ocn {

// linear equation of state; t, s are the stored (offset) tracers
template <class T>
__device__ __forceinline__ T buoyancy(const DevP<T>& P, T t, T s) {
    typedef Ex<T> E;
    return E::mul(P.g, E::sub(E::mul(P.alpha, E::sub(t, P.dT0)), E::mul(P.beta_s, E::sub(s, P.dS0))));
}

// ---------------------------------------------------------------------------------------------
// S6: one forward-backward barotropic sub-step (DESIGN.md §3.8 step 6): eta first, then U, V
// with the new eta.  eta is recomputed redundantly for the west and south neighbours so that
// one launch advances the whole sub-step.  Reads buffer `cur`, writes buffer `cur ^ 1`.
// ---------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(256) k_barotropic(const DevP<T> P, const int cur, const T am, const int first) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const int sx = P.sx, nz = P.nz, r = j + OCN_HALO;
    const long long c = (long long)r * sx + i;
    const T* __restrict__ e0 = P.eta[cur];
    const T* __restrict__ U0 = P.U[cur];
    const T* __restrict__ V0 = P.V[cur];
    const uint2 m = P.m8[c];
    const bool wet_c = (m.x & 255) < nz, wet_w = (P.m8[c - 1].x & 255) < nz, wet_s = (P.m8[c - sx].x & 255) < nz;
    const bool mu = ((m.x >> 8) & 255) < nz, mv = (m.y & 255) < nz;
    const T dy = P.dy, dtau = P.dtau;
    const T dF0 = P.dxF[r], dF1 = P.dxF[r + 1], dFm = P.dxF[r - 1];
    const T Uc = U0[c], Vc = V0[c];
    T ec = e0[c], ew = e0[c - 1], es = e0[c - sx];
    if (wet_c) ec -= dtau * (dy * (U0[c + 1] - Uc) + dF1 * V0[c + sx] - dF0 * Vc) * P.rAzC[r];
    if (wet_w) ew -= dtau * (dy * (Uc - U0[c - 1]) + dF1 * V0[c + sx - 1] - dF0 * V0[c - 1]) * P.rAzC[r];
    if (wet_s) es -= dtau * (dy * (U0[c - sx + 1] - U0[c - sx]) + dF0 * Vc - dFm * V0[c - sx]) * P.rAzC[r - 1];
    const T Un = mu ? Uc + dtau * (-P.g * P.Hu[c] * (ec - ew) * P.rdxC[r] + P.GU[c]) : T(0);
    const T Vn = mv ? Vc + dtau * (-P.g * P.Hv[c] * (ec - es) * P.rdy + P.GV[c]) : T(0);
    store_halo(P.eta[cur ^ 1], sx, P.nx, P.ny, P.px, P.py, j, i, ec);
    store_halo(P.U[cur ^ 1], sx, P.nx, P.ny, P.px, P.py, j, i, Un);
    store_halo(P.V[cur ^ 1], sx, P.nx, P.ny, P.px, P.py, j, i, Vn);
    if (first) { P.etab[c] = am * ec; P.Ub[c] = am * Un; P.Vb[c] = am * Vn; }
    else       { P.etab[c] += am * ec; P.Ub[c] += am * Un; P.Vb[c] += am * Vn; }
}

// step 7: the filtered values become the barotropic state (buffer 0, with halos)
template <class T>
__global__ void __launch_bounds__(256) k_barotropic_finish(const DevP<T> P) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const long long c = (long long)(j + OCN_HALO) * P.sx + i;
    store_halo(P.eta[0], P.sx, P.nx, P.ny, P.px, P.py, j, i, P.etab[c]);
    store_halo(P.U[0], P.sx, P.nx, P.ny, P.px, P.py, j, i, P.Ub[c]);
    store_halo(P.V[0], P.sx, P.nx, P.ny, P.px, P.py, j, i, P.Vb[c]);
}

// ---------------------------------------------------------------------------------------------
// S4 (back-substitution, top-down) + S7 (barotropic correction) + S9 (hydrostatic pressure of
// the new T, S, integrated downward from the surface in the same sweep).
// The implicit operator conserves the column integral, so sum_k dz u** = sum_k dz u* (SU from
// K1) and the correction (Ubar - SU) / Hu is known before the sweep.
// ---------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(128) k_backsub_correct(const DevP<T> P) {
    typedef Ex<T> E;
    typedef typename Pair<T>::type T2;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const int sx = P.sx, nz = P.nz;
    const long long sz = P.sz, c = (long long)(j + OCN_HALO) * sx + i;
    const uint2 m = P.m8[c];
    const int kb = m.x & 255, tx1 = (m.x >> 8) & 255, ty1 = m.y & 255;
    if (kb >= nz) return;
    const T cu = tx1 < nz ? (P.Ub[c] - P.SU[c]) * P.rHu[c] : T(0);
    const T cv = ty1 < nz ? (P.Vb[c] - P.SV[c]) * P.rHv[c] : T(0);
    const T* __restrict__ cpu = P.cp_m + min(tx1, nz - 1);
    const T* __restrict__ cpv = P.cp_m + min(ty1, nz - 1);
    const T* __restrict__ cpt = P.cp_t + kb;
    T xu = 0, xv = 0, xt = 0, xs = 0, b1 = 0, pk = 0;
    const int kuv = min(tx1, ty1);
    constexpr int NB = 4;                                  // levels whose loads are in flight together
    for (int k0 = nz - 1; k0 >= kb; k0 -= NB) {
        T2 d_ts[NB], d_uv[NB];
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            const int k = k0 - q;
            d_ts[q] = mk2(T(0), T(0)); d_uv[q] = mk2(T(0), T(0));
            if (k >= kb) {
                d_ts[q] = P.dts[k * sz + c];
                if (k >= kuv) d_uv[q] = P.duv[k * sz + c];
            }
        }
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            const int k = k0 - q;
            if (k < kb) break;
            const T ck = cpt[k * nz];
            xt = E::sub(d_ts[q].x, E::mul(ck, xt));                      // cp[nz-1] = 0
            xs = E::sub(d_ts[q].y, E::mul(ck, xs));
            store_halo(P.ts + k * sz, sx, P.nx, P.ny, P.px, P.py, j, i, mk2(xt, xs));
            const T b0 = buoyancy(P, xt, xs);
            pk = k == nz - 1 ? -E::mul(b0, P.hz_top)
                             : E::sub(pk, E::mul(E::mul(T(0.5), E::add(b1, b0)), P.dzc[k + 1]));
            b1 = b0;
            store_halo(P.p + k * sz, sx, P.nx, P.ny, P.px, P.py, j, i, pk);
            const bool mu = k >= tx1, mv = k >= ty1;
            if (mu | mv) {
                T un = 0, vn = 0;
                if (mu) { xu = E::sub(d_uv[q].x, E::mul(cpu[k * nz], xu)); un = xu + cu; }
                if (mv) { xv = E::sub(d_uv[q].y, E::mul(cpv[k * nz], xv)); vn = xv + cv; }
                store_halo(P.uv + k * sz, sx, P.nx, P.ny, P.px, P.py, j, i, mk2(un, vn));
            }
        }
    }
}

// S9 alone (ocn_set_fields): hydrostatic pressure of the current T, S
template <class T>
__global__ void __launch_bounds__(128) k_pressure(const DevP<T> P) {
    typedef Ex<T> E;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const int sx = P.sx, nz = P.nz;
    const long long sz = P.sz, c = (long long)(j + OCN_HALO) * sx + i;
    const int kb = P.m8[c].x & 255;
    T b1 = 0, pk = 0;
    for (int k = nz - 1; k >= kb; --k) {
        const typename Pair<T>::type q = P.ts[k * sz + c];
        const T b0 = buoyancy(P, q.x, q.y);
        pk = k == nz - 1 ? -E::mul(b0, P.hz_top)
                         : E::sub(pk, E::mul(E::mul(T(0.5), E::add(b1, b0)), P.dzc[k + 1]));
        b1 = b0;
        store_halo(P.p + k * sz, sx, P.nx, P.ny, P.px, P.py, j, i, pk);
    }
}

// ---------------------------------------------------------------------------------------------
// S8: w from continuity, bottom-up scan; runs through land where D = 0.
// ---------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(128) k_vertical_velocity(const DevP<T> P) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const int sx = P.sx, nz = P.nz, r = j + OCN_HALO;
    const long long sz = P.sz, c = (long long)r * sx + i;
    const T dy = P.dy, dF0 = P.dxF[r], dF1 = P.dxF[r + 1], rA = P.rAzC[r];
    double w = 0.0;
    for (int k = 0; k < nz; ++k) {
        const typename Pair<T>::type* __restrict__ q = P.uv + k * sz + c;
        const T D = (dy * (q[1].x - q[0].x) + dF1 * q[sx].y - dF0 * q[0].y) * rA;
        w -= (double)P.dz[k] * (double)D;
        store_halo(P.w + (k + 1) * sz, sx, P.nx, P.ny, P.px, P.py, j, i, (T)w);
    }
}

// U, V = sum_k dz u, v of the current state into buffer 0 (ocn_set_fields)
template <class T>
__global__ void __launch_bounds__(128) k_init_transport(const DevP<T> P) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const long long sz = P.sz, c = (long long)(j + OCN_HALO) * P.sx + i;
    double su = 0, sv = 0;
    for (int k = 0; k < P.nz; ++k) { const typename Pair<T>::type q = P.uv[k * sz + c]; su += (double)P.dz[k] * (double)q.x; sv += (double)P.dz[k] * (double)q.y; }
    store_halo(P.U[0], P.sx, P.nx, P.ny, P.px, P.py, j, i, (T)su);
    store_halo(P.V[0], P.sx, P.nx, P.ny, P.px, P.py, j, i, (T)sv);
}

// ---------------------------------------------------------------------------------------------
// scatter (contiguous interior -> halo'd plane layout, masked) and gather (back, land = 0)
// st = element stride of the device array (2 = one member of a pair array, base already offset)
// kind: 0 u, 1 v, 2 T (offset Toff), 3 S (offset Soff), 4 eta, 5 plain 2-D, 6 w (nz+1 levels, gather only)
// ---------------------------------------------------------------------------------------------
template <class T>
__device__ __forceinline__ bool cell_open(const DevP<T>& P, long long c, int k, int kind) {
    const uint2 m = P.m8[c];
    const int kb = m.x & 255, tx1 = (m.x >> 8) & 255, ty1 = m.y & 255;
    switch (kind) {
        case 0: return k >= tx1;
        case 1: return k >= ty1;
        case 2: case 3: return k >= kb;
        case 4: return kb < P.nz;
        default: return true;
    }
}

template <class T>
__global__ void __launch_bounds__(256) k_scatter(const DevP<T> P, T* __restrict__ dst, const T* __restrict__ src,
                                                 const int nl, const int kind, const int st) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const long long c = (long long)(j + OCN_HALO) * P.sx + i;
    const T off = kind == 2 ? P.Toff : kind == 3 ? P.Soff : T(0);
    for (int k = blockIdx.z; k < nl; k += gridDim.z) {
        const T v = cell_open(P, c, k, kind) ? src[((long long)k * P.ny + j) * P.nx + i] - off : T(0);
        store_halo(dst + k * P.sz * st, P.sx, P.nx, P.ny, P.px, P.py, j, i, v, st);
    }
}

template <class T, class O>
__global__ void __launch_bounds__(256) k_gather(const DevP<T> P, O* __restrict__ dst, const T* __restrict__ src,
                                                const int nl, const int kind, const int st) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const long long c = (long long)(j + OCN_HALO) * P.sx + i;
    const T off = kind == 2 ? P.Toff : kind == 3 ? P.Soff : T(0);
    for (int k = blockIdx.z; k < nl; k += gridDim.z) {
        const T v = cell_open(P, c, k, kind) ? src[(k * P.sz + c) * st] + off : T(0);
        dst[((long long)k * P.ny + j) * P.nx + i] = (O)v;
    }
}

}  // namespace ocn
