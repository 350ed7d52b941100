// kernels_mixing.cuh — the Richardson-number-based vertical mixing closure (the stored
// vertical-diffusivity diagnostic of PAPER.md:78; formulas in DESIGN.md §3.12): the face formula `ri_face` and the
// per-row Thomas elimination `ThomasRow` that K1 (kernels_tile.cuh, RI instantiation) evaluates inside the fused
// tendency pass from the (u, v) and (T, S) planes it already holds in shared memory, and K4, the stand-alone
// kernel that writes (nu, kappa) of the current state for ocn_get_mixing (not part of the time step).
#pragma once
#include "common.cuh"
#include "kernels_column.cuh"

namespace ocn {

// ---------------------------------------------------------------------------------------------
// (nu, kappa) at the face between levels k - 1 and k of a tracer column:
//   N2 = (b_k - b_{k-1}) / dzc_k,   S2 = [ (duw^2 + due^2)/2 + (dvs^2 + dvn^2)/2 ] / dzc_k^2
//   Ri = max(N2, 0) / (S2 + S2min),  f = 1 / (1 + c Ri),  conv = kconv min(1, max(-N2, 0) / N2c)
//   nu = nu_z + nu0 f^2 + conv,   kappa = kappa_z + nu0 f^3 + conv
// (t1, s1) / (t0, s0): stored tracers of level k / k - 1; duw .. dvn: u_k - u_{k-1} on the west / east, v on the south /
// north face of the column.  fp64 models: the association above in non-contracted IEEE operations, b from `buoyancy`
// (bit-identical to the oracle).  fp32 models: single precision on differenced neighbours, hardware reciprocals.
// ---------------------------------------------------------------------------------------------
template <class T>
__device__ __forceinline__ typename Pair<T>::type ri_face(const DevP<T>& P, int k, T t1, T s1, T t0, T s0,
                                                          T duw, T due, T dvs, T dvn) {
    if constexpr (sizeof(T) == 8) {
        typedef Xv<double> V;
        const V dzc(P.dzc_d[k]);
        const V N2 = (V(buoyancy(P, k, t1, s1)) - V(buoyancy(P, k - 1, t0, s0))) / dzc;
        const V S2 = (V(0.5) * (V(duw) * V(duw) + V(due) * V(due)) + V(0.5) * (V(dvs) * V(dvs) + V(dvn) * V(dvn))) / (dzc * dzc);
        const V Ri = V(fmax(N2.v, 0.0)) / (S2 + V(P.ri_s2min));
        const V f = V(1.0) / (V(1.0) + V(P.ri_c) * Ri);
        const V conv = V(P.ri_kconv) * V(fmin(1.0, (V(fmax(-N2.v, 0.0)) / V(P.ri_n2c)).v));
        const V nu = V(P.nu_z_d) + V(P.ri_nu0) * f * f + conv;
        const V kap = V(P.kappa_z_d) + V(P.ri_nu0) * f * f * f + conv;
        return mk2((T)nu.v, (T)kap.v);
    } else {
        const float rdzc = (float)P.rdzc[k];
        const float dT = (float)t1 - (float)t0, dS = (float)s1 - (float)s0;      // exact for neighbours in a column
        float db;
        if (P.eos == 1) {                               // the stored tracers are offsets from (T0, S0) in fp32 models
            const float a1 = (float)P.ath_d[k], a0 = (float)P.ath_d[k - 1];
            db = a1 * dT + (a1 - a0) * (float)t0 + (float)P.ha2_d * dT * ((float)t1 + (float)t0) - (float)P.beta_s * dS;
        } else {
            db = (float)P.alpha * dT - (float)P.beta_s * dS;
        }
        const float N2 = (float)P.g * db * rdzc;
        const float S2 = 0.5f * (((float)duw * (float)duw + (float)due * (float)due) + ((float)dvs * (float)dvs + (float)dvn * (float)dvn)) * rdzc * rdzc;
        const float Ri = __fdividef(fmaxf(N2, 0.f), S2 + (float)P.ri_s2min);     // hardware reciprocal: 2 ulp
        const float f = __fdividef(1.0f, 1.0f + (float)P.ri_c * Ri);
        const float conv = (float)P.ri_kconv * fminf(1.0f, fmaxf(-N2, 0.f) * (float)(1.0 / P.ri_n2c));
        const float g2 = (float)P.ri_nu0 * f * f;
        return mk2((T)((float)P.nu_z_d + g2 + conv), (T)((float)P.kappa_z_d + g2 * f + conv));
    }
}

// The fp32 form with its constants converted once (K1 evaluates it on every ring point of every level): same arithmetic as
// the fp32 branch of ri_face; rdzc = 1 / dzc_k from the caller's table.
struct RiConst {
    float g, alpha, beta, c, nu0, kconv, rn2c, s2min, nuz, kapz, ha2;
    int eos;
    template <class T>
    __device__ __forceinline__ void init(const DevP<T>& P) {
        g = (float)P.g; alpha = (float)P.alpha; beta = (float)P.beta_s; c = (float)P.ri_c; nu0 = (float)P.ri_nu0;
        kconv = (float)P.ri_kconv; rn2c = (float)(1.0 / P.ri_n2c); s2min = (float)P.ri_s2min; nuz = (float)P.nu_z_d;
        kapz = (float)P.kappa_z_d; ha2 = (float)P.ha2_d; eos = P.eos;
    }
};
__device__ __forceinline__ float2 ri_face_f32(const RiConst& R, const double* __restrict__ ath, int k, float rdzc, float t1, float s1,
                                              float t0, float s0, float duw, float due, float dvs, float dvn) {
    const float dT = t1 - t0, dS = s1 - s0;
    float db;
    if (R.eos == 1) {
        const float a1 = (float)ath[k], a0 = (float)ath[k - 1];
        db = a1 * dT + (a1 - a0) * t0 + R.ha2 * dT * (t1 + t0) - R.beta * dS;
    } else {
        db = R.alpha * dT - R.beta * dS;
    }
    const float N2 = R.g * db * rdzc;
    const float S2 = 0.5f * ((duw * duw + due * due) + (dvs * dvs + dvn * dvn)) * rdzc * rdzc;
    const float Ri = __fdividef(fmaxf(N2, 0.f), S2 + R.s2min);
    const float f = __fdividef(1.0f, 1.0f + R.c * Ri);
    const float conv = R.kconv * fminf(1.0f, fmaxf(-N2, 0.f) * R.rn2c);
    const float g2 = R.nu0 * f * f;
    return make_float2(R.nuz + g2 + conv, R.kapz + g2 * f + conv);
}

// ---------------------------------------------------------------------------------------------
// One row of the Thomas elimination with per-face diffusivities (DESIGN.md §3.8 step 4 with dt*kappa per face, §3.12),
// bottom-up in the order the equations are written:
//   s+ = dtk[k+1] / (dz_k dzc_{k+1}),  s- = dtk[k] / (dz_k dzc_k),  b = 1 + s+ + s-,
//   m = b - (-s-) cp_{k-1},  cp_k = (-s+) / m,  d_k = (phi*_k - (-s-) d_{k-1}) / m.
// dtk = dt * kappa for T, S; dt * (nu_{i-1} + nu_i)/2 for u; dt * (nu_{j-1} + nu_j)/2 for v.
// ---------------------------------------------------------------------------------------------
template <class T>
struct ThomasRow {
    T cp, d0, d1;                                // modified super-diagonal and two right-hand sides that share it
    // rz = 1 / dz_k, rc_lo = 1 / dzc_k, rc_hi = 1 / dzc_{k+1}: used by the fp32 form only
    __device__ __forceinline__ void step(bool first, T dtk_lo, T dtk_hi, bool has_hi, T dzk, T dzc_lo, T dzc_hi,
                                         T rz, T rc_lo, T rc_hi, T phi0, T phi1) {
        if (sizeof(T) == 8) {                    // fp64: the equations as written, true divisions (bit-identical to the oracle)
            typedef Xv<T> V;
            const V sp = has_hi ? V(dtk_hi) / (V(dzk) * V(dzc_hi)) : V(T(0));
            const V sm = first ? V(T(0)) : V(dtk_lo) / (V(dzk) * V(dzc_lo));
            const V b = V(T(1)) + sp + sm;
            const V lo = -sm, up = -sp;
            const V m = first ? b : b - lo * V(cp);
            d0 = first ? (V(phi0) / m).v : ((V(phi0) - lo * V(d0)) / m).v;
            d1 = first ? (V(phi1) / m).v : ((V(phi1) - lo * V(d1)) / m).v;
            cp = (up / m).v;
        } else {                                 // fp32: reciprocal multiplies, one division per row
            const T sp = has_hi ? dtk_hi * rz * rc_hi : T(0);
            const T sm = first ? T(0) : dtk_lo * rz * rc_lo;
            const T m = T(1) + sp + sm + sm * cp;                     // cp of the first row is 0 * sm
            const T rm = __fdividef(1.0f, (float)m);
            d0 = (phi0 + sm * d0) * rm;
            d1 = (phi1 + sm * d1) * rm;
            cp = -sp * rm;
        }
    }
};

// ---------------------------------------------------------------------------------------------
// K4: (nu, kappa) of the current state at the open vertical faces of every tracer column, bottom-up, one thread per
// column, for ocn_get_mixing (the stored vertical-diffusivity diagnostic of PAPER.md:78 as an output).  Closed faces hold 0.
// ---------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(128) k_ri_mixing(const DevP<T> P) {
    typedef typename Pair<T>::type T2;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (j >= P.ny) return;                                  // uniform over the warp (blockDim.x is a multiple of 32)
    const bool incol = i < P.nx;
    const int sx = P.sx, nz = P.nz;
    const long long sz = P.sz, c = (long long)(j + OCN_HALO) * sx + min(i, P.nx - 1);
    const int kb = incol ? (int)(P.m8[c].x & 255) : nz;
    // the lanes of a warp march together from the shallowest bottom among them, so that a level's loads and stores
    // of the warp fall into the same rows (a lane below its own bottom idles); sector-complete stores as in K3
    int kg = min(kb, __shfl_xor_sync(0xffffffffu, kb, 1));
    kg = min(kg, __shfl_xor_sync(0xffffffffu, kg, 2));
    const int k0 = __reduce_min_sync(0xffffffffu, kb);
    if (k0 >= nz - 1) return;
    const bool edge = (P.px && (i < OCN_HALO || i >= P.nx - OCN_HALO)) || (P.py && (j < OCN_HALO || j >= P.ny - OCN_HALO));
    T t0 = 0, s0 = 0, uw0 = 0, vs0 = 0, ue0 = 0, vn0 = 0;   // level k - 1
    constexpr int NB = 4;                                   // levels whose loads are in flight together
    for (int kk = k0; kk < nz; kk += NB) {
        T2 q[NB], w[NB], e[NB], n[NB];
#pragma unroll
        for (int r = 0; r < NB; ++r) {
            const int k = kk + r;
            q[r] = w[r] = e[r] = n[r] = mk2(T(0), T(0));
            if (k < nz && k >= kb) {
                const long long o = k * sz + c;
                q[r] = P.ts[o]; w[r] = P.uv[o]; e[r] = P.uv[o + 1]; n[r] = P.uv[o + sx];
            }
        }
#pragma unroll
        for (int r = 0; r < NB; ++r) {
            const int k = kk + r;
            if (k >= nz) break;
            if (k < kb) {                                   // below the own bottom: complete the sector of wet neighbours
                if (incol && k > kg) P.nk[k * sz + c] = mk2(T(0), T(0));
                continue;
            }
            const T uw1 = w[r].x, vs1 = w[r].y, ue1 = e[r].x, vn1 = n[r].y;
            if (k > kb) {
                const T2 out = ri_face(P, k, q[r].x, q[r].y, t0, s0, (X(uw1) - X(uw0)).v, (X(ue1) - X(ue0)).v,
                                       (X(vs1) - X(vs0)).v, (X(vn1) - X(vn0)).v);
                if (edge) store_halo(P.nk + k * sz, sx, P.nx, P.ny, P.px, P.py, j, i, out);
                else P.nk[k * sz + c] = out;
            } else if (k > kg) {
                P.nk[k * sz + c] = mk2(T(0), T(0));         // the face below the bottom cell is closed
            }
            t0 = q[r].x; s0 = q[r].y; uw0 = uw1; vs0 = vs1; ue0 = ue1; vn0 = vn1;
        }
    }
}

}  // namespace ocn
