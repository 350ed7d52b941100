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
// per column.  fp64 models: the association of DESIGN.md §3.12 in non-contracted IEEE operations (bit-identical
// to the oracle).  fp32 models: single precision on differenced neighbours.  Closed faces hold 0.
// ---------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(128) k_ri_mixing(const DevP<T> P) {
    typedef typename Pair<T>::type T2;
    typedef Xv<double> V;
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
    double b0 = 0;
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
            double b1 = 0;
            if (sizeof(T) == 8) b1 = buoyancy(P, q[r].x, q[r].y);
            if (k > kb) {
                T2 out;
                if (sizeof(T) == 8) {                       // fp64: the association of DESIGN.md §3.12, bit-identical to the oracle
                    const V dzc(P.dzc_d[k]);
                    const V N2 = (V(b1) - V(b0)) / dzc;
                    const V duw = V((double)uw1) - V((double)uw0), due = V((double)ue1) - V((double)ue0);
                    const V dvs = V((double)vs1) - V((double)vs0), dvn = V((double)vn1) - V((double)vn0);
                    const V S2 = (V(0.5) * (duw * duw + due * due) + V(0.5) * (dvs * dvs + dvn * dvn)) / (dzc * dzc);
                    const V Ri = V(fmax(N2.v, 0.0)) / (S2 + V(P.ri_s2min));
                    const V f = V(1.0) / (V(1.0) + V(P.ri_c) * Ri);
                    const V conv = V(P.ri_kconv) * V(fmin(1.0, (V(fmax(-N2.v, 0.0)) / V(P.ri_n2c)).v));
                    const V nu = V(P.nu_z_d) + V(P.ri_nu0) * f * f + conv;
                    const V kap = V(P.kappa_z_d) + V(P.ri_nu0) * f * f * f + conv;
                    out = mk2((T)nu.v, (T)kap.v);
                } else {                                    // fp32: difference the stored tracers first (exact for neighbours in
                    const float rdzc = (float)P.rdzc[k];         // a column), then the same formulas in single precision
                    const float N2 = (float)P.g * ((float)P.alpha * ((float)q[r].x - (float)t0) - (float)P.beta_s * ((float)q[r].y - (float)s0)) * rdzc;
                    const float duw = (float)uw1 - (float)uw0, due = (float)ue1 - (float)ue0, dvs = (float)vs1 - (float)vs0, dvn = (float)vn1 - (float)vn0;
                    const float S2 = 0.5f * ((duw * duw + due * due) + (dvs * dvs + dvn * dvn)) * rdzc * rdzc;
                    const float Ri = __fdividef(fmaxf(N2, 0.f), S2 + (float)P.ri_s2min);     // hardware reciprocal: 2 ulp
                    const float f = __fdividef(1.0f, 1.0f + (float)P.ri_c * Ri);
                    const float conv = (float)P.ri_kconv * fminf(1.0f, fmaxf(-N2, 0.f) * (float)(1.0 / P.ri_n2c));
                    const float g2 = (float)P.ri_nu0 * f * f;
                    out = mk2((T)((float)P.nu_z_d + g2 + conv), (T)((float)P.kappa_z_d + g2 * f + conv));
                }
                if (edge) store_halo(P.nk + k * sz, sx, P.nx, P.ny, P.px, P.py, j, i, out);
                else P.nk[k * sz + c] = out;
            } else if (k > kg) {
                P.nk[k * sz + c] = mk2(T(0), T(0));         // the face below the bottom cell is closed
            }
            b0 = b1; t0 = q[r].x; s0 = q[r].y; uw0 = uw1; vs0 = vs1; ue0 = ue1; vn0 = vn1;
        }
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

template <class T>
__global__ void __launch_bounds__(128) k_ri_eliminate(const DevP<T> P) {
    typedef typename Pair<T>::type T2;
    typedef Xv<T> V;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (j >= P.ny) return;                                  // uniform over the warp
    const bool incol = i < P.nx;
    const int sx = P.sx, nz = P.nz;
    const long long sz = P.sz, c = (long long)(j + OCN_HALO) * sx + min(i, P.nx - 1);
    const uint2 m8 = P.m8[c];
    const int kb = incol ? (int)(m8.x & 255) : nz, tx1 = incol ? (int)((m8.x >> 8) & 255) : nz, ty1 = incol ? (int)(m8.y & 255) : nz;
    const int kuv = min(tx1, ty1);
    // lanes of a warp march level by level together (coalesced rows); the four columns of a 32-byte sector start
    // together and the dry ones store zeros, so that no partly written sector has to be fetched (as in K3)
    int kg = min(kb, __shfl_xor_sync(0xffffffffu, kb, 1));
    kg = min(kg, __shfl_xor_sync(0xffffffffu, kg, 2));
    int kguv = min(kuv, __shfl_xor_sync(0xffffffffu, kuv, 1));
    kguv = min(kguv, __shfl_xor_sync(0xffffffffu, kguv, 2));
    const int k0 = __reduce_min_sync(0xffffffffu, kb);
    if (k0 >= nz) return;
    ThomasRow<T> rt{T(0), T(0), T(0)}, ru{T(0), T(0), T(0)}, rv{T(0), T(0), T(0)};
    T kt_lo = 0, ku_lo = 0, kv_lo = 0;                      // dt * kappa at the face below the current level
    constexpr int NB = 4;                                   // levels whose loads are in flight together
    for (int kk = k0; kk < nz; kk += NB) {
        T2 pt[NB], pm[NB];
        T kap_hi[NB], nu_hi[NB], nu_w[NB], nu_s[NB];        // face k+1: own (nu, kappa), nu of the west / south column
#pragma unroll
        for (int r = 0; r < NB; ++r) {
            const int k = kk + r;
            pt[r] = pm[r] = mk2(T(0), T(0));
            kap_hi[r] = nu_hi[r] = nu_w[r] = nu_s[r] = T(0);
            if (k < nz && k >= kb) {
                const long long o = k * sz + c;
                pt[r] = P.dts[o];
                if (k >= kuv) pm[r] = P.duv[o];
                if (k + 1 < nz) {
                    const T2 h = P.nk[o + sz];
                    kap_hi[r] = h.y; nu_hi[r] = h.x;
                    if (k >= tx1) nu_w[r] = P.nk[o + sz - 1].x;
                    if (k >= ty1) nu_s[r] = P.nk[o + sz - sx].x;
                }
            }
        }
#pragma unroll
        for (int r = 0; r < NB; ++r) {
            const int k = kk + r;
            if (k >= nz) break;
            const long long o = k * sz + c;
            if (k < kb) {
                if (incol && k >= kg) { P.dts[o] = mk2(T(0), T(0)); }
                if (incol && k >= kg) { P.cpt[o] = T(0); }
                if (incol && k >= kguv) { P.duv[o] = mk2(T(0), T(0)); P.cpuv[o] = mk2(T(0), T(0)); }
                continue;
            }
            const bool has_hi = k + 1 < nz;
            T kt_hi = 0, ku_hi = 0, kv_hi = 0;
            if (has_hi) {
                kt_hi = (V(P.dt) * V(kap_hi[r])).v;
                if (k >= tx1) ku_hi = (V(P.dt) * (V(T(0.5)) * (V(nu_w[r]) + V(nu_hi[r])))).v;
                if (k >= ty1) kv_hi = (V(P.dt) * (V(T(0.5)) * (V(nu_s[r]) + V(nu_hi[r])))).v;
            }
            const T dzk = P.dz[k], dzc_lo = k > 0 ? P.dzc[k] : T(1), dzc_hi = has_hi ? P.dzc[k + 1] : T(1);
            const T rz = P.rdz[k], rc_lo = k > 0 ? P.rdzc[k] : T(1), rc_hi = has_hi ? P.rdzc[k + 1] : T(1);
            rt.step(k == kb, kt_lo, kt_hi, has_hi, dzk, dzc_lo, dzc_hi, rz, rc_lo, rc_hi, pt[r].x, pt[r].y);
            P.dts[o] = mk2(rt.d0, rt.d1);
            P.cpt[o] = rt.cp;
            if (k >= kguv) {
                T2 dout = mk2(T(0), T(0)), cout = mk2(T(0), T(0));
                if (k >= tx1) { ru.step(k == tx1, ku_lo, ku_hi, has_hi, dzk, dzc_lo, dzc_hi, rz, rc_lo, rc_hi, pm[r].x, T(0)); dout.x = ru.d0; cout.x = ru.cp; }
                if (k >= ty1) { rv.step(k == ty1, kv_lo, kv_hi, has_hi, dzk, dzc_lo, dzc_hi, rz, rc_lo, rc_hi, pm[r].y, T(0)); dout.y = rv.d0; cout.y = rv.cp; }
                P.duv[o] = dout;
                P.cpuv[o] = cout;
            }
            kt_lo = kt_hi; ku_lo = ku_hi; kv_lo = kv_hi;
        }
    }
}

}  // namespace ocn
