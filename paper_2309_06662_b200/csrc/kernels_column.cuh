// kernels_column.cuh — column and 2-D kernels: barotropic sub-step (S6), back-substitution +
// barotropic correction (second half of S4, S7), vertical velocity scan (S8), halo-aware
// scatter / gather for ocn_set_fields / ocn_get_fields (S10 is folded into store_halo).
#pragma once
#include "common.cuh"

namespace ocn {

// linear equation of state and one level of the downward pressure integral, in fp64 with the
// rounding order of the equations as written; t, s are the stored (offset) tracers.  In fp32 runs this keeps
// the rounding of p ~ 1e2 m^2/s^2 (whose horizontal differences drive the flow) out of the momentum equation.
// eos = 1: b = g [ath[k] dT + ha2 dT dT - beta dS] with ath[k] = alpha (1 - gamma zc[k]) and ha2 = alpha2 / 2
// built on the host with the same fp64 operations the equation is written in.
template <class T>
__device__ __forceinline__ double buoyancy(const DevP<T>& P, int k, T t, T s) {
    typedef Ex<double> E;
    const double dT = E::sub((double)t, P.dT0_d), dS = E::sub((double)s, P.dS0_d);
    if (P.eos == 1)
        return E::mul(P.g_d, E::sub(E::add(E::mul(P.ath_d[k], dT), E::mul(E::mul(P.ha2_d, dT), dT)), E::mul(P.beta_d, dS)));
    return E::mul(P.g_d, E::sub(E::mul(P.alpha_d, dT), E::mul(P.beta_d, dS)));
}
template <class T>
__device__ __forceinline__ double pressure_level(const DevP<T>& P, int k, double b0, double b1, double p_above) {
    typedef Ex<double> E;
    return k == P.nz - 1 ? -E::mul(b0, P.hz_top_d)
                         : E::sub(p_above, E::mul(E::mul(0.5, E::add(b1, b0)), P.dzc_d[k + 1]));
}

// ---------------------------------------------------------------------------------------------
// S6, resident form: one launch advances `ns` (<= BT_HALO) forward-backward
// sub-steps of a (BTX x BTY) tile held in shared memory together with a halo of BT_HALO columns
// that is recomputed redundantly and shrinks by one ring per sub-step — the paper's wide-halo
// idea for the barotropic mode applied to the on-chip tile, so eta, U, V make one
// HBM round trip per `ns` sub-steps instead of one per sub-step.  Periodic directions are wrapped
// when the tile is loaded (no physical halo is needed), bounded ones read land.
// Reads buffer `cur`, writes buffer `cur ^ 1`; the filter sums live in registers during the launch.
// ---------------------------------------------------------------------------------------------
#ifndef BT_HALO
#define BT_HALO 6                  // sub-steps per launch = halo rings of the resident tile (<= 6: the launch carries six weights)
#endif

// most sub-steps one launch advances (the filter weights of the launch, a for eta and b for the transports U, V, DESIGN.md
// §3.9, §3.17, are staged from the model's device tables into shared memory)
#define BT_MAXW 12

template <class T, int BTX, int BTY>
struct BtTile {
    static constexpr int EX = BTX + 2 * BT_HALO, EY = BTY + 2 * BT_HALO, NE = EX * EY;
    static constexpr int NT = BTX * BTY >= 2048 ? 1024 : 512, PER = (NE + NT - 1) / NT;      // extended-tile points per thread
    static constexpr int SMEM = NE * (7 * (int)sizeof(T) + 1) + 6 * (EY + 1) * (int)sizeof(T) + 64 + 2 * BT_HALO * (int)sizeof(T);
};

template <class T, int BTX, int BTY>
__global__ void __launch_bounds__((BtTile<T, BTX, BTY>::NT)) k_barotropic_tile(const DevP<T> P, const int cur, const int ns, const int first, const int m0) {
    typedef BtTile<T, BTX, BTY> C;
    constexpr int EX = C::EX, EY = C::EY, NE = C::NE, NT = C::NT, H = BT_HALO;
    extern __shared__ __align__(16) unsigned char smb[];
    T* const se = (T*)smb;                 // eta
    T* const sU = se + NE;
    T* const sV = sU + NE;
    T* const sGU = sV + NE;
    T* const sGV = sGU + NE;
    T* const sHu = sGV + NE;
    T* const sHv = sHu + NE;
    T* const rAz = sHv + NE;               // per extended row: 1 / AzC, 1 / dxC, dxF (row), dxF (row + 1)
    T* const rdx = rAz + (EY + 1);
    T* const dF = rdx + (EY + 1);          // EY + 1 entries
    T* const Az = dF + (EY + 1);           // AzC, dxC per extended row (fp64 divides, fp32 multiplies by the reciprocals)
    T* const dxc = Az + (EY + 1);
    T* const saw = dxc + (EY + 1);         // filter weights of this launch: a (eta), then b (transports)
    T* const sbw = saw + BT_HALO;
    unsigned char* const smk = (unsigned char*)(sbw + BT_HALO);   // bit 0 wet, bit 1 open u face, bit 2 open v face
    const int tid = threadIdx.x;
    const int i0 = blockIdx.x * BTX, j0 = blockIdx.y * BTY;
    const int nx = P.nx, ny = P.ny, nz = P.nz, sx = P.sx;
    if (tid < ns) { saw[tid] = P.fw_a[m0 + tid]; sbw[tid] = P.fw_b[m0 + tid]; }

    // ---- load the extended tile (wrap / land) ----
    for (int q = tid; q <= EY; q += NT) {
        int jj = j0 - H + q;
        if (P.py) { while (jj < 0) jj += ny; while (jj >= ny) jj -= ny; }
        const int r = min(max(jj, -OCN_HALO), ny + OCN_HALO) + OCN_HALO;      // metric rows exist for -3 .. ny + 3
        if (q < EY) { rAz[q] = P.rAzC[r]; rdx[q] = P.rdxC[r]; Az[q] = P.AzC[r]; dxc[q] = P.dxC[r]; }
        dF[q] = P.dxF[r];
    }
    const T* __restrict__ e0 = P.eta[cur];
    const T* __restrict__ U0 = P.U[cur];
    const T* __restrict__ V0 = P.V[cur];
    {
        int cs[C::PER];                                        // source plane index of each point, -1 outside a bounded domain
        uint2 ms[C::PER];
#pragma unroll
        for (int n = 0; n < C::PER; ++n) {                     // wrap by steps: the tile reaches at most H + BTX past an edge
            const int q = n * NT + tid;
            const int x = q % EX, y = q / EX;
            int ii = i0 - H + x, jj = j0 - H + y;
            bool in = q < NE;
            if (P.px) { while (ii < 0) ii += nx; while (ii >= nx) ii -= nx; } else in = in && ii >= 0 && ii < nx;
            if (P.py) { while (jj < 0) jj += ny; while (jj >= ny) jj -= ny; } else in = in && jj >= 0 && jj < ny;
            cs[n] = in ? (jj + OCN_HALO) * sx + ii : -1;
            ms[n] = make_uint2(nz, nz);
            if (in) ms[n] = P.m8[cs[n]];
        }
#pragma unroll
        for (int n = 0; n < C::PER; ++n) {
            const int q = n * NT + tid;
            if (q < NE) {
                const uint2 m = ms[n];
                const int c = cs[n];
                T e = 0, u = 0, v = 0, gu = 0, gv = 0, hu = 0, hv = 0;
                const unsigned char mk = c < 0 ? 0 : (unsigned char)(((m.x & 255u) < (unsigned)nz ? 1 : 0) | ((((m.x >> 8) & 255u) < (unsigned)nz) ? 2 : 0) |
                                                                      (((m.y & 255u) < (unsigned)nz) ? 4 : 0));
                if (mk) { e = e0[c]; u = U0[c]; v = V0[c]; gu = P.GU[c]; gv = P.GV[c]; hu = P.Hu[c]; hv = P.Hv[c]; }
                se[q] = e; sU[q] = u; sV[q] = v; smk[q] = mk;
                sGU[q] = gu; sGV[q] = gv; sHu[q] = hu; sHv[q] = hv;
            }
        }
    }
    __syncthreads();

    // ---- filter sums of the points this thread updates (same point-to-thread map as the update loops, so no
    // other thread touches a value between its update and its accumulation); one running sum over all M
    // sub-steps (DESIGN.md §3.8 step 6), continued from the previous launch --------------------------------
    T be[C::PER], bU[C::PER], bV[C::PER];
    int cidx[C::PER];                                         // plane index of the interior points, -1 elsewhere
#pragma unroll
    for (int n = 0; n < C::PER; ++n) {
        be[n] = 0; bU[n] = 0; bV[n] = 0; cidx[n] = -1;
        const int q = n * NT + tid;
        const int x = q % EX - H, y = q / EX - H;
        const int i = i0 + x, j = j0 + y;
        if (q < NE && x >= 0 && x < BTX && y >= 0 && y < BTY && i < nx && j < ny) {
            cidx[n] = (j + OCN_HALO) * sx + i;
            if (!first) { be[n] = P.etab[cidx[n]]; bU[n] = P.Ub[cidx[n]]; bV[n] = P.Vb[cidx[n]]; }
        }
    }
    const T dy = P.dy, dtau = P.dtau, g = P.g, rdy = P.rdy;

    if constexpr (sizeof(T) == 4) {
        // fp32: everything that is constant over the sub-steps (mask, depth, metric, forcing, dtau) is folded into five
        // per-point coefficients held in registers, zero where the point is closed or on the rim of the extended tile:
        //   eta -= ce (dy (U_e - U) + dxF_n V_n - dxF V),  U += cu (eta_w - eta) + gu,  V += cv (eta_s - eta) + gv
        T ce[C::PER], cu[C::PER], cv[C::PER], gu[C::PER], gv[C::PER];
        uint32_t ypk = 0;                                      // the extended row of each point, one byte each
        static_assert(C::PER <= 4 && EY < 256, "row bytes");
#pragma unroll
        for (int n = 0; n < C::PER; ++n) {
            ce[n] = cu[n] = cv[n] = gu[n] = gv[n] = 0;
            const int q = n * NT + tid;
            if (q < NE) {
                const int x = q % EX, y = q / EX;
                const unsigned char mk = smk[q];
                ypk |= (uint32_t)y << (8 * n);
                if (x < EX - 1 && y < EY - 1 && (mk & 1)) ce[n] = dtau * rAz[y];
                if (x > 0 && (mk & 2)) { cu[n] = dtau * g * sHu[q] * rdx[y]; gu[n] = dtau * sGU[q]; }
                if (y > 0 && (mk & 4)) { cv[n] = dtau * g * sHv[q] * rdy; gv[n] = dtau * sGV[q]; }
            }
        }
        for (int s = 0; s < ns; ++s) {
#pragma unroll
            for (int n = 0; n < C::PER; ++n) {
                const int q = n * NT + tid;
                if (q < NE) {
                    const int y = (ypk >> (8 * n)) & 255u;
                    const int qe = min(q + 1, NE - 1), qn = min(q + EX, NE - 1);      // rim points: ce = 0
                    const T uc = sU[q], vc = sV[q];
                    se[q] = se[q] - ce[n] * (dy * (sU[qe] - uc) + dF[y + 1] * sV[qn] - dF[y] * vc);
                }
            }
            __syncthreads();
            const T am = saw[s], bm = sbw[s];
#pragma unroll
            for (int n = 0; n < C::PER; ++n) {
                const int q = n * NT + tid;
                if (q < NE) {
                    const T ec = se[q], ew = se[max(q - 1, 0)], es = se[max(q - EX, 0)];     // rim points: cu = cv = 0
                    const T un = sU[q] + (cu[n] * (ew - ec) + gu[n]);
                    const T vn = sV[q] + (cv[n] * (es - ec) + gv[n]);
                    sU[q] = un; sV[q] = vn;
                    if (cidx[n] >= 0) { be[n] += am * ec; bU[n] += bm * un; bV[n] += bm * vn; }
                }
            }
            __syncthreads();
        }
    } else {
    for (int s = 0; s < ns; ++s) {
        // eta: valid on [s, EX - 1 - s) x [s, EY - 1 - s) given U, V valid on [s, EX - s) x [s, EY - s)
        for (int q = tid; q < NE; q += NT) {
            const int x = q % EX, y = q / EX;
            if (x < EX - 1 && y < EY - 1 && (smk[q] & 1))
                se[q] = (X(se[q]) - xdiv(X(dtau) * (X(dy) * (X(sU[q + 1]) - X(sU[q])) + X(dF[y + 1]) * X(sV[q + EX]) - X(dF[y]) * X(sV[q])),
                                         Az[y], rAz[y])).v;
        }
        __syncthreads();
        const T am = saw[s], bm = sbw[s];
#pragma unroll
        for (int n = 0; n < C::PER; ++n) {
            const int q = n * NT + tid;
            if (q < NE) {
                const int x = q % EX, y = q / EX;
                const unsigned char mk = smk[q];
                const T ec = se[q];
                T un = sU[q], vn = sV[q];
                if (x > 0) un = (mk & 2) ? (X(un) + X(dtau) * (xdiv(-X(g) * X(sHu[q]) * (X(ec) - X(se[q - 1])), dxc[y], rdx[y]) + X(sGU[q]))).v : T(0);
                if (y > 0) vn = (mk & 4) ? (X(vn) + X(dtau) * (xdiv(-X(g) * X(sHv[q]) * (X(ec) - X(se[q - EX])), dy, rdy) + X(sGV[q]))).v : T(0);
                sU[q] = un; sV[q] = vn;
                if (cidx[n] >= 0) {
                    be[n] = (X(be[n]) + X(am) * X(ec)).v; bU[n] = (X(bU[n]) + X(bm) * X(un)).v; bV[n] = (X(bV[n]) + X(bm) * X(vn)).v;
                }
            }
        }
        __syncthreads();
    }
    }
    // ---- write back the interior ----
#pragma unroll
    for (int n = 0; n < C::PER; ++n) {
        if (cidx[n] >= 0) {
            const int q = n * NT + tid;
            const int c = cidx[n];
            P.eta[cur ^ 1][c] = se[q]; P.U[cur ^ 1][c] = sU[q]; P.V[cur ^ 1][c] = sV[q];
            P.etab[c] = be[n]; P.Ub[c] = bU[n]; P.Vb[c] = bV[n];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// S6, resident form for fp32 models, register strips: as k_barotropic_tile, but a thread owns a strip of
// four consecutive points of a row of the extended tile and keeps their eta, U, V, the five folded coefficients and the
// filter sums in REGISTERS for the whole launch.  Shared memory only carries what neighbours need: per sub-step a strip
// publishes its eta / U / V with three 128-bit stores and reads the U east of it, the eta west of it (32-bit) and the V
// row north / eta row south of it (128-bit) - 7 shared-memory instructions per four points where the point-wise kernel
// needs about fifty, which is what bounded it (LSU pipe 74 % busy, profiles/r1_ncu_summary.md).  NS <= H sub-steps per
// launch on a halo of H that is recomputed redundantly and shrinks one ring per sub-step (PAPER.md:98 on chip).
// ---------------------------------------------------------------------------------------------
template <int BTX, int BTY, int H>
struct BtStrip {
    static constexpr int EX = BTX + 2 * H, EY = BTY + 2 * H, SPR = EX / 4, NS = SPR * EY;   // strips per row, strips
    static_assert(EX % 4 == 0, "extended row must be a whole number of strips");
    static constexpr int NT = (NS + 31) / 32 * 32;
    static_assert(NT <= 1024, "one strip per thread");
    static constexpr int SMEM = 3 * EX * EY * 4 + 2 * (EY + 1) * 4 + 16 + 2 * BT_MAXW * 4;
};

template <int BTX, int BTY, int H>
__global__ void __launch_bounds__((BtStrip<BTX, BTY, H>::NT), (1024 / BtStrip<BTX, BTY, H>::NT))
k_barotropic_strip(const DevP<float> P, const int cur, const int ns, const int first, const int m0) {
    typedef BtStrip<BTX, BTY, H> C;
    constexpr int EX = C::EX, EY = C::EY, SPR = C::SPR;
    extern __shared__ __align__(16) unsigned char smb[];
    float* const se = (float*)smb;
    float* const sU = se + EX * EY;
    float* const sV = sU + EX * EY;
    float* const dF = sV + EX * EY;                 // dxF per extended row, EY + 1 entries
    float* const rAz = dF + (EY + 1);               // 1 / AzC per extended row
    float* const saw = rAz + (EY + 1) + 2;          // filter weights of this launch: a (eta), then b (transports)
    float* const sbw = saw + BT_MAXW;
    const int tid = threadIdx.x;
    const int i0 = blockIdx.x * BTX, j0 = blockIdx.y * BTY;
    const int nx = P.nx, ny = P.ny, nz = P.nz, sx = P.sx;
    for (int q = tid; q <= EY; q += C::NT) {
        int jj = j0 - H + q;
        if (P.py) { while (jj < 0) jj += ny; while (jj >= ny) jj -= ny; }
        const int r = min(max(jj, -OCN_HALO), ny + OCN_HALO) + OCN_HALO;
        dF[q] = P.dxF[r];
        if (q < EY) rAz[q] = P.rAzC[r];
    }
    if (tid < ns) { saw[tid] = P.fw_a[m0 + tid]; sbw[tid] = P.fw_b[m0 + tid]; }
    const bool on = tid < C::NS;
    const int y = on ? tid / SPR : 0, x0 = on ? 4 * (tid % SPR) : 0;
    const int qb = y * EX + x0;                     // first point of the strip in the extended tile
    const float dy = P.dy, dtau = P.dtau, g = P.g, rdy = P.rdy;
    float e[4], u[4], v[4], ce[4], cu[4], cv[4], gu[4], gv[4], be[4], bU[4], bV[4];
    int cidx[4];
    {
        int jj = j0 - H + y;
        bool iny = true;
        if (P.py) { while (jj < 0) jj += ny; while (jj >= ny) jj -= ny; } else iny = jj >= 0 && jj < ny;
        int rr = min(max(jj, -OCN_HALO), ny + OCN_HALO) + OCN_HALO;
        const float rdxr = P.rdxC[rr], rAzr = P.rAzC[rr];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int x = x0 + r;
            int ii = i0 - H + x;
            bool in = on && iny;
            if (P.px) { while (ii < 0) ii += nx; while (ii >= nx) ii -= nx; } else in = in && ii >= 0 && ii < nx;
            e[r] = u[r] = v[r] = ce[r] = cu[r] = cv[r] = gu[r] = gv[r] = be[r] = bU[r] = bV[r] = 0.f;
            cidx[r] = -1;
            if (in) {
                const int c = (jj + OCN_HALO) * sx + ii;
                const uint2 m = P.m8[c];
                const bool wet = (m.x & 255u) < (unsigned)nz, ou = ((m.x >> 8) & 255u) < (unsigned)nz, ov = (m.y & 255u) < (unsigned)nz;
                if (wet | ou | ov) { e[r] = P.eta[cur][c]; u[r] = P.U[cur][c]; v[r] = P.V[cur][c]; }
                if (x < EX - 1 && y < EY - 1 && wet) ce[r] = dtau * rAzr;
                if (x > 0 && ou) { cu[r] = dtau * g * P.Hu[c] * rdxr; gu[r] = dtau * P.GU[c]; }
                if (y > 0 && ov) { cv[r] = dtau * g * P.Hv[c] * rdy; gv[r] = dtau * P.GV[c]; }
                const int xi = x - H, yi = y - H;
                if (xi >= 0 && xi < BTX && yi >= 0 && yi < BTY && i0 + xi < nx && j0 + yi < ny) {
                    cidx[r] = c;                    // interior points are inside the domain: no wrap happened
                    if (!first) { be[r] = P.etab[c]; bU[r] = P.Ub[c]; bV[r] = P.Vb[c]; }
                }
            }
        }
    }
    if (on) {
        *(float4*)(sU + qb) = make_float4(u[0], u[1], u[2], u[3]);
        *(float4*)(sV + qb) = make_float4(v[0], v[1], v[2], v[3]);
    }
    __syncthreads();
    const int qe = min(qb + 4, EX * EY - 1);                    // U east of the strip (rim: ce = 0)
    const int qn = (y < EY - 1 ? qb + EX : qb);                 // V row north of the strip
    const int qw = max(qb - 1, 0);                              // eta west of the strip (rim: cu = 0)
    const int qs = (y > 0 ? qb - EX : qb);                      // eta row south of the strip
    const float dFs = dF[y], dFn = dF[y + 1];
    for (int s = 0; s < ns; ++s) {
        if (on) {
            const float ue = sU[qe];
            const float4 vn = *(const float4*)(sV + qn);
            e[0] = e[0] - ce[0] * (dy * (u[1] - u[0]) + dFn * vn.x - dFs * v[0]);
            e[1] = e[1] - ce[1] * (dy * (u[2] - u[1]) + dFn * vn.y - dFs * v[1]);
            e[2] = e[2] - ce[2] * (dy * (u[3] - u[2]) + dFn * vn.z - dFs * v[2]);
            e[3] = e[3] - ce[3] * (dy * (ue - u[3]) + dFn * vn.w - dFs * v[3]);
            *(float4*)(se + qb) = make_float4(e[0], e[1], e[2], e[3]);
        }
        __syncthreads();
        if (on) {
            const float am = saw[s], bm = sbw[s];
            const float ew = se[qw];
            const float4 es = *(const float4*)(se + qs);
            u[0] = u[0] + (cu[0] * (ew - e[0]) + gu[0]);
            u[1] = u[1] + (cu[1] * (e[0] - e[1]) + gu[1]);
            u[2] = u[2] + (cu[2] * (e[1] - e[2]) + gu[2]);
            u[3] = u[3] + (cu[3] * (e[2] - e[3]) + gu[3]);
            v[0] = v[0] + (cv[0] * (es.x - e[0]) + gv[0]);
            v[1] = v[1] + (cv[1] * (es.y - e[1]) + gv[1]);
            v[2] = v[2] + (cv[2] * (es.z - e[2]) + gv[2]);
            v[3] = v[3] + (cv[3] * (es.w - e[3]) + gv[3]);
#pragma unroll
            for (int r = 0; r < 4; ++r) { be[r] += am * e[r]; bU[r] += bm * u[r]; bV[r] += bm * v[r]; }
            *(float4*)(sU + qb) = make_float4(u[0], u[1], u[2], u[3]);
            *(float4*)(sV + qb) = make_float4(v[0], v[1], v[2], v[3]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        if (cidx[r] >= 0) {
            const int c = cidx[r];
            P.eta[cur ^ 1][c] = e[r]; P.U[cur ^ 1][c] = u[r]; P.V[cur ^ 1][c] = v[r];
            P.etab[c] = be[r]; P.Ub[c] = bU[r]; P.Vb[c] = bV[r];
        }
    }
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
// Rows of up to 8 plane-layout arrays <-> one contiguous buffer in ONE launch (ocn_pack_rows / ocn_unpack_rows: the overlap
// rows of a latitude band).  Every chunk is a whole number of 16-byte words (sx is a multiple of 32 elements
// and a chunk starts 4 elements before a row): plain uint4 copies, x = words of a plane's chunk, y = plane, z = array.
// ---------------------------------------------------------------------------------------------
struct RowMoves {
    struct One { const uint4* src; uint4* dst; long long src_pitch, dst_pitch; int planes; } a[8];   // pitches in 16-byte words
    unsigned w[8];                                                                                     // words of one plane's chunk
};
__global__ void __launch_bounds__(256) k_move_rows(const RowMoves R) {
    const RowMoves::One& A = R.a[blockIdx.z];
    const unsigned x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= R.w[blockIdx.z]) return;
    for (int pl = blockIdx.y; pl < A.planes; pl += gridDim.y) A.dst[pl * A.dst_pitch + x] = A.src[pl * A.src_pitch + x];
}

// ---------------------------------------------------------------------------------------------
// S4 (back-substitution, top-down) + S7 (barotropic correction) + S9 (hydrostatic pressure of
// the new T, S, integrated downward from the surface in the same sweep).
// The implicit operator conserves the column integral, so sum_k dz u** = sum_k dz u* (SU from
// K1) and the correction (Ubar - SU) / Hu is known before the sweep.
// ---------------------------------------------------------------------------------------------
// RI = true (closure 1): the modified super-diagonals come from the arrays K5 wrote instead of the tables.
// The launch covers rows Q.own_lo .. Q.own_hi - 1 (all rows of a model on its own).
// PUT (latitude bands with fused puts): what is stored in rows a neighbouring band overlaps is stored into the
// neighbour's arrays as well (Q.side; peer memory), so the new 3-D state needs no exchange afterwards.  The host launches it on
// the band's own rows; its overlap rows are not processed at all (the neighbours' puts fill them).  (Launched on the mirrored
// rows alone, with the plain kernel on the rest, it was slower: a launch of 11 rows is one latency-bound column sweep, 118 us.)
template <class T, bool RI, bool PUT = false>
__global__ void __launch_bounds__(128, sizeof(T) == 8 ? 4 : 8) k_backsub_correct(const DevP<T> P, const PeerPut<T> Q) {
    typedef Ex<T> E;
    typedef typename Pair<T>::type T2;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = Q.own_lo + blockIdx.y * blockDim.y + threadIdx.y;
    if (j >= Q.own_hi) return;                              // uniform over the warp (blockDim.x is a multiple of 32)
    const bool to0 = PUT && j >= Q.side[0].lo && j < Q.side[0].hi, to1 = PUT && j >= Q.side[1].lo && j < Q.side[1].hi;
    const bool incol = i < P.nx;
    const int sx = P.sx, nz = P.nz;
    const long long sz = P.sz, c = (long long)(j + OCN_HALO) * sx + min(i, P.nx - 1);
    const uint2 m = P.m8[c];
    const int kb = incol ? (int)(m.x & 255) : nz, tx1 = incol ? (int)((m.x >> 8) & 255) : nz, ty1 = incol ? (int)(m.y & 255) : nz;
    const int kuv = min(tx1, ty1);
    // Sector-complete stores: the four columns that share a 32-byte sector of a pair / fp64 plane start at the
    // shallowest of their first levels and the dry ones store the zeros that are there already, so that L2 never has
    // to fetch a partly written sector from HBM.
    int kg = min(kb, __shfl_xor_sync(0xffffffffu, kb, 1));
    kg = min(kg, __shfl_xor_sync(0xffffffffu, kg, 2));
    int kguv = min(kuv, __shfl_xor_sync(0xffffffffu, kuv, 1));
    kguv = min(kguv, __shfl_xor_sync(0xffffffffu, kguv, 2));
    if (kg >= nz || !incol) return;
    const T cu = tx1 < nz ? (P.Ub[c] - P.SU[c]) * P.rHu[c] : T(0);
    const T cv = ty1 < nz ? (P.Vb[c] - P.SV[c]) * P.rHv[c] : T(0);
    const T* __restrict__ cpu = P.cp_m + min(tx1, nz - 1);
    const T* __restrict__ cpv = P.cp_m + min(ty1, nz - 1);
    const T* __restrict__ cpt = P.cp_t + min(kb, nz - 1);
    T xu = 0, xv = 0, xt = 0, xs = 0;
    double b1 = 0, pk = 0;
    // columns next to a periodic edge also write their halo images; all others store straight
    const bool edge = (P.px && (i < OCN_HALO || i >= P.nx - OCN_HALO)) || (P.py && (j < OCN_HALO || j >= P.ny - OCN_HALO));
    // q0, q1: the same array of the southern / northern neighbour (PUT only)
    auto put = [&](auto* plane, auto* q0, auto* q1, int k, auto val) {
        const long long o = k * sz + c;
        if (edge) store_halo(plane + (o - c), sx, P.nx, P.ny, P.px, P.py, j, i, val);
        else plane[o] = val;
        if constexpr (PUT) {
            if (to0) store_halo(q0 + k * Q.side[0].sz, sx, P.nx, Q.side[0].ny, P.px, 0, j + Q.side[0].dj, i, val);
            if (to1) store_halo(q1 + k * Q.side[1].sz, sx, P.nx, Q.side[1].ny, P.px, 0, j + Q.side[1].dj, i, val);
        }
    };
#ifndef K3_NB
#define K3_NB 3
#endif
#ifndef K3_PF_DIST
#define K3_PF_DIST (RI ? 0 : (sizeof(T) == 8 ? 2 : 1))
#endif
    constexpr int NB = K3_NB;                              // levels whose loads are in flight together (measured best with 8 CTAs / SM)
    for (int k0 = nz - 1; k0 >= kg; k0 -= NB) {
        T2 d_ts[NB], d_uv[NB], c_uv[NB];
        T c_t[NB];
        // The lines of a later group into L2 (no registers held): the loads below then find them there.  K3 1.94 -> 1.75 ms on
        // config 4 one group ahead, 0.82 -> 0.73 ms in fp64 (config 2) two groups ahead; with the closure's two extra arrays in
        // flight it gains nothing (2.03 against 2.04 ms) and two groups ahead cost 4 %: off there (profiles/r2_ncu_summary.md §10).
        constexpr int PF = K3_PF_DIST;
        if (PF > 0) {
#pragma unroll
            for (int q = 0; q < NB; ++q) {
                const int k = k0 - PF * NB - q;
                if (k >= kb) {
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(P.dts + k * sz + c));
                    if (k >= kuv) asm volatile("prefetch.global.L2 [%0];" ::"l"(P.duv + k * sz + c));
                }
            }
        }
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            const int k = k0 - q;
            d_ts[q] = mk2(T(0), T(0)); d_uv[q] = mk2(T(0), T(0)); c_uv[q] = mk2(T(0), T(0)); c_t[q] = T(0);
            if (k >= kb) {
                d_ts[q] = P.dts[k * sz + c];
                if (RI) c_t[q] = P.cpt[k * sz + c];
                if (k >= kuv) { d_uv[q] = P.duv[k * sz + c]; if (RI) c_uv[q] = P.cpuv[k * sz + c]; }
            }
        }
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            const int k = k0 - q;
            if (k < kg) break;
            T2 ots = mk2(T(0), T(0));
            double op = 0.0;
            if (k >= kb) {
                const T ck = RI ? c_t[q] : cpt[k * nz];
                xt = E::sub(d_ts[q].x, E::mul(ck, xt));                      // cp[nz-1] = 0
                xs = E::sub(d_ts[q].y, E::mul(ck, xs));
                const double b0 = buoyancy(P, k, xt, xs);
                pk = pressure_level(P, k, b0, b1, pk);
                b1 = b0;
                ots = mk2(xt, xs); op = pk;
            }
            const long long o = k * sz + c;
            put(P.ts, Q.side[0].ts, Q.side[1].ts, k, ots);
            put(P.p, Q.side[0].p, Q.side[1].p, k, op);
            if (k >= kguv) {
                const bool mu = k >= tx1, mv = k >= ty1;
                T un = 0, vn = 0;
                if (mu) { xu = E::sub(d_uv[q].x, E::mul(RI ? c_uv[q].x : cpu[k * nz], xu)); un = xu + cu; }
                if (mv) { xv = E::sub(d_uv[q].y, E::mul(RI ? c_uv[q].y : cpv[k * nz], xv)); vn = xv + cv; }
                if (sizeof(T) == 8) { if (mu | mv) P.uv[o] = mk2(xu * T(mu), xv * T(mv)); }    // u**, corrected below
                else put(P.uv, Q.side[0].uv, Q.side[1].uv, k, mk2(un, vn));
            }
        }
    }
    if (kuv >= nz) return;
    if (sizeof(T) == 8) {
        // fp64: the correction as DESIGN.md §3.8 step 8 writes it, (Ubar - sum_k dz u**) / Hu with the sum taken
        // bottom-up over the back-substituted column (the fp32 path uses K1's sum of the predictor instead)
        double su = 0.0, sv = 0.0;
        for (int k = kuv; k < nz; ++k) {
            const T2 q = P.uv[k * sz + c];
            su = (X(su) + X((double)P.dz[k]) * X((double)q.x)).v;
            sv = (X(sv) + X((double)P.dz[k]) * X((double)q.y)).v;
        }
        const double cu2 = tx1 < nz ? ((X((double)P.Ub[c]) - X(su)) / X((double)P.Hu[c])).v : 0.0;
        const double cv2 = ty1 < nz ? ((X((double)P.Vb[c]) - X(sv)) / X((double)P.Hv[c])).v : 0.0;
        for (int k = kuv; k < nz; ++k) {
            const T2 q = P.uv[k * sz + c];
            const T un = k >= tx1 ? (T)(X((double)q.x) + X(cu2)).v : T(0);
            const T vn = k >= ty1 ? (T)(X((double)q.y) + X(cv2)).v : T(0);
            store_halo(P.uv + k * sz, sx, P.nx, P.ny, P.px, P.py, j, i, mk2(un, vn));
            if constexpr (PUT) {
                if (to0) store_halo(Q.side[0].uv + k * Q.side[0].sz, sx, P.nx, Q.side[0].ny, P.px, 0, j + Q.side[0].dj, i, mk2(un, vn));
                if (to1) store_halo(Q.side[1].uv + k * Q.side[1].sz, sx, P.nx, Q.side[1].ny, P.px, 0, j + Q.side[1].dj, i, mk2(un, vn));
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
    double b1 = 0, pk = 0;
    for (int k = nz - 1; k >= kb; --k) {
        const typename Pair<T>::type q = P.ts[k * sz + c];
        const double b0 = buoyancy(P, k, q.x, q.y);
        pk = pressure_level(P, k, b0, b1, pk);
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
    const T dy = P.dy, dF0 = P.dxF[r], dF1 = P.dxF[r + 1], rA = P.rAzC[r], A = P.AzC[r];
    double w = 0.0;
    for (int k = 0; k < nz; ++k) {
        const typename Pair<T>::type* __restrict__ q = P.uv + k * sz + c;
        const T D = xdiv(X(dy) * (X(q[1].x) - X(q[0].x)) + X(dF1) * X(q[sx].y) - X(dF0) * X(q[0].y), A, rA).v;
        w = (X(w) - X((double)P.dz[k]) * X((double)D)).v;
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
    for (int k = 0; k < P.nz; ++k) { const typename Pair<T>::type q = P.uv[k * sz + c]; su = (X(su) + X((double)P.dz[k]) * X((double)q.x)).v; sv = (X(sv) + X((double)P.dz[k]) * X((double)q.y)).v; }
    store_halo(P.U[0], P.sx, P.nx, P.ny, P.px, P.py, j, i, (T)su);
    store_halo(P.V[0], P.sx, P.nx, P.ny, P.px, P.py, j, i, (T)sv);
}

// ---------------------------------------------------------------------------------------------
// Self-test of ddiv_m (common.cuh): counts operand pairs for which the three-instruction quotient differs from __ddiv_rn.
// Operands: counter-based pseudo-random mantissas and exponents in the range the model's quantities live in, every fourth
// pair with mantissas within a few ulps of 1 or 2 (the hard cases of reciprocal-based division), every eighth with b = 6.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
    z += 0x9e3779b97f4a7c15ull; z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull; z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
    return z ^ (z >> 31);
}
__global__ void k_selftest_division(unsigned long long n, unsigned long long seed, unsigned long long* bad) {
    unsigned long long local = 0;
    for (unsigned long long q = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; q < n; q += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long ra = mix64(seed + 2 * q), rb = mix64(seed + 2 * q + 1);
        unsigned long long ma = ra & 0xfffffffffffffull, mb = rb & 0xfffffffffffffull;
        if ((q & 3) == 1) { ma = (ra >> 52 & 1) ? (ma & 7) : (0xfffffffffffffull - (ma & 7)); }
        if ((q & 3) == 2) { mb = (rb >> 52 & 1) ? (mb & 7) : (0xfffffffffffffull - (mb & 7)); }
        const int ea = 1023 + (int)((ra >> 53) % 121) - 60, eb = 1023 + (int)((rb >> 53) % 121) - 60;     // 2^-60 .. 2^60
        double a = __longlong_as_double((long long)(((unsigned long long)ea << 52) | ma | ((ra >> 63) << 63)));
        double b = __longlong_as_double((long long)(((unsigned long long)eb << 52) | mb));
        if ((q & 7) == 7) b = 6.0;
        if ((q & 1023) == 0) a = 0.0;
        const double want = __ddiv_rn(a, b);
        const double got = (q & 7) == 7 ? ddiv_m(a, 6.0, 1.0 / 6.0) : ddiv_m(a, b, __drcp_rn(b));
        local += (want != got);
    }
    if (local) atomicAdd(bad, local);
}

// ---------------------------------------------------------------------------------------------
// ocn_check_finite: counts the words of an array (any layout: halo and land hold finite zeros) that are NaN or infinite
// ---------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(256) k_count_nonfinite(const T* __restrict__ a, unsigned long long n, unsigned long long* bad) {
    unsigned long long local = 0;
    for (unsigned long long q = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; q < n; q += (unsigned long long)gridDim.x * blockDim.x)
        local += !isfinite(a[q]);
    if (local) atomicAdd(bad, local);
}

// ---------------------------------------------------------------------------------------------
// scatter (contiguous interior -> halo'd plane layout, masked) and gather (back, land = 0)
// st = element stride of the device array (2 = one member of a pair array, base already offset)
// kind: 0 u, 1 v, 2 T (offset Toff), 3 S (offset Soff), 4 eta, 5 plain 2-D, 6 w (nz+1 levels, gather only),
//       7 / 8 a 2-D surface value of T / S (offset, zero on land columns)
// ---------------------------------------------------------------------------------------------
template <class T>
__device__ __forceinline__ bool cell_open(const DevP<T>& P, long long c, int k, int kind) {
    const uint2 m = P.m8[c];
    const int kb = m.x & 255, tx1 = (m.x >> 8) & 255, ty1 = m.y & 255;
    switch (kind) {
        case 0: return k >= tx1;
        case 1: return k >= ty1;
        case 2: case 3: return k >= kb;
        case 4: case 7: case 8: return kb < P.nz;
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
    const T off = (kind == 2 || kind == 7) ? P.Toff : (kind == 3 || kind == 8) ? P.Soff : T(0);
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
