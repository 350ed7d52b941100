// common.cuh — device-side parameter block, memory layout and small device helpers of libocn.
//
// Layout: every 3-D field is [k][j][i] with i fastest, a physical halo of 3
// cells in i and j, row pitch sx = roundup(nx + 8, 32) elements, and the base pointer shifted so
// that element (k, j, i = 0) of every row starts a 128-byte line.  The prognostic groups are
// stored interleaved, one element = a pair: uv = (u, v), ts = (T, S), and likewise their AB2
// history G and eliminated right-hand sides d, so that one 8/16-byte access moves both members
// and the tracer pair shares one set of WENO weights' worth of index arithmetic.  2-D fields use
// the same plane layout (one level).  Halos of periodic directions mirror the interior (written
// by the producing kernel through store_halo); halos of bounded directions are zero forever.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define OCN_HALO 3

namespace ocn {

template <class T> struct Pair;
template <> struct Pair<float> { typedef float2 type; };
template <> struct Pair<double> { typedef double2 type; };
template <class T> __device__ __forceinline__ typename Pair<T>::type mk2(T a, T b) { typename Pair<T>::type r; r.x = a; r.y = b; return r; }

template <class T>
struct DevP {
    typedef typename Pair<T>::type T2;
    int nx, ny, nz;
    int sx, sy;            // plane pitch / rows (with halo)
    long long sz;          // level stride = sx * sy
    int px, py;            // periodic flags
    // prognostic state (time level n) as pairs, stored pressure, w (filled on demand for
    // ocn_get_fields), eliminated right-hand sides, AB2 history
    T2 *uv, *ts;
    double* p;             // hydrostatic pressure, fp64 in both precisions
    T* w;
    T2 *duv, *dts;
    T2 *Guv, *Gts;
    // 2-D (plane layout with halo)
    T *eta[2], *U[2], *V[2];       // barotropic state, double buffered inside the sub-cycle
    T *etab, *Ub, *Vb;             // weighted running averages
    T *GU, *GV;                    // barotropic forcing
    T *SU, *SV;                    // sum_k dz u*, sum_k dz v*
    T *Hu, *Hv, *rHu, *rHv;        // depth at u / v points and reciprocals (0 on closed columns)
    T *taux, *tauy;
    T2 *qts, *rts;                 // surface tracer fluxes (flux_T, flux_S) and restoring targets (stored with the tracer offsets)
    T gamma_T, gamma_S;            // restoring piston velocities
    T drag_r, drag_cd;             // bottom drag: linear [m/s] and quadratic [-] coefficients
    // compact masks (plane layout with halo): thresholds in level index
    const uint2* m8;               // bytes: kb, tx1, tx2, tx3 | ty1, ty2, ty3, 0
    const uchar4* mz;              // zu2, zu3, zv2, zv3
    // horizontal metrics per row, index j + OCN_HALO, rows -3 .. ny+3
    const T *dxC, *dxF, *AzC, *AzF, *fF, *rdxC, *rdxF, *rAzC, *rAzF;
    T dy, rdy;
    // vertical grid
    const T *dz, *rdz, *dzc;       // dzc[k] = zc[k] - zc[k-1] (k >= 1)
    const T *rdzc;                 // 1 / dzc[k] (k >= 1; entry 0 is 1)
    T hz_top;                      // zf[nz] - zc[nz-1]
    // Thomas tables, bottom-up elimination in the oracle's order.  Momentum (nu_z)
    // and tracers (kappa_z).  sm[k]: sub-diagonal s^-_k (open face below); cp/m/rm are indexed
    // [k * nz + kf] by the column's first open level kf: cp = modified super-diagonal, m = pivot,
    // rm = 1 / m.
    const T *sm_m, *cp_m, *m_m, *rm_m;
    const T *sm_t, *cp_t, *m_t, *rm_t;
    // physics
    T dt, g, alpha, beta_s, rho0, rrho0, nu_h, kappa_h;
    T Toff, Soff;          // storage offsets of the tracers: (T0, S0) in fp32, 0 in fp64
    T dT0, dS0;            // T0 - Toff, S0 - Soff: what is left to subtract in the buoyancy
    double g_d, alpha_d, beta_d, dT0_d, dS0_d, hz_top_d;   // fp64 copies for the pressure integral
    const double* dzc_d;
    T dtau;
    const T *fw_a, *fw_b;  // filter weights a_m of eta and b_m of the transports, m = 1..M at index m - 1
    // Ri-based vertical mixing closure, closure = 1 only: (nu, kappa) at the bottom face of
    // tracer cell (k, j, i) as a pair array, and the modified super-diagonals of the per-column Thomas solves
    int closure;
    T2* nk;
    T2* cpuv;
    T* cpt;
    double ri_nu0, ri_c, ri_kconv, ri_n2c, ri_s2min, nu_z_d, kappa_z_d;
    // equation of state: eos = 1 adds thermobaricity and cabbeling,
    //   b = g [ath[k] dT + ha2 dT dT - beta dS],  ath[k] = alpha (1 - gamma zc[k]),  ha2 = alpha2 / 2   (built on the host in fp64)
    int eos;
    const double* ath_d;
    double ha2_d;
    // biharmonic horizontal dissipation: scratch Laplacians and the finished terms K1 adds (bih = 1 only)
    int bih;
    T2 *Luv, *Lts, *Buv, *Bts;
    // K1: wet cells of a tile-level from which on the tile is marched with geometric ownership
    int geo_thr;
    unsigned long long* timeline;   // [8 warps][8]: cycles per phase + iterations (filled by OCN_K1_TIMELINE builds only)
};

// Latitude bands with fused puts: rows [lo, hi) of this model are ALSO stored into the neighbouring band's arrays
// (peer memory: the same device, or another GPU's over NVLink) by the kernel that produces the new 3-D state, and rows outside
// [own_lo, own_hi) are not stored at all (the neighbour that owns them stores them here the same way).  Only arrays that no
// other part of a step touches are put this way: (u, v), (T, S), p.  The 2-D state is scratch of the sub-cycle until a step ends.
template <class T>
struct PeerSide {
    typedef typename Pair<T>::type T2;
    int lo, hi;            // local rows that are mirrored (hi <= lo: none)
    int dj;                // the neighbour's row of my row j is j + dj
    int ny;                // the neighbour's ny
    long long sz;          // the neighbour's level stride (its sx is mine)
    T2 *uv, *ts;
    double* p;
};
template <class T>
struct PeerPut {
    PeerSide<T> side[2];   // 0: the band to the south, 1: the band to the north
    int own_lo, own_hi;
};

template <class T>
__device__ __forceinline__ T ldg(const T* p) { return __ldg(p); }

// Arithmetic whose rounding order is fixed (no FMA contraction) in fp64, so that the tracer /
// pressure column passes reproduce the rounding sequence of the discrete equations as written
// (DESIGN.md §6.5); fp32 lets the compiler contract and divides by multiplying with rm.
// Correctly rounded fp64 quotient from a correctly rounded reciprocal rb = RN(1 / b) (Markstein's correction: q = RN(a rb),
// r = a - q b exactly by FMA, RN(q + r rb) = RN(a / b) when nothing under- or overflows): three instructions where
// __ddiv_rn needs about twenty-five.  The reciprocals are the host's fp64 tables (1.0 / x), compile-time constants, or
// __drcp_rn.  ocn_selftest_division compares it with __ddiv_rn on random and adversarial operands (tests/test_gpu_parity.py).
__device__ __forceinline__ double ddiv_m(double a, double b, double rb) {
    const double q = __dmul_rn(a, rb);
    return __fma_rn(__fma_rn(-q, b, a), rb, q);
}
__device__ __forceinline__ double xrcp(double b, double) { return __drcp_rn(b); }
__device__ __forceinline__ float xrcp(float, float approx) { return approx; }

template <class T> struct Ex;
template <> struct Ex<double> {
    static __device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
    static __device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
    static __device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
    static __device__ __forceinline__ double div(double a, double m, double) { return ddiv_m(a, m, __drcp_rn(m)); }
};
template <> struct Ex<float> {
    static __device__ __forceinline__ float mul(float a, float b) { return a * b; }
    static __device__ __forceinline__ float add(float a, float b) { return a + b; }
    static __device__ __forceinline__ float sub(float a, float b) { return a - b; }
    static __device__ __forceinline__ float div(float a, float, float rm) { return a * rm; }
};

// store a value and its periodic halo images (up to 3 extra copies); T may be a pair type
template <class T>
__device__ __forceinline__ void store_halo(T* __restrict__ plane, int sx, int nx, int ny, int px, int py,
                                           int j, int i, T val, int st = 1) {
    // st: element stride of the plane (2 when addressing one member of a pair array as scalars)
    T* p = plane + ((long long)(j + OCN_HALO) * sx + i) * st;
    *p = val;
    const long long row = (long long)sx * st;
    int di = 0, dj = 0;
    if (px) { if (i < OCN_HALO) di = nx; else if (i >= nx - OCN_HALO) di = -nx; }
    if (py) { if (j < OCN_HALO) dj = ny; else if (j >= ny - OCN_HALO) dj = -ny; }
    if (di) p[di * st] = val;
    if (dj) p[dj * row] = val;
    if (di && dj) p[dj * row + di * st] = val;
    // very small periodic domains (n < 6): a cell can be the image of both halos
    if (px && nx < 2 * OCN_HALO) {
        if (i < OCN_HALO && i >= nx - OCN_HALO) { p[-nx * st] = val; if (dj) p[dj * row - nx * st] = val; }
    }
    if (py && ny < 2 * OCN_HALO) {
        if (j < OCN_HALO && j >= ny - OCN_HALO) {
            p[-ny * row] = val;
            if (di) p[-ny * row + di * st] = val;
            if (px && nx < 2 * OCN_HALO && i < OCN_HALO && i >= nx - OCN_HALO) p[-ny * row - nx * st] = val;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Xv<T>: a value whose arithmetic keeps the written association.  In fp64 every operator is a
// correctly rounded, non-contracted IEEE operation (__dmul_rn, ...), so an expression written in
// the order of DESIGN.md §3 rounds exactly like the equations as written; in fp32
// the operators are plain and the compiler is free to contract.  xdiv(a, b, rb) = a / b in fp64 and
// a * rb (rb = 1 / b, precomputed) in fp32.
// ---------------------------------------------------------------------------------------------
template <class T> struct Xv { T v; __device__ __forceinline__ explicit Xv(T x) : v(x) {} __device__ __forceinline__ Xv() : v(0) {} };
__device__ __forceinline__ Xv<double> operator*(Xv<double> a, Xv<double> b) { return Xv<double>(__dmul_rn(a.v, b.v)); }
__device__ __forceinline__ Xv<double> operator+(Xv<double> a, Xv<double> b) { return Xv<double>(__dadd_rn(a.v, b.v)); }
__device__ __forceinline__ Xv<double> operator-(Xv<double> a, Xv<double> b) { return Xv<double>(__dsub_rn(a.v, b.v)); }
__device__ __forceinline__ Xv<double> operator/(Xv<double> a, Xv<double> b) { return Xv<double>(ddiv_m(a.v, b.v, __drcp_rn(b.v))); }
__device__ __forceinline__ Xv<double> operator-(Xv<double> a) { return Xv<double>(-a.v); }
__device__ __forceinline__ Xv<float> operator*(Xv<float> a, Xv<float> b) { return Xv<float>(a.v * b.v); }
__device__ __forceinline__ Xv<float> operator+(Xv<float> a, Xv<float> b) { return Xv<float>(a.v + b.v); }
__device__ __forceinline__ Xv<float> operator-(Xv<float> a, Xv<float> b) { return Xv<float>(a.v - b.v); }
__device__ __forceinline__ Xv<float> operator/(Xv<float> a, Xv<float> b) { return Xv<float>(a.v / b.v); }
__device__ __forceinline__ Xv<float> operator-(Xv<float> a) { return Xv<float>(-a.v); }
// rb MUST be RN(1 / b): a host table entry or xrcp(b, .)
__device__ __forceinline__ Xv<double> xdiv(Xv<double> a, double b, double rb) { return Xv<double>(ddiv_m(a.v, b, rb)); }
__device__ __forceinline__ Xv<float> xdiv(Xv<float> a, float, float rb) { return Xv<float>(a.v * rb); }
template <class T> __device__ __forceinline__ Xv<T> X(T v) { return Xv<T>(v); }

// fp64 face value with the weights evaluated as written in DESIGN.md §3.4 (alpha_s = d_s / (eps + beta_s)^2) or, WZ, as
// written in DESIGN.md §3.15 (WENO-Z: alpha_s = d_s (1 + (tau / (eps + beta_s))^2), tau = |beta_0 - beta_{r-1}|)
template <bool WZ>
__device__ __forceinline__ double weno_face_exact(double a, double b, double c, double d, double e, double f, double vel, int order) {
    typedef Xv<double> V;
    const bool pos = vel > 0.0;
    const V qm2(pos ? a : f), qm1(pos ? b : e), q0(pos ? c : d), q1(pos ? d : c), q2(pos ? e : b);
    const V eps(1e-6), two(2.0);
    if (order >= 3) {
        // x / 6.0 with the compile-time reciprocal (correctly rounded, see ddiv_m)
        const V p0(ddiv_m((two * qm2 - V(7.0) * qm1 + V(11.0) * q0).v, 6.0, 1.0 / 6.0));
        const V p1(ddiv_m((-qm1 + V(5.0) * q0 + two * q1).v, 6.0, 1.0 / 6.0));
        const V p2(ddiv_m((two * q0 + V(5.0) * q1 - q2).v, 6.0, 1.0 / 6.0));
        const V c13(13.0 / 12.0), c4(0.25);
        const V b0 = c13 * (qm2 - two * qm1 + q0) * (qm2 - two * qm1 + q0) + c4 * (qm2 - V(4.0) * qm1 + V(3.0) * q0) * (qm2 - V(4.0) * qm1 + V(3.0) * q0);
        const V b1 = c13 * (qm1 - two * q0 + q1) * (qm1 - two * q0 + q1) + c4 * (qm1 - q1) * (qm1 - q1);
        const V b2 = c13 * (q0 - two * q1 + q2) * (q0 - two * q1 + q2) + c4 * (V(3.0) * q0 - V(4.0) * q1 + q2) * (V(3.0) * q0 - V(4.0) * q1 + q2);
        if (WZ) {
            const V tau(fabs((b0 - b2).v)), one(1.0);
            const V r0 = tau / (eps + b0), r1 = tau / (eps + b1), r2 = tau / (eps + b2);
            const V a0 = V(0.1) * (one + r0 * r0), a1 = V(0.6) * (one + r1 * r1), a2 = V(0.3) * (one + r2 * r2);
            return ((a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2)).v;
        }
        const V a0 = V(0.1) / ((eps + b0) * (eps + b0)), a1 = V(0.6) / ((eps + b1) * (eps + b1)), a2 = V(0.3) / ((eps + b2) * (eps + b2));
        return ((a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2)).v;
    }
    if (order == 2) {
        const V p0 = (-qm1 + V(3.0) * q0) * V(0.5), p1 = (q0 + q1) * V(0.5);      // x / 2 is exact
        const V b0 = (q0 - qm1) * (q0 - qm1), b1 = (q1 - q0) * (q1 - q0);
        if (WZ) {
            const V tau(fabs((b0 - b1).v)), one(1.0);
            const V r0 = tau / (eps + b0), r1 = tau / (eps + b1);
            const V a0 = V(1.0 / 3.0) * (one + r0 * r0), a1 = V(2.0 / 3.0) * (one + r1 * r1);
            return ((a0 * p0 + a1 * p1) / (a0 + a1)).v;
        }
        const V a0 = V(1.0 / 3.0) / ((eps + b0) * (eps + b0)), a1 = V(2.0 / 3.0) / ((eps + b1) * (eps + b1));
        return ((a0 * p0 + a1 * p1) / (a0 + a1)).v;
    }
    return order == 1 ? q0.v : 0.0;
}

// ---------------------------------------------------------------------------------------------
// WENO face value (Shu 1997 as cited at PAPER.md:244).  Cells n-3..n+2 are
// (a, b, c, d, e, f); the face lies between c and d; q0 is the upwind cell.
// Division-free nonlinear weights: alpha_s ~ d_s * prod_{t != s} (eps + beta_t)^2, one division.
// ---------------------------------------------------------------------------------------------
template <bool WZ>
__device__ __forceinline__ double weno_face(double a, double b, double c, double d, double e, double f, double vel, int order) {
    return weno_face_exact<WZ>(a, b, c, d, e, f, vel, order);
}
// quotient of the weighted sum: reciprocal-based in fp32 (2 ulp), exact in fp64
__device__ __forceinline__ float fquot(float a, float b) { return __fdividef(a, b); }
__device__ __forceinline__ double fquot(double a, double b) { return a / b; }
// WZ (fp32): the WENO-Z weights in the same division-free form, alpha_s ~ d_s (B_s^2 + tau^2) prod_{t != s} B_t^2 with
// B = eps + beta (>= 1e-6, so the triple products stay normal numbers)
template <bool WZ>
__device__ __forceinline__ float weno_face(float a, float b, float c, float d, float e, float f, float vel, int order) {
    typedef float T;
    const bool pos = vel > T(0);
    const T qm2 = pos ? a : f, qm1 = pos ? b : e, q0 = pos ? c : d, q1 = pos ? d : c, q2 = pos ? e : b;
    const T eps = T(1e-6);
    if (order >= 3) {
        const T p0 = (T(2) * qm2 - T(7) * qm1 + T(11) * q0) * T(1.0 / 6.0);
        const T p1 = (-qm1 + T(5) * q0 + T(2) * q1) * T(1.0 / 6.0);
        const T p2 = (T(2) * q0 + T(5) * q1 - q2) * T(1.0 / 6.0);
        const T s0 = qm2 - T(2) * qm1 + q0, t0 = qm2 - T(4) * qm1 + T(3) * q0;
        const T s1 = qm1 - T(2) * q0 + q1, t1 = qm1 - q1;
        const T s2 = q0 - T(2) * q1 + q2, t2 = T(3) * q0 - T(4) * q1 + q2;
        const T b0 = eps + T(13.0 / 12.0) * s0 * s0 + T(0.25) * t0 * t0;
        const T b1 = eps + T(13.0 / 12.0) * s1 * s1 + T(0.25) * t1 * t1;
        const T b2 = eps + T(13.0 / 12.0) * s2 * s2 + T(0.25) * t2 * t2;
        if (WZ) {
            const T tau = b0 - b2, t2 = tau * tau, q0_ = b0 * b0, q1_ = b1 * b1, q2_ = b2 * b2;
            const T a0 = T(0.1) * (q0_ + t2) * (q1_ * q2_), a1 = T(0.6) * (q1_ + t2) * (q0_ * q2_), a2 = T(0.3) * (q2_ + t2) * (q0_ * q1_);
            return fquot(a0 * p0 + a1 * p1 + a2 * p2, a0 + a1 + a2);
        }
        const T b01 = b0 * b1, b02 = b0 * b2, b12 = b1 * b2;
        const T a0 = T(0.1) * b12 * b12, a1 = T(0.6) * b02 * b02, a2 = T(0.3) * b01 * b01;
        return fquot(a0 * p0 + a1 * p1 + a2 * p2, a0 + a1 + a2);
    }
    if (order == 2) {
        const T p0 = T(0.5) * (T(3) * q0 - qm1), p1 = T(0.5) * (q0 + q1);
        const T b0 = eps + (q0 - qm1) * (q0 - qm1), b1 = eps + (q1 - q0) * (q1 - q0);
        if (WZ) {
            const T tau = b0 - b1, t2 = tau * tau, q0_ = b0 * b0, q1_ = b1 * b1;
            const T a0 = T(1.0 / 3.0) * (q0_ + t2) * q1_, a1 = T(2.0 / 3.0) * (q1_ + t2) * q0_;
            return fquot(a0 * p0 + a1 * p1, a0 + a1);
        }
        const T a0 = T(1.0 / 3.0) * b1 * b1, a1 = T(2.0 / 3.0) * b0 * b0;
        return fquot(a0 * p0 + a1 * p1, a0 + a1);
    }
    return order == 1 ? q0 : T(0);
}

// ---------------------------------------------------------------------------------------------
// fp32 pair arithmetic (Blackwell packed fp32: add/mul/fma.rn.f32x2 -> SASS FADD2 / FMUL2 / FFMA2).
// The (T, S) pair shares velocity, order and stencil geometry, and the two vorticity
// reconstructions of a cell share the arithmetic, so one packed instruction serves both members.
// The weights are the same division-free form as weno_face; the final quotient uses the
// hardware reciprocal (2 ulp), well inside the fp32 tolerance.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }

// fifth-order face value from the upwind-ordered stencil (q0 = upwind cell)
template <bool WZ>
__device__ __forceinline__ float2 weno5_pair(float2 qm2, float2 qm1, float2 q0, float2 q1, float2 q2) {
    const float2 p0 = fma2(f2(11.f / 6.f), q0, fma2(f2(-7.f / 6.f), qm1, mul2(f2(2.f / 6.f), qm2)));
    const float2 p1 = fma2(f2(2.f / 6.f), q1, fma2(f2(5.f / 6.f), q0, mul2(f2(-1.f / 6.f), qm1)));
    const float2 p2 = fma2(f2(-1.f / 6.f), q2, fma2(f2(5.f / 6.f), q1, mul2(f2(2.f / 6.f), q0)));
    const float2 s0 = fma2(f2(-2.f), qm1, add2(qm2, q0)), t0 = fma2(f2(3.f), q0, fma2(f2(-4.f), qm1, qm2));
    const float2 s1 = fma2(f2(-2.f), q0, add2(qm1, q1)), t1 = fma2(f2(-1.f), q1, qm1);
    const float2 s2 = fma2(f2(-2.f), q1, add2(q0, q2)), t2 = fma2(f2(3.f), q0, fma2(f2(-4.f), q1, q2));
    const float2 eps = f2(1e-6f), c13 = f2(13.f / 12.f), c4 = f2(0.25f);
    const float2 b0 = fma2(mul2(c13, s0), s0, fma2(mul2(c4, t0), t0, eps));
    const float2 b1 = fma2(mul2(c13, s1), s1, fma2(mul2(c4, t1), t1, eps));
    const float2 b2 = fma2(mul2(c13, s2), s2, fma2(mul2(c4, t2), t2, eps));
    float2 a0, a1, a2;
    if (WZ) {
        const float2 tau = fma2(f2(-1.f), b2, b0), t2 = mul2(tau, tau);
        const float2 r0 = mul2(b0, b0), r1 = mul2(b1, b1), r2 = mul2(b2, b2);
        a0 = mul2(mul2(f2(0.1f), add2(r0, t2)), mul2(r1, r2));
        a1 = mul2(mul2(f2(0.6f), add2(r1, t2)), mul2(r0, r2));
        a2 = mul2(mul2(f2(0.3f), add2(r2, t2)), mul2(r0, r1));
    } else {
        const float2 b01 = mul2(b0, b1), b02 = mul2(b0, b2), b12 = mul2(b1, b2);
        a0 = mul2(mul2(f2(0.1f), b12), b12); a1 = mul2(mul2(f2(0.6f), b02), b02); a2 = mul2(mul2(f2(0.3f), b01), b01);
    }
    const float2 num = fma2(a2, p2, fma2(a1, p1, mul2(a0, p0))), den = add2(add2(a0, a1), a2);
    return make_float2(__fdividef(num.x, den.x), __fdividef(num.y, den.y));
}
template <bool WZ>
__device__ __forceinline__ float2 weno3_pair(float2 qm1, float2 q0, float2 q1) {
    const float2 p0 = fma2(f2(1.5f), q0, mul2(f2(-0.5f), qm1)), p1 = mul2(f2(0.5f), add2(q0, q1));
    const float2 d0 = fma2(f2(-1.f), qm1, q0), d1 = fma2(f2(-1.f), q0, q1);
    const float2 eps = f2(1e-6f);
    const float2 b0 = fma2(d0, d0, eps), b1 = fma2(d1, d1, eps);
    float2 a0, a1;
    if (WZ) {
        const float2 tau = fma2(f2(-1.f), b1, b0), t2 = mul2(tau, tau), r0 = mul2(b0, b0), r1 = mul2(b1, b1);
        a0 = mul2(mul2(f2(1.f / 3.f), add2(r0, t2)), r1); a1 = mul2(mul2(f2(2.f / 3.f), add2(r1, t2)), r0);
    } else {
        a0 = mul2(mul2(f2(1.f / 3.f), b1), b1); a1 = mul2(mul2(f2(2.f / 3.f), b0), b0);
    }
    const float2 num = fma2(a1, p1, mul2(a0, p0)), den = add2(a0, a1);
    return make_float2(__fdividef(num.x, den.x), __fdividef(num.y, den.y));
}

// face value of a pair with one advecting velocity and one order code
template <bool WZ>
__device__ __forceinline__ double2 weno_face2(double2 a, double2 b, double2 c, double2 d, double2 e, double2 f, double vel, int order) {
    double2 r;
    r.x = weno_face<WZ>(a.x, b.x, c.x, d.x, e.x, f.x, vel, order);
    r.y = weno_face<WZ>(a.y, b.y, c.y, d.y, e.y, f.y, vel, order);
    return r;
}
template <bool WZ>
__device__ __forceinline__ float2 weno_face2(float2 a, float2 b, float2 c, float2 d, float2 e, float2 f, float vel, int order) {
    const bool pos = vel > 0.f;
    const float2 qm1 = pos ? b : e, q0 = pos ? c : d, q1 = pos ? d : c;
    if (order >= 3) return weno5_pair<WZ>(pos ? a : f, qm1, q0, q1, pos ? e : b);
    if (order == 2) return weno3_pair<WZ>(qm1, q0, q1);
    return order == 1 ? q0 : make_float2(0.f, 0.f);
}

__device__ __forceinline__ int order3(int k, int t1, int t2, int t3) {
    return (k >= t1) + (k >= t2) + (k >= t3);
}

}  // namespace ocn
