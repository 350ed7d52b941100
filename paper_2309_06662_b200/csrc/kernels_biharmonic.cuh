// kernels_biharmonic.cuh — biharmonic horizontal dissipation: the masked C-grid Laplacians
// applied twice, as a pre-pass of two launches of ONE kernel before the tendency kernel, which then only adds the finished
// term of its own cell.  Launched only when nu4_h or kappa4_h is non-zero; the default path does not know it exists.
//
//   vector field (a at u points, b at v points; masked, halo-filled):
//     Da = [dy (a[i+1] - a[i]) + dxF[j+1] b[j+1] - dxF[j] b[j]] / AzC[j]
//     Za = [dy (b[i] - b[i-1]) - (dxC[j] a[j] - dxC[j-1] a[j-1])] / AzF[j]
//     La = mu [(Da[i] - Da[i-1]) / dxC[j] - (Za[j+1] - Za[j]) / dy],  Lb = mv [(Da[j] - Da[j-1]) / dy + (Za[i+1] - Za[i]) / dxF[j]]
//   tracer pair c (no flux through closed faces):
//     fx[i] = dy (c[i] - c[i-1]) / dxC[j] mu[i],  fy[j] = dxF[j] (c[j] - c[j-1]) / dy mv[j],
//     Lc = wet [(fx[i+1] - fx[i]) + (fy[j+1] - fy[j])] / AzC[j]
//   pass 1: (Luv, Lts) = (L(uv), L(ts));  pass 2: (Buv, Bts) = (-(nu4 L(Luv)), -(kappa4 L(Lts))).
// fp64: the association above in non-contracted IEEE operations (bit-identical to the oracle).
#pragma once
#include "common.cuh"

namespace ocn {

template <class T>
__global__ void __launch_bounds__(128) k_laplacians(const DevP<T> P, const typename Pair<T>::type* __restrict__ A,
                                                    const typename Pair<T>::type* __restrict__ Cc,
                                                    typename Pair<T>::type* __restrict__ outA,
                                                    typename Pair<T>::type* __restrict__ outC, const T coefA, const T coefC,
                                                    const int second) {
    typedef typename Pair<T>::type T2;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= P.nx || j >= P.ny) return;
    const int sx = P.sx, nz = P.nz, r = j + OCN_HALO;
    const long long sz = P.sz, c = (long long)r * sx + i;
    const uint2 m = P.m8[c], me = P.m8[c + 1], mn = P.m8[c + sx];
    const int kb = m.x & 255, tx1 = (m.x >> 8) & 255, ty1 = m.y & 255, tx1e = (me.x >> 8) & 255, ty1n = mn.y & 255;
    if (kb >= nz) return;
    const T dy = P.dy, rdy = P.rdy;
    const T dxCj = P.dxC[r], dxCs = P.dxC[r - 1], rdxCj = P.rdxC[r], dxFj = P.dxF[r], dxFn = P.dxF[r + 1], dxFs = P.dxF[r - 1], rdxFj = P.rdxF[r];
    const T AzCj = P.AzC[r], rAzCj = P.rAzC[r], AzCs = P.AzC[r - 1], rAzCs = P.rAzC[r - 1];
    const T AzFj = P.AzF[r], rAzFj = P.rAzF[r], AzFn = P.AzF[r + 1], rAzFn = P.rAzF[r + 1];
    const T dxCn = P.dxC[r + 1];
    for (int k = kb; k < nz; ++k) {
        const T2* __restrict__ a = A + k * sz + c;
        const T2* __restrict__ q = Cc + k * sz + c;
        // ---- vector Laplacian ----
        T2 oA = mk2(T(0), T(0));
        if (k >= tx1 || k >= ty1) {
            const T2 v00 = a[0], ve = a[1], vw = a[-1], vn = a[sx], vs = a[-sx], vnw = a[sx - 1], vse = a[-sx + 1];
            // divergence at (i, j), (i - 1, j), (i, j - 1)
            const Xv<T> D00 = xdiv(X(dy) * (X(ve.x) - X(v00.x)) + X(dxFn) * X(vn.y) - X(dxFj) * X(v00.y), AzCj, rAzCj);
            const Xv<T> Dw = xdiv(X(dy) * (X(v00.x) - X(vw.x)) + X(dxFn) * X(vnw.y) - X(dxFj) * X(vw.y), AzCj, rAzCj);
            const Xv<T> Ds = xdiv(X(dy) * (X(vse.x) - X(vs.x)) + X(dxFj) * X(v00.y) - X(dxFs) * X(vs.y), AzCs, rAzCs);
            // vorticity at the south-west corners of (i, j), (i, j + 1), (i + 1, j)
            const Xv<T> Z00 = xdiv(X(dy) * (X(v00.y) - X(vw.y)) - (X(dxCj) * X(v00.x) - X(dxCs) * X(vs.x)), AzFj, rAzFj);
            const Xv<T> Zn = xdiv(X(dy) * (X(vn.y) - X(vnw.y)) - (X(dxCn) * X(vn.x) - X(dxCj) * X(v00.x)), AzFn, rAzFn);
            const Xv<T> Ze = xdiv(X(dy) * (X(ve.y) - X(v00.y)) - (X(dxCj) * X(ve.x) - X(dxCs) * X(vse.x)), AzFj, rAzFj);
            const T La = k >= tx1 ? (xdiv(D00 - Dw, dxCj, rdxCj) - xdiv(Zn - Z00, dy, rdy)).v : T(0);
            const T Lb = k >= ty1 ? (xdiv(D00 - Ds, dy, rdy) + xdiv(Ze - Z00, dxFj, rdxFj)).v : T(0);
            oA = second ? mk2((-(X(coefA) * X(La))).v, (-(X(coefA) * X(Lb))).v) : mk2(La, Lb);
        }
        store_halo(outA + k * sz, sx, P.nx, P.ny, P.px, P.py, j, i, oA);
        // ---- tracer Laplacian (cell (k, j, i) is wet here) ----
        {
            const T2 c0 = q[0], ce = q[1], cw = q[-1], cn = q[sx], cs = q[-sx];
            const bool ow = k >= tx1, oe = k >= tx1e, os = k >= ty1, on = k >= ty1n;
            T2 oC;
            {
                const Xv<T> fxw = ow ? xdiv(X(dy) * (X(c0.x) - X(cw.x)), dxCj, rdxCj) : X(T(0));
                const Xv<T> fxe = oe ? xdiv(X(dy) * (X(ce.x) - X(c0.x)), dxCj, rdxCj) : X(T(0));
                const Xv<T> fys = os ? xdiv(X(dxFj) * (X(c0.x) - X(cs.x)), dy, rdy) : X(T(0));
                const Xv<T> fyn = on ? xdiv(X(dxFn) * (X(cn.x) - X(c0.x)), dy, rdy) : X(T(0));
                oC.x = xdiv((fxe - fxw) + (fyn - fys), AzCj, rAzCj).v;
            }
            {
                const Xv<T> fxw = ow ? xdiv(X(dy) * (X(c0.y) - X(cw.y)), dxCj, rdxCj) : X(T(0));
                const Xv<T> fxe = oe ? xdiv(X(dy) * (X(ce.y) - X(c0.y)), dxCj, rdxCj) : X(T(0));
                const Xv<T> fys = os ? xdiv(X(dxFj) * (X(c0.y) - X(cs.y)), dy, rdy) : X(T(0));
                const Xv<T> fyn = on ? xdiv(X(dxFn) * (X(cn.y) - X(c0.y)), dy, rdy) : X(T(0));
                oC.y = xdiv((fxe - fxw) + (fyn - fys), AzCj, rAzCj).v;
            }
            if (second) oC = mk2((-(X(coefC) * X(oC.x))).v, (-(X(coefC) * X(oC.y))).v);
            store_halo(outC + k * sz, sx, P.nx, P.ny, P.px, P.py, j, i, oC);
        }
    }
}

}  // namespace ocn
