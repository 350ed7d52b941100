// grid_host.h — host-side grid: metrics, bottom index map and the compact 2-D
// level-threshold masks the kernels read instead of 3-D mask arrays.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/ocn.h"

#define OCN_HALO 3

struct ocn_grid {
    ocn_grid_desc d;
    int nx, ny, nz;
    int sx, sy;                                   // plane layout (with halo)
    std::vector<double> zf, dz, zc, dzc;
    double dy;
    std::vector<double> dxC, dxF, AzC, AzF, fF;   // rows -3 .. ny+3, index j + 3
    std::vector<int> kb;                          // ny*nx bottom index (nz = land)
    // packed thresholds in plane layout: m8 = {kb, tx1, tx2, tx3, ty1, ty2, ty3, 0}, mz = {zu2, zu3, zv2, zv3}
    std::vector<uint64_t> m8;
    std::vector<uint32_t> mz;
    std::vector<uint8_t> zu1, zv1;                // r = 1 thresholds (host only, for ocn_get_masks)

    int kbat(int j, int i) const {                // bottom index with wrap / land-halo rule
        if (d.periodic_x) i = ((i % nx) + nx) % nx; else if (i < 0 || i >= nx) return nz;
        if (d.periodic_y) j = ((j % ny) + ny) % ny; else if (j < 0 || j >= ny) return nz;
        return kb[(size_t)j * nx + i];
    }
    size_t pidx(int j, int i) const { return (size_t)(j + OCN_HALO) * sx + (i + 32); }   // into the padded host plane
};

namespace ocn_host {

inline int roundup(int a, int b) { return (a + b - 1) / b * b; }

inline std::string build_grid(ocn_grid& g, const ocn_grid_desc& d, const double* z_faces, const double* depth) {
    g.d = d; g.nx = d.nx; g.ny = d.ny; g.nz = d.nz;
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    // + 2: the TMA maps of K1 start 4 columns before i = 0, so the east halo column i = nx + 2 sits at x = nx + 6 and must
    // lie inside the row (x < sx) or the hardware zero-fills it instead of delivering the periodic image
    g.sx = roundup(nx + 2 * OCN_HALO + 2, 32);
    g.sy = ny + 2 * OCN_HALO;
    g.zf.assign(z_faces, z_faces + nz + 1);
    for (int k = 0; k <= nz; ++k) if (!std::isfinite(g.zf[k])) return "z_faces must be finite";
    for (int k = 0; k < nz; ++k) if (!(g.zf[k + 1] > g.zf[k])) return "z_faces must be strictly increasing";
    if (g.zf[nz] != 0.0) return "z_faces[nz] must be 0 (the resting surface)";
    g.dz.resize(nz); g.zc.resize(nz); g.dzc.assign(nz, 0.0);
    for (int k = 0; k < nz; ++k) { g.dz[k] = g.zf[k + 1] - g.zf[k]; g.zc[k] = 0.5 * (g.zf[k] + g.zf[k + 1]); }
    for (int k = 1; k < nz; ++k) g.dzc[k] = g.zc[k] - g.zc[k - 1];

    const int nr = ny + 2 * OCN_HALO + 1;
    g.dxC.resize(nr); g.dxF.resize(nr); g.AzC.resize(nr); g.AzF.resize(nr); g.fF.resize(nr);
    if (d.kind == 1) {
        const double rad = M_PI / 180.0, a = d.radius, dlam = d.dx * rad, dphi = d.dy * rad;
        g.dy = a * dphi;
        for (int r = 0; r < nr; ++r) {
            // j_offset: this grid is rows j_offset .. of a taller one (a latitude band): the same expression
            // in the same integers as the whole grid evaluates, so the band's metrics are bit-identical to its rows there
            const double pf = (d.y0 + (r - OCN_HALO + d.j_offset) * d.dy) * rad, pc = pf + 0.5 * dphi;
            g.dxC[r] = a * std::cos(pc) * dlam;
            g.dxF[r] = a * std::cos(pf) * dlam;
            g.AzC[r] = a * a * dlam * (std::sin(pf + dphi) - std::sin(pf));
            g.AzF[r] = a * a * dlam * (std::sin(pc) - std::sin(pc - dphi));
            g.fF[r] = 2.0 * d.rotation_rate * std::sin(pf);
        }
    } else {
        g.dy = d.dy;
        const double ymid = d.y0 + 0.5 * (d.ny_global > 0 ? d.ny_global : ny) * d.dy;
        for (int r = 0; r < nr; ++r) {
            g.dxC[r] = g.dxF[r] = d.dx;
            g.AzC[r] = g.AzF[r] = d.dx * d.dy;
            g.fF[r] = d.f0 + d.beta * ((d.y0 + (r - OCN_HALO + d.j_offset) * d.dy) - ymid);
        }
    }
    for (int r = 0; r < nr; ++r)
        if (!(g.dxC[r] > 0 && g.dxF[r] > 0 && g.AzC[r] > 0 && g.AzF[r] > 0)) return "degenerate metric (latitude range reaches a pole?)";

    // bottom index: full cells, centre test, columns with fewer than 2 wet cells are land
    g.kb.assign((size_t)ny * nx, nz);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const double h = depth[(size_t)j * nx + i];
            if (!(h >= 0.0)) return "bottom_depth must be >= 0";
            int k0 = nz;
            if (h > 0.0) for (int k = 0; k < nz; ++k) if (g.zc[k] > -h) { k0 = k; break; }
            g.kb[(size_t)j * nx + i] = (nz - k0 >= 2) ? k0 : nz;
        }

    // level thresholds
    const size_t np = (size_t)g.sy * g.sx + 64;
    uint64_t land8 = 0;
    for (int b = 0; b < 7; ++b) land8 |= (uint64_t)nz << (8 * b);
    const uint32_t landz = (uint32_t)nz * 0x01010101u;
    g.m8.assign(np, land8); g.mz.assign(np, landz);
    g.zu1.assign((size_t)ny * nx, (uint8_t)nz); g.zv1.assign((size_t)ny * nx, (uint8_t)nz);
    auto kz = [&](int j, int i) {     // corner threshold: all four cells around the SW corner wet
        return std::max(std::max(g.kbat(j - 1, i - 1), g.kbat(j - 1, i)), std::max(g.kbat(j, i - 1), g.kbat(j, i)));
    };
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            int tx[4] = {0, 0, 0, 0}, ty[4] = {0, 0, 0, 0}, zu[4] = {0, 0, 0, 0}, zv[4] = {0, 0, 0, 0};
            for (int r = 1; r <= 3; ++r) {
                int a = 0, b = 0, cc = 0, e = 0;
                for (int m = -r; m <= r - 1; ++m) { a = std::max(a, g.kbat(j, i + m)); b = std::max(b, g.kbat(j + m, i)); }
                for (int m = 1 - r; m <= r; ++m) { cc = std::max(cc, kz(j + m, i)); e = std::max(e, kz(j, i + m)); }
                tx[r] = a; ty[r] = b; zu[r] = cc; zv[r] = e;
            }
            const uint64_t w = (uint64_t)g.kb[(size_t)j * nx + i] | (uint64_t)tx[1] << 8 | (uint64_t)tx[2] << 16 | (uint64_t)tx[3] << 24
                             | (uint64_t)ty[1] << 32 | (uint64_t)ty[2] << 40 | (uint64_t)ty[3] << 48;
            g.m8[g.pidx(j, i)] = w;
            g.mz[g.pidx(j, i)] = (uint32_t)zu[2] | (uint32_t)zu[3] << 8 | (uint32_t)zv[2] << 16 | (uint32_t)zv[3] << 24;
            g.zu1[(size_t)j * nx + i] = (uint8_t)zu[1]; g.zv1[(size_t)j * nx + i] = (uint8_t)zv[1];
        }
    // halos of the packed maps: periodic wrap, else land
    for (int j = -OCN_HALO; j < ny + OCN_HALO; ++j)
        for (int i = -OCN_HALO; i < nx + OCN_HALO; ++i) {
            if (j >= 0 && j < ny && i >= 0 && i < nx) continue;
            int jj = j, ii = i;
            bool land = false;
            if (d.periodic_x) ii = ((i % nx) + nx) % nx; else if (i < 0 || i >= nx) land = true;
            if (d.periodic_y) jj = ((j % ny) + ny) % ny; else if (j < 0 || j >= ny) land = true;
            if (!land) { g.m8[g.pidx(j, i)] = g.m8[g.pidx(jj, ii)]; g.mz[g.pidx(j, i)] = g.mz[g.pidx(jj, ii)]; }
        }
    return "";
}

}  // namespace ocn_host
