// kernels_tile.cuh — K1: the fused tendency kernel (S1 + S2 + S3 + elimination half of S4 + S5 +
// S8 on the fly), one CTA per (TX x TY) tile of columns, marching k from the bottom up.
//
// Data movement: the halo'd k-planes of the tile are brought into shared memory
// by TMA (cp.async.bulk.tensor.3d) DP levels ahead of use, into small rings:
//     ts = (T, S) pairs : planes k-2 .. k+3 live (horizontal and vertical WENO stencils)
//     uv = (u, v) pairs : planes k, k+1
//     p                 : plane k
// one mbarrier per in-flight level.  Nothing on the compute path waits on a global load except
// the AB2 history read (own point, issued two phases ahead).  Per level:
//   phase 1  zeta on the halo'd tile; K, D on the tile + west/south ring; w[k+1] = w[k] - dz D
//            (S8 fused: the column accumulators live in registers of the thread that owns the point)
//   phase 2  every west / south face of the tile (+ the east / north edge) is reconstructed ONCE:
//            WENO face value of the (T, S) pair -> advective + diffusive flux, to shared memory;
//            the owning thread does the vertical face
//   phase 3  per cell: G_T, G_S from the flux planes; G_u, G_v from zeta, K, D, p, w; quasi-AB2,
//            predictor, elimination sweep of the implicit solve, barotropic forcing sums; stores.
#pragma once
#include <cuda.h>

#include <type_traits>

#include "common.cuh"
#include "kernels_mixing.cuh"

// First thread of the compacted work lists of a 256-thread CTA: v cells from 0 up, tracer cells from 64
// up, faces from 160 up (wrapping), u cells from N-1 down.  On sparse levels the four lists land on different warps; on
// half-full levels no thread carries all four.  Measured on config 4 (profiles/r1_ncu_summary.md §6).
// Wet cells of a tile-level from which on the tile is marched with GEOMETRIC ownership (thread = cell).
#ifndef K1_GEO_THR
#define K1_GEO_THR 224
#endif
#ifndef K1_TOFF
#define K1_TOFF 64
#define K1_VOFF 0
#define K1_FOFF 160
#endif

namespace ocn {

// ---- mbarrier / TMA (PTX; SASS: SYNCS.*, UTMALDG) ------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive_plain(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    const uint32_t a = smem_u32(bar);
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void tma_load_plane(void* dst, const CUtensorMap* map, uint64_t* bar, int x, int y, int z) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z) : "memory");
}

__host__ __device__ constexpr int rup128(int b) { return (b + 127) / 128 * 128; }

// RI: the instantiation that evaluates the Ri-based vertical mixing closure inside the pass: two
// more ring buffers hold (nu, kappa) at the upper face of the tile's columns (+ west / south ring).
template <class T, int TX_, int TY_, bool RI_ = false>
struct Tile {
    static constexpr bool RI = RI_;
    typedef typename Pair<T>::type T2;
    static constexpr int TX = TX_, TY = TY_, NC = TX * TY, NT = NC;   // cells = threads; a thread owns the tracers of one cell and the momentum of another
    static constexpr int BX = TX + 8, BY = TY + 6;       // TMA box: origin (i0 - 4, j0 - 3)
    static constexpr int OX = 4, OY = 3;                 // box coordinates of tile cell (0, 0)
    static constexpr int DP = 2;                         // prefetch distance in levels
    // ring lengths are powers of two (slot of level q = q & (R - 1): no loop-carried slot state); needed: DP + 5, DP + 1, DP, 3
    static constexpr int R_TS = 8, R_UV = 4, R_P = 2, R_W = 4, NB = DP;
    static_assert(DP + 5 <= R_TS && DP + 2 <= R_UV && DP <= R_P, "rings");      // RI fetches (u, v) one level earlier
    static constexpr int RX = TX + 1, RY = TY + 1;       // tile + west/south ring (K, D, w) or + east/north edge (faces, masks)
    static constexpr int PL2 = rup128(BX * BY * (int)sizeof(T2)), PL1 = rup128(BX * BY * (int)sizeof(T)),
                         PLP = rup128((TX + 4) * (TY + 1) * 8);   // pressure planes: fp64, box (TX + 4) x (TY + 1), origin (i0 - 4, j0 - 1)
    static constexpr int BYTES2 = BX * BY * (int)sizeof(T2), BYTESP = (TX + 4) * (TY + 1) * 8, PBX = TX + 4;
    // shared-memory map (byte offsets from a 128-byte aligned base)
    static constexpr int O_TS = 0;
    static constexpr int O_UV = O_TS + R_TS * PL2;
    static constexpr int O_P = O_UV + R_UV * PL2;
    static constexpr int O_ZETA = O_P + R_P * PLP;
    static constexpr int O_KD = O_ZETA + 2 * PL1;                               // 2 x T2 (K, D) on RX x RY
    static constexpr int KDB = rup128(RX * RY * (int)sizeof(T2)), WB = rup128(RX * RY * (int)sizeof(T));
    static constexpr int O_W = O_KD + 2 * KDB;                                  // R_W buffers of T on RX x RY (w at face f in slot f & 3)
    static constexpr int NFX = RX * TY, NFY = TX * RY, NF = NFX + NFY;        // west faces, then south faces
    static constexpr int FLB = rup128(NF * (int)sizeof(T2));
    static constexpr int O_FLUX = O_W + R_W * WB;                                 // 2 x T2 per face
    static constexpr int O_NK = O_FLUX + 2 * FLB;                                // RI: 2 x T2 (nu, kappa) on RX x RY, face f in slot f & 1
    static constexpr int O_M8 = O_NK + (RI ? 2 : 0) * KDB;                       // uint2 on RX x RY (not zero-filled from here on)
    static constexpr int O_MET = O_M8 + rup128(RX * RY * 8);                    // 9 row-metric arrays of BY + 1
    static constexpr int O_CELL = O_MET + rup128(9 * (BY + 1) * (int)sizeof(T)); // uint16: cells sorted by first wet level
    static constexpr int O_FS = O_CELL + rup128(NC * 2);                        // uint2: face descriptors sorted by first open level
    static constexpr int O_NC = O_FS + rup128(NF * 8);                          // uint16[256]: active cells at level k
    static constexpr int O_NF = O_NC + 512;                                     // uint16[256]: active faces at level k
    static constexpr int O_DZ = O_NF + 512;                                     // T[256] dz, T[256] 1 / dz
    static constexpr int O_DZC = O_DZ + 2 * 256 * (int)sizeof(T);               // RI: T[256] dzc, T[256] 1 / dzc
    static constexpr int O_XP = O_DZC + (RI ? 2 * 256 * (int)sizeof(T) : 0);                 // double[256][4]: column state in transit at the switch of ownership
    static constexpr int O_BAR = O_XP + 256 * 4 * 8;
    static constexpr int SMEM = O_BAR + 128 + 128;                              // + alignment slack
};


// DRAG: the "extras" instantiation: compiled with the bottom-drag term of DESIGN.md §3.14 and the add of the biharmonic terms
// of §3.18 (chosen by the host when drag_r, drag_cd, nu4_h or kappa4_h is non-zero, so that the default path does not carry
// their instructions: the drag term predicated off cost 2 %, the biharmonic flag 3 % of the default kernel).
// RI: the Ri-based closure evaluated in the pass (per-face diffusivities, per-column elimination in registers, the modified
// super-diagonals stored for K3).  WZ: WENO-Z nonlinear weights instead of Jiang-Shu's.
template <class T, int TX, int TY, int MINB, bool DRAG = false, bool RI = false, bool WZ = false>
__global__ void __launch_bounds__(TX * TY, MINB)
k_tendency_tile(const DevP<T> P, const T c0, const T c1, const __grid_constant__ CUtensorMap m_ts,
                const __grid_constant__ CUtensorMap m_uv, const __grid_constant__ CUtensorMap m_p) {
    typedef Tile<T, TX, TY, RI> C;
    typedef typename C::T2 T2;
    typedef Ex<T> E;
    constexpr int BX = C::BX, BY = C::BY, RX = C::RX, RY = C::RY, NT = C::NT, NC = C::NC, OX = C::OX, OY = C::OY;
    extern __shared__ __align__(1024) unsigned char sm[];     // dynamic only: starts the CTA's window, 1 KB aligned
    unsigned short* const s_cell = (unsigned short*)(sm + C::O_CELL);
    uint2* const s_fs = (uint2*)(sm + C::O_FS);
    unsigned short* const s_nc = (unsigned short*)(sm + C::O_NC);
    unsigned short* const s_nf = (unsigned short*)(sm + C::O_NF);
    uint2* const s_m8 = (uint2*)(sm + C::O_M8);
    T* const s_dxC = (T*)(sm + C::O_MET);
    T* const s_dxF = s_dxC + (BY + 1);
    T* const s_rAzC = s_dxF + (BY + 1);
    T* const s_rAzF = s_rAzC + (BY + 1);
    T* const s_rdxC = s_rAzF + (BY + 1);
    T* const s_AzC = s_rdxC + (BY + 1);
    T* const s_fF = s_AzC + (BY + 1);
    T* const s_rdxF = s_fF + (BY + 1);
    T* const s_AzF = s_rdxF + (BY + 1);
    T* const s_dz = (T*)(sm + C::O_DZ);
    T* const s_rdz = s_dz + 256;
    T* const s_dzc = (T*)(sm + C::O_DZC);                // RI only
    T* const s_rdzc = s_dzc + 256;
    RiConst RC;
    if constexpr (RI) RC.init(P);
    uint64_t* const bars = (uint64_t*)(sm + C::O_BAR);
    int& s_kmin = *(int*)(sm + C::O_BAR + 64);
    int& s_ks = *(int*)(sm + C::O_BAR + 68);

    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
    // rasterisation: tiles are taken in bands of RB tile-rows, y fastest inside a band, so that the
    // tiles resident together form a compact patch and their halo planes are shared through L2
    constexpr int RB = 4;
    const int bid = blockIdx.x + gridDim.x * blockIdx.y;
    const int band = bid / (RB * (int)gridDim.x), inb = bid - band * RB * (int)gridDim.x;
    const int rows = min(RB, (int)gridDim.y - band * RB);
    const int i0 = (inb / rows) * TX, j0 = (band * RB + inb % rows) * TY;
    const int nz = P.nz, sx = P.sx;
    const long long sz = P.sz;

    // ---- masks of the tile (+ east / north edge) and the first level with any open cell -----
    if (tid == 0) { s_kmin = nz; s_ks = nz; }
    __syncthreads();
    {
        const uint32_t nzb = (uint32_t)nz;
        const uint2 land = make_uint2(nzb * 0x01010101u, nzb * 0x00010101u);
        int kloc = nz;
        for (int q = tid; q < (TX + 2) * (TY + 2); q += NT) {
            const int qx = q % (TX + 2) - 1, qy = q / (TX + 2) - 1;
            const int ii = i0 + qx, jj = j0 + qy;
            uint2 m = land;
            if (ii < P.nx + OCN_HALO && jj < P.ny + OCN_HALO) m = P.m8[(long long)(jj + OCN_HALO) * sx + ii];
            kloc = min(kloc, (int)(m.x & 255u));
            if (qx >= 0 && qy >= 0) s_m8[qy * RX + qx] = m;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) kloc = min(kloc, __shfl_xor_sync(0xffffffffu, kloc, o));
        if ((tid & 31) == 0) atomicMin(&s_kmin, kloc);
    }
    __syncthreads();
    const int kmin = s_kmin;
    if (kmin >= nz) return;                              // all land: forcing sums stay zero

    int gT = 0, gU = 0, gV = 0;                          // this thread's cell in the tracer, u and v orders
    // ---- compaction lists: cells sorted by their first wet level, faces by their
    // first open level (stable counting sort on the 8-bit level), so that at level k the active work
    // is a dense prefix of each list and keeps the geometric order (coalescing) within a level ------
    {
        constexpr int MAXR = (C::NF + NT - 1) / NT;           // rounds of NT items
        unsigned short* const cnt = (unsigned short*)sm;                  // [virtual warp][key], scratch in the unused ts ring
        int* const base = (int*)(sm + MAXR * (NT / 32) * 256 * 2);        // [key] exclusive prefix, then [256 + w] warp sums
        static_assert(MAXR * (NT / 32) * 512 + 2048 <= C::O_M8, "sort scratch");
        const int lane = tid & 31, wrp = tid >> 5;
        // sorts items 0 .. n-1 by keyf(q) in [0, 255]; emit(q, rank); nle[k] = number of items with key <= k
        auto csort = [&](const int n, auto keyf, auto emit, unsigned short* nle) {
            const int nr = (n + NT - 1) / NT;
            for (int q = tid; q < nr * (NT / 32) * 256; q += NT) cnt[q] = 0;
            __syncthreads();
            int kq[MAXR], lr[MAXR];
#pragma unroll
            for (int r = 0; r < MAXR; ++r) {
                const int q = r * NT + tid;
                const bool on = r < nr && q < n;
                const unsigned act = __ballot_sync(0xffffffffu, on);
                kq[r] = 0; lr[r] = 0;
                if (on) {
                    kq[r] = keyf(q);
                    const unsigned peers = __match_any_sync(act, kq[r]);
                    lr[r] = __popc(peers & ((1u << lane) - 1u));
                    if (lr[r] == 0) cnt[(r * (NT / 32) + wrp) * 256 + kq[r]] = (unsigned short)__popc(peers);
                }
            }
            __syncthreads();
            // per key: offsets of the virtual warps within the key, and the key total (into base[])
            for (int kt = tid; kt < 256; kt += NT) {
                int run = 0;
                for (int vw = 0; vw < nr * (NT / 32); ++vw) {
                    const int cc = cnt[vw * 256 + kt];
                    cnt[vw * 256 + kt] = (unsigned short)run;
                    run += cc;
                }
                base[kt] = run;
            }
            __syncthreads();
            if (wrp == 0) {                                               // exclusive scan of the 256 key totals by one warp
                int tot[8], sum = 0;
#pragma unroll
                for (int e = 0; e < 8; ++e) { tot[e] = base[lane * 8 + e]; sum += tot[e]; }
                int inc = sum;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
                int off = inc - sum;
#pragma unroll
                for (int e = 0; e < 8; ++e) { base[lane * 8 + e] = off; off += tot[e]; nle[lane * 8 + e] = (unsigned short)off; }
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < MAXR; ++r) {
                const int q = r * NT + tid;
                if (r < nr && q < n) emit(q, base[kq[r]] + (int)cnt[(r * (NT / 32) + wrp) * 256 + kq[r]] + lr[r]);
            }
            __syncthreads();
        };
        // three orders of the tile's cells: by first wet level (tracers), by first open west face (u), by first
        // open south face (v); the thread keeps its entry of each, so one shared list serves all three
        auto cell_key = [&](int q, int which) {
            const int gx = q % TX, gy = q / TX;
            if (!(i0 + gx < P.nx && j0 + gy < P.ny)) return nz;
            const uint2 m = s_m8[gy * RX + gx];
            return (int)(which == 0 ? (m.x & 255u) : which == 1 ? ((m.x >> 8) & 255u) : (m.y & 255u));
        };
        auto cell_emit = [&](int q, int rank) { s_cell[rank] = (unsigned short)q; };
        csort(NC, [&](int q) { return cell_key(q, 0); }, cell_emit, s_nc);
        // first level at which the tile is dense enough for geometric ownership (the fill never decreases with k)
        for (int k = tid; k < nz; k += NT) if (s_nc[k] >= P.geo_thr) atomicMin(&s_ks, k);
        constexpr int TOFF = K1_TOFF, VOFF = K1_VOFF;                     // first thread of the tracer and v lists (u runs from N-1 down, faces from K1_FOFF up)
        gT = s_cell[(tid + NC - TOFF) % NC];
        {
            csort(NC, [&](int q) { return cell_key(q, 1); }, cell_emit, s_nc);
            gU = s_cell[NC - 1 - tid];
            csort(NC, [&](int q) { return cell_key(q, 2); }, cell_emit, s_nc);
            gV = s_cell[(tid + NC - VOFF) % NC];
        }
        {
            // faces: fid < NFX = west face of cell (fid % RX, fid / RX); else south face of cell (g % TX, g / TX), g = fid - NFX
            auto face_cell = [&](int fid, bool& isy, int& fx, int& fy) {
                isy = fid >= C::NFX;
                const int g = isy ? fid - C::NFX : fid;
                fx = isy ? g % TX : g % RX; fy = isy ? g / TX : g / RX;
            };
            csort(C::NF,
                  [&](int q) { bool isy; int fx, fy; face_cell(q, isy, fx, fy);
                               const uint2 m = s_m8[fy * RX + fx];
                               return (int)(isy ? (m.y & 255u) : ((m.x >> 8) & 255u)); },
                  [&](int fid, int rank) { bool isy; int fx, fy; face_cell(fid, isy, fx, fy);
                               const uint2 m = s_m8[fy * RX + fx];
                               const uint32_t thr = isy ? (m.y & 0xffffffu) : (m.x >> 8);
                               const uint32_t bb = (uint32_t)((fy + OY) * BX + fx + OX);
                               s_fs[rank] = make_uint2(bb | ((uint32_t)(fy + OY) << 10) | ((isy ? 1u : 0u) << 14) | ((uint32_t)fid << 16), thr); },
                  s_nf);
        }
    }

    // ---- one-time shared-memory setup --------------------------------------------------------
    for (int q = tid; q < C::O_M8 / 16; q += NT) ((uint4*)sm)[q] = make_uint4(0u, 0u, 0u, 0u);
    {
        const int nr = P.ny + 2 * OCN_HALO + 1;
        for (int q = tid; q <= BY; q += NT) {
            const int r = min(j0 + q, nr - 1);
            s_dxC[q] = P.dxC[r]; s_dxF[q] = P.dxF[r]; s_rAzC[q] = P.rAzC[r]; s_rAzF[q] = P.rAzF[r]; s_rdxC[q] = P.rdxC[r];
            s_AzC[q] = P.AzC[r]; s_fF[q] = P.fF[r]; s_rdxF[q] = P.rdxF[r]; s_AzF[q] = P.AzF[r];
        }
    }
    for (int q = tid; q < nz; q += NT) {
        s_dz[q] = P.dz[q]; s_rdz[q] = P.rdz[q];
        if constexpr (RI) { s_dzc[q] = q > 0 ? P.dzc[q] : T(1); s_rdzc[q] = q > 0 ? P.rdzc[q] : T(1); }
    }
    if (tid == 0) {
#pragma unroll
        for (int b = 0; b < C::NB; ++b) mbar_init(&bars[b], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // zero fill (generic) before TMA writes (async)
    __syncthreads();

    // Iteration m of the march does parts A(m) = phases 1 + 2 of level m and B(m - 1) = phase 3 of level
    // m - 1, then ONE block barrier.  group(m) = the planes iteration m needs beyond those of iteration
    // m - 1: ts(m + 2) (vertical stencil of B(m - 1)), uv(m), p(m - 1).
    auto issue_group = [&](int m, bool first) {
        uint64_t* bar = &bars[(m - kmin) % C::NB];
        uint32_t bytes = 0;
        const int tlo = first ? max(m - 3, 0) : m + 2, thi = min(m + 2, nz - 1);
        // (u, v): plane m; RI needs plane m + 1 in iteration m (shear across the face above level m), so it runs one ahead
        const int ulo = RI ? (first ? m : m + 1) : m, uhi = min(RI ? m + 1 : m, nz - 1);
        if (thi >= tlo) bytes += (uint32_t)(thi - tlo + 1) * C::BYTES2;
        if (uhi >= ulo) bytes += (uint32_t)(uhi - ulo + 1) * C::BYTES2;
        if (m - 1 >= kmin) bytes += C::BYTESP;
        if (bytes == 0) { mbar_arrive_plain(bar); return; }          // nothing to load for this iteration
        mbar_expect_tx(bar, bytes);
        for (int q = tlo; q <= thi; ++q) tma_load_plane(sm + C::O_TS + (q % C::R_TS) * C::PL2, &m_ts, bar, 2 * i0, j0, q);
        for (int q = ulo; q <= uhi; ++q) tma_load_plane(sm + C::O_UV + (q % C::R_UV) * C::PL2, &m_uv, bar, 2 * i0, j0, q);
        if (m - 1 >= kmin) tma_load_plane(sm + C::O_P + ((m - 1) % C::R_P) * C::PLP, &m_p, bar, i0, j0 + 2, m - 1);
    };
    // the TMA producer is a thread of a warp without part-A / part-B work on sparse levels (v cells run from thread 0,
    // tracer cells from 64, faces from 160, u cells from N-1 down): its issue latency stays off the critical path
    constexpr int PROD = 32;                 // warp 1: measured best of 32 / 96 / 128 (9.98 / 10.06 / 10.04 ms)
    if (tid == PROD) {
        issue_group(kmin, true);
#pragma unroll
        for (int d = 1; d < C::DP; ++d) if (kmin + d <= nz) issue_group(kmin + d, false);
    }

    // ---- per-thread column state ------------------------------------------------------------
    // COMPACT ownership (sparse levels of the tile): a thread owns the TRACERS of the cell of rank
    // t - K1_TOFF (mod N) in the order by first wet level, the U of the cell of rank N-1-t in the order by first open west
    // face and the V of the cell of rank t - K1_VOFF (mod N) in the order by first open south face: every block of part B
    // runs on a dense run of threads, and on sparse levels the runs land on different warps instead of one after the other.
    // GEOMETRIC ownership (from the first level with >= K1_GEO_THR wet cells on): thread (tx, ty) owns tracers, u and v of
    // cell (tx, ty) and the west / south face fluxes of that cell: shared-memory accesses of a warp fall into one row of
    // the box (no bank conflicts), global accesses are contiguous, and no list is decoded.
    // t1 = first level of the role the descriptor serves (which = 0: tracers, first wet level; 1: u, first open west face;
    // 2: v, first open south face); z2, z3: thresholds of the vorticity reconstruction orders
    struct Cell { int cx, cy, t1, bo, by; unsigned c; bool incol; unsigned char z2, z3; };
    auto make_cell = [&](int g, int which) {
        Cell X;
        X.cx = g % TX; X.cy = g / TX;
        const int i = i0 + X.cx, j = j0 + X.cy;
        X.incol = i < P.nx && j < P.ny;
        X.c = (unsigned)((j + OCN_HALO) * sx + i);
        const uint2 mo = s_m8[X.cy * RX + X.cx];
        const int kb = X.incol ? (int)(mo.x & 255u) : nz;
        X.t1 = !X.incol ? nz : which == 0 ? kb : which == 1 ? (int)((mo.x >> 8) & 255u) : (int)(mo.y & 255u);
        X.z2 = X.z3 = 255;
        if (which != 0 && kb < nz) { const uchar4 mz = P.mz[X.c]; X.z2 = which == 1 ? mz.x : mz.z; X.z3 = which == 1 ? mz.y : mz.w; }
        X.by = X.cy + OY; X.bo = X.by * BX + X.cx + OX;
        return X;
    };
    Cell cT = make_cell(gT, 0), cU = make_cell(gU, 1), cV = make_cell(gV, 2);
    const T dy = P.dy, rdy = P.rdy;
    const int ks = s_ks;                                 // iterations m <= ks run compact, m > ks geometric

    double wacc0 = 0.0, wacc1 = 0.0;                     // w accumulators of this thread's ring points
    // RI: first wet level of the columns of this thread's ring points (the face above level k is open from there on; the
    // coefficients of closed faces are never read, so they are not evaluated)
    int kbr0 = nz, kbr1 = nz;
    if constexpr (RI) {
#pragma unroll
        for (int n = 0; n < 2; ++n) {
            const int q = n * NT + (NT - 1 - tid);
            if (q < RX * RY) {
                const int ii = i0 - 1 + q % RX, jj = j0 - 1 + q / RX;
                int kb = nz;
                if (ii < P.nx + OCN_HALO && jj < P.ny + OCN_HALO) kb = (int)(P.m8[(long long)(jj + OCN_HALO) * sx + ii].x & 255u);
                (n == 0 ? kbr0 : kbr1) = kb;
            }
        }
    }
    T2 fz_bot = mk2(T(0), T(0));                         // vertical tracer flux through the face below
    T u_dn = 0, v_dn = 0;
    double aGU = 0, aGV = 0, aSU = 0, aSV = 0;
    // Thomas rows of this thread's columns: d0 (, d1) = eliminated right-hand sides of the level below; RI also carries the
    // modified super-diagonal cp and dt * diffusivity at the face below the current level
    ThomasRow<T> rt{T(0), T(0), T(0)}, ru{T(0), T(0), T(0)}, rv{T(0), T(0), T(0)};
    T kt_lo = 0, ku_lo = 0, kv_lo = 0;

    // advective + diffusive flux of the (T, S) pair through one face: b = box index of the cell east / north
    // of the face, st = box stride across it, row = box row (metrics)
    auto face_flux = [&](const T2* __restrict__ s_ts, const T2* __restrict__ s_uv, const int b, const bool isy, const int st,
                         const int row, const int ord, const T dzk) -> T2 {
        const T2 uvf = s_uv[b];
        const T vel = isy ? uvf.y : uvf.x;
        const T len = isy ? s_dxF[row] : dy;                       // face length; the face area is len * dz
        const T dd = isy ? dy : s_dxC[row], rdd = isy ? rdy : s_rdxC[row];   // centre-to-centre distance
        const T2 cm = s_ts[b - st], cc = s_ts[b];
        const T2 fv = weno_face2<WZ>(s_ts[b - 3 * st], s_ts[b - 2 * st], cm, cc, s_ts[b + st], s_ts[b + 2 * st], vel, ord);
        const Xv<T> adv = X(vel) * X(len) * X(dzk), dif = X(P.kappa_h) * X(len) * X(dzk);
        T2 flux;
        flux.x = (adv * X(fv.x) - xdiv(dif * (X(cc.x) - X(cm.x)), dd, rdd)).v;
        flux.y = (adv * X(fv.y) - xdiv(dif * (X(cc.y) - X(cm.y)), dd, rdd)).v;
        return flux;
    };

    // one iteration of the march: parts A(m) and B(m - 1), then ONE block barrier.  GEO selects the ownership (a compile-time
    // tag: the geometric body has one cell descriptor, constant strides and no lists)
    // OCN_K1_TIMELINE (diagnostic builds only, `OCN_NVCC_FLAGS=-DOCN_K1_TIMELINE python -m paper_2309_06662_b200.build --force`):
    // every warp accumulates the SM cycles it spends in each phase of an iteration; read with ocn_get_timeline.  Note that
    // BAR.SYNC does not block at issue: the time a warp waits at the block barrier shows up in the NEXT phase (the prologue).
#ifdef OCN_K1_TIMELINE
    long long tl_acc[6] = {0, 0, 0, 0, 0, 0}, tl_last = clock64();
#define TLA(i) { const long long now_ = clock64(); tl_acc[i] += now_ - tl_last; tl_last = now_; }
#else
#define TLA(i)
#endif
    auto iteration = [&](auto geo_tag, const int m, const Cell& XT, const Cell& XU, const Cell& XV) {
        constexpr bool GEO = decltype(geo_tag)::value;
        const int kB = m - 1;                                 // level of part B (phase 3) in this iteration
        const bool doB = kB >= kmin, wetT = doB && kB >= XT.t1, wetU = doB && kB >= XU.t1, wetV = doB && kB >= XV.t1;
        // AB2 history and pivots of level kB: issued now, consumed after part A.  A warp without an active cell or
        // face at this level (most warps on sparsely wet levels) skips this and all of part B.
        const bool anyB = __any_sync(0xffffffffu, wetT | wetU | wetV);
        T2 gm_ts = mk2(T(0), T(0));
        T gm_u = 0, gm_v = 0;
        T piv_t = 1, piv_u = 1, piv_v = 1;
        const long long okB = (long long)kB * sz;             // warp-uniform level base; the column offsets are 32-bit
        T2 bih_ts = mk2(T(0), T(0));                          // biharmonic terms of the own cell (pre-pass)
        T bih_u = 0, bih_v = 0;
        if (DRAG && P.bih && anyB) {                          // (the extras instantiation; the default one has no trace of it)
            if (wetT) bih_ts = (P.Bts + okB)[XT.c];
            if (wetU) bih_u = ((const T*)(P.Buv + okB + XU.c))[0];
            if (wetV) bih_v = ((const T*)(P.Buv + okB + XV.c))[1];
        }
        if (anyB) {
            if (wetT) {
                gm_ts = (P.Gts + okB)[XT.c];
                if (!RI) piv_t = sizeof(T) == 8 ? P.m_t[kB * nz + XT.t1] : P.rm_t[kB * nz + XT.t1];
            }
            if (GEO) {
                if (wetU | wetV) {
                    const T2 g2 = (P.Guv + okB)[XU.c];
                    gm_u = g2.x; gm_v = g2.y;
                }
            } else {
                if (wetU) gm_u = ((const T*)(P.Guv + okB + XU.c))[0];
                if (wetV) gm_v = ((const T*)(P.Guv + okB + XV.c))[1];
            }
            if (!RI) {
                if (wetU) piv_u = sizeof(T) == 8 ? P.m_m[kB * nz + XU.t1] : P.rm_m[kB * nz + XU.t1];
                if (wetV) piv_v = sizeof(T) == 8 ? P.m_m[kB * nz + XV.t1] : P.rm_m[kB * nz + XV.t1];
            }
        }
        TLA(0)
        mbar_wait(&bars[(m - kmin) % C::NB], (uint32_t)(((m - kmin) / C::NB) & 1));
        TLA(1)

        if (m < nz) {                                         // ---------------- part A: level k = m ----------------
            const int k = m;
            const T dzk = s_dz[k];
            const T2* __restrict__ s_uv = (const T2*)(sm + C::O_UV + (k & (C::R_UV - 1)) * C::PL2);
            T* __restrict__ s_zeta = (T*)(sm + C::O_ZETA + (k & 1) * C::PL1);
            T2* __restrict__ s_kd = (T2*)(sm + C::O_KD + (k & 1) * C::KDB);
            T* __restrict__ s_w1 = (T*)(sm + C::O_W + ((k + 1) & (C::R_W - 1)) * C::WB);
            T2* __restrict__ s_flux = (T2*)(sm + C::O_FLUX + (k & 1) * C::FLB);
            // ================= phase 1: zeta, K, D, w[k+1] =================
            {
        #pragma unroll
                for (int h = 0; h < (BX - 1) * (BY - 1); h += NT) {
                    const int q = h + (NT - 1 - tid);
                    if (q < (BX - 1) * (BY - 1)) {
                        const int px = 1 + q % (BX - 1), py = 1 + q / (BX - 1);
                        const T2 a = s_uv[py * BX + px], as = s_uv[(py - 1) * BX + px], aw = s_uv[py * BX + px - 1];
                        s_zeta[py * BX + px] = xdiv(X(dy) * (X(a.y) - X(aw.y)) - (X(s_dxC[py]) * X(a.x) - X(s_dxC[py - 1]) * X(as.x)),
                                                    s_AzF[py], s_rAzF[py]).v;
                    }
                }
            }
    #pragma unroll
            for (int h = 0, n = 0; h < RX * RY; h += NT, ++n) {
                const int q = h + (NT - 1 - tid);
                if (q < RX * RY) {
                    const int qx = q % RX, qy = q / RX;
                    const int px = qx + OX - 1, py = qy + OY - 1;          // cells i0 - 1 + qx, j0 - 1 + qy
                    const T2 a = s_uv[py * BX + px], ae = s_uv[py * BX + px + 1], an = s_uv[(py + 1) * BX + px];
                    const T Kc = (X(T(0.25)) * (X(a.x) * X(a.x) + X(ae.x) * X(ae.x)) + X(T(0.25)) * (X(a.y) * X(a.y) + X(an.y) * X(an.y))).v;
                    const T Dc = xdiv(X(dy) * (X(ae.x) - X(a.x)) + X(s_dxF[py + 1]) * X(an.y) - X(s_dxF[py]) * X(a.y), s_AzC[py], s_rAzC[py]).v;
                    s_kd[q] = mk2(Kc, Dc);
                    double& wa = n == 0 ? wacc0 : wacc1;
                    wa = (X(wa) - X((double)dzk) * X((double)Dc)).v;
                    s_w1[q] = (T)wa;
                    if constexpr (RI) if (k + 1 < nz && k >= (n == 0 ? kbr0 : kbr1)) {     // (nu, kappa) at the face above level k of this column
                        const T2* __restrict__ s_uvh = (const T2*)(sm + C::O_UV + ((k + 1) & (C::R_UV - 1)) * C::PL2);
                        const T2 b = s_uvh[py * BX + px], be = s_uvh[py * BX + px + 1], bn = s_uvh[(py + 1) * BX + px];
                        const T2 t0 = ((const T2*)(sm + C::O_TS + (k & (C::R_TS - 1)) * C::PL2))[py * BX + px];
                        const T2 t1 = ((const T2*)(sm + C::O_TS + ((k + 1) & (C::R_TS - 1)) * C::PL2))[py * BX + px];
                        T2* const s_nkw = (T2*)(sm + C::O_NK + ((k + 1) & 1) * C::KDB);
                        if constexpr (sizeof(T) == 4)
                            s_nkw[q] = ri_face_f32(RC, P.ath_d, k + 1, s_rdzc[k + 1], t1.x, t1.y, t0.x, t0.y, b.x - a.x, be.x - ae.x, b.y - a.y, bn.y - an.y);
                        else
                            s_nkw[q] = ri_face(P, k + 1, t1.x, t1.y, t0.x, t0.y, (X(b.x) - X(a.x)).v, (X(be.x) - X(ae.x)).v,
                                               (X(b.y) - X(a.y)).v, (X(bn.y) - X(an.y)).v);
                    }
                }
            }
            TLA(2)
            // ================= phase 2: tracer face fluxes, each open face once =================
            const T2* __restrict__ s_ts = (const T2*)(sm + C::O_TS + (k & (C::R_TS - 1)) * C::PL2);
            if constexpr (GEO) {
                // the west and the south face of the own cell (thresholds of the cell's own mask word), then the east edge of
                // the tile by lanes 0 .. TY-1 of warp 0 and the north edge by warp 1
                const uint2 mo = s_m8[XT.cy * RX + XT.cx];
                const int ox = order3(k, (mo.x >> 8) & 255u, (mo.x >> 16) & 255u, mo.x >> 24);
                const int oy = order3(k, mo.y & 255u, (mo.y >> 8) & 255u, (mo.y >> 16) & 255u);
                if (ox > 0) s_flux[XT.cy * RX + XT.cx] = face_flux(s_ts, s_uv, XT.bo, false, 1, XT.by, ox, dzk);
                if (oy > 0) s_flux[C::NFX + XT.cy * TX + XT.cx] = face_flux(s_ts, s_uv, XT.bo, true, BX, XT.by, oy, dzk);
                if (tid < TY) {
                    const uint2 me = s_m8[tid * RX + TX];
                    const int oe = order3(k, (me.x >> 8) & 255u, (me.x >> 16) & 255u, me.x >> 24);
                    if (oe > 0) s_flux[tid * RX + TX] = face_flux(s_ts, s_uv, (tid + OY) * BX + TX + OX, false, 1, tid + OY, oe, dzk);
                } else if (tid >= 32 && tid < 32 + TX) {
                    const int fx = tid - 32;
                    const uint2 mn = s_m8[TY * RX + fx];
                    const int on = order3(k, mn.y & 255u, (mn.y >> 8) & 255u, (mn.y >> 16) & 255u);
                    if (on > 0) s_flux[C::NFX + TY * TX + fx] = face_flux(s_ts, s_uv, (TY + OY) * BX + fx + OX, true, BX, TY + OY, on, dzk);
                }
            } else {
                const int nface = s_nf[k];
                for (int f = (tid + NT - K1_FOFF) % NT; f < nface; f += NT) {
                    const uint2 d = s_fs[f];
                    const int b = d.x & 1023u, row = (d.x >> 10) & 15u, fid = d.x >> 16;
                    const bool isy = (d.x >> 14) & 1u;
                    const int ord = order3(k, d.y & 255u, (d.y >> 8) & 255u, (d.y >> 16) & 255u);   // >= 1 here
                    s_flux[fid] = face_flux(s_ts, s_uv, b, isy, isy ? BX : 1, row, ord, dzk);
                }
            }
        }
        TLA(3)
        if (anyB) {                                           // ---------------- part B: level k = m - 1 ----------------
            const int k = kB;
            const T dzk = s_dz[k], rdzk = s_rdz[k];
            const T2* __restrict__ s_uv = (const T2*)(sm + C::O_UV + (k & (C::R_UV - 1)) * C::PL2);
            const T2* __restrict__ s_uv1 = (const T2*)(sm + C::O_UV + ((k + 1) & (C::R_UV - 1)) * C::PL2);
            const double* __restrict__ s_p = (const double*)(sm + C::O_P + (k & (C::R_P - 1)) * C::PLP);
            const T* __restrict__ s_w0 = (const T*)(sm + C::O_W + (k & (C::R_W - 1)) * C::WB);
            const T* __restrict__ s_w1 = (const T*)(sm + C::O_W + ((k + 1) & (C::R_W - 1)) * C::WB);
            const T* __restrict__ s_zeta = (const T*)(sm + C::O_ZETA + (k & 1) * C::PL1);
            const T2* __restrict__ s_kd = (const T2*)(sm + C::O_KD + (k & 1) * C::KDB);
            const T2* __restrict__ s_flux = (const T2*)(sm + C::O_FLUX + (k & 1) * C::FLB);
            const bool has_hi = k + 1 < nz;
            // RI: vertical spacings around level k for the per-column elimination
            [[maybe_unused]] T dzc_lo = T(1), dzc_hi = T(1), rc_lo = T(1), rc_hi = T(1);
            [[maybe_unused]] const T2* __restrict__ s_nk1 = nullptr;
            if constexpr (RI) {
                dzc_lo = s_dzc[k]; rc_lo = s_rdzc[k];
                if (has_hi) { dzc_hi = s_dzc[k + 1]; rc_hi = s_rdzc[k + 1]; }
                s_nk1 = (const T2*)(sm + C::O_NK + ((k + 1) & 1) * C::KDB);
            }
            // ---------- tracer half ----------
            T2 fz_top = mk2(T(0), T(0));
            if (wetT) {
                const int cx = XT.cx, cy = XT.cy, kb = XT.t1, bo = XT.bo, by = XT.by;
                const T AzCj = s_AzC[by], rAzCj = s_rAzC[by];
                const T w_c1 = s_w1[(cy + 1) * RX + cx + 1];
                // vertical face above cell k (own column)
                {
                    const int ozt = has_hi ? min(3, min(k + 1 - kb, nz - k - 1)) : 0;
                    if (ozt > 0) {
                        auto tsz = [&](int dk) -> T2 {           // plane of level k + dk, dk = -2 .. 3
                            return ((const T2*)(sm + C::O_TS + ((k + dk) & (C::R_TS - 1)) * C::PL2))[bo];
                        };
                        const T2 fv = weno_face2<WZ>(tsz(-2), tsz(-1), tsz(0), tsz(1), tsz(2), tsz(3), w_c1, ozt);
                        fz_top.x = (X(w_c1) * X(AzCj) * X(fv.x)).v;
                        fz_top.y = (X(w_c1) * X(AzCj) * X(fv.y)).v;
                    }
                }
                // ---- tracers ----
                const T2 fw = s_flux[cy * RX + cx], fe = s_flux[cy * RX + cx + 1];
                const T2 fs = s_flux[C::NFX + cy * TX + cx], fn = s_flux[C::NFX + (cy + 1) * TX + cx];
                const T2 tsc = ((const T2*)(sm + C::O_TS + (k & (C::R_TS - 1)) * C::PL2))[bo];
                const T vol = (X(AzCj) * X(dzk)).v, rvol = xrcp(vol, rAzCj * rdzk);
                T GT, GS;
                if constexpr (sizeof(T) == 8) {    // the flux divergence summed in the order of DESIGN.md §3.7
                    GT = xdiv(-(X(fe.x) - X(fw.x) + X(fn.x) - X(fs.x) + X(fz_top.x) - X(fz_bot.x)), vol, rvol).v;
                    GS = xdiv(-(X(fe.y) - X(fw.y) + X(fn.y) - X(fs.y) + X(fz_top.y) - X(fz_bot.y)), vol, rvol).v;
                } else {                           // fp32: difference the like fluxes first (they nearly cancel)
                    GT = -((fe.x - fw.x) + (fn.x - fs.x) + (fz_top.x - fz_bot.x)) * rvol;
                    GS = -((fe.y - fw.y) + (fn.y - fs.y) + (fz_top.y - fz_bot.y)) * rvol;
                }
                if (k == nz - 1) {                 // tracers are stored as offsets from (Toff, Soff): exact source
                    const T src = w_c1 * rdzk;     // of the constant under the zero-top-flux linear free surface
                    GT += P.Toff * src; GS += P.Soff * src;
                    // surface tracer forcing: flux into the ocean + restoring toward the target
                    const T2 qf = P.qts[XT.c], rtg = P.rts[XT.c];
                    GT = (X(GT) + xdiv(X(qf.x) + X(P.gamma_T) * (X(rtg.x) - X(tsc.x)), dzk, rdzk)).v;
                    GS = (X(GS) + xdiv(X(qf.y) + X(P.gamma_S) * (X(rtg.y) - X(tsc.y)), dzk, rdzk)).v;
                }
                if constexpr (DRAG) if (P.bih) { GT = (X(GT) + X(bih_ts.x)).v; GS = (X(GS) + X(bih_ts.y)).v; }
                // ---- quasi-AB2, predictor, elimination sweep (S3, S4) ----
                const T Ght = (X(c0) * X(GT) - X(c1) * X(gm_ts.x)).v, Ghs = (X(c0) * X(GS) - X(c1) * X(gm_ts.y)).v;
                (P.Gts + okB)[XT.c] = mk2(GT, GS);
                if constexpr (RI) {               // per-face diffusivity: kappa of the own column at the face above
                    const T kt_hi = has_hi ? (X(P.dt) * X(s_nk1[(cy + 1) * RX + cx + 1].y)).v : T(0);
                    rt.step(k == kb, kt_lo, kt_hi, has_hi, dzk, dzc_lo, dzc_hi, rdzk, rc_lo, rc_hi,
                            E::add(tsc.x, E::mul(P.dt, Ght)), E::add(tsc.y, E::mul(P.dt, Ghs)));
                    (P.cpt + okB)[XT.c] = rt.cp;
                    kt_lo = kt_hi;
                } else {
                    const T smk = k > kb ? P.sm_t[k] : T(0);
                    rt.d0 = E::div(E::add(E::add(tsc.x, E::mul(P.dt, Ght)), E::mul(smk, rt.d0)), piv_t, piv_t);
                    rt.d1 = E::div(E::add(E::add(tsc.y, E::mul(P.dt, Ghs)), E::mul(smk, rt.d1)), piv_t, piv_t);
                }
                (P.dts + okB)[XT.c] = mk2(rt.d0, rt.d1);
            }
            // ---------- momentum: the u face and the v face this thread owns ----------
            T Gu_out = 0, du_out = 0, cpu_out = 0;
            if (wetU) {
                const int cx = XU.cx, cy = XU.cy, tx1 = XU.t1, bo = XU.bo, by = XU.by;
                const int qo = (cy + 1) * RX + cx + 1;                       // this column in the ring arrays
                const T w_c1 = s_w1[qo], w_c0 = s_w0[qo];
                const T dxFj = s_dxF[by], dxFn = s_dxF[by + 1], dxCj = s_dxC[by], rdxCj = s_rdxC[by];
                const T AzCj = s_AzC[by], rAzCj = s_rAzC[by];
                const T fFj = s_fF[by], fFn = s_fF[by + 1];
                const T2 uvc = s_uv[bo];
                const T u_c = uvc.x, v_c = uvc.y;
                const T2 uv_w = s_uv[bo - 1], uv_n = s_uv[bo + BX], uv_nw = s_uv[bo + BX - 1];
                const T u_up = has_hi ? s_uv1[bo].x : T(0);
                const T z00 = s_zeta[bo];
                const T2 kdc = s_kd[qo];
                const int pbo = (cy + 1) * C::PBX + cx + 4;
                const Xv<T> half(T(0.5)), quart(T(0.25)), nuh(P.nu_h);
                const T vold = (X(AzCj) * X(dzk)).v;
                const Xv<T> vsum_s = X(uv_w.y) + X(v_c), vsum_n = X(uv_nw.y) + X(uv_n.y);
                const T vhat = xdiv(quart * (X(dxFj) * vsum_s + X(dxFn) * vsum_n), dxCj, rdxCj).v;
                const int ozu = 1 + (k >= XU.z2) + (k >= XU.z3);
                const T z01 = s_zeta[bo + BX];
                const T zt = ozu == 1 ? (vhat > T(0) ? z00 : z01)
                                      : weno_face<WZ>(s_zeta[bo - 2 * BX], s_zeta[bo - BX], z00, z01, s_zeta[bo + 2 * BX],
                                                      s_zeta[bo + 3 * BX], vhat, ozu);
                const Xv<T> Cu = xdiv(half * (X(fFj) * half * X(dxFj) * vsum_s + X(fFn) * half * X(dxFn) * vsum_n), dxCj, rdxCj);
                const T2 kdw = s_kd[qo - 1];
                const Xv<T> dK = xdiv(X(kdc.x) - X(kdw.x), dxCj, rdxCj);
                const Xv<T> dP = xdiv(X((T)(s_p[pbo] - s_p[pbo - 1])), dxCj, rdxCj);
                const Xv<T> dlo((k >= 1 && k - 1 >= tx1) ? (X(u_c) - X(u_dn)).v : T(0));
                const Xv<T> dhi(has_hi ? (X(u_up) - X(u_c)).v : T(0));
                const Xv<T> Whi = half * X(AzCj) * (X(s_w1[qo - 1]) + X(w_c1)), Wlo = half * X(AzCj) * (X(s_w0[qo - 1]) + X(w_c0));
                const Xv<T> Au = xdiv(half * (Whi * dhi + Wlo * dlo), vold, xrcp(vold, rAzCj * rdzk));
                const Xv<T> Vu = nuh * (xdiv(X(kdc.y) - X(kdw.y), dxCj, rdxCj) - xdiv(X(z01) - X(z00), dy, rdy));
                const T rhodz = (X(P.rho0) * X(dzk)).v;
                const Xv<T> tau((k == nz - 1) ? xdiv(X(P.taux[XU.c]), rhodz, xrcp(rhodz, P.rrho0 * rdzk)).v : T(0));
                T Gu = (X(zt) * X(vhat) + Cu - dK - dP - Au + Vu + tau).v;
                if constexpr (DRAG) {             // bottom drag on the lowest open level of the column
                    const Xv<T> drag(k == tx1 ? xdiv((X(P.drag_r) + X(P.drag_cd) * X((T)sqrt((X(u_c) * X(u_c) + X(vhat) * X(vhat)).v))) * X(u_c), dzk, rdzk).v : T(0));
                    Gu = (X(Gu) - drag).v;
                }
                if constexpr (DRAG) if (P.bih) Gu = (X(Gu) + X(bih_u)).v;
                // ---- quasi-AB2, predictor, elimination sweep (S3, S4, S5) ----
                const T Ghu = (X(c0) * X(Gu) - X(c1) * X(gm_u)).v;
                const T us = E::add(u_c, E::mul(P.dt, Ghu));
                aGU = (X(aGU) + X((double)dzk) * X((double)Ghu)).v; aSU = (X(aSU) + X((double)dzk) * X((double)us)).v;
                if constexpr (RI) {               // nu at the u face = mean of the two tracer columns that share it
                    const T ku_hi = has_hi ? (X(P.dt) * (X(T(0.5)) * (X(s_nk1[qo - 1].x) + X(s_nk1[qo].x)))).v : T(0);
                    ru.step(k == tx1, ku_lo, ku_hi, has_hi, dzk, dzc_lo, dzc_hi, rdzk, rc_lo, rc_hi, us, T(0));
                    ku_lo = ku_hi;
                } else {
                    const T smk = k > tx1 ? P.sm_m[k] : T(0);
                    ru.d0 = E::div(E::add(us, E::mul(smk, ru.d0)), piv_u, piv_u);
                }
                if constexpr (GEO) { Gu_out = Gu; du_out = ru.d0; cpu_out = ru.cp; }
                else {
                    ((T*)(P.Guv + okB + XU.c))[0] = Gu; ((T*)(P.duv + okB + XU.c))[0] = ru.d0;
                    if constexpr (RI) ((T*)(P.cpuv + okB + XU.c))[0] = ru.cp;
                }
                u_dn = u_c;
            }
            T Gv_out = 0, dv_out = 0, cpv_out = 0;
            if (wetV) {
                const int cx = XV.cx, cy = XV.cy, ty1 = XV.t1, bo = XV.bo, by = XV.by;
                const int qo = (cy + 1) * RX + cx + 1;
                const T w_c1 = s_w1[qo], w_c0 = s_w0[qo];
                const T dxFj = s_dxF[by], rdxFj = s_rdxF[by];
                const T AzCj = s_AzC[by], AzCs = s_AzC[by - 1], AzFj = s_AzF[by], rAzFj = s_rAzF[by];
                const T fFj = s_fF[by];
                const T2 uvc = s_uv[bo];
                const T u_c = uvc.x, v_c = uvc.y;
                const T2 uv_s = s_uv[bo - BX], uv_e = s_uv[bo + 1], uv_se = s_uv[bo - BX + 1];
                const T v_up = has_hi ? s_uv1[bo].y : T(0);
                const T z00 = s_zeta[bo];
                const T2 kdc = s_kd[qo];
                const int pbo = (cy + 1) * C::PBX + cx + 4;
                const Xv<T> half(T(0.5)), quart(T(0.25)), nuh(P.nu_h);
                const T uhat = (quart * (X(uv_s.x) + X(u_c) + X(uv_se.x) + X(uv_e.x))).v;
                const int ozv = 1 + (k >= XV.z2) + (k >= XV.z3);
                const T z10 = s_zeta[bo + 1];
                const T zt = ozv == 1 ? (uhat > T(0) ? z00 : z10)
                                      : weno_face<WZ>(s_zeta[bo - 2], s_zeta[bo - 1], z00, z10, s_zeta[bo + 2], s_zeta[bo + 3], uhat, ozv);
                const Xv<T> Cv = X(fFj) * X(uhat);
                const T2 kds = s_kd[qo - RX];
                const Xv<T> dK = xdiv(X(kdc.x) - X(kds.x), dy, rdy);
                const Xv<T> dP = xdiv(X((T)(s_p[pbo] - s_p[pbo - C::PBX])), dy, rdy);
                const Xv<T> dlo((k >= 1 && k - 1 >= ty1) ? (X(v_c) - X(v_dn)).v : T(0));
                const Xv<T> dhi(has_hi ? (X(v_up) - X(v_c)).v : T(0));
                const Xv<T> Whi = half * (X(AzCs) * X(s_w1[qo - RX]) + X(AzCj) * X(w_c1));
                const Xv<T> Wlo = half * (X(AzCs) * X(s_w0[qo - RX]) + X(AzCj) * X(w_c0));
                const T volf = (X(AzFj) * X(dzk)).v;
                const Xv<T> Av = xdiv(half * (Whi * dhi + Wlo * dlo), volf, xrcp(volf, rAzFj * rdzk));
                const Xv<T> Vv = nuh * (xdiv(X(kdc.y) - X(kds.y), dy, rdy) + xdiv(X(z10) - X(z00), dxFj, rdxFj));
                const T rhodz = (X(P.rho0) * X(dzk)).v;
                const Xv<T> tau((k == nz - 1) ? xdiv(X(P.tauy[XV.c]), rhodz, xrcp(rhodz, P.rrho0 * rdzk)).v : T(0));
                T Gv = (-X(zt) * X(uhat) - Cv - dK - dP - Av + Vv + tau).v;
                if constexpr (DRAG) {
                    const Xv<T> drag(k == ty1 ? xdiv((X(P.drag_r) + X(P.drag_cd) * X((T)sqrt((X(uhat) * X(uhat) + X(v_c) * X(v_c)).v))) * X(v_c), dzk, rdzk).v : T(0));
                    Gv = (X(Gv) - drag).v;
                }
                if constexpr (DRAG) if (P.bih) Gv = (X(Gv) + X(bih_v)).v;
                const T Ghv = (X(c0) * X(Gv) - X(c1) * X(gm_v)).v;
                const T vs2 = E::add(v_c, E::mul(P.dt, Ghv));
                aGV = (X(aGV) + X((double)dzk) * X((double)Ghv)).v; aSV = (X(aSV) + X((double)dzk) * X((double)vs2)).v;
                if constexpr (RI) {
                    const T kv_hi = has_hi ? (X(P.dt) * (X(T(0.5)) * (X(s_nk1[qo - RX].x) + X(s_nk1[qo].x)))).v : T(0);
                    rv.step(k == ty1, kv_lo, kv_hi, has_hi, dzk, dzc_lo, dzc_hi, rdzk, rc_lo, rc_hi, vs2, T(0));
                    kv_lo = kv_hi;
                } else {
                    const T smk = k > ty1 ? P.sm_m[k] : T(0);
                    rv.d0 = E::div(E::add(vs2, E::mul(smk, rv.d0)), piv_v, piv_v);
                }
                if constexpr (GEO) { Gv_out = Gv; dv_out = rv.d0; cpv_out = rv.cp; }
                else {
                    ((T*)(P.Guv + okB + XV.c))[1] = Gv; ((T*)(P.duv + okB + XV.c))[1] = rv.d0;
                    if constexpr (RI) ((T*)(P.cpuv + okB + XV.c))[1] = rv.cp;
                }
                v_dn = v_c;
            }
            // stores of the momentum group: one pair store per array in geometric ownership (the same cell), member stores else
            if constexpr (GEO) {
                if (wetU | wetV) {
                    (P.Guv + okB)[XU.c] = mk2(Gu_out, Gv_out);       // closed members hold 0, as they always have
                    (P.duv + okB)[XU.c] = mk2(du_out, dv_out);
                    if constexpr (RI) (P.cpuv + okB)[XU.c] = mk2(cpu_out, cpv_out);
                }
            }
            fz_bot = fz_top;
        }
        TLA(4)
        __syncthreads();                       // planes of level m - 1 are dead: refill the ring
        TLA(5)
        if (tid == PROD && m + C::DP <= nz) {
            const int g = m + C::DP;
            if (g + 2 < nz) {                  // steady state: one plane of each array (the general form handles the ends)
                uint64_t* bar = &bars[(g - kmin) % C::NB];
                mbar_expect_tx(bar, 2 * C::BYTES2 + C::BYTESP);
                tma_load_plane(sm + C::O_TS + ((g + 2) % C::R_TS) * C::PL2, &m_ts, bar, 2 * i0, j0, g + 2);
                tma_load_plane(sm + C::O_UV + ((g + (RI ? 1 : 0)) % C::R_UV) * C::PL2, &m_uv, bar, 2 * i0, j0, g + (RI ? 1 : 0));
                tma_load_plane(sm + C::O_P + ((g - 1) % C::R_P) * C::PLP, &m_p, bar, i0, j0 + 2, g - 1);
            } else {
                issue_group(g, false);
            }
        }
    };

    typedef std::true_type GeoTag;
    typedef std::false_type CmpTag;
    int m = kmin;
    for (; m <= nz && m <= ks; ++m) iteration(CmpTag{}, m, cT, cU, cV);
    if (m <= nz) {
        // ---- switch of ownership: the column state travels through shared memory to the thread of the cell's own position.
        // Every cell is owned by exactly one thread in each of the three compact orders, so every slot is written once.
        double* const xp = (double*)(sm + C::O_XP);
        auto travel = [&](const int gold, double a, double b, double c, double d, double (&out)[4]) {
            xp[gold * 4 + 0] = a; xp[gold * 4 + 1] = b; xp[gold * 4 + 2] = c; xp[gold * 4 + 3] = d;
            __syncthreads();
#pragma unroll
            for (int q = 0; q < 4; ++q) out[q] = xp[tid * 4 + q];
            __syncthreads();
        };
        double r[4];
        travel(gT, (double)rt.cp, (double)rt.d0, (double)rt.d1, (double)kt_lo, r);
        rt.cp = (T)r[0]; rt.d0 = (T)r[1]; rt.d1 = (T)r[2]; kt_lo = (T)r[3];
        travel(gT, (double)fz_bot.x, (double)fz_bot.y, 0.0, 0.0, r);
        fz_bot = mk2((T)r[0], (T)r[1]);
        travel(gU, (double)ru.cp, (double)ru.d0, (double)ku_lo, (double)u_dn, r);
        ru.cp = (T)r[0]; ru.d0 = (T)r[1]; ku_lo = (T)r[2]; u_dn = (T)r[3];
        travel(gU, aGU, aSU, 0.0, 0.0, r);
        aGU = r[0]; aSU = r[1];
        travel(gV, (double)rv.cp, (double)rv.d0, (double)kv_lo, (double)v_dn, r);
        rv.cp = (T)r[0]; rv.d0 = (T)r[1]; kv_lo = (T)r[2]; v_dn = (T)r[3];
        travel(gV, aGV, aSV, 0.0, 0.0, r);
        aGV = r[0]; aSV = r[1];
        cT = make_cell(tid, 0); cU = make_cell(tid, 1); cV = make_cell(tid, 2);
        for (; m <= nz; ++m) iteration(GeoTag{}, m, cT, cU, cV);
    }
#ifdef OCN_K1_TIMELINE
    if ((tid & 31) == 0) {
        for (int q = 0; q < 6; ++q) atomicAdd(&P.timeline[(tid >> 5) * 8 + q], (unsigned long long)tl_acc[q]);
        atomicAdd(&P.timeline[(tid >> 5) * 8 + 6], (unsigned long long)(nz + 1 - kmin));
    }
#endif
    if (cU.incol && cU.t1 < nz) { P.GU[cU.c] = (T)aGU; P.SU[cU.c] = (T)aSU; }     // never-open faces keep their zeros
    if (cV.incol && cV.t1 < nz) { P.GV[cV.c] = (T)aGV; P.SV[cV.c] = (T)aSV; }
}
}  // namespace ocn
