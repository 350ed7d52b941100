// ocn_api.cu — the C ABI of libocn (include/ocn.h): host-side scheduling only.  Every step of the
// hot path runs in the kernels of kernels_tend.cuh / kernels_column.cuh.
#include <cuda.h>
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "grid_host.h"
#include "kernels_column.cuh"
#include "kernels_tile.cuh"
#include "kernels_mixing.cuh"
#include "kernels_biharmonic.cuh"

// Scratch of the allocation-free entry point ocn_get_mixing_noalloc (include/ocn.h): the halo'd (nu, kappa) pair array that
// k_ri_mixing writes before it is gathered into the caller's buffers.  A file-scope device array of a fixed, modest size:
// every GPU that loads the library holds these bytes until the process exits.  In HOST code this name is only a stand-in
// for the symbol, not a device address: the address a kernel may use comes from cudaGetSymbolAddress (noalloc_scratch).
#define OCN_NOALLOC_SCRATCH_BYTES (16u << 20)
static __device__ __align__(256) unsigned char g_noalloc_scratch[OCN_NOALLOC_SCRATCH_BYTES];

namespace {

thread_local std::string g_err;
ocn_status fail(ocn_status s, const std::string& m) { g_err = m; return s; }

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? OCN_ENOMEM : OCN_ECUDA,                  \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                       \
    } while (0)

// a device call of model construction: skipped in the dry run that sizes a workspace (M->measure)
#define DEV(call) do { if (!M->measure) CK(call); } while (0)

constexpr int LEAD = 32;   // elements before the first row so that i = 0 starts a 128-byte line

// Every entry point that touches the device switches to the model's device and restores the caller's on return.
struct DeviceGuard {
    int prev = -1;
    cudaError_t err;
    explicit DeviceGuard(int dev) {
        if (dev < 0) { err = cudaSuccess; return; }        // (host-only call: nothing to switch)
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        err = cudaSetDevice(dev);
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define ON_DEVICE(dev)                 \
    DeviceGuard guard_(dev);           \
    CK(guard_.err)

}  // namespace

struct ocn_model {
    const ocn_grid* g = nullptr;
    ocn_model_desc d{};
    int prec = 64;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    std::vector<double> a_w, b_w;       // filter weights of eta and of the transports (b_w = a_w unless filter_weights_uv was given)
    double dtau = 0;
    bool have_history = false;
    std::vector<void*> allocs;
    unsigned long long bytes = 0;
    // caller-supplied device memory (ocn_model_desc.workspace): allocations are carved from it in order; `measure` is the
    // dry run of ocn_model_workspace_bytes (same code path, no device call, addresses from a made-up base)
    char* ws = nullptr;
    size_t ws_cap = 0, ws_used = 0;
    bool measure = false;
    ocn::DevP<float> pf{};
    ocn::DevP<double> pd{};
    // host <-> device staging: copies run on a stream of their own beside the steps; one big region for
    // 3-D fields and a ring of small ones for 2-D fields (per-step forcing in, eta out), each guarded by two events
    struct Stage {
        void* buf = nullptr;
        size_t bytes = 0;
        cudaEvent_t filled = nullptr;   // H2D copy done (copy stream) / gather done (main stream)
        cudaEvent_t freed = nullptr;    // last consumer done: scatter (main stream) / D2H copy (copy stream)
    };
    static constexpr int NSMALL = 8, NTICKET = 64;
    Stage big, small_[NSMALL];
    int next_small = 0;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ticket_ev[NTICKET] = {};
    unsigned long long tickets = 0;     // async read-backs issued so far (ticket t lives in ticket_ev[t % NTICKET])
    cudaGraphExec_t graph = nullptr;    // one steady-state (AB2) step
    CUtensorMap tm_ts{}, tm_uv{}, tm_p{};   // TMA descriptors of the halo'd (T,S), (u,v) and p arrays
    int launches_per_step = 0;
    // split step (ocn_step_part): the next part expected, and whether the step in progress is the Euler start
    int split_next = 0;
    bool split_euler = false;
    bool nvtx = false;                  // ocn_tune("nvtx", 1): host ranges around steps, parts and profiled stages
    // fused puts into neighbouring bands (ocn_peer_attach): what the last part of a step also stores into peer memory
    bool put = false;
    ocn::PeerPut<float> qf{};
    ocn::PeerPut<double> qd{};
    std::vector<void*> ipc_open;        // bases mapped with cudaIpcOpenMemHandle
    // per-stage timing (ocn_profile_*)
    bool profiling = false;
    std::vector<cudaEvent_t> ev_pool;   // OCN_NSTAGES + 1 events per profiled step
    size_t ev_used = 0;
    double prof_ms[OCN_NSTAGES] = {0, 0, 0, 0};
    long long prof_launches[OCN_NSTAGES] = {0, 0, 0, 0};
};

namespace {

// ipc: an array a neighbouring band in another process maps through CUDA IPC (ocn_peer_export).  The driver carves small
// allocations out of shared 2 MiB pages and an IPC handle names the whole page, so these get whole pages of their own.
// bytes from the library (cudaMalloc) or, 256-byte aligned and in call order, from the caller's workspace
inline ocn_status raw_alloc(ocn_model* M, size_t total, void** out, bool ipc) {
    if (M->ws || M->measure) {
        const size_t off = (M->ws_used + 255) / 256 * 256;
        if (!M->measure && off + total > M->ws_cap)
            return fail(OCN_ENOMEM, "workspace too small: ocn_model_workspace_bytes gives the size for this grid and these parameters");
        *out = (M->measure ? (char*)(uintptr_t)0x100000000ull : M->ws) + off;
        M->ws_used = off + total;
    } else {
        if (ipc) total = (total + ((size_t)2 << 20) - 1) / ((size_t)2 << 20) * ((size_t)2 << 20);
        CK(cudaMalloc(out, total));
        M->allocs.push_back(*out);
    }
    M->bytes += total;
    return OCN_OK;
}

template <class T>
ocn_status dev_alloc(ocn_model* M, size_t n, T** out, bool lead, bool ipc = false) {
    void* p = nullptr;
    const size_t total = (n + (lead ? 2 * LEAD : 0)) * sizeof(T);
    const ocn_status sa = raw_alloc(M, total, &p, ipc);
    if (sa != OCN_OK) return sa;
    DEV(cudaMemsetAsync(p, 0, total, M->stream));
    *out = reinterpret_cast<T*>(p) + (lead ? LEAD : 0);
    return OCN_OK;
}

template <class T>
ocn_status upload(ocn_model* M, const std::vector<double>& src, const T** out) {
    std::vector<T> tmp(src.begin(), src.end());
    T* p = nullptr;
    ocn_status s = dev_alloc(M, tmp.size(), &p, false);
    if (s != OCN_OK) return s;
    DEV(cudaMemcpyAsync(p, tmp.data(), tmp.size() * sizeof(T), cudaMemcpyHostToDevice, M->stream));
    DEV(cudaStreamSynchronize(M->stream));
    *out = p;
    return OCN_OK;
}

template <class T> ocn::PeerPut<T>& peer_put(ocn_model* M);
template <> ocn::PeerPut<float>& peer_put<float>(ocn_model* M) { return M->qf; }
template <> ocn::PeerPut<double>& peer_put<double>(ocn_model* M) { return M->qd; }

template <class T>
ocn::DevP<T>& params(ocn_model* M);
template <> ocn::DevP<float>& params<float>(ocn_model* M) { return M->pf; }
template <> ocn::DevP<double>& params<double>(ocn_model* M) { return M->pd; }

constexpr int TILE_X = 32, TILE_Y = 8;    // K1 tile (kernels_tile.cuh)
constexpr int BT_X = 32, BT_Y = 32;       // barotropic tile of the point-wise kernel (fp64 models; kernels_column.cuh)
#ifndef BS_X
#define BS_X 64
#define BS_Y 28
#define BS_H 10
#endif                                    // tile and halo (= sub-steps per launch) of the register-strip kernel (fp32 models);
                                          // measured on config 4 (M = 40): 64x32/6 1.13 ms, 64x32/8 0.86, 64x28/10 0.855 (4 launches)
template <class T> constexpr int bt_substeps_per_launch() { return sizeof(T) == 4 ? BS_H : BT_HALO; }

// TMA descriptor of a halo'd 3-D array seen as [levels][rows][inner] scalars
ocn_status make_tmap(CUtensorMap* tm, bool f64, void* base, unsigned long long inner, unsigned long long rows,
                     unsigned long long levels, unsigned box_inner, unsigned box_rows) {
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) == cudaSuccess && fn &&
            qr == cudaDriverEntryPointSuccess)
            encode = reinterpret_cast<encode_fn>(fn);
    });
    if (!encode) return fail(OCN_ECUDA, "cuTensorMapEncodeTiled not available");
    const unsigned long long es = f64 ? 8 : 4;
    const cuuint64_t dims[3] = {inner, rows, levels};
    const cuuint64_t strides[2] = {inner * es, inner * rows * es};
    const cuuint32_t box[3] = {box_inner, box_rows, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = encode(tm, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, dims,
                              strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(OCN_ECUDA, "cuTensorMapEncodeTiled failed (code " + std::to_string((int)r) + ")");
    return OCN_OK;
}

// K1 instantiations.  MINB = CTAs per SM the register allocation is bounded for.  drag: carries the bottom-drag term
// (drag_r or drag_cd non-zero); ri: evaluates the Ri-based closure in the pass (closure = 1); wz: WENO-Z weights (advection = 1).
template <class T> using k1_fn = void (*)(const ocn::DevP<T>, const T, const T, const CUtensorMap, const CUtensorMap, const CUtensorMap);
template <class T, bool DRAG, bool RI, bool WZ> k1_fn<T> k1_inst() {
    return ocn::k_tendency_tile<T, TILE_X, TILE_Y, (sizeof(T) == 4 ? 2 : 1), DRAG, RI, WZ>;
}
template <class T> k1_fn<T> k1_fused(bool drag, bool ri, bool wz) {
    const int id = (drag ? 4 : 0) | (ri ? 2 : 0) | (wz ? 1 : 0);
    switch (id) {
        case 0: return k1_inst<T, false, false, false>();
        case 1: return k1_inst<T, false, false, true>();
        case 2: return k1_inst<T, false, true, false>();
        case 3: return k1_inst<T, false, true, true>();
        case 4: return k1_inst<T, true, false, false>();
        case 5: return k1_inst<T, true, false, true>();
        case 6: return k1_inst<T, true, true, false>();
        default: return k1_inst<T, true, true, true>();
    }
}
template <class T> int k1_smem(bool ri) { return ri ? ocn::Tile<T, TILE_X, TILE_Y, true>::SMEM : ocn::Tile<T, TILE_X, TILE_Y, false>::SMEM; }

dim3 grid2(const ocn_grid* g, dim3 b, int z = 1) { return dim3((g->nx + b.x - 1) / b.x, (g->ny + b.y - 1) / b.y, z); }

template <class T>
ocn_status build_model(ocn_model* M) {
    const ocn_grid* g = M->g;
    ocn::DevP<T>& P = params<T>(M);
    const int nz = g->nz;
    P.nx = g->nx; P.ny = g->ny; P.nz = nz; P.sx = g->sx; P.sy = g->sy; P.sz = (long long)g->sx * g->sy;
    P.px = g->d.periodic_x != 0; P.py = g->d.periodic_y != 0;
    const size_t n3 = (size_t)P.sz * nz, n2 = (size_t)P.sz;
    ocn_status s;
    // plane-layout arrays: allocation starts LEAD elements before row -3; cell (j, i) is at
    // base[(j+3)*sx + i] and i = 0 is 128-byte aligned (sx is a multiple of 32 elements)
    auto plane = [&](size_t n, T** out) -> ocn_status {
        return dev_alloc(M, n, out, true);
    };
    typedef typename ocn::Pair<T>::type T2;
    T2** f3[] = {&P.uv, &P.ts, &P.duv, &P.dts, &P.Guv, &P.Gts};
    for (T2** f : f3) if ((s = dev_alloc(M, n3, f, true, f == &P.uv || f == &P.ts)) != OCN_OK) return s;
    if ((s = dev_alloc(M, n3, &P.p, true, true)) != OCN_OK) return s;
    if ((s = plane(n3 + n2, &P.w)) != OCN_OK) return s;
    P.closure = M->d.closure; P.nk = nullptr; P.cpuv = nullptr; P.cpt = nullptr;
    if (M->d.closure == 1) {                       // the per-column super-diagonals K1 leaves for K3
        if ((s = dev_alloc(M, n3, &P.cpuv, true)) != OCN_OK || (s = dev_alloc(M, n3, &P.cpt, true)) != OCN_OK) return s;
    }                                              // (nu, kappa) as an output array: allocated by the first ocn_get_mixing
    P.bih = (M->d.nu4_h != 0.0 || M->d.kappa4_h != 0.0) ? 1 : 0;
    P.Luv = P.Lts = P.Buv = P.Bts = nullptr;
    if (P.bih) {                                   // two scratch Laplacians and the two finished terms
        T2** fb[] = {&P.Luv, &P.Lts, &P.Buv, &P.Bts};
        for (T2** f : fb) if ((s = dev_alloc(M, n3, f, true)) != OCN_OK) return s;
    }
    P.ri_nu0 = M->d.ri_nu0; P.ri_c = M->d.ri_c; P.ri_kconv = M->d.ri_kconv; P.ri_n2c = M->d.ri_n2c; P.ri_s2min = M->d.ri_s2min;
    P.nu_z_d = M->d.nu_z; P.kappa_z_d = M->d.kappa_z;
    T** f2[] = {&P.eta[0], &P.eta[1], &P.U[0], &P.U[1], &P.V[0], &P.V[1], &P.etab, &P.Ub, &P.Vb, &P.GU, &P.GV,
                &P.SU, &P.SV, &P.Hu, &P.Hv, &P.rHu, &P.rHv, &P.taux, &P.tauy};
    for (T** f : f2) if ((s = plane(n2, f)) != OCN_OK) return s;
    if ((s = dev_alloc(M, n2, &P.qts, true)) != OCN_OK || (s = dev_alloc(M, n2, &P.rts, true)) != OCN_OK) return s;
    P.gamma_T = (T)M->d.gamma_T; P.gamma_S = (T)M->d.gamma_S;
    P.drag_r = (T)M->d.drag_r; P.drag_cd = (T)M->d.drag_cd;
    // masks
    {
        uint2* p8 = nullptr; uchar4* pz = nullptr;
        if ((s = dev_alloc(M, g->m8.size(), &p8, false)) != OCN_OK) return s;
        if ((s = dev_alloc(M, g->mz.size(), &pz, false)) != OCN_OK) return s;
        DEV(cudaMemcpyAsync(p8, g->m8.data(), g->m8.size() * 8, cudaMemcpyHostToDevice, M->stream));
        DEV(cudaMemcpyAsync(pz, g->mz.data(), g->mz.size() * 4, cudaMemcpyHostToDevice, M->stream));
        P.m8 = p8 + LEAD; P.mz = pz + LEAD;          // host planes were built with the same lead
    }
    // metrics (+ reciprocals), vertical grid
    auto recip = [](const std::vector<double>& a) { std::vector<double> r(a.size()); for (size_t q = 0; q < a.size(); ++q) r[q] = 1.0 / a[q]; return r; };
    if ((s = upload(M, g->dxC, &P.dxC)) != OCN_OK || (s = upload(M, g->dxF, &P.dxF)) != OCN_OK ||
        (s = upload(M, g->AzC, &P.AzC)) != OCN_OK || (s = upload(M, g->AzF, &P.AzF)) != OCN_OK ||
        (s = upload(M, g->fF, &P.fF)) != OCN_OK || (s = upload(M, recip(g->dxC), &P.rdxC)) != OCN_OK ||
        (s = upload(M, recip(g->dxF), &P.rdxF)) != OCN_OK || (s = upload(M, recip(g->AzC), &P.rAzC)) != OCN_OK ||
        (s = upload(M, recip(g->AzF), &P.rAzF)) != OCN_OK || (s = upload(M, g->dz, &P.dz)) != OCN_OK ||
        (s = upload(M, recip(g->dz), &P.rdz)) != OCN_OK || (s = upload(M, g->dzc, &P.dzc)) != OCN_OK)
        return s;
    {
        std::vector<double> r(g->dzc.size(), 1.0);
        for (size_t q = 1; q < r.size(); ++q) r[q] = 1.0 / g->dzc[q];
        if ((s = upload(M, r, &P.rdzc)) != OCN_OK) return s;
    }
    {
        const double* dzc_d = nullptr;
        if ((s = upload<double>(M, g->dzc, &dzc_d)) != OCN_OK) return s;
        P.dzc_d = dzc_d;
    }
    P.dy = (T)g->dy; P.rdy = (T)(1.0 / g->dy);
    P.hz_top = (T)(g->zf[nz] - g->zc[nz - 1]);
    // Thomas tables: bottom-up elimination started at the column's first open
    // level kf; sub-diagonal sm[k], and per (k, kf) the pivot m, its reciprocal and the modified
    // super-diagonal cp, computed in fp64 exactly as the equations of DESIGN.md §3.8 step 4 are written
    for (int pass = 0; pass < 2; ++pass) {
        // (closure 1 eliminates with per-face coefficients inside K1 and does not read these tables)
        const double dtk = M->d.dt * (pass == 0 ? M->d.nu_z : M->d.kappa_z);
        std::vector<double> sm(nz, 0.0), cp((size_t)nz * nz, 0.0), mm((size_t)nz * nz, 1.0), rm((size_t)nz * nz, 1.0);
        for (int k = 1; k < nz; ++k) sm[k] = dtk / (g->dz[k] * g->dzc[k]);
        for (int kf = 0; kf < nz; ++kf) {
            double cprev = 0.0;
            for (int k = kf; k < nz; ++k) {
                const double sp = (k + 1 <= nz - 1) ? dtk / (g->dz[k] * g->dzc[k + 1]) : 0.0;
                const double smk = (k > kf) ? sm[k] : 0.0;
                const double b = 1.0 + sp + smk;
                const double lo = -smk, up = -sp;
                const double m = (k == kf) ? b : b - lo * cprev;
                cprev = up / m;
                cp[(size_t)k * nz + kf] = cprev; mm[(size_t)k * nz + kf] = m; rm[(size_t)k * nz + kf] = 1.0 / m;   // [k][kf]: a warp works at one k
            }
        }
        if (pass == 0) {
            if ((s = upload(M, sm, &P.sm_m)) != OCN_OK || (s = upload(M, cp, &P.cp_m)) != OCN_OK ||
                (s = upload(M, mm, &P.m_m)) != OCN_OK || (s = upload(M, rm, &P.rm_m)) != OCN_OK) return s;
        } else {
            if ((s = upload(M, sm, &P.sm_t)) != OCN_OK || (s = upload(M, cp, &P.cp_t)) != OCN_OK ||
                (s = upload(M, mm, &P.m_t)) != OCN_OK || (s = upload(M, rm, &P.rm_t)) != OCN_OK) return s;
        }
    }
    P.dt = (T)M->d.dt; P.g = (T)M->d.g; P.alpha = (T)M->d.alpha; P.beta_s = (T)M->d.beta_s;
    P.Toff = sizeof(T) == 4 ? (T)M->d.T0 : T(0); P.Soff = sizeof(T) == 4 ? (T)M->d.S0 : T(0);
    P.dT0 = (T)(M->d.T0 - (double)P.Toff); P.dS0 = (T)(M->d.S0 - (double)P.Soff);
    P.rho0 = (T)M->d.rho0; P.rrho0 = (T)(1.0 / M->d.rho0);
    P.g_d = M->d.g; P.alpha_d = M->d.alpha; P.beta_d = M->d.beta_s; P.hz_top_d = g->zf[nz] - g->zc[nz - 1];
    P.dT0_d = M->d.T0 - (double)P.Toff; P.dS0_d = M->d.S0 - (double)P.Soff;
    P.nu_h = (T)M->d.nu_h; P.kappa_h = (T)M->d.kappa_h; P.dtau = (T)M->dtau;
    if ((s = upload(M, M->a_w, &P.fw_a)) != OCN_OK || (s = upload(M, M->b_w, &P.fw_b)) != OCN_OK) return s;
    // equation of state: per-level thermal expansion alpha (1 - gamma zc[k]) and alpha2 / 2, in the fp64
    // operations the equation is written in
    if ((s = dev_alloc(M, 64, &P.timeline, false)) != OCN_OK) return s;
    P.geo_thr = sizeof(T) == 4 ? K1_GEO_THR : 1 << 20;   // fp64: lane efficiency decides (measured on config 2: 9.0 ms compact, 11.6 geometric)
    P.eos = M->d.eos; P.ha2_d = 0.5 * M->d.eos_alpha2;
    {
        std::vector<double> ath(nz);
        for (int k = 0; k < nz; ++k) ath[k] = M->d.alpha * (1.0 - M->d.eos_gamma * g->zc[k]);
        const double* a = nullptr;
        if ((s = upload<double>(M, ath, &a)) != OCN_OK) return s;
        P.ath_d = a;
    }
    // Hu, Hv = sum_k dz over open faces, and reciprocals
    {
        std::vector<T> hu(n2 + 2 * LEAD, T(0)), hv(hu), rhu(hu), rhv(hu);
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                const uint64_t w = g->m8[g->pidx(j, i)];
                const int tx1 = (w >> 8) & 255, ty1 = (w >> 32) & 255;
                double a = 0, b = 0;
                for (int k = 0; k < nz; ++k) { if (k >= tx1) a += g->dz[k]; if (k >= ty1) b += g->dz[k]; }
                const size_t q = g->pidx(j, i);
                hu[q] = (T)a; hv[q] = (T)b; rhu[q] = a > 0 ? (T)(1.0 / a) : T(0); rhv[q] = b > 0 ? (T)(1.0 / b) : T(0);
            }
        const size_t nb = hu.size() * sizeof(T);
        DEV(cudaMemcpyAsync(P.Hu - LEAD, hu.data(), nb, cudaMemcpyHostToDevice, M->stream));
        DEV(cudaMemcpyAsync(P.Hv - LEAD, hv.data(), nb, cudaMemcpyHostToDevice, M->stream));
        DEV(cudaMemcpyAsync(P.rHu - LEAD, rhu.data(), nb, cudaMemcpyHostToDevice, M->stream));
        DEV(cudaMemcpyAsync(P.rHv - LEAD, rhv.data(), nb, cudaMemcpyHostToDevice, M->stream));
        DEV(cudaStreamSynchronize(M->stream));
    }
    {
        auto mk = [&](ocn_model::Stage& st, size_t bytes) -> ocn_status {
            const ocn_status sa = raw_alloc(M, bytes, &st.buf, false);
            if (sa != OCN_OK) return sa;
            st.bytes = bytes;
            DEV(cudaEventCreateWithFlags(&st.filled, cudaEventDisableTiming));
            DEV(cudaEventCreateWithFlags(&st.freed, cudaEventDisableTiming));
            return OCN_OK;
        };
        if ((s = mk(M->big, (size_t)(nz + 1) * g->ny * g->nx * sizeof(double))) != OCN_OK) return s;
        for (auto& st : M->small_) if ((s = mk(st, (size_t)g->ny * g->nx * sizeof(double))) != OCN_OK) return s;
        DEV(cudaStreamCreateWithFlags(&M->copy_stream, cudaStreamNonBlocking));
        for (auto& e : M->ticket_ev) DEV(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    if (M->measure) return OCN_OK;                 // everything below allocates nothing
    M->launches_per_step = (M->d.substeps + bt_substeps_per_launch<T>() - 1) / bt_substeps_per_launch<T>() + 3 + (P.bih ? 2 : 0);
    // TMA descriptors: box origin (i0 - 4, j0 - 3), so the map starts 4 elements before (row -3, i = 0)
    {
        typedef ocn::Tile<T, TILE_X, TILE_Y> C;
        const bool f64 = sizeof(T) == 8;
        const unsigned long long sxu = (unsigned long long)g->sx, syu = (unsigned long long)g->sy;
        if ((s = make_tmap(&M->tm_ts, f64, (T*)P.ts - 2 * C::OX, 2 * sxu, syu, nz, 2 * C::BX, C::BY)) != OCN_OK ||
            (s = make_tmap(&M->tm_uv, f64, (T*)P.uv - 2 * C::OX, 2 * sxu, syu, nz, 2 * C::BX, C::BY)) != OCN_OK ||
            (s = make_tmap(&M->tm_p, true, P.p - C::OX, sxu, syu, nz, C::PBX, TILE_Y + 1)) != OCN_OK)
            return s;
        for (int id = 0; id < 8; ++id)
            CK(cudaFuncSetAttribute(k1_fused<T>(id & 4, id & 2, id & 1), cudaFuncAttributeMaxDynamicSharedMemorySize, k1_smem<T>(id & 2)));
        CK(cudaFuncSetAttribute(ocn::k_barotropic_tile<T, BT_X, BT_Y>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                ocn::BtTile<T, BT_X, BT_Y>::SMEM));
        CK(cudaFuncSetAttribute(ocn::k_barotropic_strip<BS_X, BS_Y, BS_H>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                ocn::BtStrip<BS_X, BS_Y, BS_H>::SMEM));
    }
    return OCN_OK;
}

}  // namespace

// =================================================================================================
// step scheduling
// =================================================================================================
namespace {

ocn_status prof_flush(ocn_model* M) {           // fold recorded events into the per-stage totals
    M->ev_used -= M->ev_used % (OCN_NSTAGES + 1);   // a step that failed between two marks left an incomplete group: drop it
    if (M->ev_used == 0) return OCN_OK;
    CK(cudaStreamSynchronize(M->stream));
    for (size_t q = 0; q + OCN_NSTAGES < M->ev_used; q += OCN_NSTAGES + 1)
        for (int s = 0; s < OCN_NSTAGES; ++s) {
            static const int in_time_order[OCN_NSTAGES] = {0, 1, 3, 2};   // the closure stage runs before K3
            float ms = 0.f;
            CK(cudaEventElapsedTime(&ms, M->ev_pool[q + s], M->ev_pool[q + s + 1]));
            M->prof_ms[in_time_order[s]] += ms;
        }
    M->ev_used = 0;
    return OCN_OK;
}

ocn_status prof_mark(ocn_model* M) {
    if (!M->profiling) return OCN_OK;
    if (M->ev_used == M->ev_pool.size()) {
        cudaEvent_t e;
        CK(cudaEventCreate(&e));
        M->ev_pool.push_back(e);
    }
    CK(cudaEventRecord(M->ev_pool[M->ev_used++], M->stream));
    return OCN_OK;
}

// number of launches of the barotropic sub-cycle (each advances bt_substeps_per_launch sub-steps)
template <class T> int bt_launches(const ocn_model* M) { return (M->d.substeps + bt_substeps_per_launch<T>() - 1) / bt_substeps_per_launch<T>(); }

// part < 0: the whole step.  Else one part of it (ocn_step_part): 0 = tendency pass, 1 + q = launch q of the sub-cycle,
// bt_launches + 1 = end of the sub-cycle, back-substitution and correction.
template <class T>
ocn_status launch_step(ocn_model* M, bool euler, int part = -1) {
    const ocn_grid* g = M->g;
    ocn_status ps;
    const int last_part = bt_launches<T>(M) + 1;
    M->ev_used -= M->ev_used % (OCN_NSTAGES + 1);   // groups start on a step boundary (see prof_flush)
    if (M->profiling && M->ev_used + OCN_NSTAGES + 1 > 4096 && (ps = prof_flush(M)) != OCN_OK) return ps;
#define MARK(stage, n)                                                   \
    do {                                                                 \
        if (part >= 0) break;                   /* parts are not profiled */ \
        if ((ps = prof_mark(M)) != OCN_OK) return ps;                    \
        if (M->profiling && (stage) >= 0) M->prof_launches[stage] += (n); \
    } while (0)
    const ocn::DevP<T>& P = params<T>(M);
    const T c0 = euler ? T(1) : (T)(1.5 + M->d.chi), c1 = euler ? T(0) : (T)(0.5 + M->d.chi);
    const dim3 bc(32, 4), b2(32, 8);
    MARK(-1, 0);
    if (part < 0 || part == 0) {
        const dim3 bt(TILE_X, TILE_Y), gt = grid2(g, bt);
        if (P.bih) {                               // biharmonic pre-pass: L of the state, then -coefficient L(L)
            ocn::k_laplacians<T><<<grid2(g, bc), bc, 0, M->stream>>>(P, P.uv, P.ts, P.Luv, P.Lts, T(1), T(1), 0);
            ocn::k_laplacians<T><<<grid2(g, bc), bc, 0, M->stream>>>(P, P.Luv, P.Lts, P.Buv, P.Bts, (T)M->d.nu4_h, (T)M->d.kappa4_h, 1);
        }
        // the extras instantiation carries bottom drag and the biharmonic add
        const bool drag = M->d.drag_r != 0.0 || M->d.drag_cd != 0.0 || P.bih, ri = M->d.closure == 1, wz = M->d.advection == 1;
        k1_fused<T>(drag, ri, wz)<<<gt, bt, k1_smem<T>(ri), M->stream>>>(P, c0, c1, M->tm_ts, M->tm_uv, M->tm_p);
    }
    MARK(0, P.bih ? 3 : 1);
    if constexpr (sizeof(T) == 4) {                // register-strip kernel, BS_H sub-steps per launch
        typedef ocn::BtStrip<BS_X, BS_Y, BS_H> B;
        const dim3 gb((g->nx + BS_X - 1) / BS_X, (g->ny + BS_Y - 1) / BS_Y);
        int cur = 0;
        for (int m0 = 0, q = 0; m0 < M->d.substeps; m0 += BS_H, ++q) {
            const int ns = std::min(BS_H, M->d.substeps - m0);
            if (part < 0 || part == 1 + q)
                ocn::k_barotropic_strip<BS_X, BS_Y, BS_H><<<gb, B::NT, B::SMEM, M->stream>>>(P, cur, ns, m0 == 0 ? 1 : 0, m0);
            cur ^= 1;
        }
    } else {
        typedef ocn::BtTile<T, BT_X, BT_Y> B;
        const dim3 gb((g->nx + BT_X - 1) / BT_X, (g->ny + BT_Y - 1) / BT_Y);
        int cur = 0;
        for (int m0 = 0, q = 0; m0 < M->d.substeps; m0 += BT_HALO, ++q) {
            const int ns = std::min(BT_HALO, M->d.substeps - m0);
            if (part < 0 || part == 1 + q)
                ocn::k_barotropic_tile<T, BT_X, BT_Y><<<gb, B::NT, B::SMEM, M->stream>>>(P, cur, ns, m0 == 0 ? 1 : 0, m0);
            cur ^= 1;
        }
    }
    if (part >= 0 && part != last_part) { CK(cudaGetLastError()); return OCN_OK; }
    const ocn::PeerPut<T>& Q = peer_put<T>(M);
    ocn::k_barotropic_finish<T><<<grid2(g, b2), b2, 0, M->stream>>>(P);
    MARK(1, (M->d.substeps + bt_substeps_per_launch<T>() - 1) / bt_substeps_per_launch<T>() + 1);
    MARK(3, 0);                                    // (the closure is evaluated inside K1: stage 3 is empty)
    {
        // rows lo .. hi - 1 with the plain kernel or with the one that also stores into the neighbours' arrays
        auto k3 = [&](int lo, int hi, bool put) {
            if (hi <= lo) return;
            ocn::PeerPut<T> R = Q;
            R.own_lo = lo; R.own_hi = hi;
            const dim3 gk((g->nx + bc.x - 1) / bc.x, (hi - lo + bc.y - 1) / bc.y);
            const bool ri = M->d.closure == 1;
            if (put) {
                if (ri) ocn::k_backsub_correct<T, true, true><<<gk, bc, 0, M->stream>>>(P, R);
                else ocn::k_backsub_correct<T, false, true><<<gk, bc, 0, M->stream>>>(P, R);
            } else {
                if (ri) ocn::k_backsub_correct<T, true><<<gk, bc, 0, M->stream>>>(P, R);
                else ocn::k_backsub_correct<T, false><<<gk, bc, 0, M->stream>>>(P, R);
            }
        };
        if (!M->put) k3(0, g->ny, false);
        else k3(Q.own_lo, Q.own_hi, true);         // own rows only; the mirrored rows among them also go to the neighbours
    }
    MARK(2, 1);
#undef MARK
    CK(cudaGetLastError());
    return OCN_OK;
}

template <class T>
ocn_status run_steps(ocn_model* M, int n) {
    ocn_status s;
    while (n > 0 && !M->have_history) {          // Euler start after ocn_set_fields
        if ((s = launch_step<T>(M, true)) != OCN_OK) return s;
        M->have_history = true; --n;
    }
    if (n <= 0) return OCN_OK;
    if (M->profiling) {                           // direct launches with stage events
        for (int q = 0; q < n; ++q) if ((s = launch_step<T>(M, false)) != OCN_OK) return s;
        return OCN_OK;
    }
    if (!M->graph) {                              // capture one steady-state step once
        cudaGraph_t gr = nullptr;
        CK(cudaStreamBeginCapture(M->stream, cudaStreamCaptureModeThreadLocal));
        s = launch_step<T>(M, false);
        cudaError_t e = cudaStreamEndCapture(M->stream, &gr);
        if (s != OCN_OK) { if (gr) cudaGraphDestroy(gr); return s; }
        CK(e);
        CK(cudaGraphInstantiate(&M->graph, gr, 0));
        CK(cudaGraphDestroy(gr));
    }
    for (int q = 0; q < n; ++q) CK(cudaGraphLaunch(M->graph, M->stream));
    return OCN_OK;
}

// a staging region for `bytes`: 2-D fields take the next small region of the ring, 3-D fields the big one
ocn_model::Stage& stage_for(ocn_model* M, size_t bytes) {
    if (bytes > M->small_[0].bytes) return M->big;
    ocn_model::Stage& st = M->small_[M->next_small];
    M->next_small = (M->next_small + 1) % ocn_model::NSMALL;
    return st;
}

// host -> device: the copy runs on the copy stream (beside whatever the main stream is doing), the masked scatter into the
// halo'd layout on the main stream after it; the host waits for the DMA only, so its buffer is reusable on return
template <class T>
ocn_status set_one(ocn_model* M, const void* src, T* dst, int nl, int kind, bool on_device, int st = 1) {
    const ocn_grid* g = M->g;
    const size_t n = (size_t)nl * g->ny * g->nx;
    const T* dsrc = static_cast<const T*>(src);
    ocn_model::Stage* sg = nullptr;
    if (!on_device) {
        sg = &stage_for(M, n * sizeof(T));
        CK(cudaStreamWaitEvent(M->copy_stream, sg->freed, 0));          // its last consumer (an event never recorded is complete)
        CK(cudaMemcpyAsync(sg->buf, src, n * sizeof(T), cudaMemcpyHostToDevice, M->copy_stream));
        CK(cudaEventRecord(sg->filled, M->copy_stream));
        CK(cudaStreamWaitEvent(M->stream, sg->filled, 0));
        dsrc = static_cast<const T*>(sg->buf);
    }
    const dim3 b(32, 8);
    ocn::k_scatter<T><<<grid2(g, b, nl < 64 ? nl : 64), b, 0, M->stream>>>(params<T>(M), dst, dsrc, nl, kind, st);
    CK(cudaGetLastError());
    if (sg) {
        CK(cudaEventRecord(sg->freed, M->stream));
        CK(cudaEventSynchronize(sg->filled));
    }
    return OCN_OK;
}

template <class T>
ocn_status set_fields_t(ocn_model* M, const ocn_fields* f) {
    ocn::DevP<T>& P = params<T>(M);
    const int nz = M->g->nz;
    const bool dev = f->on_device != 0;
    ocn_status s;
    if (f->u && (s = set_one<T>(M, f->u, (T*)P.uv, nz, 0, dev, 2)) != OCN_OK) return s;
    if (f->v && (s = set_one<T>(M, f->v, (T*)P.uv + 1, nz, 1, dev, 2)) != OCN_OK) return s;
    if (f->T && (s = set_one<T>(M, f->T, (T*)P.ts, nz, 2, dev, 2)) != OCN_OK) return s;
    if (f->S && (s = set_one<T>(M, f->S, (T*)P.ts + 1, nz, 3, dev, 2)) != OCN_OK) return s;
    if (f->eta && (s = set_one<T>(M, f->eta, P.eta[0], 1, 4, dev)) != OCN_OK) return s;
    if (f->tau_x && (s = set_one<T>(M, f->tau_x, P.taux, 1, 5, dev)) != OCN_OK) return s;
    if (f->tau_y && (s = set_one<T>(M, f->tau_y, P.tauy, 1, 5, dev)) != OCN_OK) return s;
    if (f->flux_T && (s = set_one<T>(M, f->flux_T, (T*)P.qts, 1, 4, dev, 2)) != OCN_OK) return s;
    if (f->flux_S && (s = set_one<T>(M, f->flux_S, (T*)P.qts + 1, 1, 4, dev, 2)) != OCN_OK) return s;
    if (f->restore_T && (s = set_one<T>(M, f->restore_T, (T*)P.rts, 1, 7, dev, 2)) != OCN_OK) return s;
    if (f->restore_S && (s = set_one<T>(M, f->restore_S, (T*)P.rts + 1, 1, 8, dev, 2)) != OCN_OK) return s;
    if (f->u || f->v || f->T || f->S || f->eta) {
        const dim3 bc(32, 4);
        ocn::k_init_transport<T><<<grid2(M->g, bc), bc, 0, M->stream>>>(P);
        ocn::k_pressure<T><<<grid2(M->g, bc), bc, 0, M->stream>>>(P);
        CK(cudaGetLastError());
        M->have_history = false;
        M->split_next = 0;                     // a split step in progress is abandoned with the state it was advancing
    }
    return OCN_OK;
}

// device -> host: gather into a staging region on the main stream, copy out on the copy stream; `last` receives the event
// that marks the completion of the copy (the caller waits for it, or hands it out as a ticket)
template <class T, class O>
ocn_status get_one(ocn_model* M, void* dst, const T* src, int nl, int kind, bool on_device, int st = 1, cudaEvent_t* last = nullptr) {
    const ocn_grid* g = M->g;
    const size_t n = (size_t)nl * g->ny * g->nx;
    ocn_model::Stage* sg = nullptr;
    O* ddst = static_cast<O*>(dst);
    if (!on_device) {
        sg = &stage_for(M, n * sizeof(O));
        CK(cudaStreamWaitEvent(M->stream, sg->freed, 0));
        ddst = static_cast<O*>(sg->buf);
    }
    const dim3 b(32, 8);
    ocn::k_gather<T, O><<<grid2(g, b, nl < 64 ? nl : 64), b, 0, M->stream>>>(params<T>(M), ddst, src, nl, kind, st);
    CK(cudaGetLastError());
    if (sg) {
        CK(cudaEventRecord(sg->filled, M->stream));
        CK(cudaStreamWaitEvent(M->copy_stream, sg->filled, 0));
        CK(cudaMemcpyAsync(dst, sg->buf, n * sizeof(O), cudaMemcpyDeviceToHost, M->copy_stream));
        CK(cudaEventRecord(sg->freed, M->copy_stream));
        if (last) *last = sg->freed;
        else CK(cudaEventSynchronize(sg->freed));
    }
    return OCN_OK;
}

// ticket: NULL = blocking (returns when every copy has landed); else the copies are left in flight and *ticket names them
template <class T>
ocn_status get_fields_t(ocn_model* M, ocn_fields* f, unsigned long long* ticket) {
    ocn::DevP<T>& P = params<T>(M);
    const int nz = M->g->nz;
    const bool dev = f->on_device != 0;
    ocn_status s;
    cudaEvent_t last = nullptr;
    if (f->u && (s = get_one<T, T>(M, f->u, (T*)P.uv, nz, 0, dev, 2, &last)) != OCN_OK) return s;
    if (f->v && (s = get_one<T, T>(M, f->v, (T*)P.uv + 1, nz, 1, dev, 2, &last)) != OCN_OK) return s;
    if (f->T && (s = get_one<T, T>(M, f->T, (T*)P.ts, nz, 2, dev, 2, &last)) != OCN_OK) return s;
    if (f->S && (s = get_one<T, T>(M, f->S, (T*)P.ts + 1, nz, 3, dev, 2, &last)) != OCN_OK) return s;
    if (f->w) {                                   // w is diagnosed on demand (K1 recomputes it on the fly)
        const dim3 bc(32, 4);
        ocn::k_vertical_velocity<T><<<grid2(M->g, bc), bc, 0, M->stream>>>(P);
        CK(cudaGetLastError());
    }
    if (f->w && (s = get_one<T, T>(M, f->w, P.w, nz + 1, 6, dev, 1, &last)) != OCN_OK) return s;
    if (f->eta && (s = get_one<T, T>(M, f->eta, P.eta[0], 1, 4, dev, 1, &last)) != OCN_OK) return s;
    if (f->tau_x && (s = get_one<T, T>(M, f->tau_x, P.taux, 1, 5, dev, 1, &last)) != OCN_OK) return s;
    if (f->tau_y && (s = get_one<T, T>(M, f->tau_y, P.tauy, 1, 5, dev, 1, &last)) != OCN_OK) return s;
    if (ticket) {                                 // the copy stream is in order: its position after the last copy covers them all
        cudaEvent_t e = M->ticket_ev[M->tickets % ocn_model::NTICKET];
        if (dev) CK(cudaEventRecord(e, M->stream)); else CK(cudaEventRecord(e, M->copy_stream));
        *ticket = M->tickets++;
        return OCN_OK;
    }
    if (dev || !last) CK(cudaStreamSynchronize(M->stream));
    else CK(cudaEventSynchronize(last));          // implies everything the main stream did before the last gather
    CK(cudaGetLastError());
    return OCN_OK;
}

template <class T>
ocn_status get_debug_t(ocn_model* M, double* Gu, double* Gv, double* GT, double* GS, double* U, double* V) {
    ocn::DevP<T>& P = params<T>(M);
    const int nz = M->g->nz;
    ocn_status s;
    if (Gu && (s = get_one<T, double>(M, Gu, (T*)P.Guv, nz, 5, false, 2)) != OCN_OK) return s;
    if (Gv && (s = get_one<T, double>(M, Gv, (T*)P.Guv + 1, nz, 5, false, 2)) != OCN_OK) return s;
    if (GT && (s = get_one<T, double>(M, GT, (T*)P.Gts, nz, 5, false, 2)) != OCN_OK) return s;
    if (GS && (s = get_one<T, double>(M, GS, (T*)P.Gts + 1, nz, 5, false, 2)) != OCN_OK) return s;
    if (U && (s = get_one<T, double>(M, U, P.U[0], 1, 5, false)) != OCN_OK) return s;
    if (V && (s = get_one<T, double>(M, V, P.V[0], 1, 5, false)) != OCN_OK) return s;
    return OCN_OK;
}

template <class T>
ocn_status get_mixing_t(ocn_model* M, double* nu, double* kappa) {
    ocn::DevP<T>& P = params<T>(M);
    const int nz = M->g->nz;
    const dim3 bc(32, 4);
    if (!P.nk) {                                   // the output array of the diagnostic (the step itself keeps (nu, kappa) on chip)
        char* const ws = M->ws;                    // allocated by the library on first use, also for a model in a workspace
        M->ws = nullptr;
        const ocn_status sa = dev_alloc(M, (size_t)P.sz * nz, &P.nk, true);
        M->ws = ws;
        if (sa != OCN_OK) return sa;
    }
    ocn::k_ri_mixing<T><<<grid2(M->g, bc), bc, 0, M->stream>>>(P);
    CK(cudaGetLastError());
    ocn_status s;
    if (nu && (s = get_one<T, double>(M, nu, (T*)P.nk, nz, 5, false, 2)) != OCN_OK) return s;
    if (kappa && (s = get_one<T, double>(M, kappa, (T*)P.nk + 1, nz, 5, false, 2)) != OCN_OK) return s;
    return OCN_OK;
}

// Device address of g_noalloc_scratch on `device`, which must be the CURRENT device; looked up once per device.
ocn_status noalloc_scratch(int device, void** out) {
    constexpr int MAXDEV = 64;
    static std::mutex mu;
    static void* addr[MAXDEV] = {};
    std::lock_guard<std::mutex> lock(mu);
    if (device >= 0 && device < MAXDEV && addr[device]) { *out = addr[device]; return OCN_OK; }
    void* p = nullptr;
    CK(cudaGetSymbolAddress(&p, g_noalloc_scratch));
    if (!p) return fail(OCN_ECUDA, "cudaGetSymbolAddress returned a null address for the scratch array");
    if (device >= 0 && device < MAXDEV) addr[device] = p;
    *out = p;
    return OCN_OK;
}

// ocn_get_mixing without any allocation: k_ri_mixing writes into the static scratch array instead of a cudaMalloc'ed one.
// The kernel only stores open faces (and the zeros that complete a sector), and relies on everything else being zero, so
// the part of the scratch this model uses is cleared first: the array keeps whatever the last call (of any model) left.
template <class T>
ocn_status get_mixing_noalloc_t(ocn_model* M, double* nu, double* kappa) {
    typedef typename ocn::Pair<T>::type T2;
    ocn::DevP<T> P = params<T>(M);                 // a copy: the model's own parameter block (and its nk, if any) stays as it is
    const int nz = M->g->nz;
    const size_t bytes = ((size_t)P.sz * nz + 2 * LEAD) * sizeof(T2);
    if (bytes > (size_t)OCN_NOALLOC_SCRATCH_BYTES)
        return fail(OCN_EUNSUPPORTED, "ocn_get_mixing_noalloc: the (nu, kappa) planes of this model need " + std::to_string(bytes) +
                                      " bytes, the static scratch holds " + std::to_string((size_t)OCN_NOALLOC_SCRATCH_BYTES) +
                                      " (use ocn_get_mixing)");
    void* base = nullptr;
    ocn_status s = noalloc_scratch(M->d.device, &base);
    if (s != OCN_OK) return s;
    CK(cudaMemsetAsync(base, 0, bytes, M->stream));
    P.nk = reinterpret_cast<T2*>(base) + LEAD;
    const dim3 bc(32, 4);
    ocn::k_ri_mixing<T><<<grid2(M->g, bc), bc, 0, M->stream>>>(P);
    CK(cudaGetLastError());
    if (nu && (s = get_one<T, double>(M, nu, (T*)P.nk, nz, 5, false, 2)) != OCN_OK) return s;
    if (kappa && (s = get_one<T, double>(M, kappa, (T*)P.nk + 1, nz, 5, false, 2)) != OCN_OK) return s;
    return OCN_OK;
}

}  // namespace

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

const char* ocn_last_error(void) { return g_err.c_str(); }
const char* ocn_version(void) { return "libocn 0.1 (sm_100a)"; }

ocn_status ocn_grid_create(const ocn_grid_desc* d, const double* z_faces, const double* depth, ocn_grid** out) {
    if (!d || !z_faces || !depth || !out) return fail(OCN_EINVAL, "null argument");
    if (d->nx < OCN_HALO || d->ny < OCN_HALO || d->nz < 2) return fail(OCN_EINVAL, "grid too small (nx, ny >= 3, nz >= 2)");
    if (d->nz > 250) return fail(OCN_EUNSUPPORTED, "nz > 250 (level thresholds are stored in 8 bits)");
    if (d->kind != 0 && d->kind != 1) return fail(OCN_EINVAL, "kind must be 0 (cartesian) or 1 (lat-lon)");
    if (d->kind == 1 && d->periodic_y) return fail(OCN_EINVAL, "a lat-lon grid cannot be periodic in latitude");
    if (!(d->dx > 0) || !(d->dy > 0)) return fail(OCN_EINVAL, "dx, dy must be positive");
    if (d->j_offset < 0 || d->ny_global < 0 || (d->ny_global > 0 && d->j_offset + d->ny > d->ny_global) ||
        (d->ny_global == 0 && d->j_offset != 0))
        return fail(OCN_EINVAL, "j_offset / ny_global: the band must lie inside the whole grid (0, 0 = a grid of its own)");
    if (d->ny_global > 0 && d->periodic_y) return fail(OCN_EINVAL, "a latitude band is bounded in y (periodic_y = 0)");

    ocn_grid* g = new (std::nothrow) ocn_grid();
    if (!g) return fail(OCN_ENOMEM, "host allocation failed");
    try {
        const std::string e = ocn_host::build_grid(*g, *d, z_faces, depth);
        if (!e.empty()) { delete g; return fail(OCN_EINVAL, e); }
    } catch (const std::exception& ex) { delete g; return fail(OCN_ENOMEM, ex.what()); }
    *out = g;
    return OCN_OK;
}

ocn_status ocn_grid_destroy(ocn_grid* g) { delete g; return OCN_OK; }

ocn_status ocn_get_masks(const ocn_grid* g, unsigned char* wet, unsigned char* ox, unsigned char* oy,
                         unsigned char* oz, unsigned char* ozu, unsigned char* ozv) {
    if (!g) return fail(OCN_EINVAL, "null grid");
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    for (int k = 0; k <= nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const uint64_t m = g->m8[g->pidx(j, i)];
                const uint32_t z = g->mz[g->pidx(j, i)];
                const int kb = m & 255, tx1 = (m >> 8) & 255, tx2 = (m >> 16) & 255, tx3 = (m >> 24) & 255;
                const int ty1 = (m >> 32) & 255, ty2 = (m >> 40) & 255, ty3 = (m >> 48) & 255;
                const size_t n = ((size_t)k * ny + j) * nx + i;
                if (oz) oz[n] = (unsigned char)((k >= 1 && k < nz) ? std::max(0, std::min(3, std::min(k - kb, nz - k))) : 0);
                if (k == nz) continue;
                if (wet) wet[n] = k >= kb;
                if (ox) ox[n] = (unsigned char)((k >= tx1) + (k >= tx2) + (k >= tx3));
                if (oy) oy[n] = (unsigned char)((k >= ty1) + (k >= ty2) + (k >= ty3));
                if (ozu) ozu[n] = (unsigned char)(k >= tx1 ? 1 + (k >= (int)(z & 255)) + (k >= (int)((z >> 8) & 255)) : 0);
                if (ozv) ozv[n] = (unsigned char)(k >= ty1 ? 1 + (k >= (int)((z >> 16) & 255)) + (k >= (int)(z >> 24)) : 0);
            }
    return OCN_OK;
}

// measure_bytes != nullptr: the dry run of ocn_model_workspace_bytes (no device call, no model returned)
static ocn_status create_impl(const ocn_grid* g, const ocn_model_desc* d, ocn_model** out, unsigned long long* measure_bytes) {
    const bool measure = measure_bytes != nullptr;
    if (!g || !d || (!out && !measure)) return fail(OCN_EINVAL, "null argument");
    if (d->precision != 32 && d->precision != 64) return fail(OCN_EINVAL, "precision must be 32 or 64");
    if (!(d->dt > 0) || d->substeps < 1) return fail(OCN_EINVAL, "dt must be > 0 and substeps >= 1");
    if (!(d->rho0 > 0)) return fail(OCN_EINVAL, "rho0 must be > 0");
    {
        const double nonneg[] = {d->chi, d->g, d->nu_h, d->kappa_h, d->nu_z, d->kappa_z};
        for (double x : nonneg) if (!(x >= 0) || !std::isfinite(x)) return fail(OCN_EINVAL, "chi, g, nu_h, kappa_h, nu_z, kappa_z must be finite and >= 0");
        const double fin[] = {d->dt, d->alpha, d->beta_s, d->T0, d->S0, d->rho0, d->gamma_T, d->gamma_S, d->drag_r, d->drag_cd};
        for (double x : fin) if (!std::isfinite(x)) return fail(OCN_EINVAL, "model parameters must be finite");
    }
    if (!(d->gamma_T >= 0) || !(d->gamma_S >= 0)) return fail(OCN_EINVAL, "gamma_T, gamma_S must be >= 0");
    if (!(d->drag_r >= 0) || !(d->drag_cd >= 0)) return fail(OCN_EINVAL, "drag_r, drag_cd must be >= 0");
    if (d->closure != 0 && d->closure != 1) return fail(OCN_EINVAL, "closure must be 0 (constant) or 1 (Ri-based)");
    if (!(d->nu4_h >= 0 && d->kappa4_h >= 0) || !std::isfinite(d->nu4_h) || !std::isfinite(d->kappa4_h))
        return fail(OCN_EINVAL, "nu4_h, kappa4_h must be finite and >= 0");
    if (d->eos != 0 && d->eos != 1) return fail(OCN_EINVAL, "eos must be 0 (linear) or 1 (nonlinear)");
    if (d->eos == 1 && !(std::isfinite(d->eos_alpha2) && std::isfinite(d->eos_gamma))) return fail(OCN_EINVAL, "eos_alpha2, eos_gamma must be finite");
    if (d->advection != 0 && d->advection != 1) return fail(OCN_EINVAL, "advection must be 0 (WENO-JS) or 1 (WENO-Z)");
    if (d->closure == 1 && !(d->ri_n2c > 0 && d->ri_s2min > 0 && d->ri_c >= 0 && d->ri_nu0 >= 0 && d->ri_kconv >= 0))
        return fail(OCN_EINVAL, "Ri closure: ri_n2c, ri_s2min must be > 0 and ri_c, ri_nu0, ri_kconv >= 0");
    if (!measure && d->workspace && ((uintptr_t)d->workspace & 255u))
        return fail(OCN_EINVAL, "workspace must be 256-byte aligned device memory");
    int ndev = 0;
    if (!measure) {
        if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
            return fail(OCN_ECUDA, "no CUDA device: libocn has no CPU fallback");
        if (d->device < 0 || d->device >= ndev) return fail(OCN_EINVAL, "bad device ordinal");
    }
    DeviceGuard guard_(measure ? -1 : d->device);
    if (!measure) CK(guard_.err);
    ocn_model* M = new (std::nothrow) ocn_model();
    if (!M) return fail(OCN_ENOMEM, "host allocation failed");
    M->g = g; M->d = *d; M->prec = d->precision;
    M->measure = measure;
    if (!measure && d->workspace) { M->ws = static_cast<char*>(d->workspace); M->ws_cap = (size_t)d->workspace_bytes; }
    M->d.workspace = nullptr;
    // filter weights: power law p = 2, q = 4 unless given; dtau centres the average on t^{n+1}
    const int Ms = d->substeps;
    M->a_w.resize(Ms);
    if (d->filter_weights) {
        double sum = 0;
        for (int m = 0; m < Ms; ++m) { M->a_w[m] = d->filter_weights[m]; sum += M->a_w[m]; }
        if (!std::isfinite(sum) || std::fabs(sum - 1.0) > 1e-9) {
            delete M;
            return fail(OCN_EINVAL, "filter_weights must be finite and sum to 1 (they average eta, U, V over the sub-cycle)");
        }
    } else {
        double sum = 0;
        for (int m = 1; m <= Ms; ++m) { const double s = (double)m / (double)(Ms + 1); M->a_w[m - 1] = s * s * (1.0 - s * s * s * s); sum += M->a_w[m - 1]; }
        for (int m = 0; m < Ms; ++m) M->a_w[m] /= sum;
    }
    double first = 0;
    for (int m = 1; m <= Ms; ++m) first += m * M->a_w[m - 1];
    if (!(first > 0)) { delete M; return fail(OCN_EINVAL, "filter weights have no positive first moment"); }
    M->dtau = d->dt * (1.0 / first);
    M->d.filter_weights = nullptr;
    M->b_w = M->a_w;
    if (d->filter_weights_uv) {
        double sum = 0;
        for (int m = 0; m < Ms; ++m) { M->b_w[m] = d->filter_weights_uv[m]; sum += M->b_w[m]; }
        if (!std::isfinite(sum) || std::fabs(sum - 1.0) > 1e-9) {
            delete M;
            return fail(OCN_EINVAL, "filter_weights_uv must be finite and sum to 1");
        }
    }
    M->d.filter_weights_uv = nullptr;
    if (measure) {
        const ocn_status s = d->precision == 32 ? build_model<float>(M) : build_model<double>(M);
        *measure_bytes = (unsigned long long)((M->ws_used + 255) / 256 * 256);
        delete M;
        return s;
    }
    if (d->stream) M->stream = static_cast<cudaStream_t>(d->stream);
    else {
        cudaError_t e = cudaStreamCreateWithFlags(&M->stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) { delete M; return fail(OCN_ECUDA, cudaGetErrorString(e)); }
        M->own_stream = true;
    }
    const ocn_status s = d->precision == 32 ? build_model<float>(M) : build_model<double>(M);
    if (s != OCN_OK) { const std::string keep = g_err; ocn_model_destroy(M); g_err = keep; return s; }
    *out = M;
    return OCN_OK;
}

ocn_status ocn_model_create(const ocn_grid* g, const ocn_model_desc* d, ocn_model** out) {
    if (!out) return fail(OCN_EINVAL, "null argument");
    return create_impl(g, d, out, nullptr);
}

ocn_status ocn_model_workspace_bytes(const ocn_grid* g, const ocn_model_desc* d, unsigned long long* bytes) {
    if (!bytes) return fail(OCN_EINVAL, "null argument");
    return create_impl(g, d, nullptr, bytes);
}

ocn_status ocn_model_destroy(ocn_model* M) {
    if (!M) return OCN_OK;
    DeviceGuard guard_(M->d.device);
    if (M->stream) cudaStreamSynchronize(M->stream);
    if (M->graph) cudaGraphExecDestroy(M->graph);
    for (cudaEvent_t e : M->ev_pool) cudaEventDestroy(e);
    for (void* p : M->allocs) cudaFree(p);
    if (M->copy_stream) { cudaStreamSynchronize(M->copy_stream); cudaStreamDestroy(M->copy_stream); }
    for (ocn_model::Stage* st : {&M->big, &M->small_[0], &M->small_[1], &M->small_[2], &M->small_[3], &M->small_[4], &M->small_[5],
                                 &M->small_[6], &M->small_[7]}) {
        if (st->filled) cudaEventDestroy(st->filled);      // (the buffer is in `allocs` or in the caller's workspace)
        if (st->freed) cudaEventDestroy(st->freed);
    }
    for (cudaEvent_t e : M->ticket_ev) if (e) cudaEventDestroy(e);
    for (void* b : M->ipc_open) cudaIpcCloseMemHandle(b);
    if (M->own_stream && M->stream) cudaStreamDestroy(M->stream);
    delete M;
    return OCN_OK;
}

ocn_status ocn_set_fields(ocn_model* M, const ocn_fields* f) {
    if (!M || !f) return fail(OCN_EINVAL, "null argument");
    if (f->w) return fail(OCN_EINVAL, "w is diagnostic (get only)");
    ON_DEVICE(M->d.device);
    return M->prec == 32 ? set_fields_t<float>(M, f) : set_fields_t<double>(M, f);
}

ocn_status ocn_time_step(ocn_model* M, int n) {
    if (!M || n < 0) return fail(OCN_EINVAL, "bad argument");
    if (M->split_next != 0) return fail(OCN_ESTATE, "a split step is in progress (ocn_step_part): finish its parts first");
    ON_DEVICE(M->d.device);
    if (M->nvtx) nvtxRangePushA("ocn_time_step");
    const ocn_status s = M->prec == 32 ? run_steps<float>(M, n) : run_steps<double>(M, n);
    if (M->nvtx) nvtxRangePop();
    return s;
}

// ---- the step in parts, and rows of the arrays a neighbouring band needs (latitude bands) ----
extern "C++" {
namespace {
int step_parts(const ocn_model* M) { return (M->prec == 32 ? bt_launches<float>(M) : bt_launches<double>(M)) + 2; }

// the arrays of a row group: base pointer (plane layout), bytes per element, planes
struct RowArray { char* base; size_t es; int planes; };
template <class T>
int row_arrays(ocn_model* M, int group, RowArray* out) {
    ocn::DevP<T>& P = params<T>(M);
    const int nz = M->g->nz;
    int n = 0;
    auto add = [&](void* b, size_t es, int planes) { out[n++] = RowArray{(char*)b, es, planes}; };
    switch (group) {
        case OCN_ROWS_STATE:
            add(P.uv, 2 * sizeof(T), nz); add(P.ts, 2 * sizeof(T), nz); add(P.p, sizeof(double), nz);
            add(P.eta[0], sizeof(T), 1); add(P.U[0], sizeof(T), 1); add(P.V[0], sizeof(T), 1);
            break;
        case OCN_ROWS_STATE_2D: add(P.eta[0], sizeof(T), 1); add(P.U[0], sizeof(T), 1); add(P.V[0], sizeof(T), 1); break;
        case OCN_ROWS_FORCING: add(P.GU, sizeof(T), 1); add(P.GV, sizeof(T), 1); break;
        case OCN_ROWS_BAROTROPIC_0: case OCN_ROWS_BAROTROPIC_1: {
            const int b = group - OCN_ROWS_BAROTROPIC_0;
            add(P.eta[b], sizeof(T), 1); add(P.U[b], sizeof(T), 1); add(P.V[b], sizeof(T), 1);
            break;
        }
        default: return -1;
    }
    return n;
}
int row_arrays_any(ocn_model* M, int group, RowArray* out) {
    return M->prec == 32 ? row_arrays<float>(M, group, out) : row_arrays<double>(M, group, out);
}
// Rows j_begin .. j_begin + nrows - 1 of every plane of the group's arrays <-> one contiguous device buffer, array after
// array, plane after plane.  A chunk is nrows * sx elements from 4 elements before (row j_begin, i = 0): the rows with
// their x-halo images (the padding between rows rides along).
ocn_status move_rows(ocn_model* M, int group, int j_begin, int nrows, char* buf, bool pack) {
    RowArray arr[8];
    const int na = row_arrays_any(M, group, arr);
    if (na < 0) return fail(OCN_EINVAL, "unknown row group");
    const ocn_grid* g = M->g;
    if (nrows < 0 || j_begin < 0 || j_begin + nrows > g->ny) return fail(OCN_EINVAL, "rows outside the grid");
    if (nrows == 0) return OCN_OK;
    const size_t chunk = (size_t)nrows * g->sx, sz = (size_t)g->sx * g->sy;
    const long long off = (long long)(j_begin + OCN_HALO) * g->sx - 4;
    if (((uintptr_t)buf & 15u) != 0) return fail(OCN_EINVAL, "the row buffer must be 16-byte aligned");
    ocn::RowMoves R{};
    unsigned wmax = 0;
    int pmax = 1;
    for (int a = 0; a < na; ++a) {
        char* dev = arr[a].base + off * (long long)arr[a].es;
        const size_t w = chunk * arr[a].es;                 // bytes of one plane's chunk: a multiple of 128
        ocn::RowMoves::One& A = R.a[a];
        A.planes = arr[a].planes;
        if (pack) { A.src = (const uint4*)dev; A.dst = (uint4*)buf; A.src_pitch = (long long)(sz * arr[a].es / 16); A.dst_pitch = (long long)(w / 16); }
        else { A.src = (const uint4*)buf; A.dst = (uint4*)dev; A.src_pitch = (long long)(w / 16); A.dst_pitch = (long long)(sz * arr[a].es / 16); }
        R.w[a] = (unsigned)(w / 16);
        wmax = std::max(wmax, R.w[a]);
        pmax = std::max(pmax, arr[a].planes);
        buf += w * arr[a].planes;
    }
    ocn::k_move_rows<<<dim3((wmax + 255) / 256, std::min(pmax, 32), na), 256, 0, M->stream>>>(R);
    CK(cudaGetLastError());
    return OCN_OK;
}
}  // namespace
}  // extern "C++"

ocn_status ocn_step_parts(const ocn_model* M, int* parts) {
    if (!M || !parts) return fail(OCN_EINVAL, "null argument");
    *parts = step_parts(M);
    return OCN_OK;
}

ocn_status ocn_step_part(ocn_model* M, int part) {
    if (!M) return fail(OCN_EINVAL, "null model");
    const int np = step_parts(M);
    if (part < 0 || part >= np) return fail(OCN_EINVAL, "no such part of a step");
    if (part != M->split_next) return fail(OCN_ESTATE, "parts of a step run in order, 0 .. ocn_step_parts - 1 (next expected: " + std::to_string(M->split_next) + ")");
    ON_DEVICE(M->d.device);
    if (part == 0) M->split_euler = !M->have_history;
    if (M->nvtx) nvtxRangePushA(part == 0 ? "ocn_step_part tendency" : part == np - 1 ? "ocn_step_part backsub_correct" : "ocn_step_part barotropic");
    const ocn_status s = M->prec == 32 ? launch_step<float>(M, M->split_euler, part) : launch_step<double>(M, M->split_euler, part);
    if (M->nvtx) nvtxRangePop();
    if (s != OCN_OK) return s;
    if (part == np - 1) { M->have_history = true; M->split_next = 0; }
    else M->split_next = part + 1;
    return OCN_OK;
}

// ---- checkpoint / resume and the finite check ----
extern "C++" {
namespace {
struct CkptHeader {
    char magic[8];
    int nx, ny, nz, precision, sx, sy, have_history, reserved;
    unsigned long long payload;
};
struct CkptArray { char* base; size_t bytes; };
// everything a step reads that an earlier step or the caller wrote: state, pressure, AB2 history, the barotropic state a
// step starts from, and the forcing fields; each as its whole plane-layout allocation (halo images included)
template <class T>
int ckpt_arrays(ocn_model* M, CkptArray* out) {
    ocn::DevP<T>& P = params<T>(M);
    const size_t n3 = (size_t)P.sz * P.nz, n2 = (size_t)P.sz;
    int n = 0;
    auto add = [&](void* p, size_t es, size_t cnt) { out[n++] = CkptArray{(char*)p - LEAD * es, (cnt + 2 * LEAD) * es}; };
    add(P.uv, 2 * sizeof(T), n3); add(P.ts, 2 * sizeof(T), n3); add(P.p, sizeof(double), n3);
    add(P.Guv, 2 * sizeof(T), n3); add(P.Gts, 2 * sizeof(T), n3);
    add(P.eta[0], sizeof(T), n2); add(P.U[0], sizeof(T), n2); add(P.V[0], sizeof(T), n2);
    add(P.taux, sizeof(T), n2); add(P.tauy, sizeof(T), n2); add(P.qts, 2 * sizeof(T), n2); add(P.rts, 2 * sizeof(T), n2);
    return n;
}
int ckpt_arrays_any(ocn_model* M, CkptArray* out) { return M->prec == 32 ? ckpt_arrays<float>(M, out) : ckpt_arrays<double>(M, out); }
template <class T>
ocn_status count_nonfinite(ocn_model* M, unsigned long long* bad) {
    ocn::DevP<T>& P = params<T>(M);
    const unsigned long long n3 = (unsigned long long)P.sz * P.nz * 2, n2 = (unsigned long long)P.sz;
    unsigned long long* d = P.timeline + 63;               // a spare device word of the model (the timeline uses 8 x 7)
    CK(cudaMemsetAsync(d, 0, sizeof(*d), M->stream));
    ocn::k_count_nonfinite<T><<<592, 256, 0, M->stream>>>((const T*)P.uv, n3, d);
    ocn::k_count_nonfinite<T><<<592, 256, 0, M->stream>>>((const T*)P.ts, n3, d);
    ocn::k_count_nonfinite<T><<<64, 256, 0, M->stream>>>((const T*)P.eta[0], n2, d);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(bad, d, sizeof(*d), cudaMemcpyDeviceToHost, M->stream));
    CK(cudaStreamSynchronize(M->stream));
    return OCN_OK;
}
}  // namespace
}  // extern "C++"

ocn_status ocn_check_finite(ocn_model* M, unsigned long long* nonfinite) {
    if (!M || !nonfinite) return fail(OCN_EINVAL, "null argument");
    ON_DEVICE(M->d.device);
    return M->prec == 32 ? count_nonfinite<float>(M, nonfinite) : count_nonfinite<double>(M, nonfinite);
}

ocn_status ocn_checkpoint_bytes(const ocn_model* M, unsigned long long* bytes) {
    if (!M || !bytes) return fail(OCN_EINVAL, "null argument");
    CkptArray arr[16];
    const int n = ckpt_arrays_any(const_cast<ocn_model*>(M), arr);
    unsigned long long b = sizeof(CkptHeader);
    for (int a = 0; a < n; ++a) b += arr[a].bytes;
    *bytes = b;
    return OCN_OK;
}

ocn_status ocn_checkpoint_save(ocn_model* M, void* host) {
    if (!M || !host) return fail(OCN_EINVAL, "null argument");
    if (M->split_next != 0) return fail(OCN_ESTATE, "a split step is in progress");
    ON_DEVICE(M->d.device);
    CkptArray arr[16];
    const int n = ckpt_arrays_any(M, arr);
    CkptHeader h{};
    std::memcpy(h.magic, "OCNCKPT1", 8);
    h.nx = M->g->nx; h.ny = M->g->ny; h.nz = M->g->nz; h.precision = M->prec; h.sx = M->g->sx; h.sy = M->g->sy;
    h.have_history = M->have_history ? 1 : 0;
    char* dst = (char*)host + sizeof(h);
    for (int a = 0; a < n; ++a) {
        CK(cudaMemcpyAsync(dst, arr[a].base, arr[a].bytes, cudaMemcpyDeviceToHost, M->stream));
        dst += arr[a].bytes;
    }
    h.payload = (unsigned long long)(dst - (char*)host) - sizeof(h);
    CK(cudaStreamSynchronize(M->stream));
    std::memcpy(host, &h, sizeof(h));
    return OCN_OK;
}

ocn_status ocn_checkpoint_load(ocn_model* M, const void* host, unsigned long long bytes) {
    if (!M || !host) return fail(OCN_EINVAL, "null argument");
    CkptHeader h;
    if (bytes < sizeof(h)) return fail(OCN_EINVAL, "not a checkpoint (too short)");
    std::memcpy(&h, host, sizeof(h));
    if (std::memcmp(h.magic, "OCNCKPT1", 8) != 0) return fail(OCN_EINVAL, "not a checkpoint (bad magic)");
    if (h.nx != M->g->nx || h.ny != M->g->ny || h.nz != M->g->nz || h.precision != M->prec || h.sx != M->g->sx || h.sy != M->g->sy)
        return fail(OCN_EINVAL, "the checkpoint was written by a model of another size or precision");
    ON_DEVICE(M->d.device);
    CkptArray arr[16];
    const int n = ckpt_arrays_any(M, arr);
    unsigned long long need = 0;
    for (int a = 0; a < n; ++a) need += arr[a].bytes;
    if (h.payload != need || bytes != need + sizeof(h)) return fail(OCN_EINVAL, "checkpoint size mismatch");
    const char* src = (const char*)host + sizeof(h);
    for (int a = 0; a < n; ++a) {
        CK(cudaMemcpyAsync(arr[a].base, src, arr[a].bytes, cudaMemcpyHostToDevice, M->stream));
        src += arr[a].bytes;
    }
    CK(cudaStreamSynchronize(M->stream));
    M->have_history = h.have_history != 0;
    M->split_next = 0;
    return OCN_OK;
}

// ---- fused puts: the arrays of the new state as seen by a neighbouring band ----
extern "C++" {
namespace {
template <class T>
void peer_arrays(ocn_model* M, void** out) {
    ocn::DevP<T>& P = params<T>(M);
    out[0] = P.uv; out[1] = P.ts; out[2] = P.p;
}
template <class T>
void peer_fill(ocn_model* M, int side, void* const* a, int lo, int rows, int dj, int peer_ny, long long peer_sz) {
    typedef typename ocn::Pair<T>::type T2;
    ocn::PeerPut<T>& Q = peer_put<T>(M);
    ocn::PeerSide<T>& S = Q.side[side];
    S.lo = lo; S.hi = lo + rows; S.dj = dj; S.ny = peer_ny; S.sz = peer_sz;
    S.uv = (T2*)a[0]; S.ts = (T2*)a[1]; S.p = (double*)a[2];
    if (side == 0) Q.own_lo = lo; else Q.own_hi = lo + rows;
}
}  // namespace
}  // extern "C++"

ocn_status ocn_peer_export(ocn_model* M, ocn_peer* out) {
    if (!M || !out) return fail(OCN_EINVAL, "null argument");
    ON_DEVICE(M->d.device);
    std::memset(out, 0, sizeof(*out));
    out->nx = M->g->nx; out->ny = M->g->ny; out->nz = M->g->nz; out->precision = M->prec; out->sx = M->g->sx; out->sy = M->g->sy;
    out->device = M->d.device;
    if (M->prec == 32) peer_arrays<float>(M, out->ptr); else peer_arrays<double>(M, out->ptr);
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "ipc handle size");
    for (int a = 0; a < OCN_PEER_ARRAYS; ++a) {
        if (M->ws) continue;                       // in the caller's workspace: reachable in this process only (no IPC handle)
        void* base = nullptr;                      // the allocation that holds the array (the largest base below it)
        for (void* b : M->allocs) if (b <= out->ptr[a] && (!base || b > base)) base = b;
        if (!base) return fail(OCN_ESTATE, "array without an allocation");
        cudaIpcMemHandle_t h;
        CK(cudaIpcGetMemHandle(&h, base));
        std::memcpy(out->ipc[a], &h, 64);
        out->ipc_offset[a] = (unsigned long long)((char*)out->ptr[a] - (char*)base);
    }
    return OCN_OK;
}

ocn_status ocn_peer_attach(ocn_model* M, int side, const ocn_peer* peer, int my_first_row, int peer_first_row, int rows, int same_process) {
    if (!M || !peer) return fail(OCN_EINVAL, "null argument");
    if (side != 0 && side != 1) return fail(OCN_EINVAL, "side must be 0 (south) or 1 (north)");
    if (peer->nx != M->g->nx || peer->nz != M->g->nz || peer->precision != M->prec || peer->sx != M->g->sx)
        return fail(OCN_EINVAL, "the neighbouring band must have the same nx, nz and precision");
    if (rows < 1 || my_first_row < 0 || my_first_row + rows > M->g->ny || peer_first_row < 0 || peer_first_row + rows > peer->ny)
        return fail(OCN_EINVAL, "rows outside a grid");
    if (M->split_next != 0) return fail(OCN_ESTATE, "a split step is in progress");
    ON_DEVICE(M->d.device);
    void* arr[OCN_PEER_ARRAYS];
    for (int a = 0; a < OCN_PEER_ARRAYS; ++a) {
        if (same_process) { arr[a] = peer->ptr[a]; continue; }
        cudaIpcMemHandle_t h;
        std::memcpy(&h, peer->ipc[a], 64);
        void* base = nullptr;
        CK(cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess));
        M->ipc_open.push_back(base);
        arr[a] = (char*)base + peer->ipc_offset[a];
    }
    const long long psz = (long long)peer->sx * peer->sy;
    if (M->prec == 32) peer_fill<float>(M, side, arr, my_first_row, rows, peer_first_row - my_first_row, peer->ny, psz);
    else peer_fill<double>(M, side, arr, my_first_row, rows, peer_first_row - my_first_row, peer->ny, psz);
    if (!M->put) {                                 // first attachment: the other side has no neighbour yet
        if (side == 0) { M->qf.own_hi = M->qd.own_hi = M->g->ny; M->qf.side[1].lo = M->qf.side[1].hi = M->qd.side[1].lo = M->qd.side[1].hi = 0; }
        else { M->qf.own_lo = M->qd.own_lo = 0; M->qf.side[0].lo = M->qf.side[0].hi = M->qd.side[0].lo = M->qd.side[0].hi = 0; }
    }
    M->put = true;
    if (M->graph) { cudaGraphExecDestroy(M->graph); M->graph = nullptr; }     // the captured step stored without puts
    return OCN_OK;
}

int ocn_band_overlap(int precision, int substeps) {
    if ((precision != 32 && precision != 64) || substeps < 1) return -1;
    return std::max(std::min(substeps, precision == 32 ? bt_substeps_per_launch<float>() : bt_substeps_per_launch<double>()), OCN_HALO) + 1;
}

ocn_status ocn_rows_bytes(const ocn_model* M, int group, int nrows, unsigned long long* bytes) {
    if (!M || !bytes) return fail(OCN_EINVAL, "null argument");
    RowArray arr[8];
    const int na = row_arrays_any(const_cast<ocn_model*>(M), group, arr);
    if (na < 0) return fail(OCN_EINVAL, "unknown row group");
    if (nrows < 0 || nrows > M->g->ny) return fail(OCN_EINVAL, "rows outside the grid");
    unsigned long long b = 0;
    for (int a = 0; a < na; ++a) b += (unsigned long long)nrows * M->g->sx * arr[a].es * arr[a].planes;
    *bytes = b;
    return OCN_OK;
}

ocn_status ocn_pack_rows(ocn_model* M, int group, int j_begin, int nrows, void* dst) {
    if (!M || !dst) return fail(OCN_EINVAL, "null argument");
    ON_DEVICE(M->d.device);
    return move_rows(M, group, j_begin, nrows, (char*)dst, true);
}

ocn_status ocn_unpack_rows(ocn_model* M, int group, int j_begin, int nrows, const void* src) {
    if (!M || !src) return fail(OCN_EINVAL, "null argument");
    ON_DEVICE(M->d.device);
    return move_rows(M, group, j_begin, nrows, (char*)const_cast<void*>(src), false);
}

ocn_status ocn_get_fields(ocn_model* M, ocn_fields* f) {
    if (!M || !f) return fail(OCN_EINVAL, "null argument");
    ON_DEVICE(M->d.device);
    return M->prec == 32 ? get_fields_t<float>(M, f, nullptr) : get_fields_t<double>(M, f, nullptr);
}

ocn_status ocn_get_fields_async(ocn_model* M, ocn_fields* f, unsigned long long* ticket) {
    if (!M || !f || !ticket) return fail(OCN_EINVAL, "null argument");
    ON_DEVICE(M->d.device);
    return M->prec == 32 ? get_fields_t<float>(M, f, ticket) : get_fields_t<double>(M, f, ticket);
}

ocn_status ocn_wait(ocn_model* M, unsigned long long ticket) {
    if (!M) return fail(OCN_EINVAL, "null model");
    if (ticket >= M->tickets) return fail(OCN_EINVAL, "ticket was never issued");
    ON_DEVICE(M->d.device);
    // a ticket whose event slot has been reused is older than NTICKET later read-backs on the same in-order stream: wait for
    // the oldest event still held, which was recorded after it
    const unsigned long long held = M->tickets > ocn_model::NTICKET ? M->tickets - ocn_model::NTICKET : 0;
    CK(cudaEventSynchronize(M->ticket_ev[(ticket < held ? held : ticket) % ocn_model::NTICKET]));
    CK(cudaGetLastError());
    return OCN_OK;
}

ocn_status ocn_synchronize(ocn_model* M) {
    if (!M) return fail(OCN_EINVAL, "null model");
    ON_DEVICE(M->d.device);
    CK(cudaStreamSynchronize(M->stream));
    CK(cudaStreamSynchronize(M->copy_stream));
    return OCN_OK;
}

ocn_status ocn_model_info(const ocn_model* M, int* launches, unsigned long long* bytes) {
    if (!M) return fail(OCN_EINVAL, "null model");
    if (launches) *launches = M->launches_per_step;
    if (bytes) *bytes = M->bytes;
    return OCN_OK;
}

ocn_status ocn_profile_enable(ocn_model* M, int on) {
    if (!M) return fail(OCN_EINVAL, "null model");
    ON_DEVICE(M->d.device);
    if (!on) { const ocn_status s = prof_flush(M); if (s != OCN_OK) return s; }
    M->profiling = on != 0;
    return OCN_OK;
}

ocn_status ocn_profile_read(ocn_model* M, double* ms, long long* launches, int reset) {
    if (!M) return fail(OCN_EINVAL, "null model");
    ON_DEVICE(M->d.device);
    const ocn_status s = prof_flush(M);
    if (s != OCN_OK) return s;
    for (int q = 0; q < OCN_NSTAGES; ++q) {
        if (ms) ms[q] = M->prof_ms[q];
        if (launches) launches[q] = M->prof_launches[q];
        if (reset) { M->prof_ms[q] = 0; M->prof_launches[q] = 0; }
    }
    return OCN_OK;
}

ocn_status ocn_tune(ocn_model* M, const char* key, double value) {
    if (!M || !key) return fail(OCN_EINVAL, "null argument");
    ON_DEVICE(M->d.device);
    if (std::string(key) == "nvtx") { M->nvtx = value != 0; return OCN_OK; }
    if (std::string(key) == "k1_geo_threshold") {
        if (!(value >= 0 && value <= 1e6)) return fail(OCN_EINVAL, "k1_geo_threshold out of range");
        M->pf.geo_thr = (int)value; M->pd.geo_thr = (int)value;
    } else {
        return fail(OCN_EINVAL, std::string("unknown tuning key: ") + key);
    }
    if (M->graph) { CK(cudaStreamSynchronize(M->stream)); cudaGraphExecDestroy(M->graph); M->graph = nullptr; }   // re-capture with the new arguments
    return OCN_OK;
}

ocn_status ocn_selftest_division(int device, unsigned long long n, unsigned long long seed, unsigned long long* mismatches) {
    if (!mismatches) return fail(OCN_EINVAL, "null argument");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return fail(OCN_ECUDA, "no such CUDA device");
    ON_DEVICE(device);
    unsigned long long* d = nullptr;
    CK(cudaMalloc(&d, 8));
    CK(cudaMemset(d, 0, 8));
    ocn::k_selftest_division<<<148 * 8, 256>>>(n, seed, d);
    CK(cudaGetLastError());
    CK(cudaMemcpy(mismatches, d, 8, cudaMemcpyDeviceToHost));
    CK(cudaFree(d));
    return OCN_OK;
}

ocn_status ocn_get_timeline(ocn_model* M, double* cycles, int reset) {
    if (!M || !cycles) return fail(OCN_EINVAL, "null argument");
#ifndef OCN_K1_TIMELINE
    (void)reset;
    return fail(OCN_EUNSUPPORTED, "libocn was built without -DOCN_K1_TIMELINE");
#else
    ON_DEVICE(M->d.device);
    unsigned long long* d = M->prec == 32 ? M->pf.timeline : M->pd.timeline;
    unsigned long long h[64];
    CK(cudaStreamSynchronize(M->stream));
    CK(cudaMemcpy(h, d, sizeof(h), cudaMemcpyDeviceToHost));
    if (reset) CK(cudaMemset(d, 0, sizeof(h)));
    for (int q = 0; q < 64; ++q) cycles[q] = (double)h[q];
    return OCN_OK;
#endif
}

const char* ocn_stage_name(int stage) {
    static const char* names[OCN_NSTAGES] = {"tendency", "barotropic", "backsub_correct_pressure", "vertical_mixing"};
    return (stage >= 0 && stage < OCN_NSTAGES) ? names[stage] : "";
}

ocn_status ocn_get_debug(ocn_model* M, double* Gu, double* Gv, double* GT, double* GS, double* U, double* V) {
    if (!M) return fail(OCN_EINVAL, "null model");
    ON_DEVICE(M->d.device);
    return M->prec == 32 ? get_debug_t<float>(M, Gu, Gv, GT, GS, U, V) : get_debug_t<double>(M, Gu, Gv, GT, GS, U, V);
}

ocn_status ocn_get_mixing(ocn_model* M, double* nu, double* kappa) {
    if (!M) return fail(OCN_EINVAL, "null model");
    if (M->d.closure != 1) return fail(OCN_ESTATE, "model was created with closure = 0");
    ON_DEVICE(M->d.device);
    return M->prec == 32 ? get_mixing_t<float>(M, nu, kappa) : get_mixing_t<double>(M, nu, kappa);
}

ocn_status ocn_get_mixing_noalloc(ocn_model* M, double* nu, double* kappa) {
    if (!M) return fail(OCN_EINVAL, "null model");
    if (M->d.closure != 1) return fail(OCN_ESTATE, "model was created with closure = 0");
    ON_DEVICE(M->d.device);
    return M->prec == 32 ? get_mixing_noalloc_t<float>(M, nu, kappa) : get_mixing_noalloc_t<double>(M, nu, kappa);
}

unsigned long long ocn_noalloc_scratch_bytes(void) { return (unsigned long long)OCN_NOALLOC_SCRATCH_BYTES; }

}  // extern "C"
