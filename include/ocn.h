/* ocn.h — C ABI of libocn: the B200-native (sm_100a) hydrostatic free-surface time step.
 *
 * One call of ocn_time_step(model, n) advances the hydrostatic Boussinesq equations on a
 * staggered C-grid (§5.2) by n baroclinic steps: fused WENO-upwind tendency
 * kernels, quasi-AB2 + backward-Euler vertical diffusion by a tridiagonal
 * solve, the split-explicit barotropic sub-cycle, the barotropic
 * correction and the column diagnostics.  Every step of that path runs in CUDA kernels of this
 * library; there is no CPU fallback.  The discrete equations are fixed in DESIGN.md §3.
 *
 * Conventions
 *   - Field buffers crossing the ABI are `precision`-bit floats (32 or 64), INTERIOR cells only,
 *     layout [k][j][i] with i (longitude / x) fastest and k = 0 the bottom layer.  u is stored on
 *     the west face of cell i, v on the south face of cell j, w on the bottom face of cell k
 *     (nz+1 levels).  eta, tau_x (at u points), tau_y (at v points) are [j][i].
 *   - Handles and all device memory are owned by the library.  I/O buffers are owned by the
 *     caller and never retained.  A grid must outlive the models created from it.
 *   - Every call returns ocn_status and never throws; ocn_last_error() gives the message of the
 *     last non-OK status on the calling thread.  Asynchronous CUDA faults surface at the next
 *     ocn_get_fields / ocn_synchronize.
 */
#ifndef OCN_H
#define OCN_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ocn_grid ocn_grid;
typedef struct ocn_model ocn_model;

typedef enum {
    OCN_OK = 0, OCN_EINVAL = 1, OCN_ENOMEM = 2, OCN_ECUDA = 3, OCN_ESTATE = 4, OCN_EUNSUPPORTED = 5
} ocn_status;

/* Horizontal grid.  PAPER.md:102-104 (§6): the realistic domains "span the entire longitudinal extent of the sphere and
 * cover the latitudinal range from 75 S to 75 N", periodic in longitude, with bathymetry; PAPER.md:84 (§5.2): finite volume
 * on a staggered C-grid.  Metrics of the curvilinear cells: DESIGN.md §3.1-3.2. */
typedef struct {
    int kind;                       /* 0 cartesian (f/beta-plane), 1 latitude-longitude */
    int nx, ny, nz;                 /* nx, ny >= 3; 2 <= nz <= 250 */
    int periodic_x, periodic_y;     /* non-periodic edges are solid walls (land halo) */
    double x0, dx;                  /* metres, or degrees longitude (uniform) */
    double y0, dy;                  /* metres, or degrees latitude  (uniform) */
    double radius, rotation_rate;   /* lat-lon: sphere radius [m], Omega [1/s] */
    double f0, beta;                /* cartesian: f = f0 + beta (y - y_mid) */
    /* Latitude bands: this grid is rows j_offset .. j_offset + ny - 1 of a grid of ny_global
     * rows that starts at y0 — its metrics are evaluated with the whole grid's row numbers, so they are bit-identical to
     * the whole grid's.  0, 0 = a grid of its own.  A band is bounded in y (periodic_y = 0). */
    int j_offset, ny_global;
} ocn_grid_desc;

/* ocn_grid_create — the grid and the immersed-boundary bathymetry of PAPER.md:102-104; builds the metrics and the compact
 * 2-D level-threshold masks the kernels read.
 * z_faces: HOST, nz+1 finite doubles, strictly increasing, z_faces[nz] = 0 (the resting surface).
 * bottom_depth: HOST, ny*nx doubles, metres >= 0, 0 = land.  Immersed boundary = full cells,
 * cell wet iff its centre lies above the bottom; columns with < 2 wet cells are land
 * (DESIGN.md §3.3).  Host-only: allocates nothing on the device.
 * Errors: OCN_EINVAL (null pointer, sizes, non-monotonic or non-finite z_faces, z_faces[nz] != 0, negative depth, a
 * latitude range that reaches a pole), OCN_EUNSUPPORTED (nz > 250), OCN_ENOMEM. */
ocn_status ocn_grid_create(const ocn_grid_desc* desc, const double* z_faces, const double* bottom_depth,
                           ocn_grid** out);
ocn_status ocn_grid_destroy(ocn_grid* grid);

/* Model parameters. */
typedef struct {
    int precision;                  /* 32 or 64: dtype of every field buffer crossing the ABI and
                                       of all device fields, tendencies and metrics (PAPER.md:26, 143:
                                       the paper runs and reports both FP32 and FP64) */
    double dt;                      /* baroclinic time step [s] */
    int substeps;                   /* barotropic sub-steps M per baroclinic step */
    double chi;                     /* quasi-AB2 offset (0.1) */
    double g, alpha, beta_s, T0, S0, rho0;      /* linear equation of state, reference density */
    double nu_h, kappa_h, nu_z, kappa_z;        /* constant viscosities / diffusivities [m^2/s] */
    const double* filter_weights;   /* HOST, `substeps` doubles a_1..a_M, or NULL = power-law
                                       default of DESIGN.md §3.9; copied at creation */
    int device;                     /* CUDA device ordinal */
    void* stream;                   /* cudaStream_t of the caller (e.g. torch's): all work of the model is enqueued on it.
                                       NULL = the library creates a PRIVATE non-blocking stream (it does not synchronise
                                       with the legacy default stream): device buffers passed with on_device = 1 must
                                       then be complete before the call (caller synchronises its producer) */
    /* Vertical mixing closure ("Richardson-number-based parameterization for vertical
     * mixing due to unresolved shear and convective turbulence"; its coefficient is the second stored
     * diagnostic of PAPER.md:78; formulas: DESIGN.md §3.12).  closure = 0: constant nu_z / kappa_z.
     * closure = 1: at every open vertical face of a tracer column
     *   nu = nu_z + ri_nu0 f^2 + conv,  kappa = kappa_z + ri_nu0 f^3 + conv,  f = 1 / (1 + ri_c Ri),
     *   Ri = max(N2, 0) / (S2 + ri_s2min),  conv = ri_kconv min(1, max(-N2, 0) / ri_n2c),
     * evaluated from state n inside the fused tendency kernel; ri_n2c, ri_s2min > 0, the others >= 0.  Costs three more
     * 3-D words per cell (the modified super-diagonals of the per-column solves). */
    int closure;
    double ri_nu0, ri_c, ri_kconv, ri_n2c, ri_s2min;
    /* Surface restoring of the top-cell tracers toward ocn_fields.restore_T / restore_S with piston velocities
     * gamma_T, gamma_S [m/s]; 0 = off. */
    double gamma_T, gamma_S;
    /* Bottom drag on the lowest open level of every u / v column:
     * G_u -= (drag_r + drag_cd |u|) u / dz with |u| the speed at the point; drag_r [m/s], drag_cd [-], >= 0, 0 = off. */
    double drag_r, drag_cd;
    /* Equation of state.  0 = linear (north_star).  1 = nonlinear:
     * b = g [alpha (1 - eos_gamma z) (T - T0) + eos_alpha2 / 2 (T - T0)^2 - beta_s (S - S0)], z <= 0 the cell-centre depth:
     * thermobaricity eos_gamma [1/m] and cabbeling eos_alpha2 [1/K^2]; both 0 reproduces eos = 0 bit for bit. */
    int eos;
    double eos_alpha2, eos_gamma;
    /* Nonlinear weights of the WENO reconstructions ("based on WENO reconstructions", the family of refs
     * PAPER.md:244-245): 0 = Jiang-Shu (north_star reading), 1 = WENO-Z. */
    int advection;
    /* Separate filter weights b_1..b_M for the barotropic TRANSPORTS: HOST, `substeps`
     * doubles that sum to 1, or NULL = the weights of eta (filter_weights).  eta-bar = sum a_m eta^m, U-bar = sum b_m U^m,
     * V-bar likewise; dtau is still set by the first moment of a.  Copied at creation. */
    const double* filter_weights_uv;
    /* Biharmonic horizontal dissipation: viscosity nu4_h and tracer diffusivity kappa4_h
     * [m^4/s], >= 0, 0 = off.  G -= coefficient x L(L(.)) with the masked C-grid Laplacians of the second-order terms.
     * Costs two pre-pass launches per step and four more 3-D pair arrays; the default path is unchanged. */
    double nu4_h, kappa4_h;
    /* Caller-supplied device memory ("optionally a caller-supplied torch workspace"): 256-byte aligned DEVICE
     * memory of at least ocn_model_workspace_bytes bytes on `device`, e.g. a torch tensor; the model lives in it (no cudaMalloc
     * at creation or while stepping) and the caller frees it after ocn_model_destroy.  NULL = the library allocates.  Not in it:
     * the output array of ocn_get_mixing (allocated by the library on first use).  A model in a workspace cannot be reached
     * from another process (ocn_peer_export leaves the IPC handles empty). */
    void* workspace;
    unsigned long long workspace_bytes;
} ocn_model_desc;

/* ocn_model_create — the model of PAPER.md:84 (§5.2: hydrostatic Boussinesq, IMEX quasi-AB2, backward-Euler vertical
 * diffusion) with the split-explicit free surface of PAPER.md:94-98 (§5.3) on `grid`.  Allocates all device state
 * (14 3-D arrays + 2-D arrays + tables) on `device`; the calling thread's current device is restored on return (as it is
 * by every call below).  Parameters must be finite; chi, g, the viscosities / diffusivities, gamma_*, drag_* >= 0; user
 * filter_weights must sum to 1 (1e-9) and have a positive first moment (dtau = dt / sum_m m a_m).
 * Errors: OCN_EINVAL, OCN_ENOMEM (device allocation), OCN_ECUDA (no device: there is no CPU fallback). */
ocn_status ocn_model_create(const ocn_grid* grid, const ocn_model_desc* desc, ocn_model** out);
ocn_status ocn_model_destroy(ocn_model* model);
/* Bytes of device memory a model of this grid and these parameters takes (all its arrays, tables and staging regions): the size
 * of ocn_model_desc.workspace, and what ocn_model_create will allocate itself otherwise (2 MiB page rounding of the arrays a
 * neighbouring band may map aside).  Host-only dry run of the construction; validates the parameters like ocn_model_create. */
ocn_status ocn_model_workspace_bytes(const ocn_grid* grid, const ocn_model_desc* desc, unsigned long long* bytes);

/* Field set.  NULL member = skip.  on_device = 0: HOST pointers; 1: DEVICE pointers on the
 * model's device (contiguous, same layout). */
typedef struct {
    void *u, *v, *T, *S;            /* nz*ny*nx */
    void *w;                        /* (nz+1)*ny*nx, get only */
    void *eta;                      /* ny*nx */
    void *tau_x, *tau_y;            /* ny*nx, N/m^2, set only */
    /* Surface tracer forcing ("forced by realistic surface momentum, heat, and salinity fluxes";
     * DESIGN.md §3.13), ny*nx, set only: kinematic fluxes into the ocean flux_T [K m/s], flux_S [psu m/s] and the
     * restoring targets restore_T [K], restore_S [psu].  Top-cell tendency: G += (flux + gamma (target - c)) / dz_top.
     * All four default to 0. */
    void *flux_T, *flux_S, *restore_T, *restore_S;
    int on_device;
} ocn_fields;

/* ocn_set_fields — initial / boundary data of the problem of PAPER.md:102-104 (state, and the "surface momentum, heat, and
 * salinity fluxes" that force it).  Copies fields in (masking closed faces / land), on the model's stream.  If any of u, v,
 * T, S, eta is given: re-derives U, V = sum(u dz), w, p and resets the AB2 history (the next step is an Euler step).
 * DEPARTURE from SURVEY.md §8(b)'s proposed contract ("resets AB2 history" on every call): a call that carries ONLY forcing
 * fields (tau_x, tau_y, flux_*, restore_*) keeps the state and the AB2 history, so that time-varying forcing can be re-sent
 * before each step without an Euler restart (reading 19); the oracle's ocn_ref_set_fields does the same.
 * Host buffers may be reused as soon as the call returns.  Errors: OCN_EINVAL (null, w given), OCN_ECUDA. */
ocn_status ocn_set_fields(ocn_model* model, const ocn_fields* fields);
/* ocn_time_step — n baroclinic steps of the algorithm of PAPER.md:84 (§5.2) and PAPER.md:94-98 (§5.3): fused tendency
 * kernel, quasi-AB2, implicit vertical diffusion, split-explicit barotropic sub-cycle with filter
 * weights, barotropic correction, diagnostics.  Enqueues on the stream; no host synchronisation.
 * Errors: OCN_EINVAL (n < 0), OCN_ECUDA (launch failure; asynchronous faults surface at the next synchronising call). */
ocn_status ocn_time_step(ocn_model* model, int n);
/* ocn_get_fields — the prognostic state (u, v, T, S, eta) and the diagnosed w.  Copies fields out (land /
 * closed faces = 0); returns after the copies have completed (host buffers are valid on return).
 * Errors: OCN_EINVAL, OCN_ECUDA (including asynchronous faults of earlier steps). */
ocn_status ocn_get_fields(ocn_model* model, ocn_fields* fields);
/* The same read-back left in flight: returns as soon as the gathers and copies are enqueued (they run on a copy stream of
 * the library beside later steps) and writes a ticket; the buffers are valid after ocn_wait(model, ticket) — or after any
 * later blocking ocn_get_fields / ocn_synchronize.  Lets a caller enqueue step n+1 while the result of step n travels
 * (one exchange per step, overlapped as the paper overlaps its communication). */
ocn_status ocn_get_fields_async(ocn_model* model, ocn_fields* fields, unsigned long long* ticket);
/* Blocks until the read-back named by `ticket` (and every earlier one) has landed.  OCN_EINVAL for a ticket never issued. */
ocn_status ocn_wait(ocn_model* model, unsigned long long ticket);
/* Blocks until everything enqueued by earlier calls (steps and copies) has completed. */
ocn_status ocn_synchronize(ocn_model* model);

/* Expanded 3-D integer masks for the bit-exact test (HOST buffers, NULL = skip): wet, order_x,
 * order_y, order_zeta_u, order_zeta_v: nz*ny*nx; order_z: (nz+1)*ny*nx.  Expanded on the host
 * from the same compact 2-D threshold maps the kernels read. */
ocn_status ocn_get_masks(const ocn_grid* grid, unsigned char* wet, unsigned char* order_x,
                         unsigned char* order_y, unsigned char* order_z,
                         unsigned char* order_zeta_u, unsigned char* order_zeta_v);

/* Number of kernel launches enqueued by one baroclinic step, and device bytes held by the model. */
ocn_status ocn_model_info(const ocn_model* model, int* launches_per_step, unsigned long long* device_bytes);

/* Per-stage device timing (used by bench.py for the roofline of the dominant kernel).
 * Stages: 0 = K1 fused tendency / AB2 / elimination, 1 = barotropic sub-cycle (all M sub-steps +
 * finish; the sub-cycle runs BT_HALO sub-steps per launch on shared-memory tiles), 2 = K3 back-substitution / correction / pressure,
 * 3 = unused since the vertical mixing closure is evaluated inside stage 0 (always 0 launches; kept so that the stage
 * indices are stable).  (w is recomputed on the fly inside
 * K1 and written out only when ocn_get_fields asks for it.)
 * While enabled, ocn_time_step launches the kernels of a step directly (no CUDA graph) and
 * records a CUDA event on the model's stream between stages.  ocn_profile_read synchronises
 * the stream and returns the milliseconds and kernel launches accumulated per stage since the
 * last reset (HOST arrays of OCN_NSTAGES entries; NULL = skip). */
#define OCN_NSTAGES 4
ocn_status ocn_profile_enable(ocn_model* model, int on);
ocn_status ocn_profile_read(ocn_model* model, double* ms, long long* launches, int reset);
const char* ocn_stage_name(int stage);

/* Knobs that do not change results (bit for bit).  "nvtx" (0 / 1): NVTX host ranges around ocn_time_step and the parts of
 * ocn_step_part for timeline tools (PAPER.md:116 profiles with Nsight Systems + NVTX ranges; header-only NVTX 3, a no-op
 * without a tool attached).  "k1_geo_threshold": number of wet cells of a 32 x 8 tile-level
 * from which on the tendency kernel marches the tile with geometric (thread = cell) instead of compacted ownership
 * (default K1_GEO_THR of kernels_tile.cuh; 0 = always geometric, > 256 = never).  OCN_EINVAL for an unknown key. */
ocn_status ocn_tune(ocn_model* model, const char* key, double value);

/* Diagnostic builds only (nvcc -DOCN_K1_TIMELINE; OCN_EUNSUPPORTED otherwise): SM cycles every warp of the tendency kernel
 * has spent per phase of its march since the last reset, summed over all CTAs.  cycles: HOST, 64 doubles = [8 warps][8]:
 * 0 prologue (history loads; includes the wait at the previous block barrier), 1 wait for the TMA planes, 2 phase 1
 * (zeta, K, D, w), 3 face fluxes, 4 part B, 5 barrier issue, 6 iterations executed, 7 unused. */
ocn_status ocn_get_timeline(ocn_model* model, double* cycles, int reset);

/* Self-test of the fp64 path's three-instruction division (reciprocal + Markstein correction, csrc/common.cuh) against the
 * correctly rounded __ddiv_rn on n pseudo-random operand pairs (a quarter of them within a few ulps of a power of two, an
 * eighth with the divisor 6): *mismatches must come back 0.  Runs on `device`, synchronous. */
ocn_status ocn_selftest_division(int device, unsigned long long n, unsigned long long seed, unsigned long long* mismatches);

/* Debug / parity hooks (HOST double buffers, NULL = skip): the AB2 history G^{n-1} of each
 * prognostic field (nz*ny*nx each) and the barotropic transports U, V (ny*nx). */
ocn_status ocn_get_debug(ocn_model* model, double* Gu, double* Gv, double* GT, double* GS,
                         double* U, double* V);

/* closure = 1 only (OCN_ESTATE otherwise): the mixing coefficients of the CURRENT state (K4 is run on it), HOST double
 * buffers nz*ny*nx, value at the bottom face of tracer cell (k, j, i), 0 on closed faces and at k = 0; NULL = skip. */
ocn_status ocn_get_mixing(ocn_model* model, double* nu, double* kappa);

/* The same diagnostic for callers that must not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): calls no cudaMalloc, cudaFree or allocating library routine.  ocn_get_mixing keeps the
 * halo'd (nu, kappa) pair array in a buffer it cudaMallocs on first use; here that scratch is a file-scope static device
 * array of ocn_noalloc_scratch_bytes() = 16 MiB, which every GPU that loads the library holds until the process exits.
 * Limit: (sx * sy * nz + 64) pairs of `precision`-bit values must fit, sx = roundup(nx + 8, 32), sy = ny + 6 (e.g. up to about
 * 360 x 150 x 25 in fp32); a larger model is rejected with OCN_EUNSUPPORTED and a message that names both sizes.
 * Results are identical to ocn_get_mixing.  The array is SHARED by every call and every model of the process and keeps the
 * last call's contents: each call first clears the part it uses, on the model's stream.  Calls that overlap on the GPU
 * (two models on different streams, or two host threads) race on it: serialise them. */
ocn_status ocn_get_mixing_noalloc(ocn_model* model, double* nu, double* kappa);
unsigned long long ocn_noalloc_scratch_bytes(void);

/* ---- Checkpoint / resume and the finite check ("a restart re-starts AB2 with an Euler step unless G- is added") ----
 * ocn_set_fields / ocn_get_fields move the prognostic state only, and a model restarted from them takes an Euler step.  A
 * checkpoint holds everything a step reads that an earlier step or the caller wrote — (u, v), (T, S), p, the quasi-AB2 history
 * G^- (DESIGN.md §3.8), the barotropic state (eta, U, V) and the forcing fields — as raw device words, so a model of
 * the same grid and parameters that loads it continues BIT FOR BIT where the saved one stood (tests/test_gpu_checkpoint.py).
 * ocn_checkpoint_bytes: size of the blob.  ocn_checkpoint_save: blob -> HOST buffer of that size (blocks until it is there).
 * ocn_checkpoint_load: HOST blob of `bytes` bytes -> model (blocks); the blob must come from a model of the same nx, ny, nz
 * and precision (OCN_EINVAL otherwise: bad magic, size, shape).  The format is the library version's own (not portable).
 * ocn_check_finite: number of NaN / infinite words in u, v, T, S, eta (0 = healthy); blocks.  Cheap enough to call every few
 * hundred steps (three small reductions). */
ocn_status ocn_checkpoint_bytes(const ocn_model* model, unsigned long long* bytes);
ocn_status ocn_checkpoint_save(ocn_model* model, void* host_buffer);
ocn_status ocn_checkpoint_load(ocn_model* model, const void* host_buffer, unsigned long long bytes);
ocn_status ocn_check_finite(ocn_model* model, unsigned long long* nonfinite);

/* ---- Latitude bands: the one exchange step of the path ----------------------------------
 * PAPER.md:98 (§5.3): the barotropic sub-cycle is stepped with a wide halo so that neighbours exchange once per group of
 * sub-steps instead of once per sub-step; one exchange of the 3-D halos per baroclinic step.  A band is an
 * ordinary model on rows j_offset - h .. of the whole grid (ocn_grid_desc.j_offset, ny_global) with h overlap rows on each
 * inner side; its own rows stay bit-identical to the whole-grid model as long as, after each part of a step, the overlap
 * rows are overwritten with the neighbour's rows of the group that part made stale (paper_2309_06662_b200/bands.py):
 *   part 0 (tendency pass)            -> OCN_ROWS_FORCING (G^U, G^V)
 *   part 1 + q (launch q of the sub-cycle, not the last) -> OCN_ROWS_BAROTROPIC_0 + ((q + 1) & 1) (eta, U, V of that buffer)
 *   last part (end of sub-cycle, back-substitution, correction) -> OCN_ROWS_STATE (u, v, T, S, p, eta, U, V)
 * h must cover what one part reaches: ocn_band_overlap(precision, substeps) rows.
 *
 * ocn_step_parts: number of parts of one baroclinic step (2 + launches of the sub-cycle).
 * ocn_step_part: enqueues part `part` of the next step on the model's stream; parts run in order 0 .. parts - 1 (OCN_ESTATE
 *   otherwise, and ocn_time_step returns OCN_ESTATE while a split step is in progress).  All parts of a step = ocn_time_step(1),
 *   bit for bit (same kernels, launched directly instead of through the captured graph).
 * ocn_rows_bytes: size of the packed rows of a group.  ocn_pack_rows / ocn_unpack_rows: rows j_begin .. j_begin + nrows - 1
 *   (with their x-halo images) of every array of the group -> / <- one contiguous DEVICE buffer of that size, enqueued on
 *   the model's stream (one copy kernel per call; no host synchronisation; nothing is allocated).  The 16-byte aligned buffer is the
 *   caller's (e.g. a torch tensor handed to NCCL send / recv); it must stay valid until the stream has passed the call.
 *   Packing from one model and unpacking into another of the same nx, nz and precision is the whole exchange.
 * Errors: OCN_EINVAL (null, rows outside the grid, unknown group), OCN_ESTATE, OCN_ECUDA. */
enum { OCN_ROWS_STATE = 0, OCN_ROWS_FORCING = 1, OCN_ROWS_BAROTROPIC_0 = 2, OCN_ROWS_BAROTROPIC_1 = 3,
       OCN_ROWS_STATE_2D = 4 /* eta, U, V only: what is left to exchange after the last part with fused puts */ };
ocn_status ocn_step_parts(const ocn_model* model, int* parts);
ocn_status ocn_step_part(ocn_model* model, int part);
ocn_status ocn_rows_bytes(const ocn_model* model, int group, int nrows, unsigned long long* bytes);
ocn_status ocn_pack_rows(ocn_model* model, int group, int j_begin, int nrows, void* dst_device);
ocn_status ocn_unpack_rows(ocn_model* model, int group, int j_begin, int nrows, const void* src_device);
/* Fused puts ("peer memory"): instead of packing, sending and unpacking the new 3-D state after the last part of a
 * step — 99 % of the exchanged bytes — the kernel that produces it (back-substitution + correction + pressure) stores the rows
 * a neighbouring band overlaps straight into the neighbour's arrays, and leaves the rows it overlaps itself to the neighbour:
 * compute and transfer in one kernel, stores over NVLink when the neighbour lives on another GPU.  Only (u, v), (T, S) and p
 * travel this way — no other part of a step touches them, so a put can only race with the tendency pass of the NEXT step; the
 * 2-D state (eta, U, V: scratch of the sub-cycle) still goes through OCN_ROWS_STATE_2D after the last part, and the arrival of
 * those rows is the signal that the neighbour's puts are complete (they were enqueued before the rows were packed).
 * ocn_peer_export: what a neighbour needs to reach this model's arrays (u,v), (T,S), p: their addresses (valid in this
 *   process) and CUDA IPC handles + offsets (for another process on the same node).  Plain data: send it as bytes.
 * ocn_peer_attach: from now on rows my_first_row .. + rows - 1 of this model's new state are also stored at rows
 *   peer_first_row .. of the neighbour on `side` (0 = south, 1 = north), and this model no longer stores ITS overlap rows on
 *   that side (everything south of my_first_row for side 0, north of my_first_row + rows for side 1: the neighbour's puts fill
 *   them).  same_process = 1 uses the addresses, 0 opens the IPC handles (peer access is enabled lazily by the driver).
 *   After attaching, the bands of a grid step in parts and exchange OCN_ROWS_STATE_2D instead of OCN_ROWS_STATE after the last
 *   part (bands.py).
 * Errors: OCN_EINVAL (null, side, mismatched nx / nz / precision, rows outside a grid), OCN_ESTATE (a split step in progress),
 * OCN_ECUDA (IPC). */
#define OCN_PEER_ARRAYS 3
typedef struct {
    int nx, ny, nz, precision, sx, sy, device;
    void* ptr[OCN_PEER_ARRAYS];                      /* (u,v), (T,S), p */
    unsigned char ipc[OCN_PEER_ARRAYS][64];          /* cudaIpcMemHandle_t of the allocation that holds each */
    unsigned long long ipc_offset[OCN_PEER_ARRAYS];  /* byte offset of the array in that allocation */
} ocn_peer;
ocn_status ocn_peer_export(ocn_model* model, ocn_peer* out);
ocn_status ocn_peer_attach(ocn_model* model, int side, const ocn_peer* peer, int my_first_row, int peer_first_row, int rows,
                           int same_process);
/* Overlap rows a band of a model of this precision (32 / 64) and sub-step count needs on each inner side: what ONE part
 * of a step reaches (every exchange resets the overlap rows, so the reaches do not add up) — the larger of the sub-steps
 * one launch of the sub-cycle advances (the error of the band's artificial wall travels one row per sub-step) and the 3
 * rows of the widest stencil of the tendency pass — + 1 for the staggering of the v faces.  -1 for bad arguments.  Host-only. */
int ocn_band_overlap(int precision, int substeps);

const char* ocn_last_error(void);
const char* ocn_version(void);

#ifdef __cplusplus
}
#endif
#endif
