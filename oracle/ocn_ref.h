/* ocn_ref.h — C ABI of the CPU ORACLE for the hydrostatic free-surface time step.
 *
 * TEST INFRASTRUCTURE ONLY.  This is the plain, slow, serial (optionally OpenMP-over-rows,
 * bit-identical) fp64 restatement of the discrete equations in DESIGN.md §3, written from
 * the paper's problem statement (PAPER.md:84 hydrostatic Boussinesq / finite volume / C-grid
 * / IMEX AB2 / backward-Euler tridiagonal; PAPER.md:86 WENO advection
 * split-explicit barotropic sub-cycling; PAPER.md:102-104 lat-lon domain with bathymetry;
 * PAPER.md:78, 114 Ri-based vertical mixing).  Parity unpinned: nothing
 * (pins: tests/test_oracle_*.py, listed in DESIGN.md §5).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load it.  It shares no code, header, table or helper with the CUDA library (libocn).
 *
 * All buffers are HOST pointers, fp64, interior only, layout [k][j][i] (i = longitude fastest,
 * k = 0 is the bottom layer).  u is stored on the west face of cell i, v on the south face
 * of cell j, w on the bottom face of cell k (nz+1 levels).
 */
#ifndef OCN_REF_H
#define OCN_REF_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ocn_ref_grid ocn_ref_grid;
typedef struct ocn_ref_model ocn_ref_model;

typedef struct {
    int kind;                 /* 0 cartesian (f/beta-plane), 1 latitude-longitude */
    int nx, ny, nz;
    int periodic_x, periodic_y;
    double x0, dx;            /* metres, or degrees longitude */
    double y0, dy;            /* metres, or degrees latitude  */
    double radius, rotation_rate;   /* lat-lon */
    double f0, beta;                /* cartesian */
} ocn_ref_grid_desc;

typedef struct {
    double dt;
    int substeps;
    double chi;
    double g, alpha, beta_s, T0, S0, rho0;
    double nu_h, kappa_h, nu_z, kappa_z;
    const double* filter_weights;   /* host, `substeps` entries, or NULL = DESIGN.md §3.9 default */
    /* vertical mixing closure: 0 = constant nu_z / kappa_z,
     * 1 = Richardson-number based with convective adjustment, nu_z / kappa_z as background */
    int closure;
    double ri_nu0, ri_c, ri_kconv, ri_n2c, ri_s2min;
    /* surface restoring piston velocities [m/s] of T and S (0 = off) */
    double gamma_T, gamma_S;
    /* bottom drag on the lowest open u / v level: linear coefficient [m/s], quadratic [-]; 0 = off */
    double drag_r, drag_cd;
    /* equation of state: 0 = linear, 1 = b = g [alpha (1 - eos_gamma z) (T - T0) + eos_alpha2 / 2 (T - T0)^2
     * - beta_s (S - S0)] (thermobaricity eos_gamma [1/m], cabbeling eos_alpha2 [1/K^2]) */
    int eos;
    double eos_alpha2, eos_gamma;
    /* nonlinear WENO weights: 0 = Jiang-Shu, 1 = WENO-Z */
    int advection;
    /* separate filter weights b_m (m = 1..M) for the barotropic transports U, V; NULL = the weights of eta */
    const double* filter_weights_uv;
    /* biharmonic horizontal dissipation: viscosity nu4_h and diffusivity kappa4_h [m^4/s], 0 = off */
    double nu4_h, kappa4_h;
} ocn_ref_model_desc;

typedef struct {
    double *u, *v, *T, *S;    /* nz*ny*nx */
    double *w;                /* (nz+1)*ny*nx, get only */
    double *eta;              /* ny*nx */
    double *tau_x, *tau_y;    /* ny*nx, N/m^2, set only */
    /* surface tracer forcing ("surface momentum, heat, and salinity fluxes"), ny*nx, set only:
     * kinematic fluxes into the ocean [K m/s], [psu m/s] and restoring targets [K], [psu] */
    double *flux_T, *flux_S, *restore_T, *restore_S;
} ocn_ref_fields;

/* 0 = ok, non-zero = error (message via ocn_ref_last_error) */
int ocn_ref_grid_create(const ocn_ref_grid_desc*, const double* z_faces, const double* bottom_depth,
                        ocn_ref_grid** out);
int ocn_ref_grid_destroy(ocn_ref_grid*);
int ocn_ref_model_create(const ocn_ref_grid*, const ocn_ref_model_desc*, ocn_ref_model** out);
int ocn_ref_model_destroy(ocn_ref_model*);
/* copies in; if any of u, v, T, S, eta is given: masks, re-derives U, V, w, p and resets the AB2 history (the next
 * step is an Euler step); a forcing-only call (tau, flux, restore) keeps state and history */
int ocn_ref_set_fields(ocn_ref_model*, const ocn_ref_fields*);
int ocn_ref_time_step(ocn_ref_model*, int n);
int ocn_ref_get_fields(ocn_ref_model*, ocn_ref_fields*);
const char* ocn_ref_last_error(void);

/* expanded 3-D byte masks / order codes, each nz*ny*nx (order_z: (nz+1)*ny*nx); NULL = skip.
 * order_x/order_y: tracer face order 0..3 at the west/south face; order_z at the bottom face;
 * order_zeta_u / order_zeta_v: vorticity reconstruction order at u / v points (0 on closed faces). */
int ocn_ref_get_masks(const ocn_ref_grid*, unsigned char* wet, unsigned char* order_x,
                      unsigned char* order_y, unsigned char* order_z,
                      unsigned char* order_zeta_u, unsigned char* order_zeta_v);
/* metrics per row j = 0..ny-1: dxC, dxF, AzC, AzF, fF (each ny), dy (1 value) */
int ocn_ref_get_metrics(const ocn_ref_grid*, double* dxC, double* dxF, double* AzC, double* AzF,
                        double* fF, double* dy);

/* ---- pieces exposed for the pin tests (tests/test_oracle_*.py) ---- */
/* WENO face value at the interface between c[2] and c[3] of the six cells c[0..5]
 * (= cells n-3..n+2), order 1..3, upwinded by the sign of vel. */
double ocn_ref_weno(const double c[6], int order, double vel);
/* the same with the weight family chosen: scheme 0 = Jiang-Shu, 1 = WENO-Z */
double ocn_ref_weno_scheme(const double c[6], int order, double vel, int scheme);
/* backward-Euler vertical diffusion of one column, in place (DESIGN.md §3.8 step 4).
 * open[k], k = 0..nz: 1 if the face below cell k is open (open[0], open[nz] ignored = closed). */
int ocn_ref_implicit_column(int nz, const double* z_faces, const unsigned char* open,
                            double dt_kappa, double* phi);
/* the same solve with a diffusivity per face: dt_kappa[k], k = 0..nz, is dt * kappa at the face
 * below cell k (entries of closed faces are ignored) — DESIGN.md §3.12. */
int ocn_ref_implicit_column_var(int nz, const double* z_faces, const unsigned char* open,
                                const double* dt_kappa, double* phi);
/* Ri-based closure of the CURRENT state: viscosity nu and diffusivity kappa at
 * the bottom face of tracer cell (k, j, i), each nz*ny*nx (level 0 and closed faces hold 0);
 * error if the model was created with closure = 0.  NULL = skip. */
int ocn_ref_get_mixing(ocn_ref_model*, double* nu, double* kappa);
/* default filter weights a_m (m = 1..M) and dtau/dt */
int ocn_ref_filter_weights(int M, double* a, double* dtau_over_dt);
/* tendencies G^n of the CURRENT state (recomputed, no side effects); each nz*ny*nx or NULL */
int ocn_ref_get_tendencies(ocn_ref_model*, double* Gu, double* Gv, double* GT, double* GS);
/* stored diagnostics of the current state: p (nz*ny*nx), U, V (ny*nx); NULL = skip */
int ocn_ref_get_diagnostics(ocn_ref_model*, double* p, double* U, double* V);
/* the intermediates of the momentum tendency of the CURRENT state: relative vorticity zeta at the
 * south-west corner of cell (k, j, i), kinetic energy K and horizontal divergence D at its centre; nz*ny*nx each, NULL = skip */
int ocn_ref_get_momentum_diagnostics(ocn_ref_model*, double* zeta, double* K, double* D);
/* m raw barotropic sub-steps of (eta, U, V) with time step dtau and forcing G^U = G^V = 0,
 * no averaging (for the gravity-wave closed form); 3-D state untouched. */
int ocn_ref_barotropic_raw(ocn_ref_model*, int m, double dtau);
/* number of OpenMP threads the oracle will use (1 if built without OpenMP) */
int ocn_ref_num_threads(void);
void ocn_ref_set_num_threads(int n);

#ifdef __cplusplus
}
#endif
#endif
