/* dgswem_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, independent CPU oracle (fp64; -DORC_F32: fp32) of the DG-SWEM hot path
 * (arxiv 2508.21208; PAPER.md).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may use it.  It shares no
 * code with paper_2508_21208_b200/ (the CUDA path) and neither includes the other.
 *
 * What is pinned by tests (-m "not gpu"): basis/mass/quadrature tables, geometry,
 * LLF flux, RHS (constant state, lake at rest, rotation, brute force on tiny
 * meshes), conservation, SSP-RK order, seiche period/convergence, limiter and
 * wet/dry properties, det_exp/det_log, Holland closed-form values.
 * PARITY UNPINNED (paper gives no algorithm): the CHOICE
 * of limiter (c.2), of wet/dry redistribution (c.3), of friction law and of the
 * Holland/Garratt constants -- only their self-consistency properties are pinned.
 */
#ifndef DGSWEM_ORACLE_H
#define DGSWEM_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Working precision: binary64 (default; the BASELINE metric) or, built with -DORC_F32, binary32 (the paper's own runs use
 * single precision, PAPER.md:158 "-r4", :529).  Same source, same expression trees: every literal is written RL(x) and
 * every operation has operands of type `real`, so the f32 build performs one IEEE binary32 operation where the f64
 * build performs one binary64 operation.  Time, time step, tidal parameters and the storm track stay binary64. */
#ifdef ORC_F32
typedef float real;
#else
typedef double real;
#endif
#define RL(x) ((real)(x))

#define ORC_MAXDOF 10
#define ORC_MAXQA 12
#define ORC_MAXQE 4

typedef struct {
  int32_t p;          /* 1, 2 or 3 */
  int32_t rk_order;   /* 2: SSP(2,2), 3: SSP(3,3) */
  real g, cf, coriolis_f, h0_dry;
  int32_t limiter;    /* 0 off, 1 edge-neighbour Barth-Jespersen [R-7], 2 vertex-neighbourhood Barth-Jespersen [R-18] */
  int32_t wetdry;
  int32_t flux;       /* 0 local Lax-Friedrichs [R-3], 1 Roe [R-17] */
  int32_t rk_stages;  /* 0: = rk_order (SSP(2,2) / SSP(3,3)); many-stage schemes [R-19]: (order 2: 3 or 4 stages), (order 3: 4 stages) */
} orc_params;

typedef struct { double x0, y0, vx, vy, rmax, dp, B, rho_air, rho_water, f; } orc_holland;   /* binary64 in every build */

/* element-independent tables (Table 4: PHI_AREA, PHI_EDGE, SRFAC, EDGEFAC) */
typedef struct {
  int32_t p, ndof, nqe, nqa;
  real ge[ORC_MAXQE], we[ORC_MAXQE];            /* Gauss-Legendre on [-1,1], weights sum 2 */
  real elam[ORC_MAXQE][2];                      /* (lambda_a, lambda_b) of edge point j */
  real la[ORC_MAXQA][3], wa[ORC_MAXQA];         /* area points (barycentric), weights sum 2 */
  real invM[ORC_MAXDOF];                        /* 1/M_k, M_k reference mass */
  real phiA[ORC_MAXQA][ORC_MAXDOF];             /* PHI_AREA[k,i] */
  real dphiA1[ORC_MAXQA][ORC_MAXDOF];           /* d phi_k / d xi_1 at area point i */
  real dphiA2[ORC_MAXQA][ORC_MAXDOF];
  real phiE[3][ORC_MAXQE][ORC_MAXDOF];          /* PHI_EDGE: local edge l, point j */
  real wfac[ORC_MAXQA][ORC_MAXDOF];             /* wa[i]*invM[k] */
  real srfac[ORC_MAXQA][ORC_MAXDOF];            /* wfac*phiA  (SRFAC without geometry) */
  real efac[3][ORC_MAXQE][ORC_MAXDOF];          /* (we[j]*invM[k])*phiE  (EDGEFAC) */
  real phiV[3][ORC_MAXDOF];                     /* basis at the three vertices */
} orc_tables;

typedef struct orc_model orc_model;

/* ---- pieces exposed for the pins ---- */
void   orc_basis(real lam0, real lam1, real lam2, real* phi /*[6]*/, real* d1 /*[6]*/, real* d2 /*[6]*/);
int    orc_make_tables(int p, orc_tables* T);
void   orc_llf_flux(real g, real h0, real nx, real ny, real hq,
                    real zp, real qxp, real qyp, real zm, real qxm, real qym,
                    int bc, real zeta_b, real* fz, real* fqx, real* fqy);
void   orc_roe_flux(real g, real h0, real nx, real ny, real hq,
                    real zp, real qxp, real qyp, real zm, real qxm, real qym,
                    int bc, real zeta_b, real* fz, real* fqx, real* fqy);
real orc_det_exp(real x);
real orc_det_log(real x);
void   orc_holland_node(const orc_holland* h, double cx, double cy, real x, real y, real* tsx, real* tsy, real* V);
/* ... with the surface-pressure anomaly as a water column, eta_p = (p - p_n)/(rho_0 g) (etap may be NULL) */
void   orc_holland_node_p(const orc_holland* h, real g, double cx, double cy, real x, real y,
                          real* tsx, real* tsy, real* V, real* etap);
/* limiter on one element, one variable; mean_nb[3] neighbour means, has_nb[3] flags */
real orc_limit_var(int p, real* w /*[ndof]*/, const real* mean_nb, const int* has_nb);
/* vertex-neighbourhood variant: vmin[3], vmax[3] = extrema of the means of all elements sharing vertex v */
real orc_limit_var_vertex(int p, real* w /*[ndof]*/, const real* vmin, const real* vmax);
/* wet/dry on one element: modes [ndof] of ze,qx,qy, vertex bathymetry hv[3]; returns wet flag */
int    orc_wetdry_elem(const orc_tables* T, real h0, const real* hv, real* ze, real* qx, real* qy);
/* generic SSP-RK step: w <- one step of size dt, with user RHS and post-stage hooks */
typedef void (*orc_rhs_fn)(void* ctx, int stage, double t_stage, const real* w, real* rhs);
typedef void (*orc_post_fn)(void* ctx, int stage, real* w);
int    orc_ssprk_step_s(int order, int stages, int64_t n, real* w, real* w0, real* rhs, double t, double dt,
                        orc_rhs_fn rhs_fn, orc_post_fn post_fn, void* ctx);
int    orc_ssprk_step(int order, int64_t n, real* w, real* w0, real* rhs, double t, double dt,
                      orc_rhs_fn rhs_fn, orc_post_fn post_fn, void* ctx);

/* ---- model ---- */
orc_model* orc_create(const orc_params* prm,
                      int64_t n_nodes, const real* xy, const real* bathy,
                      int64_t n_elem, const int32_t* tri,
                      int64_t n_edge, const int32_t* edge_elem, const int8_t* edge_local,
                      const int32_t* edge_bc, const int32_t* elem_edge);
void orc_destroy(orc_model*);
const orc_tables* orc_get_tables(const orc_model*);
void orc_set_state(orc_model*, double t, const real* ze, const real* qx, const real* qy);
/* test hooks: state + wet flags as given (no initial wet/dry pass); the post-stage sequence limiter -> wet/dry on the current state */
void orc_set_state_raw(orc_model*, double t, const real* ze, const real* qx, const real* qy, const uint8_t* wet);
void orc_apply_post(orc_model*, int do_limiter, int do_wetdry);
void orc_set_tide(orc_model*, double amp, double omega, double phase);
void orc_set_wind_holland(orc_model*, const orc_holland* /* NULL = off */);
void orc_set_wind_forcing(orc_model*, int stress_on, int press_on);   /* parts of the Holland forcing in use (default 1, 0) */
void orc_set_rain(orc_model*, real rate);                           /* uniform mass source R, m/s */
void orc_step(orc_model*, int64_t nsteps, double dt);
/* L_h(current state) at t (stage-1 time); scale arrays (may be NULL) receive the sum of
 * absolute values of all contributions to each entry (the error-norm denominator). */
void orc_eval_rhs(orc_model*, real* rze, real* rqx, real* rqy, real* sze, real* sqx, real* sqy);
void orc_get_flux(orc_model*, real* flux /*[3][nqe][n_edge]*/);   /* of the last RHS evaluation */
void orc_get_state(orc_model*, double* t, real* ze, real* qx, real* qy);
void orc_get_wetdry(orc_model*, uint8_t* wet);
void orc_get_nodal(orc_model*, real* zn, real* qxn, real* qyn);   /* [n_nodes] each: element-averaged nodal output */
void orc_get_geometry(orc_model*, real* area /*[n_elem]*/, real* jinv /*[4][n_elem]*/, real* lfac /*[3][n_elem]*/,
                      real* enx /*[n_edge]*/, real* eny /*[n_edge]*/);
void orc_get_wind(orc_model*, real* tau /*[2][n_nodes]*/);
void orc_get_pressure(orc_model*, real* etap /*[n_nodes]*/);
int  orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
