/* dgswem.h -- C ABI of the B200-native DG-SWEM hot path (arxiv 2508.21208).
 *
 * The library evaluates, on ONE sm_100a GPU in fp64 (or, on request, fp32), the per-RK-stage discontinuous Galerkin
 * right-hand side of the 2-D shallow water equations on an unstructured triangular mesh
 * (eqs (1)-(5); kernels EDGE / GATHER / AREA = PAPER.md Alg. 2 / 3 / 1) and the
 * SSP Runge-Kutta stage update followed by slope limiting and wetting/drying.
 * Readings of everything the paper leaves open: DESIGN.md section 3.
 *
 * Conventions
 *   - every pointer argument is HOST memory owned by the caller; it is copied in or out during
 *     the call and never retained (only exception: the halo buffers of dgswem_halo_pack / _unpack when
 *     flagged buf_on_device).  All other device memory is owned by the handle.
 *   - element arrays are [ndof][n_elem] doubles, mode index slow, in the CALLER's element order
 *     (any internal reordering is invisible); ndof = (p+1)(p+2)/2; mode order 00,01,10,(02,11,20),(03,12,21,30).
 *   - triangles are counter-clockwise, 0-based; local edge l joins local vertices (l+1)%3 -> (l+2)%3.
 *   - return value 0 = success; <0 = error (DGSWEM_E_*), text via dgswem_last_error().
 *   - calls on one handle must not be concurrent.  Work is enqueued on the handle's stream;
 *     get_* calls synchronise it.
 *   - environment, read by dgswem_create (tuning / test knobs; every setting gives the same bits):
 *     DGSWEM_FUSED=0..3 form of the RK stage (see dgswem_stage_form), DGSWEM_GRAPH=0 plain stream launches instead of
 *     CUDA-graph replay in dgswem_step, DGSWEM_PERSISTENT_CTAS=n cap (0: off) on the persistent kernels' grids,
 *     DGSWEM_PF_DIST=n tiles ahead that the stage kernel pulls into L2 (0: off; default on for meshes larger than L2).
 */
#ifndef DGSWEM_H
#define DGSWEM_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DGSWEM_OK          0
#define DGSWEM_E_ARG      -1   /* bad argument (NULL, size, parameter range) */
#define DGSWEM_E_MESH     -2   /* inconsistent mesh tables (orientation, edge/element tables) */
#define DGSWEM_E_CUDA     -3   /* CUDA runtime error */
#define DGSWEM_E_NONFINITE -4  /* non-finite state found by dgswem_get_state */

typedef struct dgswem dgswem_t;   /* opaque */

typedef struct {
  int32_t p;            /* polynomial degree 1, 2 or 3 (paper runs p=1; p = 3 runs the edge + element
                           kernel pair only)                                                      */
  int32_t rk_order;     /* order of the SSP Runge-Kutta scheme, 2 or 3 (R-2); see rk_stages */
  double  g;            /* gravity, e.g. 9.81                                                    */
  double  cf;           /* quadratic bottom friction coefficient, 0 = off (R-6)        */
  double  coriolis_f;   /* Coriolis parameter, 0 = off                             */
  double  h0_dry;       /* dry tolerance H0 > 0; also the depth floor in denominators (R-6, R-8) */
  int32_t limiter;      /* slope limiter after every stage: 0 off, 1 edge-neighbour
                           Barth-Jespersen (R-7), 2 vertex-neighbourhood Barth-Jespersen (R-18)   */
  int32_t wetdry;       /* 0/1: wet/dry pass after every stage (R-8)               */
  int32_t reorder;      /* internal renumbering (invisible at this ABI; north_star (b)): 0 keep the caller's numbering,
                           1 Hilbert curve through the element centroids, 2 reverse Cuthill-McKee on the element graph */
  int32_t device;       /* CUDA device ordinal                                                   */
  int32_t flux;         /* numerical flux: 0 local Lax-Friedrichs (R-3), 1 Roe (R-17)      */
  int32_t precision;    /* working precision of state, tables and kernels: 64 (or 0; default, the BASELINE
                           metric) or 32 (the paper's own runs, PAPER.md:158 "-r4", :529).
                           Every pointer of this ABI stays binary64: values are rounded on the way in and are
                           exact on the way out; time, time step, tide and storm track stay binary64 inside */
  int32_t rk_stages;    /* 0: as many stages as rk_order (SSP(2,2), SSP(3,3)).  Many-stage SSP schemes (PAPER.md:109
                           "optimized ... SSPRK"; R-19), two-register Shu-Osher form: rk_order 2 with 3 or 4
                           stages (optimal SSP(s,2), SSP coefficient s-1), rk_order 3 with 4 stages (SSP(4,3), coefficient 2) */
} dgswem_params;

/* Holland (1980) vortex, R-9: centre (x0+vx t, y0+vy t), radius of max wind rmax [m],
 * pressure deficit dp [Pa], shape B, densities [kg/m3], Coriolis f used in the gradient wind. */
typedef struct { double x0, y0, vx, vy, rmax, dp, B, rho_air, rho_water, f; } dgswem_holland;

/* Optional device-memory hooks (the Python binding backs them with torch allocations) and the
 * CUDA stream (a cudaStream_t cast to void*; NULL = the library creates its own stream). */
typedef struct {
  void* (*alloc)(size_t bytes, void* user);   /* returns a device pointer, 256-byte aligned, or NULL */
  void  (*free)(void* ptr, void* user);
  void* user;
  void* stream;
} dgswem_devhooks;

/* Build a model.  xy[n_nodes][2], bathy[n_nodes] (positive down), tri[n_elem][3],
 * edge_elem[n_edge][2] = (e+, e-) with e- = -1 on a boundary edge, edge_local[n_edge][2] = local
 * edge number of e+ / of e- (-1), edge_bc[n_edge] = 0 interior, 1 land/wall, 2 ocean elevation,
 * elem_edge[n_elem][3] = global edge of local edge l  (the paper's NEDEL / LED / NIEDN tables,
 * PAPER.md:341-354).  The tables are validated (E_MESH).  hooks may be NULL. */
int dgswem_create(dgswem_t** out, const dgswem_params* prm, const dgswem_devhooks* hooks,
                  int64_t n_nodes, const double* xy, const double* bathy,
                  int64_t n_elem, const int32_t* tri,
                  int64_t n_edge, const int32_t* edge_elem, const int8_t* edge_local,
                  const int32_t* edge_bc, const int32_t* elem_edge);

/* Load the modal state at time t.  If wetdry is on, one wet/dry pass is applied (it initialises
 * the wet mask and may modify the state); otherwise every element is flagged wet. */
int dgswem_set_state(dgswem_t*, double t, const double* ze, const double* qx, const double* qy);

/* Ocean-boundary elevation zeta_b(t) = amp sin(omega t + phase) on edge_bc == 2 edges (R-4). */
int dgswem_set_tide(dgswem_t*, double amp, double omega, double phase);

/* Moving Holland vortex wind stress (R-9); NULL switches the wind off. */
int dgswem_set_wind_holland(dgswem_t*, const dgswem_holland*);

/* Which parts of the Holland forcing enter the momentum source while a vortex is set: the wind stress (R-9; default
 * on) and the surface-pressure gradient -(H/rho_0) grad p_a = -g H grad eta_p with the Holland pressure profile
 * p(r) = p_c + dp exp(-(R/r)^B) evaluated at the nodes by the WIND kernel ("Wind forcing and pressure
 * calculations"; R-15; default off). */
int dgswem_set_wind_forcing(dgswem_t*, int stress_on, int pressure_on);

/* Uniform mass source R in the continuity equation ("such as rain"; R-16), in m/s; 0 = off. */
int dgswem_set_rain(dgswem_t*, double rate);

/* Advance nsteps time steps of size dt: per step WIND at the nodes, then per
 * stage EDGE -> GATHER+AREA+RK update -> limiter -> wet/dry.  Asynchronous on the stream. */
int dgswem_step(dgswem_t*, int64_t nsteps, double dt);

/* ---- Stage-granular stepping and halo lists: building blocks of a domain-decomposed run (
 * PAPER.md:476-519 "Multiple GPUs").  A driver splits the mesh into partitions with one layer of edge-neighbour
 * ghost elements (whose outer edges it closes as land edges), creates one handle per partition and, for every step,
 * calls  begin_step;  for s in 0..n_stage-1: { stage_rhs(s); [limiter on: exchange what=1; stage_limit(s);]
 * exchange what=0 };  end_step  -- where "exchange" = halo_pack on the owner, transport, halo_unpack on the ghost side.
 * The ghost elements' own results are meaningless and are overwritten by every exchange; owned elements then get the
 * same bits as in an undivided run.  dgswem_step must not be called between begin_step and end_step.
 * With the vertex-neighbourhood limiter (limiter = 2) the ghost layer must hold every foreign element that shares a NODE
 * with an owned element (the limiter takes the extrema of the means around each vertex), not only the edge-neighbours.
 *   dgswem_set_halo: element ids (caller numbering of this handle) to pack (owned elements that are ghosts elsewhere)
 *   and to unpack (this handle's ghosts); copied.  what = 0: the stage buffer written last (3*ndof rows; the current
 *   state between steps), what = 1: the RK-updated means (3 rows).  buf: [rows][n_send] resp. [rows][n_recv] doubles,
 *   host memory (buf_on_device = 0, synchronous) or device memory (1, asynchronous on the handle's stream). */
int dgswem_begin_step(dgswem_t*, double dt);
int dgswem_stage_rhs(dgswem_t*, int s);
/* The same in two halves, so that the halo exchange can overlap the interior elements ("overlapping
 * computation and communication"): part = 1 evaluates the stage on the send-list elements only (after which
 * dgswem_halo_pack may be enqueued and the packed buffer sent), part = 2 on all the others; part = 0 is
 * dgswem_stage_rhs.  Same bits as the undivided call (every element's arithmetic is independent of the launch it runs
 * in).  Stage forms that cannot run on a subset (DGSWEM_FUSED = 0, 2, 3) do the whole stage in part 1 and nothing in
 * part 2. */
int dgswem_stage_rhs_part(dgswem_t*, int s, int part);
int dgswem_stage_limit(dgswem_t*, int s);
int dgswem_end_step(dgswem_t*);
/* Recording a stage-granular step into the CALLER's CUDA graph (a decomposed run: every partition's kernels and the
 * exchange between them in one graph per step).  Kernel arguments are frozen in
 * a graph, so while capture mode is on the per-stage scalars (tidal elevation, storm centre) are passed as references
 * into the handle's device table, row = a device step counter, and dgswem_end_step records the counter's increment
 * instead of advancing the handle's time: the caller brackets ONE begin_step ... end_step sequence (and its
 * halo_pack / halo_unpack calls with device buffers) with dgswem_capture_mode(1) ... (0) while its own stream capture
 * is active on streams that include this handle's.  Before replaying the graph n <= 4096 times the caller calls
 * dgswem_graph_steps(n, dt) -- dt as recorded --: it tabulates the scalars of the next n steps, uploads them on the
 * handle's stream, resets the counter and advances the handle's time by n dt.  Same bits as the unrecorded calls.
 * While capture mode is on, dgswem_step and every call that synchronises the handle's stream (set_state, eval_rhs, all
 * get_* calls, sync, profile_read, test_math, fp64_peak, halo_pack / halo_unpack with host buffers) return
 * DGSWEM_E_ARG: a synchronisation inside a stream capture would invalidate the capture. */
int dgswem_capture_mode(dgswem_t*, int on);
int dgswem_graph_steps(dgswem_t*, int64_t nsteps, double dt);
int dgswem_set_halo(dgswem_t*, int64_t n_send, const int32_t* send_ids, int64_t n_recv, const int32_t* recv_ids);
int dgswem_halo_pack(dgswem_t*, int what, double* buf, int buf_on_device);
int dgswem_halo_unpack(dgswem_t*, int what, const double* buf, int buf_on_device);

/* TEST HOOK: L_h(current state) (eq. (5)) at the current time, each [ndof][n_elem]. */
int dgswem_eval_rhs(dgswem_t*, double* rze, double* rqx, double* rqy);

/* TEST HOOK: per-edge numerical flux buffer [3][nq_e][n_edge] (caller's edge order; point j numbered along e+'s local
 * edge; Alg. 2 l.25).  Edge + element form: the buffer of the last RHS evaluation.  Element-centric form (no
 * buffer exists): EDGE is evaluated on the current state at the current time for this call.  Neither this call (in the
 * element-centric form) nor dgswem_eval_rhs may be used between dgswem_begin_step and dgswem_end_step (E_ARG). */
int dgswem_get_flux(dgswem_t*, double* flux);

/* Copy the modal state of PAPER.md:193-195 (ZE, QX, QY[k, e]) back, and the time if t != NULL; synchronises;
 * E_NONFINITE if any value is not finite (the arrays are still filled). */
int dgswem_get_state(dgswem_t*, double* t, double* ze, double* qx, double* qy);

/* Wet (1) / dry (0) flag per element after the last WETDRY pass (R-8), caller's order; synchronises. */
int dgswem_get_wetdry(dgswem_t*, uint8_t* wet);

/* Nodal output ("we convert the modal representation to a nodal representation by averaging the
 * neighboring elements of each node"): for every node the mean over its incident elements of the element's polynomial
 * evaluated at that node (summed in ascending caller element id); zn, qxn, qyn: [n_nodes] each, host.  Synchronises. */
int dgswem_get_nodal(dgswem_t*, double* zn, double* qxn, double* qyn);

/* ---- Nodal output without any allocation (csrc/dgswem_static.cu).
 * For callers that cannot allocate device memory at the moment they want nodal fields, and so can neither create a handle
 * nor let one grow: code running while a stream capture is open (cudaMalloc is forbidden there and breaks the capture),
 * a solver living inside an application whose memory pool already holds the whole GPU (cudaMalloc fails), a time loop
 * that must not stall (cudaMalloc / cudaFree synchronise the device).  Same result, bit for bit, as dgswem_get_nodal
 * on a binary64 handle holding the same mesh and state: per node the mean, over the elements touching it in ascending
 * element id, of the element's polynomial at that node; a node no element touches gets 0.
 *   ALL pointers are DEVICE memory on `device`, owned by the caller, in the caller's numbering: tri [n_elem][3] node ids
 *   (an entry outside [0, n_nodes) is left out of the averages -- it is not reported); ze, qx, qy [ndof][n_elem],
 *   ndof = (p+1)(p+2)/2, p = 1, 2 or 3; outputs zn, qxn, qyn [n_nodes].  stream: a cudaStream_t cast to void*
 *   (NULL = the default stream).  The call only enqueues kernels on that stream; it does not synchronise.
 *   Limits: n_elem <= DGSWEM_STATIC_MAX_ELEM and n_nodes <= DGSWEM_STATIC_MAX_NODES, else DGSWEM_E_ARG (nothing is
 *   launched).  The node -> element table is rebuilt on every call in one file-scope device array of
 *   DGSWEM_STATIC_SCRATCH_BYTES (20 MiB), which every GPU that loads this library holds until the process exits.
 *   The call uses no cudaMalloc, cudaFree or allocating library routine.
 *   The FIRST call on each device looks up that device's address of the array (cudaGetSymbolAddress); make that first
 *   call before starting any stream capture.  All calls share the one array: it keeps the previous call's contents (the
 *   parts that must start at zero are cleared by each call), and two calls whose kernels can overlap on the same GPU
 *   -- different streams or host threads without an ordering between them -- race on it and give wrong results.
 *   Errors: 0, DGSWEM_E_ARG or DGSWEM_E_CUDA; text from dgswem_nodal_static_error (per host thread, valid until that
 *   thread's next call). */
#define DGSWEM_STATIC_MAX_ELEM      524288      /* 2^19: BASELINE configs[1]'s mesh just fits */
#define DGSWEM_STATIC_MAX_NODES     524288
#define DGSWEM_STATIC_SCRATCH_BYTES 20971520    /* 2^21 sort keys of 8 bytes + 2 x 2^19 int32 */
int dgswem_nodal_static(int device, void* stream, int p, int64_t n_nodes, int64_t n_elem, const int32_t* tri,
                        const double* ze, const double* qx, const double* qy, double* zn, double* qxn, double* qyn);
const char* dgswem_nodal_static_error(void);

/* Nodal kinematic wind stress tau_s/rho_0 of the last WIND evaluation, [2][n_nodes] (test hook). */
int dgswem_get_wind(dgswem_t*, double* tau);

/* Nodal surface-pressure anomaly as a water column, eta_p = (p - p_n)/(rho_0 g), of the last WIND evaluation, [n_nodes] (test hook). */
int dgswem_get_pressure(dgswem_t*, double* etap);

/* TEST HOOK: the kernels' reciprocal and square-root routines next to the IEEE
 * operators, on n caller-supplied arguments x (host): out (host, [4][n]) = rcp_rn(x), sqrt_rn(x), 1.0/x, sqrt(x).
 * Arguments outside the routines' stated range give unspecified values in rows 0 and 1. */
int dgswem_test_math(dgswem_t*, int64_t n, const double* x, double* out);

/* MEASUREMENT HOOK: the device's double-precision FMA rate (second roof of the stage kernel: "builder
 * measures it with a DFMA microbenchmark"): 8 independent chains of dependent DFMAs per thread on 8 CTAs of 256 threads
 * per SM, best of 3 timed launches (CUDA events on the handle's stream); *dfma_per_s = thread-level DFMAs per second
 * (x 2 = flop/s).  Synchronises. */
int dgswem_fp64_peak(dgswem_t*, double* dfma_per_s);

/* Which form of the RK stage this handle runs (DGSWEM_FUSED=0..3 in the environment of dgswem_create overrides the
 * default): 0 = edge kernel + element kernel with the per-edge flux buffer (default for p = 2; the only form at p = 3),
 * 1 = element-centric stage kernel without it (default for p = 1), 2 = the same with a shared-memory edge tile (each
 * tile-interior flux evaluated once), 3 = the same with TMA-staged operands.  All give the same bits. */
int dgswem_stage_form(const dgswem_t*);

/* Working precision of the handle: 64 or 32 (dgswem_params.precision). */
int dgswem_precision(const dgswem_t*);

/* Number of kernels launched by this handle so far (for bench.py's gpu_launches). */
int64_t dgswem_launch_count(const dgswem_t*);

/* Per-kernel timing for bench.py's roofline: while enabled, every kernel launch of dgswem_step /
 * dgswem_eval_rhs is bracketed by CUDA events recorded on the handle's stream (at most 32768
 * launches are recorded between reads).  dgswem_profile_read synchronises, returns the summed
 * device time in milliseconds and the launch count per kernel kind
 * (0 WIND, 1 EDGE, 2 ELEMENT = GATHER+AREA+RK(+wet/dry), 3 LIMITER+WETDRY; arrays of 4) and clears the records. */
int dgswem_profile(dgswem_t*, int enable);
int dgswem_profile_read(dgswem_t*, double* ms, int64_t* count);

/* Block until all enqueued work is done (the paper's `!$acc wait`). */
int dgswem_sync(dgswem_t*);

const char* dgswem_last_error(const dgswem_t*);   /* valid until the next call on the handle; NULL handle: creation error */
/* Release the handle and every device buffer it owns (the library owns all device memory); NULL is a no-op. */
void dgswem_destroy(dgswem_t*);

#ifdef __cplusplus
}
#endif
#endif
