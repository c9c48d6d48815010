// dgswem.cu -- the C ABI of include/dgswem.h.  The implementation (handle, validation, element-independent tables,
// geometry, Hilbert renumbering, device layout, per-step launch sequence: dgswem_impl.inl) and the kernels
// (dgswem_kernels.cuh) are compiled twice, in binary64 (namespaces imp64 / dgk64; the default, the BASELINE metric) and in
// binary32 (imp32 / dgk32, the paper's own precision).  dgswem_params.precision
// picks one at dgswem_create; every other entry point dispatches on the handle.  The ABI itself is binary64 in both.
// No torch types here; device memory comes from the hooks (or cudaMalloc), work goes to one stream.
#include "dgswem.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <numeric>
#include <string>
#include <vector>

#include <cuda_runtime.h>

// what both precisions' handles share (the opaque dgswem_t of the ABI)
struct dgswem {
  int precision = 64;
  std::string err;
  virtual ~dgswem() {}
};

namespace {
thread_local std::string g_create_error;
}

#define DGK_NS dgk64
#define DGK_REAL double
#define DGK_F32 0
#define DGK_IMPL_NS imp64
#include "dgswem_kernels.cuh"
#include "dgswem_impl.inl"
#undef DGK_NS
#undef DGK_REAL
#undef DGK_F32
#undef DGK_IMPL_NS

#define DGK_NS dgk32
#define DGK_REAL float
#define DGK_F32 1
#define DGK_IMPL_NS imp32
#include "dgswem_kernels.cuh"
#include "dgswem_impl.inl"
#undef DGK_NS
#undef DGK_REAL
#undef DGK_F32
#undef DGK_IMPL_NS

// call the implementation of the handle's precision
#define DISPATCH(h, fn, ...) \
  ((h)->precision == 32 ? imp32::fn(static_cast<imp32::Handle*>(h), ##__VA_ARGS__) : imp64::fn(static_cast<imp64::Handle*>(h), ##__VA_ARGS__))
#define DISPATCH_C(h, fn, ...)                                                           \
  ((h)->precision == 32 ? imp32::fn(static_cast<const imp32::Handle*>(h), ##__VA_ARGS__) \
                        : imp64::fn(static_cast<const imp64::Handle*>(h), ##__VA_ARGS__))

extern "C" {

const char* dgswem_last_error(const dgswem_t* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int dgswem_create(dgswem_t** out, const dgswem_params* prm, const dgswem_devhooks* hooks, int64_t n_nodes, const double* xy,
                  const double* bathy, int64_t n_elem, const int32_t* tri, int64_t n_edge, const int32_t* edge_elem,
                  const int8_t* edge_local, const int32_t* edge_bc, const int32_t* elem_edge) {
  if (!out) { g_create_error = "out is NULL"; return DGSWEM_E_ARG; }
  *out = nullptr;
  if (prm && prm->precision != 0 && prm->precision != 64 && prm->precision != 32) {
    g_create_error = "precision must be 64 (or 0) or 32";
    return DGSWEM_E_ARG;
  }
  if (prm && prm->precision == 32)
    return imp32::api_create(out, prm, hooks, n_nodes, xy, bathy, n_elem, tri, n_edge, edge_elem, edge_local, edge_bc, elem_edge);
  return imp64::api_create(out, prm, hooks, n_nodes, xy, bathy, n_elem, tri, n_edge, edge_elem, edge_local, edge_bc, elem_edge);
}

void dgswem_destroy(dgswem_t* h) { if (h) DISPATCH(h, api_destroy); }

int dgswem_end_step(dgswem_t* h) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_end_step); }
int dgswem_capture_mode(dgswem_t* h, int on) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_capture_mode, on); }
int dgswem_graph_steps(dgswem_t* h, int64_t nsteps, double dt) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_graph_steps, nsteps, dt); }
int dgswem_sync(dgswem_t* h) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_sync); }
int dgswem_set_state(dgswem_t* h, double t, const double* ze, const double* qx, const double* qy) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_set_state, t, ze, qx, qy); }
int dgswem_set_tide(dgswem_t* h, double amp, double omega, double phase) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_set_tide, amp, omega, phase); }
int dgswem_set_wind_holland(dgswem_t* h, const dgswem_holland* hol) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_set_wind_holland, hol); }
int dgswem_set_wind_forcing(dgswem_t* h, int stress_on, int pressure_on) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_set_wind_forcing, stress_on, pressure_on); }
int dgswem_set_rain(dgswem_t* h, double rate) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_set_rain, rate); }
int dgswem_step(dgswem_t* h, int64_t nsteps, double dt) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_step, nsteps, dt); }
int dgswem_begin_step(dgswem_t* h, double dt) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_begin_step, dt); }
int dgswem_stage_rhs(dgswem_t* h, int s) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_stage_rhs, s, 0); }
int dgswem_stage_rhs_part(dgswem_t* h, int s, int part) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_stage_rhs, s, part); }
int dgswem_stage_limit(dgswem_t* h, int s) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_stage_limit, s); }
int dgswem_set_halo(dgswem_t* h, int64_t n_send, const int32_t* send_ids, int64_t n_recv, const int32_t* recv_ids) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_set_halo, n_send, send_ids, n_recv, recv_ids); }
int dgswem_halo_pack(dgswem_t* h, int what, double* buf, int buf_on_device) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_halo_pack, what, buf, buf_on_device); }
int dgswem_halo_unpack(dgswem_t* h, int what, const double* buf, int buf_on_device) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_halo_unpack, what, buf, buf_on_device); }
int dgswem_eval_rhs(dgswem_t* h, double* rze, double* rqx, double* rqy) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_eval_rhs, rze, rqx, rqy); }
int dgswem_get_flux(dgswem_t* h, double* flux) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_get_flux, flux); }
int dgswem_get_state(dgswem_t* h, double* t, double* ze, double* qx, double* qy) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_get_state, t, ze, qx, qy); }
int dgswem_get_wetdry(dgswem_t* h, uint8_t* wet) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_get_wetdry, wet); }
int dgswem_get_nodal(dgswem_t* h, double* zn, double* qxn, double* qyn) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_get_nodal, zn, qxn, qyn); }
int dgswem_get_wind(dgswem_t* h, double* tau) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_get_wind, tau); }
int dgswem_get_pressure(dgswem_t* h, double* etap) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_get_pressure, etap); }
int dgswem_test_math(dgswem_t* h, int64_t n, const double* x, double* out) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_test_math, n, x, out); }
int dgswem_fp64_peak(dgswem_t* h, double* dfma_per_s) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_fp64_peak, dfma_per_s); }
int dgswem_stage_form(const dgswem_t* h) { return h ? DISPATCH_C(h, api_stage_form) : 0; }
int dgswem_precision(const dgswem_t* h) { return h ? h->precision : 0; }
int64_t dgswem_launch_count(const dgswem_t* h) { return h ? DISPATCH_C(h, api_launch_count) : 0; }
int dgswem_profile(dgswem_t* h, int enable) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_profile, enable); }
int dgswem_profile_read(dgswem_t* h, double* ms, int64_t* count) { if (!h) return DGSWEM_E_ARG; return DISPATCH(h, api_profile_read, ms, count); }

}  // extern "C"
