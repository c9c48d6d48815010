// dgswem_impl.inl -- host side of the C ABI (include/dgswem.h) in the working precision `real` of the enclosing
// inclusion (dgswem.cu includes this file once per precision, after dgswem_kernels.cuh): handle, validation,
// element-independent tables, geometry, Hilbert renumbering, device layout and the per-step launch sequence.
// Everything the ABI passes is binary64; tables and geometry are computed here in `real` from the caller's values
// rounded once (same expression trees as the specification in that precision); time, time step,
// tidal parameters and the storm track stay binary64.
namespace DGK_IMPL_NS {

using namespace DGK_NS;

namespace {

constexpr real kG_edge1 = RL(0.57735026918962576);   // 1/sqrt(3)
constexpr real kG_edge2 = RL(0.77459666924148338);   // sqrt(3/5)

inline long long round_up(long long n, long long m) { return (n + m - 1) / m * m; }

// ------------------------------------------------------------------------------------ tables
// Dubiner basis (eq. (4)), mode order 00,01,10, 02,11,20, 03,12,21,30, from barycentrics:
// phi_ij = A_i B_j^(2i+1)(xi_2), A_i = P_i(eta_1) s^i in the collapsed coordinate (A_1 = a = xi_1 + (1 + xi_2)/2,
// A_2 = (3 a^2 - s^2)/2, A_3 = (5 a^3 - 3 a s^2)/2, s = (1 - xi_2)/2), B_j^(alpha) = Jacobi P_j^(alpha,0).
void dubiner(real l1, real l2, real* phi, real* g1, real* g2) {
  const real xi1 = RL(2.0) * l1 - RL(1.0);
  const real xi2 = RL(2.0) * l2 - RL(1.0);
  const real s = RL(0.5) * (RL(1.0) - xi2);
  const real r = RL(0.5) * (RL(5.0) * xi2 + RL(3.0));
  phi[0] = RL(1.0);
  phi[1] = RL(0.5) * (RL(3.0) * xi2 + RL(1.0));
  phi[2] = xi1 + RL(0.5) * (RL(1.0) + xi2);
  phi[3] = RL(0.5) * (((RL(5.0) * xi2) * xi2 + RL(2.0) * xi2) - RL(1.0));
  phi[4] = phi[2] * r;
  phi[5] = RL(0.5) * ((RL(3.0) * phi[2]) * phi[2] - s * s);
  g1[0] = RL(0.0);           g2[0] = RL(0.0);
  g1[1] = RL(0.0);           g2[1] = RL(1.5);
  g1[2] = RL(1.0);           g2[2] = RL(0.5);
  g1[3] = RL(0.0);           g2[3] = RL(5.0) * xi2 + RL(1.0);
  g1[4] = r;             g2[4] = RL(0.5) * r + RL(2.5) * phi[2];
  g1[5] = RL(3.0) * phi[2];  g2[5] = RL(0.5) * (RL(3.0) * phi[2] + s);
  {   // p = 3
    const real y = xi2, a = phi[2];
    const real b3 = RL(0.125) * ((((RL(35.0) * y) * y) * y + (RL(15.0) * y) * y) - RL(15.0) * y - RL(3.0));
    const real db3 = RL(0.125) * (((RL(105.0) * y) * y + RL(30.0) * y) - RL(15.0));
    const real b2 = RL(0.25) * (((RL(21.0) * y) * y + RL(18.0) * y) + RL(1.0));
    const real db2 = RL(0.25) * (RL(42.0) * y + RL(18.0));
    const real b1 = RL(0.5) * (RL(7.0) * y + RL(5.0));
    const real a2 = phi[5];
    const real da2x = g1[5], da2y = g2[5];
    const real a3 = RL(0.5) * (((RL(5.0) * a) * a) * a - ((RL(3.0) * a) * s) * s);
    const real da3x = RL(0.5) * ((RL(15.0) * a) * a - (RL(3.0) * s) * s);
    const real da3y = RL(0.5) * (((RL(7.5) * a) * a - (RL(1.5) * s) * s) + (RL(3.0) * a) * s);
    phi[6] = b3;       g1[6] = RL(0.0);    g2[6] = db3;
    phi[7] = a * b2;   g1[7] = b2;         g2[7] = RL(0.5) * b2 + a * db2;
    phi[8] = a2 * b1;  g1[8] = da2x * b1;  g2[8] = da2y * b1 + RL(3.5) * a2;
    phi[9] = a3;       g1[9] = da3x;       g2[9] = da3y;
  }
}

void make_tables(int p, Tables& T) {
  std::memset(&T, 0, sizeof(T));
  const int ndof = (p + 1) * (p + 2) / 2, nqe = p + 1, nqa = (p == 1) ? 3 : (p == 2) ? 6 : 12;
  real ge[4] = {0, 0, 0, 0}, we[4] = {0, 0, 0, 0}, wa[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
  if (p == 1) {
    ge[0] = -kG_edge1; ge[1] = kG_edge1; we[0] = RL(1.0); we[1] = RL(1.0);
    for (int i = 0; i < 3; ++i) {
      for (int v = 0; v < 3; ++v) T.la[i][v] = (v == i) ? RL(2.0) / RL(3.0) : RL(1.0) / RL(6.0);
      wa[i] = RL(2.0) / RL(3.0);
    }
  } else if (p == 3) {   // 4-point Gauss-Legendre; the classical 12-point degree-6 rule (two 3-point orbits, one 6-point orbit)
    ge[0] = -RL(0.86113631159405258); ge[1] = -RL(0.33998104358485626); ge[2] = RL(0.33998104358485626); ge[3] = RL(0.86113631159405258);
    we[0] = RL(0.34785484513745386); we[1] = RL(0.65214515486254614); we[2] = RL(0.65214515486254614); we[3] = RL(0.34785484513745386);
    const real a1 = RL(0.249286745170910), w1 = RL(0.116786275726379);
    const real a2 = RL(0.063089014491502), w2 = RL(0.050844906370207);
    const real b3 = RL(0.053145049844817), c3 = RL(0.310352451033784), w3 = RL(0.082851075618374);
    for (int i = 0; i < 3; ++i) {
      for (int v = 0; v < 3; ++v) {
        T.la[i][v] = (v == i) ? RL(1.0) - RL(2.0) * a1 : a1;
        T.la[3 + i][v] = (v == i) ? RL(1.0) - RL(2.0) * a2 : a2;
      }
      wa[i] = RL(2.0) * w1;
      wa[3 + i] = RL(2.0) * w2;
    }
    static const int perm[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
    const real tri3[3] = {b3, c3, (RL(1.0) - b3) - c3};
    for (int q = 0; q < 6; ++q) {
      for (int v = 0; v < 3; ++v) T.la[6 + q][v] = tri3[perm[q][v]];
      wa[6 + q] = RL(2.0) * w3;
    }
  } else {
    ge[0] = -kG_edge2; ge[1] = RL(0.0); ge[2] = kG_edge2;
    we[0] = RL(5.0) / RL(9.0); we[1] = RL(8.0) / RL(9.0); we[2] = RL(5.0) / RL(9.0);
    const real a1 = RL(0.445948490915965), w1 = RL(0.223381589678011);
    const real a2 = RL(0.091576213509771), w2 = RL(0.109951743655322);
    for (int i = 0; i < 3; ++i) {
      for (int v = 0; v < 3; ++v) {
        T.la[i][v] = (v == i) ? RL(1.0) - RL(2.0) * a1 : a1;
        T.la[3 + i][v] = (v == i) ? RL(1.0) - RL(2.0) * a2 : a2;
      }
      wa[i] = RL(2.0) * w1;
      wa[3 + i] = RL(2.0) * w2;
    }
  }
  const real mass[10] = {RL(2.0), RL(1.0), RL(1.0) / RL(3.0), RL(2.0) / RL(3.0), RL(2.0) / RL(9.0), RL(2.0) / RL(15.0),
                         RL(0.5), RL(1.0) / RL(6.0), RL(0.1), RL(1.0) / RL(14.0)};
  real invM[10];
  for (int k = 0; k < 10; ++k) invM[k] = RL(1.0) / mass[k];
  real phi[10], g1[10], g2[10];
  for (int i = 0; i < nqa; ++i) {
    dubiner(T.la[i][1], T.la[i][2], phi, g1, g2);
    for (int k = 0; k < ndof; ++k) {
      T.phiA[i][k] = phi[k]; T.dA1[i][k] = g1[k]; T.dA2[i][k] = g2[k];
      T.wfac[i][k] = wa[i] * invM[k];
      T.srfac[i][k] = T.wfac[i][k] * phi[k];
    }
  }
  for (int j = 0; j < nqe; ++j) {
    T.elam[j][0] = RL(0.5) * (RL(1.0) - ge[j]);
    T.elam[j][1] = RL(0.5) * (RL(1.0) + ge[j]);
  }
  for (int l = 0; l < 3; ++l) {
    const int va = (l + 1) % 3, vb = (l + 2) % 3;
    for (int j = 0; j < nqe; ++j) {
      real lam[3] = {RL(0.0), RL(0.0), RL(0.0)};
      lam[va] = T.elam[j][0]; lam[vb] = T.elam[j][1];
      dubiner(lam[1], lam[2], phi, g1, g2);
      for (int k = 0; k < ndof; ++k) {
        T.phiE[l][j][k] = phi[k];
        T.efac[l][j][k] = (we[j] * invM[k]) * phi[k];
      }
    }
  }
  for (int v = 0; v < 3; ++v) {
    real lam[3] = {RL(0.0), RL(0.0), RL(0.0)};
    lam[v] = RL(1.0);
    dubiner(lam[1], lam[2], phi, g1, g2);
    for (int k = 0; k < ndof; ++k) T.phiV[v][k] = phi[k];
  }
}

// ------------------------------------------------------------------------------------ Hilbert
// index of (x, y) in [0, 2^16)^2 along the Hilbert curve
inline uint32_t hilbert_d(uint32_t x, uint32_t y) {
  const uint32_t n = 1u << 16;
  uint32_t d = 0;
  for (uint32_t s = n >> 1; s > 0; s >>= 1) {
    const uint32_t rx = (x & s) ? 1u : 0u, ry = (y & s) ? 1u : 0u;
    d += s * s * ((3u * rx) ^ ry);
    if (ry == 0) {   // rotate / flip the quadrant
      if (rx == 1) { x = (n - 1u) - x; y = (n - 1u) - y; }
      const uint32_t t = x; x = y; y = t;
    }
  }
  return d;
}

std::vector<int> hilbert_order(const std::vector<double>& px, const std::vector<double>& py) {
  const size_t n = px.size();
  double x0 = 1e300, x1 = -1e300, y0 = 1e300, y1 = -1e300;
  for (size_t i = 0; i < n; ++i) {
    x0 = std::min(x0, px[i]); x1 = std::max(x1, px[i]);
    y0 = std::min(y0, py[i]); y1 = std::max(y1, py[i]);
  }
  const double span = std::max(std::max(x1 - x0, y1 - y0), 1e-300);
  std::vector<uint64_t> key(n);
  for (size_t i = 0; i < n; ++i) {
    const uint32_t ix = (uint32_t)std::min(65535.0, (px[i] - x0) / span * 65535.0);
    const uint32_t iy = (uint32_t)std::min(65535.0, (py[i] - y0) / span * 65535.0);
    key[i] = ((uint64_t)hilbert_d(ix, iy) << 32) | (uint64_t)i;
  }
  std::sort(key.begin(), key.end());
  std::vector<int> order(n);
  for (size_t i = 0; i < n; ++i) order[i] = (int)(key[i] & 0xffffffffu);
  return order;   // order[new] = old
}

// Reverse Cuthill-McKee on the element adjacency graph (two elements are adjacent when they share an edge): breadth-first
// levels from a low-degree start element, neighbours by ascending degree (ties by index), every component in turn,
// the whole order reversed.  The other renumbering north_star names; narrows the distance between edge neighbours.
std::vector<int> rcm_order(long long ne, long long nd, const int32_t* edge_elem) {
  std::vector<int> adj(3 * ne, -1), deg(ne, 0);
  for (long long d = 0; d < nd; ++d) {
    const int a = edge_elem[2 * d], b = edge_elem[2 * d + 1];
    if (b < 0) continue;
    adj[3 * (long long)a + deg[a]++] = b;
    adj[3 * (long long)b + deg[b]++] = a;
  }
  std::vector<int> order; order.reserve(ne);
  std::vector<char> seen(ne, 0);
  std::vector<int> starts(ne);
  std::iota(starts.begin(), starts.end(), 0);
  std::stable_sort(starts.begin(), starts.end(), [&](int x, int y) { return deg[x] < deg[y]; });
  for (int s0 : starts) {
    if (seen[s0]) continue;
    seen[s0] = 1;
    size_t head = order.size();
    order.push_back(s0);
    while (head < order.size()) {
      const int e = order[head++];
      int nb[3]; int k = 0;
      for (int l = 0; l < deg[e]; ++l) { const int q = adj[3 * (long long)e + l]; if (!seen[q]) { seen[q] = 1; nb[k++] = q; } }
      std::sort(nb, nb + k, [&](int x, int y) { return deg[x] != deg[y] ? deg[x] < deg[y] : x < y; });
      for (int i = 0; i < k; ++i) order.push_back(nb[i]);
    }
  }
  std::reverse(order.begin(), order.end());
  return order;   // order[new] = old
}

}  // namespace

// ------------------------------------------------------------------------------------ handle
struct RkScheme { int ns; real a[4], b[4]; double beta[4], c[4]; };   // see rk_get

struct Handle : ::dgswem {
  dgswem_params prm{};
  RkScheme rk{};
  int ndof = 0, nqe = 0, nqa = 0, nstage = 0;
  long long nn = 0, ne = 0, nd = 0, ld = 0, ldd = 0, ldn = 0;
  cudaStream_t stream = nullptr;
  bool own_stream = false;
  dgswem_devhooks hooks{};
  bool have_hooks = false;
  std::vector<void*> allocs;
  long long launches = 0;
  int res_edge[3] = {0, 0, 0};   // resident grid of the persistent edge kernel [p-1]
  int res_limwd = 0;          // same for the limiter kernel of this handle's p

  // optional per-kernel timing (dgswem_profile): CUDA events recorded on the stream around every launch
  struct ProfRec { int kind; cudaEvent_t a, b; };
  bool profiling = false;
  std::vector<ProfRec> prof;
  cudaEvent_t prof_start = nullptr;

  // device
  real* W[3] = {nullptr, nullptr, nullptr};
  real* nmm = nullptr;   // [6][ldn] node extrema of the means (vertex-neighbourhood limiter)
  real *flux = nullptr, *mean = nullptr, *jinv = nullptr, *lfac = nullptr, *hv = nullptr;
  real *en = nullptr, *ehb = nullptr, *tau = nullptr, *etap = nullptr, *nxy = nullptr;
  double* stage_buf = nullptr;   // binary64 staging in the caller's layout (set_state / get_* conversions)
  int2* edge_elem = nullptr;
  int *einfo = nullptr, *elem_edge = nullptr, *nbr = nullptr, *tri = nullptr, *nbinfo = nullptr;
  real* enl = nullptr;
  bool fused = false;         // element-centric stage kernel (k_stage) instead of k_edge + k_elem
  bool tiled = false;         // ... in its shared-memory edge-tile form (k_stage_tile): each tile evaluates its unique edges once
  bool staged = false;        // ... with TMA-staged operands (k_stage_stg)
  int pf_dist = 0;            // k_stage: L2 prefetch distance in tiles (DGSWEM_PF_DIST; 0 = off)
  int *nbs = nullptr, *stg_nb = nullptr;
  int2* stg_info = nullptr;
  int stg_cap1 = 0, res_stg[2] = {0, 0};
  int2* tile_info = nullptr;
  unsigned char* it_blob = nullptr;
  int *it_nb = nullptr, *eslot = nullptr;
  int tile_cap = 0, tile_cap1 = 0, res_tile[2] = {0, 0};   // resident grid of k_stage_tile without / with the wind block
  int *node_ptr = nullptr, *node_ev = nullptr;   // node -> (internal element * 4 + vertex), ascending caller element id
  int *perm_e = nullptr, *inv_e = nullptr, *inv_d = nullptr;   // perm_e[new]=old, inv_e[old]=new, inv_d[old]=new
  unsigned char *wet = nullptr, *wet_stage = nullptr;
  int* nf_flag = nullptr;
  size_t stage_bytes = 0;

  // CUDA-graph replay of whole time steps (dgswem_step): per-call scalar table + device step counter
  bool graphs_on = true;      // DGSWEM_GRAPH=0 switches to plain stream launches
  bool capturing = false;     // launch helpers pass table references instead of values
  double* scal_tab = nullptr; // [cap][kScalStride]
  double* scal_host = nullptr; // pinned staging copy of the table (so that dgswem_step stays asynchronous)
  cudaEvent_t scal_ev = nullptr;   // recorded after the table's upload: the staging copy may be rewritten after it
  long long scal_cap = 0;
  int* step_ctr = nullptr;
  struct StepGraph { cudaGraphExec_t exec = nullptr; int steps = 0; long long launches = 0; };
  StepGraph graph_many, graph_one;
  double graph_dt = 0.0; bool graph_wind = false; bool graph_tide = false;

  // stage-granular stepping and halo lists (dgswem_begin_step ... dgswem_halo_unpack)
  double step_dt = 0.0;        // dt of the step in progress (0: none)
  real* last_out = nullptr;  // stage buffer written by the last dgswem_stage_rhs (W[0] between steps)
  int *halo_send = nullptr, *halo_recv = nullptr;   // internal element ids
  int* send_uniq = nullptr;            // the send list without repeats (an element may go to several neighbours)
  unsigned char* send_mask = nullptr;  // [ld] 1 where the element is in the send list
  long long n_send_uniq = 0;
  long long n_send = 0, n_recv = 0;
  double* halo_buf = nullptr;  // device staging for host-side pack/unpack, [rows][max(n_send, n_recv)]

  double t = 0.0;
  double tide_amp = 0.0, tide_omega = 0.0, tide_phase = 0.0;
  bool wind_on = false;
  bool stress_on = true, press_on = false;   // parts of the Holland forcing in the momentum source (R-9, R-15)
  double rain = 0.0;                         // uniform mass source (R-16)
  dgswem_holland hol{};

  int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof(buf), fmt, ap); va_end(ap);
    err = buf;
    return code;
  }
  int cuda_fail(cudaError_t e, const char* what) { return fail(DGSWEM_E_CUDA, "%s: %s", what, cudaGetErrorString(e)); }

  void* dalloc(size_t bytes) {
    void* p = nullptr;
    if (bytes == 0) bytes = 256;
    if (have_hooks) {
      p = hooks.alloc(bytes, hooks.user);
    } else if (cudaMalloc(&p, bytes) != cudaSuccess) {
      p = nullptr;
    }
    if (p) allocs.push_back(p);
    return p;
  }
  void dfree(void* p) {   // give one allocation back before the handle dies (scratch, replaced halo lists)
    if (!p) return;
    auto it = std::find(allocs.begin(), allocs.end(), p);
    if (it == allocs.end()) return;
    allocs.erase(it);
    if (have_hooks) hooks.free(p, hooks.user); else cudaFree(p);
  }
  void release_all() {
    for (void* p : allocs) {
      if (have_hooks) hooks.free(p, hooks.user); else cudaFree(p);
    }
    allocs.clear();
  }
};

#define CK(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return h->cuda_fail(e__, #call); } while (0)
// entry points that synchronise the handle's stream: a synchronisation inside a stream capture invalidates the capture
#define NO_CAPTURE() do { if (h->capturing) return h->fail(DGSWEM_E_ARG, "capture mode is on and this call synchronises the stream, which would invalidate the capture (dgswem_capture_mode(0) first)"); } while (0)
#define CKL(name) do { cudaError_t e__ = cudaGetLastError(); if (e__ != cudaSuccess) return h->cuda_fail(e__, name); h->launches++; } while (0)

enum ProfKind { PK_WIND = 0, PK_EDGE = 1, PK_ELEM = 2, PK_LIMWD = 3, PK_COUNT = 4 };
constexpr size_t kMaxProfRecords = 1 << 15;
static inline void prof_begin(Handle* h, int kind) {
  if (!h->profiling || h->prof.size() >= kMaxProfRecords) return;
  Handle::ProfRec r; r.kind = kind; r.a = nullptr; r.b = nullptr;
  if (cudaEventCreate(&r.a) != cudaSuccess || cudaEventCreate(&r.b) != cudaSuccess) {
    if (r.a) cudaEventDestroy(r.a);
    (void)cudaGetLastError();   // a failed profiling event must not surface as the next launch's error
    return;
  }
  cudaEventRecord(r.a, h->stream);
  h->prof.push_back(r);
  h->prof_start = r.a;
}
static inline void prof_end(Handle* h) {
  if (!h->profiling || h->prof_start == nullptr) return;
  cudaEventRecord(h->prof.back().b, h->stream);
  h->prof_start = nullptr;
}

namespace {

template <typename T>
int upload(Handle* h, T*& dptr, const std::vector<T>& host) {
  dptr = (T*)h->dalloc(host.size() * sizeof(T));
  if (!dptr) return h->fail(DGSWEM_E_CUDA, "device allocation of %zu bytes failed", host.size() * sizeof(T));
  CK(cudaMemcpyAsync(dptr, host.data(), host.size() * sizeof(T), cudaMemcpyHostToDevice, h->stream));
  CK(cudaStreamSynchronize(h->stream));   // host vector may die after return
  return 0;
}

inline int grid_for(long long n, int block) { return (int)((n + block - 1) / block); }

int validate_mesh(Handle* h, long long nn, const double* xy, long long ne, const int32_t* tri, long long nd,
                  const int32_t* edge_elem, const int8_t* edge_local, const int32_t* edge_bc, const int32_t* elem_edge) {
  for (long long e = 0; e < ne; ++e) {
    for (int v = 0; v < 3; ++v)
      if (tri[3 * e + v] < 0 || tri[3 * e + v] >= nn) return h->fail(DGSWEM_E_MESH, "element %lld: node id out of range", e);
    const double* a = xy + 2 * (long long)tri[3 * e], *b = xy + 2 * (long long)tri[3 * e + 1], *c = xy + 2 * (long long)tri[3 * e + 2];
    const double A2 = (b[0] - a[0]) * (c[1] - a[1]) - (c[0] - a[0]) * (b[1] - a[1]);
    if (!(A2 > 0.0)) return h->fail(DGSWEM_E_MESH, "element %lld is not counter-clockwise (or degenerate)", e);
    for (int l = 0; l < 3; ++l) {
      const long long d = elem_edge[3 * e + l];
      if (d < 0 || d >= nd) return h->fail(DGSWEM_E_MESH, "elem_edge[%lld][%d] out of range", e, l);
      const bool plus = edge_elem[2 * d] == e && edge_local[2 * d] == l;
      const bool minus = edge_elem[2 * d + 1] == e && edge_local[2 * d + 1] == l;
      if (plus == minus) return h->fail(DGSWEM_E_MESH, "elem_edge[%lld][%d]=%lld does not point back to the element", e, l, d);
    }
  }
  for (long long d = 0; d < nd; ++d) {
    const long long ep = edge_elem[2 * d], em = edge_elem[2 * d + 1];
    const int lp = edge_local[2 * d], lm = edge_local[2 * d + 1];
    const int bc = edge_bc[d];
    if (ep < 0 || ep >= ne || lp < 0 || lp > 2) return h->fail(DGSWEM_E_MESH, "edge %lld: bad e+ / local edge", d);
    if (elem_edge[3 * ep + lp] != d) return h->fail(DGSWEM_E_MESH, "edge %lld: e+ does not list it", d);
    if (em >= 0) {
      if (em >= ne || lm < 0 || lm > 2 || em == ep) return h->fail(DGSWEM_E_MESH, "edge %lld: bad e- / local edge", d);
      if (elem_edge[3 * em + lm] != d) return h->fail(DGSWEM_E_MESH, "edge %lld: e- does not list it", d);
      if (bc != 0) return h->fail(DGSWEM_E_MESH, "edge %lld: interior edge with boundary code %d", d, bc);
      // the two sides must share the same two nodes, traversed in opposite directions
      const int a1 = tri[3 * ep + (lp + 1) % 3], b1 = tri[3 * ep + (lp + 2) % 3];
      const int a2 = tri[3 * em + (lm + 1) % 3], b2 = tri[3 * em + (lm + 2) % 3];
      if (a1 != b2 || b1 != a2) return h->fail(DGSWEM_E_MESH, "edge %lld: the two sides do not share the same nodes", d);
    } else {
      if (bc != 1 && bc != 2) return h->fail(DGSWEM_E_MESH, "edge %lld: boundary edge needs code 1 or 2, got %d", d, bc);
    }
  }
  return 0;
}

// resident grid of a persistent kernel: CTAs per SM (occupancy API) x SM count
template <typename K>
int resident_ctas(K kernel, int threads, size_t smem, int device) {
  int per_sm = 0, sms = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem) != cudaSuccess) { (void)cudaGetLastError(); return 0; }
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) { (void)cudaGetLastError(); return 0; }
  return per_sm * sms;
}

// a scalar argument: by value on a stream launch, by table reference while a step graph is being captured
inline ScalRef scal(const Handle* h, int idx, double val) {
  ScalRef r;
  r.tab = h->capturing ? h->scal_tab : nullptr; r.ctr = h->capturing ? h->step_ctr : nullptr; r.idx = idx; r.val = val;
  return r;
}

template <int P>
int launch_edge(Handle* h, const real* w, ScalRef zeta_b) {
  EdgeArgs a;
  a.w = w; a.edge_elem = h->edge_elem; a.einfo = h->einfo; a.en = h->en; a.ehb = h->ehb; a.flux = h->flux;
  a.nd = (int)h->nd; a.ld = h->ld; a.ldd = h->ldd;
  a.ph = Phys{(real)h->prm.g, (real)h->prm.h0_dry, (real)h->prm.cf, (real)h->prm.coriolis_f};
  a.zeta = zeta_b;
  const int ntiles = grid_for(h->nd, DGK_EDGE_THREADS);
  const int resident = h->res_edge[P - 1];
  prof_begin(h, PK_EDGE);
  const bool pipe = DGK_PIPE_EDGE && resident > 0 && ntiles > resident;
  if (h->prm.flux == 1) {
    if (pipe) k_edge_pipe<P, 1><<<resident, DGK_EDGE_THREADS, 0, h->stream>>>(a, ntiles);
    else k_edge<P, 1><<<ntiles, DGK_EDGE_THREADS, 0, h->stream>>>(a);
  } else {
    if (pipe) k_edge_pipe<P, 0><<<resident, DGK_EDGE_THREADS, 0, h->stream>>>(a, ntiles);
    else k_edge<P, 0><<<ntiles, DGK_EDGE_THREADS, 0, h->stream>>>(a);
  }
  prof_end(h);
  CKL("k_edge");
  return 0;
}

// compile-time specialisation of the element / stage kernels: bit 0 first RK stage, bit 1 Holland forcing, bit 2 its
// pressure gradient; -1 (flags read from the arguments) when a rarely used option is on (rain)
inline int stage_variant(const Handle* h, int first) {
  if (h->rain != 0.0) return -1;
  return (first ? 1 : 0) | (h->wind_on ? 2 : 0) | ((h->wind_on && h->press_on) ? 4 : 0);
}

template <int P, int MODE>
int launch_elem(Handle* h, const real* win, const real* w0, real* wout, double dt, real a, real b,
                int first, bool fuse_wd, bool write_mean) {
  ElemArgs A;
  A.win = win; A.w0 = w0; A.wout = wout; A.flux = h->flux; A.elem_edge = h->elem_edge; A.jinv = h->jinv;
  A.lfac = h->lfac; A.hv = h->hv; A.tri = h->tri; A.tau = h->tau; A.wet = h->wet;
  A.etap = h->etap; A.stress = h->stress_on ? 1 : 0; A.press = h->press_on ? 1 : 0; A.rain = (real)h->rain;
  A.nbinfo = nullptr; A.enl = nullptr; A.zeta = scal(h, 0, 0.0);
  A.mean = write_mean ? h->mean : nullptr;
  A.ne = (int)h->ne; A.ld = h->ld; A.ldd = h->ldd; A.ldn = h->ldn;
  A.ph = Phys{(real)h->prm.g, (real)h->prm.h0_dry, (real)h->prm.cf, (real)h->prm.coriolis_f};
  A.dt = (real)dt; A.a = a; A.b = b; A.first_stage = first; A.wind = h->wind_on ? 1 : 0; A.fuse_wetdry = fuse_wd ? 1 : 0;
  // (a persistent form with next-tile index prefetch, as for the edge kernel, was measured slower: it needs
  // more registers than the 128 the 4-CTA budget leaves, and the spills cost more than the prefetch saves)
  prof_begin(h, PK_ELEM);
  const int grid = grid_for(h->ne, DGK_ELEM_THREADS);
  if constexpr (MODE == MODE_UPDATE) {
    switch (stage_variant(h, first)) {   // specialised on (first stage, wind, pressure), as k_stage
      case 0: k_elem<P, MODE, 0><<<grid, DGK_ELEM_THREADS, 0, h->stream>>>(A); break;
      case 1: k_elem<P, MODE, 1><<<grid, DGK_ELEM_THREADS, 0, h->stream>>>(A); break;
      case 2: k_elem<P, MODE, 2><<<grid, DGK_ELEM_THREADS, 0, h->stream>>>(A); break;
      case 3: k_elem<P, MODE, 3><<<grid, DGK_ELEM_THREADS, 0, h->stream>>>(A); break;
      case 6: k_elem<P, MODE, 6><<<grid, DGK_ELEM_THREADS, 0, h->stream>>>(A); break;
      case 7: k_elem<P, MODE, 7><<<grid, DGK_ELEM_THREADS, 0, h->stream>>>(A); break;
      default: k_elem<P, MODE, -1><<<grid, DGK_ELEM_THREADS, 0, h->stream>>>(A); break;
    }
  } else {
    k_elem<P, MODE, -1><<<grid, DGK_ELEM_THREADS, 0, h->stream>>>(A);
  }
  prof_end(h);
  CKL("k_elem");
  return 0;
}

// the instantiation of k_stage_tile for (flux, stage variant): specialised like k_stage for p = 1 / LLF, generic otherwise
using TileKernel = void (*)(const ElemArgs, const int);
template <int P, int MODE>
TileKernel tile_kernel(int flux, int variant) {
  if (flux == 1) return k_stage_tile<P, MODE, -1, 1>;
  if constexpr (P == 1 && MODE == MODE_UPDATE) {
    switch (variant) {
      case 0: return k_stage_tile<P, MODE, 0>;
      case 1: return k_stage_tile<P, MODE, 1>;
      case 2: return k_stage_tile<P, MODE, 2>;
      case 3: return k_stage_tile<P, MODE, 3>;
      case 6: return k_stage_tile<P, MODE, 6>;
      case 7: return k_stage_tile<P, MODE, 7>;
      default: break;
    }
  }
  return k_stage_tile<P, MODE, -1>;
}
// (the attribute belongs to the function, not to the handle: always the largest tile possible, 3 x 128 items)
template <int P>
int tile_kernel_attrs(Handle* h, int smem) {
  for (int flux = 0; flux < 2; ++flux)
    for (int v = -1; v < 8; ++v) {
      CK(cudaFuncSetAttribute(tile_kernel<P, MODE_UPDATE>(flux, v), cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
      CK(cudaFuncSetAttribute(tile_kernel<P, MODE_RHS>(flux, v), cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    }
  return 0;
}

// the same for k_stage_stg
template <int P, int MODE>
TileKernel stg_kernel(int flux, int variant) {
  if (flux == 1) return k_stage_stg<P, MODE, -1, 1>;
  if constexpr (P == 1 && MODE == MODE_UPDATE) {
    switch (variant) {
      case 0: return k_stage_stg<P, MODE, 0>;
      case 1: return k_stage_stg<P, MODE, 1>;
      case 2: return k_stage_stg<P, MODE, 2>;
      case 3: return k_stage_stg<P, MODE, 3>;
      case 6: return k_stage_stg<P, MODE, 6>;
      case 7: return k_stage_stg<P, MODE, 7>;
      default: break;
    }
  }
  return k_stage_stg<P, MODE, -1>;
}
template <int P>
int stg_kernel_attrs(Handle* h, int smem) {
  for (int flux = 0; flux < 2; ++flux)
    for (int v = -1; v < 8; ++v) {
      CK(cudaFuncSetAttribute(stg_kernel<P, MODE_UPDATE>(flux, v), cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
      CK(cudaFuncSetAttribute(stg_kernel<P, MODE_RHS>(flux, v), cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    }
  return 0;
}

// A1-A5 (+A7) in one launch (element-centric form, no flux buffer)
template <int P, int MODE>
int launch_stage(Handle* h, const real* win, const real* w0, real* wout, double dt, real a, real b,
                 int first, bool fuse_wd, bool write_mean, ScalRef zeta_b, int part = 0) {
  // part: 0 the whole mesh; 1 the send-list elements only, 2 all the others (form 1; the other forms do everything in part 1)
  const bool split = part != 0 && !h->tiled && !h->staged && h->n_send_uniq > 0;
  if (part == 2 && !split) return 0;
  ElemArgs A;
  A.subset = h->send_uniq; A.skip = h->send_mask; A.nsub = (int)h->n_send_uniq; A.pf_dist = h->pf_dist;
  A.win = win; A.w0 = w0; A.wout = wout; A.flux = h->flux; A.elem_edge = h->elem_edge; A.jinv = h->jinv;
  A.lfac = h->lfac; A.hv = h->hv; A.tri = h->tri; A.tau = h->tau; A.wet = h->wet;
  A.etap = h->etap; A.stress = h->stress_on ? 1 : 0; A.press = h->press_on ? 1 : 0; A.rain = (real)h->rain;
  A.nbinfo = h->nbinfo; A.enl = h->enl; A.zeta = zeta_b;
  A.mean = write_mean ? h->mean : nullptr;
  A.ne = (int)h->ne; A.ld = h->ld; A.ldd = h->ldd; A.ldn = h->ldn;
  A.ph = Phys{(real)h->prm.g, (real)h->prm.h0_dry, (real)h->prm.cf, (real)h->prm.coriolis_f};
  A.dt = (real)dt; A.a = a; A.b = b; A.first_stage = first; A.wind = h->wind_on ? 1 : 0; A.fuse_wetdry = fuse_wd ? 1 : 0;
  // (persistent forms were measured slower on C3: next-tile neighbour-table prefetch 425 us, per-warp cp.async
  // staging of the next tile's rows in shared memory 445 us, against 374 us)
  if (h->staged) {          // TMA-staged operands, persistent CTAs
    A.tile_info = h->stg_info; A.it_nb = h->stg_nb; A.nbs = h->nbs; A.cap1 = h->stg_cap1; A.cap = 0;
    const int ntiles = grid_for(h->ne, kTile);
    const int res = h->res_stg[h->wind_on ? 1 : 0];
    const int grid = std::max(1, std::min(ntiles, res > 0 ? res : ntiles));
    prof_begin(h, PK_ELEM);
    stg_kernel<P, MODE>(h->prm.flux, MODE == MODE_UPDATE ? stage_variant(h, first) : -1)
        <<<grid, kTile, StageStg<P>::smem(h->stg_cap1, h->wind_on), h->stream>>>(A, ntiles);
    prof_end(h);
    CKL("k_stage_stg");
    return 0;
  }
  if (h->tiled) {           // shared-memory edge-tile form: one CTA per tile of 128 elements
    A.tile_info = h->tile_info; A.it_blob = h->it_blob; A.it_nb = h->it_nb; A.eslot = h->eslot;
    A.cap = h->tile_cap; A.cap1 = h->tile_cap1;
    const int ntiles = grid_for(h->ne, kTile);
    const int res = h->res_tile[h->wind_on ? 1 : 0];
    const int grid = std::max(1, std::min(ntiles, res > 0 ? res : ntiles));
    prof_begin(h, PK_ELEM);
    tile_kernel<P, MODE>(h->prm.flux, MODE == MODE_UPDATE ? stage_variant(h, first) : -1)
        <<<grid, kTile, StageTile<P>::smem(h->tile_cap, h->tile_cap1, h->wind_on), h->stream>>>(A, ntiles);
    prof_end(h);
    CKL("k_stage_tile");
    return 0;
  }
  if (split) {   // the listed elements (small: generic-flag kernel) / all but the flagged ones (specialised like the full launch)
    if (part == 1 && h->n_send_uniq == 0) return 0;
    prof_begin(h, PK_ELEM);
    const int grid = grid_for(part == 1 ? h->n_send_uniq : h->ne, DGK_STAGE_THREADS);
    if (h->prm.flux == 1) {
      if (part == 1) k_stage<P, MODE, -1, 1, 1><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A);
      else k_stage<P, MODE, -1, 1, 2><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A);
    } else if (part == 1) {
      k_stage<P, MODE, -1, 0, 1><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A);
    } else if constexpr (MODE == MODE_UPDATE && P == 1) {
      switch (stage_variant(h, first)) {
        case 0: k_stage<P, MODE, 0, 0, 2><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
        case 1: k_stage<P, MODE, 1, 0, 2><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
        case 2: k_stage<P, MODE, 2, 0, 2><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
        case 3: k_stage<P, MODE, 3, 0, 2><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
        case 6: k_stage<P, MODE, 6, 0, 2><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
        case 7: k_stage<P, MODE, 7, 0, 2><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
        default: k_stage<P, MODE, -1, 0, 2><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
      }
    } else {
      k_stage<P, MODE, -1, 0, 2><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A);
    }
    prof_end(h);
    CKL("k_stage (part)");
    return 0;
  }
  prof_begin(h, PK_ELEM);
  const int grid = grid_for(h->ne, DGK_STAGE_THREADS);
  constexpr int PFV = (P == 1) ? 1 : 0;          // the prefetching kernels exist for p = 1 (where this form is the default)
  const bool pf = PFV != 0 && h->pf_dist > 0;
  if (h->prm.flux == 1) {   // Roe: the generic-flag kernel only
    k_stage<P, MODE, -1, 1><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A);
  } else if constexpr (MODE == MODE_UPDATE) {
    // specialised on (first stage, wind): no w^n registers in stage 1, no wind registers without wind
    switch (stage_variant(h, first)) {
      case 0: if (pf) k_stage<P, MODE, 0, 0, 0, PFV><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); else k_stage<P, MODE, 0><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
      case 1: if (pf) k_stage<P, MODE, 1, 0, 0, PFV><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); else k_stage<P, MODE, 1><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
      case 2: if (pf) k_stage<P, MODE, 2, 0, 0, PFV><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); else k_stage<P, MODE, 2><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
      case 3: if (pf) k_stage<P, MODE, 3, 0, 0, PFV><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); else k_stage<P, MODE, 3><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
      case 6: if (pf) k_stage<P, MODE, 6, 0, 0, PFV><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); else k_stage<P, MODE, 6><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
      case 7: if (pf) k_stage<P, MODE, 7, 0, 0, PFV><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); else k_stage<P, MODE, 7><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
      default: if (pf) k_stage<P, MODE, -1, 0, 0, PFV><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); else k_stage<P, MODE, -1><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A); break;
    }
  } else {
    k_stage<P, MODE, -1><<<grid, DGK_STAGE_THREADS, 0, h->stream>>>(A);
  }
  prof_end(h);
  CKL("k_stage");
  return 0;
}

template <int P>
int launch_limwd(Handle* h, real* w) {
  LimArgs A;
  A.w = w; A.mean = h->mean; A.nbr = h->nbr; A.hv = h->hv; A.wet = h->wet; A.ne = (int)h->ne; A.ld = h->ld;
  A.tri = h->tri; A.nmm = h->nmm; A.ldn = h->ldn;
  A.h0 = (real)h->prm.h0_dry; A.limiter = h->prm.limiter; A.wetdry = h->prm.wetdry;
  prof_begin(h, PK_LIMWD);
  const int ntiles = grid_for(h->ne, 128);
  const int grid = std::max(1, std::min(ntiles, h->res_limwd > 0 ? h->res_limwd : ntiles));
  if (h->prm.limiter == 2) {   // vertex neighbourhood: extrema of the means around every node first
    k_node_minmax<<<grid_for(h->nn, 256), 256, 0, h->stream>>>(h->nmm, h->ldn, h->mean, h->node_ptr, h->node_ev, (int)h->nn);
    CKL("k_node_minmax");   // a failed launch must not let the limiter run on stale node extrema
    k_limwd_tma<P, 2><<<grid, 128, LimTile<P>::kSmem, h->stream>>>(A, ntiles);
  } else {
    k_limwd_tma<P, 1><<<grid, 128, LimTile<P>::kSmem, h->stream>>>(A, ntiles);
  }
  prof_end(h);
  CKL("k_limwd");
  return 0;
}

int launch_wind(Handle* h, double t) {
  WindArgs A;
  A.nxy = h->nxy; A.tau = h->tau; A.etap = h->etap; A.g = (real)h->prm.g; A.nn = (int)h->nn; A.ldn = h->ldn;
  A.cx = scal(h, 4, h->hol.x0 + h->hol.vx * t); A.cy = scal(h, 5, h->hol.y0 + h->hol.vy * t);
  A.rmax = (real)h->hol.rmax; A.dp = (real)h->hol.dp; A.B = (real)h->hol.B; A.rho_air = (real)h->hol.rho_air;
  A.rho_water = (real)h->hol.rho_water; A.f = (real)h->hol.f;
  prof_begin(h, PK_WIND);
  k_wind<<<grid_for(h->nn, 256), 256, 0, h->stream>>>(A);
  prof_end(h);
  CKL("k_wind");
  return 0;
}

double tide_value(const Handle* h, double t) {
  if (h->tide_amp == 0.0) return 0.0;
  return h->tide_amp * std::sin(h->tide_omega * t + h->tide_phase);
}

// one RK stage, first part: EDGE -> GATHER+AREA+RK (+wet/dry when no limiter follows)
template <int P>
int run_stage_rhs(Handle* h, const real* win, const real* w0, real* wout, double dt, real a, real b, int first,
                  double t_stage, int stage, int part = 0) {
  const bool lim = h->prm.limiter != 0;
  const bool wd = h->prm.wetdry != 0;
  int rc = 0;
  bool done = false;
  if constexpr (P <= 2) {
    if (h->fused) {
      rc = launch_stage<P, MODE_UPDATE>(h, win, w0, wout, dt, a, b, first, wd && !lim, lim, scal(h, stage, tide_value(h, t_stage)), part);
      done = true;
    }
  }
  if (!done) {
    if (part == 2) return 0;   // the edge + element pair does the whole stage in part 1
    rc = launch_edge<P>(h, win, scal(h, stage, tide_value(h, t_stage)));
    if (rc) return rc;
    rc = launch_elem<P, MODE_UPDATE>(h, win, w0, wout, dt, a, b, first, wd && !lim, lim);
  }
  return rc;
}

// one RK stage: first part, then the limiter + wet/dry pass over the RK-updated means (limiter on)
template <int P>
int run_stage(Handle* h, const real* win, const real* w0, real* wout, double dt, real a, real b, int first,
              double t_stage, int stage) {
  int rc = run_stage_rhs<P>(h, win, w0, wout, dt, a, b, first, t_stage, stage);
  if (rc) return rc;
  if (h->prm.limiter != 0) rc = launch_limwd<P>(h, wout);
  return rc;
}

// Two-register Shu-Osher SSP Runge-Kutta schemes (R-2, R-19): stage s is
//   u = w^(s-1) + (beta_s dt) L(w^(s-1), t + c_s dt);  w^(s) = u  (plain stage)  or  a_s w^n + b_s u.
// (order, stages): (2,2), (3,3), the optimal many-stage schemes (2,3), (2,4) and (3,4).
inline bool rk_get(int order, int stages, RkScheme& k) {
  if (stages == 0) stages = order;
  k.ns = stages;
  for (int s = 0; s < 4; ++s) { k.a[s] = RL(0.0); k.b[s] = RL(1.0); k.beta[s] = 1.0; k.c[s] = 0.0; }
  if (order == 2 && stages == 2) {
    k.a[1] = RL(0.5); k.b[1] = RL(0.5); k.c[1] = 1.0;
  } else if (order == 3 && stages == 3) {
    k.a[1] = RL(0.75); k.b[1] = RL(0.25); k.c[1] = 1.0;
    k.a[2] = RL(1.0) / RL(3.0); k.b[2] = RL(2.0) / RL(3.0); k.c[2] = 0.5;
  } else if (order == 2 && (stages == 3 || stages == 4)) {
    for (int s = 0; s < stages; ++s) { k.beta[s] = 1.0 / (double)(stages - 1); k.c[s] = (double)s / (double)(stages - 1); }
    k.a[stages - 1] = RL(1.0) / (real)stages; k.b[stages - 1] = (real)(stages - 1) / (real)stages;
  } else if (order == 3 && stages == 4) {
    for (int s = 0; s < 4; ++s) k.beta[s] = 0.5;
    k.c[1] = 0.5; k.c[2] = 1.0; k.c[3] = 0.5;
    k.a[2] = RL(2.0) / RL(3.0); k.b[2] = RL(1.0) / RL(3.0);
  } else {
    return false;
  }
  return true;
}

// buffers and coefficients of stage s: w^n stays in W[0] until the last stage overwrites it; the stages in between
// alternate W[1], W[2]
struct StageBufs { const real* win; const real* w0; real* wout; real a, b; double c, beta; int first; };
inline StageBufs stage_bufs(Handle* h, int s) {
  const RkScheme& K = h->rk;
  StageBufs B;
  B.a = K.a[s]; B.b = K.b[s]; B.c = K.c[s]; B.beta = K.beta[s];
  B.first = (K.a[s] == RL(0.0) && K.b[s] == RL(1.0)) ? 1 : 0;   // plain stage: no combine with w^n (and no read of it)
  B.w0 = h->W[0];
  B.win = s == 0 ? h->W[0] : h->W[1 + ((s - 1) & 1)];
  B.wout = s == K.ns - 1 ? h->W[0] : h->W[1 + (s & 1)];
  return B;
}

// enqueue the kernels of one time step starting at time t (values) or at table row *step_ctr (capturing)
template <int P>
int enqueue_step(Handle* h, double dt, double t) {
  if (h->wind_on) { int rc = launch_wind(h, t); if (rc) return rc; }
  for (int s = 0; s < h->rk.ns; ++s) {
    const StageBufs B = stage_bufs(h, s);
    const int rc = run_stage<P>(h, B.win, B.w0, B.wout, B.beta * dt, B.a, B.b, B.first, t + B.c * dt, s);
    if (rc) return rc;
  }
  return 0;
}

void drop_graphs(Handle* h) {
  if (h->graph_many.exec) cudaGraphExecDestroy(h->graph_many.exec);
  if (h->graph_one.exec) cudaGraphExecDestroy(h->graph_one.exec);
  h->graph_many = Handle::StepGraph(); h->graph_one = Handle::StepGraph();
}

// capture `steps` consecutive time steps (each followed by k_advance when a scalar table is in use) into one graph
template <int P>
int capture_steps(Handle* h, int steps, double dt, bool need_tab, Handle::StepGraph& out) {
  const long long l0 = h->launches;
  CK(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeRelaxed));
  h->capturing = need_tab;
  int rc = 0;
  for (int i = 0; i < steps && rc == 0; ++i) {
    rc = enqueue_step<P>(h, dt, 0.0);
    if (rc == 0 && need_tab) { k_advance<<<1, 1, 0, h->stream>>>(h->step_ctr); if (cudaGetLastError() != cudaSuccess) rc = DGSWEM_E_CUDA; else h->launches++; }
  }
  h->capturing = false;
  cudaGraph_t g = nullptr;
  const cudaError_t e = cudaStreamEndCapture(h->stream, &g);
  out.launches = h->launches - l0;
  h->launches = l0;   // nothing has run yet: replays are counted when they are launched
  if (rc) { if (g) cudaGraphDestroy(g); return rc; }
  if (e != cudaSuccess) return h->cuda_fail(e, "cudaStreamEndCapture");
  const cudaError_t e2 = cudaGraphInstantiate(&out.exec, g, 0);
  cudaGraphDestroy(g);
  if (e2 != cudaSuccess) { out.exec = nullptr; return h->cuda_fail(e2, "cudaGraphInstantiate"); }
  out.steps = steps;
  return 0;
}

// The per-step scalars of a replayed graph (tidal elevation of every stage, storm centre): device table + pinned staging
// copy + the event that guards the staging copy, created once per handle
constexpr long long kScalRows = 4096;   // steps per table upload (256 KiB); longer calls go in chunks
int ensure_scalar_table(Handle* h) {
  if (h->scal_cap != 0) return 0;
  // all three resources first, then published together: a failure leaves the handle as it was (scal_cap == 0)
  double* tab = (double*)h->dalloc((size_t)kScalRows * kScalStride * sizeof(double));
  if (!tab) return h->fail(DGSWEM_E_CUDA, "device allocation failed");
  double* host = nullptr;
  cudaEvent_t ev = nullptr;
  cudaError_t e = cudaMallocHost((void**)&host, (size_t)kScalRows * kScalStride * sizeof(double));
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
  if (e != cudaSuccess) {
    if (host) cudaFreeHost(host);
    h->dfree(tab);
    return h->cuda_fail(e, "scalar table setup");
  }
  h->scal_tab = tab; h->scal_host = host; h->scal_ev = ev; h->scal_cap = kScalRows;
  return 0;
}
// rows for the `chunk` steps that start at h->t, tabulated on the host exactly as the stream path computes them, uploaded on
// the handle's stream; the device step counter goes back to row 0
int upload_scalar_rows(Handle* h, long long chunk, double dt) {
  const double* c = h->rk.c;
  CK(cudaEventSynchronize(h->scal_ev));   // the previous upload has left the pinned staging copy
  double t = h->t;
  for (long long n = 0; n < chunk; ++n) {
    double* row = h->scal_host + (size_t)n * kScalStride;
    for (int i = 0; i < kScalStride; ++i) row[i] = 0.0;
    for (int st = 0; st < h->nstage; ++st) row[st] = tide_value(h, t + c[st] * dt);
    row[4] = h->hol.x0 + h->hol.vx * t; row[5] = h->hol.y0 + h->hol.vy * t;
    t = t + dt;
  }
  // stream order keeps earlier replays' reads of the device table ahead of this overwrite
  CK(cudaMemcpyAsync(h->scal_tab, h->scal_host, (size_t)chunk * kScalStride * sizeof(double), cudaMemcpyHostToDevice, h->stream));
  CK(cudaEventRecord(h->scal_ev, h->stream));
  CK(cudaMemsetAsync(h->step_ctr, 0, sizeof(int), h->stream));
  return 0;
}

template <int P>
int run_steps(Handle* h, long long nsteps, double dt) {
  if (!h->graphs_on || h->profiling || nsteps == 0) {
    for (long long n = 0; n < nsteps; ++n) {
      int rc = enqueue_step<P>(h, dt, h->t);
      if (rc) return rc;
      h->t = h->t + dt;
    }
    return 0;
  }
  // ---- graph replay: the step's kernel sequence is captured once per (dt, forcing on/off) and replayed;
  // the scalars that change from step to step (tidal elevation per stage, storm centre) are tabulated here
  // on the host exactly as the stream path computes them, and read by row on the device.
  const bool tide_on = h->tide_amp != 0.0;
  const bool need_tab = tide_on || h->wind_on;
  if (h->graph_one.exec && (h->graph_dt != dt || h->graph_wind != h->wind_on || h->graph_tide != tide_on)) drop_graphs(h);
  if (need_tab) { int rc = ensure_scalar_table(h); if (rc) return rc; }
  const int many = h->ne < 65536 ? 8 : (h->ne < 1000000 ? 2 : 1);
  if (!h->graph_one.exec) {
    int rc = capture_steps<P>(h, 1, dt, need_tab, h->graph_one);
    if (rc) return rc;
    if (many > 1 && (rc = capture_steps<P>(h, many, dt, need_tab, h->graph_many))) return rc;
    h->graph_dt = dt; h->graph_wind = h->wind_on; h->graph_tide = tide_on;
  }
  long long done = 0;
  while (done < nsteps) {
    const long long chunk = need_tab ? std::min(nsteps - done, h->scal_cap) : nsteps - done;
    if (need_tab) { int rc = upload_scalar_rows(h, chunk, dt); if (rc) return rc; }
    long long left = chunk;
    while (left > 0) {
      Handle::StepGraph& g = (h->graph_many.exec && left >= h->graph_many.steps) ? h->graph_many : h->graph_one;
      CK(cudaGraphLaunch(g.exec, h->stream));
      h->launches += g.launches;
      left -= g.steps;
    }
    for (long long n = 0; n < chunk; ++n) h->t = h->t + dt;
    done += chunk;
  }
  return 0;
}

}  // namespace

// ------------------------------------------------------------------------------------ C ABI


void api_destroy(Handle* h) {
  if (!h) return;
  // (a handle whose creation failed before a device was chosen owns nothing on any device: its ordinal may be the
  // rejected one and must not be made current)
  if (h->stream || !h->allocs.empty()) cudaSetDevice(h->prm.device);
  if (h->stream) cudaStreamSynchronize(h->stream);
  for (auto& r : h->prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  h->prof.clear();
  if (h->graph_many.exec) cudaGraphExecDestroy(h->graph_many.exec);
  if (h->graph_one.exec) cudaGraphExecDestroy(h->graph_one.exec);
  if (h->scal_ev) cudaEventDestroy(h->scal_ev);
  if (h->scal_host) cudaFreeHost(h->scal_host);
  h->release_all();
  if (h->own_stream && h->stream) cudaStreamDestroy(h->stream);
  delete h;
  (void)cudaGetLastError();   // nothing ignored above may stay pending for the next launch check of another handle
}

int api_create(dgswem_t** out, const dgswem_params* prm, const dgswem_devhooks* hooks, int64_t n_nodes,
                  const double* xy, const double* bathy, int64_t n_elem, const int32_t* tri, int64_t n_edge,
                  const int32_t* edge_elem, const int8_t* edge_local, const int32_t* edge_bc, const int32_t* elem_edge) {
  if (!out) { g_create_error = "out is NULL"; return DGSWEM_E_ARG; }
  *out = nullptr;
  Handle* h = new Handle();
  h->precision = DGK_F32 ? 32 : 64;
  auto bail = [&](int code) { g_create_error = h->err; api_destroy(h); return code; };
  if (!prm || !xy || !bathy || !tri || !edge_elem || !edge_local || !edge_bc || !elem_edge)
    return bail(h->fail(DGSWEM_E_ARG, "NULL argument"));
  if (n_nodes < 3 || n_elem < 1 || n_edge < 3 || n_elem > 0x1fffffff || n_edge > 0x7ffffff0 || n_nodes > 0x7ffffff0)
    return bail(h->fail(DGSWEM_E_ARG, "bad sizes"));
  if (prm->p < 1 || prm->p > 3) return bail(h->fail(DGSWEM_E_ARG, "p must be 1, 2 or 3"));
  if (!rk_get(prm->rk_order, prm->rk_stages, h->rk))
    return bail(h->fail(DGSWEM_E_ARG, "(rk_order, rk_stages) must be (2, 0|2), (3, 0|3), (2, 3), (2, 4) or (3, 4)"));
  if (prm->reorder < 0 || prm->reorder > 2) return bail(h->fail(DGSWEM_E_ARG, "reorder must be 0 (none), 1 (Hilbert curve) or 2 (reverse Cuthill-McKee)"));
  if (prm->flux < 0 || prm->flux > 1 || prm->limiter < 0 || prm->limiter > 2)
    return bail(h->fail(DGSWEM_E_ARG, "flux must be 0 (LLF) or 1 (Roe), limiter 0, 1 (edge neighbours) or 2 (vertex neighbourhood)"));
  if (!(prm->h0_dry > 0.0) || !(prm->g > 0.0) || prm->cf < 0.0)
    return bail(h->fail(DGSWEM_E_ARG, "need h0_dry > 0, g > 0, cf >= 0"));
  // range of the kernels' reciprocal / square-root routines (rcp_rn, sqrt_rn): arguments are H_c >= h0_dry and g * H_c
  if (!(prm->h0_dry >= 1e-100) || !(prm->g * prm->h0_dry >= 1e-100) || !(prm->g <= 1e100) || !(prm->h0_dry <= 1e100))
    return bail(h->fail(DGSWEM_E_ARG, "need 1e-100 <= h0_dry <= 1e100, g <= 1e100 and g*h0_dry >= 1e-100"));
  h->prm = *prm;
  h->ndof = (prm->p + 1) * (prm->p + 2) / 2; h->nqe = prm->p + 1; h->nqa = prm->p == 1 ? 3 : prm->p == 2 ? 6 : 12; h->nstage = h->rk.ns;
  h->nn = n_nodes; h->ne = n_elem; h->nd = n_edge;
  h->ld = round_up(n_elem, 256); h->ldd = round_up(n_edge, 256); h->ldn = round_up(n_nodes, 64);
  int rc = validate_mesh(h, n_nodes, xy, n_elem, tri, n_edge, edge_elem, edge_local, edge_bc, elem_edge);
  if (rc) return bail(rc);

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return bail(h->fail(DGSWEM_E_CUDA, "no CUDA device"));
  if (prm->device < 0 || prm->device >= ndev) return bail(h->fail(DGSWEM_E_ARG, "device ordinal out of range"));
  if (cudaSetDevice(prm->device) != cudaSuccess) return bail(h->fail(DGSWEM_E_CUDA, "cudaSetDevice failed"));
  if (hooks && hooks->alloc && hooks->free) { h->hooks = *hooks; h->have_hooks = true; }
  if (hooks && hooks->stream) {
    h->stream = (cudaStream_t)hooks->stream;
  } else {
    if (cudaStreamCreateWithFlags(&h->stream, cudaStreamNonBlocking) != cudaSuccess)
      return bail(h->fail(DGSWEM_E_CUDA, "cudaStreamCreate failed"));
    h->own_stream = true;
  }

  auto body = [&]() -> int {
    // ---- tables to constant memory (both degrees; identical for every handle)
    Tables T1, T2, T3;
    make_tables(1, T1); make_tables(2, T2); make_tables(3, T3);
    static TablesT<1> C1; static TablesT<2> C2;      // (static: the asynchronous copies below read them)
    copy_tables<1>(T1, C1); copy_tables<2>(T2, C2);
    CK(cudaMemcpyToSymbolAsync(c_tab1, &C1, sizeof(C1), 0, cudaMemcpyHostToDevice, h->stream));
    CK(cudaMemcpyToSymbolAsync(c_tab2, &C2, sizeof(C2), 0, cudaMemcpyHostToDevice, h->stream));
    CK(cudaMemcpyToSymbolAsync(c_tab3, &T3, sizeof(T3), 0, cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));

    h->res_edge[0] = resident_ctas(k_edge_pipe<1>, DGK_EDGE_THREADS, 0, prm->device);
    h->res_edge[1] = resident_ctas(k_edge_pipe<2>, DGK_EDGE_THREADS, 0, prm->device);
    h->res_edge[2] = resident_ctas(k_edge_pipe<3>, DGK_EDGE_THREADS, 0, prm->device);
    // tuning / test knob: DGSWEM_PERSISTENT_CTAS=n caps the persistent grid at n CTAs (so that small
    // meshes walk several tiles per CTA); 0 switches the persistent kernel off
    CK(cudaFuncSetAttribute(k_limwd_tma<1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LimTile<1>::kSmem));
    CK(cudaFuncSetAttribute(k_limwd_tma<2, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LimTile<2>::kSmem));
    CK(cudaFuncSetAttribute(k_limwd_tma<1, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LimTile<1>::kSmem));
    CK(cudaFuncSetAttribute(k_limwd_tma<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LimTile<2>::kSmem));
    CK(cudaFuncSetAttribute(k_limwd_tma<3, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LimTile<3>::kSmem));
    CK(cudaFuncSetAttribute(k_limwd_tma<3, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LimTile<3>::kSmem));
    if (prm->limiter == 2)
      h->res_limwd = prm->p == 1 ? resident_ctas(k_limwd_tma<1, 2>, 128, LimTile<1>::kSmem, prm->device)
                   : prm->p == 2 ? resident_ctas(k_limwd_tma<2, 2>, 128, LimTile<2>::kSmem, prm->device)
                                 : resident_ctas(k_limwd_tma<3, 2>, 128, LimTile<3>::kSmem, prm->device);
    else
      h->res_limwd = prm->p == 1 ? resident_ctas(k_limwd_tma<1, 1>, 128, LimTile<1>::kSmem, prm->device)
                   : prm->p == 2 ? resident_ctas(k_limwd_tma<2, 1>, 128, LimTile<2>::kSmem, prm->device)
                                 : resident_ctas(k_limwd_tma<3, 1>, 128, LimTile<3>::kSmem, prm->device);
    if (const char* env = std::getenv("DGSWEM_PERSISTENT_CTAS")) {
      const int cap = std::atoi(env);

      for (int& r : h->res_edge) r = cap <= 0 ? 0 : std::min(r, cap);
      h->res_limwd = cap <= 0 ? 0 : std::min(h->res_limwd, cap);
    }

    // DGSWEM_FUSED=1/0: element-centric stage kernel (no flux buffer) on/off; default: on for p = 1
    h->fused = prm->p == 1;
    h->tiled = false;
    // k_stage's L2 prefetch: on where a stage buffer does not stay in the 126 MB L2 anyway (C3: 336 -> 305 us per launch at any
    // distance from 50 to 600 tiles; C4, whose state fits, gains nothing)
    h->pf_dist = ((size_t)3 * h->ndof * h->ld * sizeof(real) > ((size_t)100 << 20)) ? 200 : 0;
    if (const char* env = std::getenv("DGSWEM_PF_DIST")) h->pf_dist = std::max(0, std::atoi(env));
    if (const char* env = std::getenv("DGSWEM_FUSED")) { h->fused = std::atoi(env) != 0; h->tiled = std::atoi(env) == 2; h->staged = std::atoi(env) == 3; }
    if (prm->p == 3) { h->fused = false; h->tiled = false; h->staged = false; }   // p = 3: the edge + element pair only (the element-centric forms would need > 255 registers)

    const long long ne = h->ne, nd = h->nd, nn = h->nn, ld = h->ld, ldd = h->ldd, ldn = h->ldn;
    // ---- renumbering (internal only): perm_e[new] = old
    std::vector<int> perm_e(ne), inv_e(ne), perm_d(nd), inv_d(nd);
    if (prm->reorder == 1) {
      std::vector<double> cx(ne), cy(ne);
      for (long long e = 0; e < ne; ++e) {
        const int* t = tri + 3 * e;
        cx[e] = (xy[2 * (long long)t[0]] + xy[2 * (long long)t[1]] + xy[2 * (long long)t[2]]) / 3.0;
        cy[e] = (xy[2 * (long long)t[0] + 1] + xy[2 * (long long)t[1] + 1] + xy[2 * (long long)t[2] + 1]) / 3.0;
      }
      perm_e = hilbert_order(cx, cy);
    } else if (prm->reorder == 2) {
      perm_e = rcm_order(ne, nd, edge_elem);
    } else {
      std::iota(perm_e.begin(), perm_e.end(), 0);
      std::iota(perm_d.begin(), perm_d.end(), 0);
    }
    for (long long i = 0; i < ne; ++i) inv_e[perm_e[i]] = (int)i;
    if (prm->reorder != 0) {
      // edges follow the elements: sorted by (first, second) of their two elements in the new element
      // numbering, so an edge sits next to the first element that needs it and the
      // state gather of consecutive edges walks consecutive elements
      std::vector<uint64_t> key(nd);
      for (long long d = 0; d < nd; ++d) {
        const uint32_t ip = (uint32_t)inv_e[edge_elem[2 * d]];
        const uint32_t im = edge_elem[2 * d + 1] >= 0 ? (uint32_t)inv_e[edge_elem[2 * d + 1]] : ip;
        key[d] = ((uint64_t)std::min(ip, im) << 32) | (uint64_t)std::max(ip, im);
      }
      std::iota(perm_d.begin(), perm_d.end(), 0);
      std::stable_sort(perm_d.begin(), perm_d.end(), [&](int x, int y) { return key[x] < key[y]; });
    }
    for (long long i = 0; i < nd; ++i) inv_d[perm_d[i]] = (int)i;

    // ---- element geometry in internal order (same expression trees as the spec), computed in the
    // working precision from the caller's coordinates and bathymetry rounded once
    auto X = [&](long long n) -> real { return (real)xy[2 * n]; };
    auto Y = [&](long long n) -> real { return (real)xy[2 * n + 1]; };
    std::vector<real> jinv(4 * ld, RL(0.0)), lfac(3 * ld, RL(0.0)), hv(3 * ld, RL(0.0));
    std::vector<int> ee_packed(3 * ld, 0), nbr(3 * ld, -1), trin(3 * ld, 0), nbinfo(3 * ld, (int)0x80000001);
    std::vector<real> enl(6 * ld, RL(0.0));
    for (long long i = 0; i < ne; ++i) {
      const long long e = perm_e[i];
      const int* t = tri + 3 * e;
      const real x0 = X(t[0]), y0 = Y(t[0]);
      const real x1 = X(t[1]), y1 = Y(t[1]);
      const real x2 = X(t[2]), y2 = Y(t[2]);
      const real dx1 = x1 - x0, dy1 = y1 - y0, dx2 = x2 - x0, dy2 = y2 - y0;
      const real A = RL(0.5) * (dx1 * dy2 - dx2 * dy1);
      const real rA = RL(1.0) / A;
      jinv[tix(4, 0, i)] = dy2 * rA;
      jinv[tix(4, 1, i)] = (-dx2) * rA;
      jinv[tix(4, 2, i)] = (-dy1) * rA;
      jinv[tix(4, 3, i)] = dx1 * rA;
      for (int l = 0; l < 3; ++l) {
        const long long na = t[(l + 1) % 3], nb = t[(l + 2) % 3];
        const real ex = X(nb) - X(na), ey = Y(nb) - Y(na);
        const real L = std::sqrt(ex * ex + ey * ey);
        lfac[tix(3, l, i)] = L * rA;
        hv[tix(3, l, i)] = (real)bathy[t[l]];
        trin[tix(3, l, i)] = t[l];
        const long long d = elem_edge[3 * e + l];
        const bool plus = edge_elem[2 * d] == e && edge_local[2 * d] == l;
        ee_packed[tix(3, l, i)] = inv_d[d] | (plus ? 0 : (int)0x80000000);
        const long long other = plus ? edge_elem[2 * d + 1] : edge_elem[2 * d];
        nbr[tix(3, l, i)] = other >= 0 ? inv_e[other] : -1;
        // element-centric form: neighbour id | its local edge << 29 (or bit 31 | boundary code), and the
        // outward normal: the e+ side's normal (computed from the e+ vertices, as for the edge kernel) or its negative
        const int lo = plus ? edge_local[2 * d + 1] : edge_local[2 * d];
        nbinfo[tix(3, l, i)] = other >= 0 ? (inv_e[other] | (lo << 29)) : (int)(0x80000000u | (unsigned)edge_bc[d]);
        const long long ep = edge_elem[2 * d];
        const int lp = edge_local[2 * d];
        const long long pa = tri[3 * ep + (lp + 1) % 3], pb = tri[3 * ep + (lp + 2) % 3];
        const real px = X(pb) - X(pa), py = Y(pb) - Y(pa);
        const real rL = RL(1.0) / std::sqrt(px * px + py * py);
        const real nx = py * rL, ny = (-px) * rL;
        enl[tix(6, 2 * l, i)] = plus ? nx : -nx;
        enl[tix(6, 2 * l + 1, i)] = plus ? ny : -ny;
      }
    }
    // ---- shared-memory edge-tile form: per tile of 128 elements the list of its unique edges ("items").  An edge whose
    // two elements sit in the same tile is listed once, under the element with the lower index (side a; the other
    // element reads the slot negated, in reversed point order); an edge to another tile or to the boundary is listed
    // under its element of this tile.  Items are in (a, la) order; every tile's list starts at a multiple of 32.
    const long long ntiles = ld / kTile;
    std::vector<int2> tile_info(ntiles, make_int2(0, 0));
    std::vector<unsigned char> it_blob;
    std::vector<int> it_nb, eslot(ld, 0);
    int tile_cap = 8, tile_cap1 = 8;
    if (h->tiled) {
      struct Item { int rec, nb; real nx, ny; };
      std::vector<Item> items; items.reserve((size_t)(1.8 * ne) + 64);
      std::vector<long long> first(ntiles + 1, 0);
      for (long long t = 0; t < ntiles; ++t) {
        int cnt = 0, n1 = 0;
        // items to other tiles first (their neighbour rows are prefetched into slots 0 .. n1-1), then the rest
        for (int pass = 0; pass < 2; ++pass) {
          for (long long i = t * kTile; i < std::min<long long>((t + 1) * kTile, ne); ++i) {
            for (int l = 0; l < 3; ++l) {
              const int nbi = nbinfo[tix(3, l, i)];
              const bool bnd = nbi < 0;
              const long long nb = bnd ? -1 : (nbi & 0x1fffffff);
              const int lo = bnd ? 0 : ((nbi >> 29) & 3);
              const bool in_tile = !bnd && (nb / kTile) == t;
              if (in_tile && nb < i) continue;   // listed under the lower element
              const int kind = bnd ? ((nbi & 3) == 2 ? 3 : 2) : (in_tile ? 0 : 1);
              if ((kind == 1) != (pass == 0)) continue;
              const int a = (int)(i - t * kTile), b = in_tile ? (int)(nb - t * kTile) : 0;
              items.push_back(Item{a | (l << 7) | (kind << 9) | (b << 11) | (lo << 18), kind == 1 ? (int)nb : 0,
                                   enl[tix(6, 2 * l, i)], enl[tix(6, 2 * l + 1, i)]});
              eslot[i] |= cnt << (10 * l);
              if (in_tile) eslot[nb] |= (cnt | 512) << (10 * lo);
              ++cnt;
            }
          }
          if (pass == 0) n1 = cnt;
        }
        tile_info[t] = make_int2(cnt, n1);
        first[t + 1] = first[t] + cnt;
        tile_cap = std::max(tile_cap, (cnt + 7) / 8 * 8);
        tile_cap1 = std::max(tile_cap1, (n1 + 7) / 8 * 8);
      }
      // fixed-size blocks per tile, so that one bulk copy of known size moves each
      const size_t ib = (size_t)(4 + 2 * sizeof(real)) * tile_cap;
      it_blob.assign(ib * ntiles, 0);
      it_nb.assign((size_t)tile_cap1 * ntiles, 0);
      for (long long t = 0; t < ntiles; ++t) {
        int* rec = reinterpret_cast<int*>(it_blob.data() + ib * t);
        real* nrm = reinterpret_cast<real*>(it_blob.data() + ib * t + 4 * (size_t)tile_cap);
        for (long long k = first[t]; k < first[t + 1]; ++k) {
          const long long i = k - first[t];
          rec[i] = items[k].rec; nrm[i] = items[k].nx; nrm[tile_cap + i] = items[k].ny;
          if (i < tile_info[t].y) it_nb[(size_t)tile_cap1 * t + i] = items[k].nb;
        }
      }
      h->tile_cap = tile_cap; h->tile_cap1 = tile_cap1;
      if (std::getenv("DGSWEM_TILE_STATS"))
        std::fprintf(stderr, "dgswem tile stats: %lld tiles, items/tile mean %.1f max-cap %d, to other tiles mean %.1f max-cap %d\n", ntiles,
                     (double)first[ntiles] / ntiles, tile_cap, [&] { double s1 = 0; for (auto& q : tile_info) s1 += q.y; return s1 / ntiles; }(), tile_cap1);
    }
    // ---- TMA-staged element-centric form: per tile the (deduplicated) list of neighbours in other tiles, and per
    // (element, local edge) the column of the neighbour's modes in the staged rows: its index in the tile, or 128 + its
    // position in that list; | neighbour's local edge << 9; boundary: bit 31 | code
    std::vector<int> nbs(3 * ld, (int)0x80000001), stg_nb;
    std::vector<int2> stg_info(ntiles, make_int2(0, 0));
    int stg_cap1 = 8;
    if (h->staged) {
      std::vector<std::vector<int>> lists(ntiles);
      for (long long t = 0; t < ntiles; ++t) {
        std::vector<int>& L = lists[t];
        for (long long i = t * kTile; i < std::min<long long>((t + 1) * kTile, ne); ++i) {
          for (int l = 0; l < 3; ++l) {
            const int nbi = nbinfo[tix(3, l, i)];
            if (nbi < 0) { nbs[tix(3, l, i)] = nbi; continue; }
            const long long nb = nbi & 0x1fffffff;
            const int lo = (nbi >> 29) & 3;
            int col;
            if (nb / kTile == t) {
              col = (int)(nb - t * kTile);
            } else {
              auto itf = std::find(L.begin(), L.end(), (int)nb);
              if (itf == L.end()) { L.push_back((int)nb); col = kTile + (int)L.size() - 1; } else col = kTile + (int)(itf - L.begin());
            }
            nbs[tix(3, l, i)] = col | (lo << 9);
          }
        }
        stg_info[t] = make_int2(0, (int)L.size());
        stg_cap1 = std::max(stg_cap1, ((int)L.size() + 7) / 8 * 8);
      }
      stg_nb.assign((size_t)stg_cap1 * ntiles, 0);
      for (long long t = 0; t < ntiles; ++t) std::copy(lists[t].begin(), lists[t].end(), stg_nb.begin() + (size_t)stg_cap1 * t);
      h->stg_cap1 = stg_cap1;
      if (std::getenv("DGSWEM_TILE_STATS")) {
        double s1 = 0; for (auto& q : stg_info) s1 += q.y;
        std::fprintf(stderr, "dgswem staged form: %lld tiles, neighbours in other tiles mean %.1f cap %d\n", ntiles, s1 / ntiles, stg_cap1);
      }
    }
    // ---- edge geometry in internal order, from the e+ side
    std::vector<int2> ee(ldd, make_int2(0, -1));
    std::vector<int> einfo(ldd, 1 << 4);
    std::vector<real> en(2 * ldd, RL(0.0)), ehb(2 * ldd, RL(0.0));
    for (long long i = 0; i < nd; ++i) {
      const long long d = perm_d[i];
      const long long ep = edge_elem[2 * d], em = edge_elem[2 * d + 1];
      const int lp = edge_local[2 * d], lm = em >= 0 ? edge_local[2 * d + 1] : 0;
      const long long na = tri[3 * ep + (lp + 1) % 3], nb = tri[3 * ep + (lp + 2) % 3];
      const real ex = X(nb) - X(na), ey = Y(nb) - Y(na);
      const real L = std::sqrt(ex * ex + ey * ey);
      const real rL = RL(1.0) / L;
      en[i] = ey * rL;
      en[ldd + i] = (-ex) * rL;
      ehb[i] = (real)bathy[na];
      ehb[ldd + i] = (real)bathy[nb];
      ee[i] = make_int2(inv_e[ep], em >= 0 ? inv_e[em] : -1);
      einfo[i] = lp | (lm << 2) | (edge_bc[d] << 4);
    }
    // node -> incident (element, vertex) lists for the nodal output, in ascending caller element id
    std::vector<int> node_ptr(nn + 1, 0), node_ev(3 * ne, 0);
    for (long long e = 0; e < ne; ++e) for (int v = 0; v < 3; ++v) node_ptr[tri[3 * e + v] + 1]++;
    for (long long n = 0; n < nn; ++n) node_ptr[n + 1] += node_ptr[n];
    {
      std::vector<int> fill(node_ptr.begin(), node_ptr.end() - 1);
      for (long long e = 0; e < ne; ++e) for (int v = 0; v < 3; ++v) node_ev[fill[tri[3 * e + v]]++] = inv_e[e] * 4 + v;
    }
    std::vector<real> nxy(2 * ldn, RL(0.0));
    for (long long i = 0; i < nn; ++i) { nxy[i] = X(i); nxy[ldn + i] = Y(i); }

    int r;
    if ((r = upload(h, h->jinv, jinv))) return r;
    if ((r = upload(h, h->lfac, lfac))) return r;
    if ((r = upload(h, h->hv, hv))) return r;
    if ((r = upload(h, h->elem_edge, ee_packed))) return r;
    if ((r = upload(h, h->nbr, nbr))) return r;
    if ((r = upload(h, h->nbinfo, nbinfo))) return r;
    if ((r = upload(h, h->enl, enl))) return r;
    if (h->staged) {
      if ((r = prm->p == 1 ? stg_kernel_attrs<1>(h, (int)StageStg<1>::smem(3 * kTile, true)) : stg_kernel_attrs<2>(h, (int)StageStg<2>::smem(3 * kTile, true)))) return r;
      for (int wnd = 0; wnd < 2; ++wnd) {
        const size_t sm = prm->p == 1 ? StageStg<1>::smem(stg_cap1, wnd != 0) : StageStg<2>::smem(stg_cap1, wnd != 0);
        h->res_stg[wnd] = prm->p == 1 ? resident_ctas(stg_kernel<1, MODE_UPDATE>(prm->flux, wnd ? 2 : 0), kTile, sm, prm->device)
                                      : resident_ctas(stg_kernel<2, MODE_UPDATE>(prm->flux, -1), kTile, sm, prm->device);
        if (const char* env = std::getenv("DGSWEM_PERSISTENT_CTAS")) { const int c = std::atoi(env); if (c > 0) h->res_stg[wnd] = std::min(h->res_stg[wnd], c); }
      }
      if ((r = upload(h, h->nbs, nbs))) return r;
      if ((r = upload(h, h->stg_nb, stg_nb))) return r;
      if ((r = upload(h, h->stg_info, stg_info))) return r;
    }
    if (h->tiled) {
      if ((r = prm->p == 1 ? tile_kernel_attrs<1>(h, (int)StageTile<1>::smem(3 * kTile, 3 * kTile, true)) : tile_kernel_attrs<2>(h, (int)StageTile<2>::smem(3 * kTile, 3 * kTile, true)))) return r;
      for (int wnd = 0; wnd < 2; ++wnd) {   // resident grid of the persistent kernel at this handle's shared-memory size
        const size_t sm = prm->p == 1 ? StageTile<1>::smem(tile_cap, tile_cap1, wnd != 0) : StageTile<2>::smem(tile_cap, tile_cap1, wnd != 0);
        h->res_tile[wnd] = prm->p == 1 ? resident_ctas(tile_kernel<1, MODE_UPDATE>(prm->flux, wnd ? 2 : 0), kTile, sm, prm->device)
                                       : resident_ctas(tile_kernel<2, MODE_UPDATE>(prm->flux, -1), kTile, sm, prm->device);
        if (const char* env = std::getenv("DGSWEM_PERSISTENT_CTAS")) { const int c = std::atoi(env); if (c > 0) h->res_tile[wnd] = std::min(h->res_tile[wnd], c); }
      }
      if ((r = upload(h, h->tile_info, tile_info))) return r;
      if ((r = upload(h, h->it_blob, it_blob))) return r;
      if ((r = upload(h, h->it_nb, it_nb))) return r;
      if ((r = upload(h, h->eslot, eslot))) return r;
    }
    if ((r = upload(h, h->tri, trin))) return r;
    if ((r = upload(h, h->edge_elem, ee))) return r;
    if ((r = upload(h, h->einfo, einfo))) return r;
    if ((r = upload(h, h->en, en))) return r;
    if ((r = upload(h, h->ehb, ehb))) return r;
    if ((r = upload(h, h->nxy, nxy))) return r;
    if ((r = upload(h, h->node_ptr, node_ptr))) return r;
    if ((r = upload(h, h->node_ev, node_ev))) return r;
    if (prm->reorder != 0) {
      if ((r = upload(h, h->perm_e, perm_e))) return r;
      if ((r = upload(h, h->inv_e, inv_e))) return r;
      if ((r = upload(h, h->inv_d, inv_d))) return r;
    }
    const size_t wbytes = (size_t)3 * h->ndof * ld * sizeof(real);
    for (int i = 0; i < std::min(h->nstage, 3); ++i) {
      h->W[i] = (real*)h->dalloc(wbytes);
      if (!h->W[i]) return h->fail(DGSWEM_E_CUDA, "device allocation of %zu bytes failed", wbytes);
      CK(cudaMemsetAsync(h->W[i], 0, wbytes, h->stream));
    }
    const size_t fbytes = (size_t)3 * h->nqe * ldd * sizeof(real);
    // staging in the caller's layout, binary64 whatever the working precision: a state, a flux buffer, or nodal rows
    h->stage_bytes = std::max((size_t)3 * h->ndof * ld, (size_t)3 * h->nqe * ldd) * sizeof(double);
    h->flux = (real*)h->dalloc(fbytes);
    h->mean = (real*)h->dalloc((size_t)3 * ld * sizeof(real));
    h->tau = (real*)h->dalloc((size_t)2 * ldn * sizeof(real));
    h->etap = (real*)h->dalloc((size_t)ldn * sizeof(real));
    if (prm->limiter == 2) {
      h->nmm = (real*)h->dalloc((size_t)6 * ldn * sizeof(real));
      if (!h->nmm) return h->fail(DGSWEM_E_CUDA, "device allocation failed");
    }
    h->stage_buf = (double*)h->dalloc(h->stage_bytes);
    h->wet = (unsigned char*)h->dalloc((size_t)ld);
    h->wet_stage = (unsigned char*)h->dalloc((size_t)ld);
    h->nf_flag = (int*)h->dalloc(256);
    h->step_ctr = (int*)h->dalloc(256);
    h->last_out = h->W[0];
    if (const char* env = std::getenv("DGSWEM_GRAPH")) h->graphs_on = std::atoi(env) != 0;
    if (!h->flux || !h->mean || !h->tau || !h->etap || !h->stage_buf || !h->wet || !h->wet_stage || !h->nf_flag || !h->step_ctr)
      return h->fail(DGSWEM_E_CUDA, "device allocation failed");
    CK(cudaMemsetAsync(h->flux, 0, fbytes, h->stream));
    CK(cudaMemsetAsync(h->mean, 0, (size_t)3 * ld * sizeof(real), h->stream));
    CK(cudaMemsetAsync(h->tau, 0, (size_t)2 * ldn * sizeof(real), h->stream));
    CK(cudaMemsetAsync(h->etap, 0, (size_t)ldn * sizeof(real), h->stream));
    CK(cudaMemsetAsync(h->wet, 1, (size_t)ld, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return 0;
  };
  rc = body();
  if (rc) return bail(rc);
  *out = h;
  return DGSWEM_OK;
}

int api_set_state(Handle* h, double t, const double* ze, const double* qx, const double* qy) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (!ze || !qx || !qy) return h->fail(DGSWEM_E_ARG, "NULL state pointer");
  CK(cudaSetDevice(h->prm.device));
  const double* src[3] = {ze, qx, qy};
  const size_t row = (size_t)h->ne * sizeof(double);
  // stage in caller order (rows of length ne, leading dimension ld), then renumber into the tiled layout on the device
  double* stage = h->stage_buf;
  for (int c = 0; c < 3; ++c)
    CK(cudaMemcpy2DAsync(stage + (size_t)c * h->ndof * h->ld, (size_t)h->ld * sizeof(double), src[c], row, row, h->ndof,
                         cudaMemcpyHostToDevice, h->stream));
  k_rows_to_tiled<<<dim3(grid_for(h->ne, 256), 3 * h->ndof), 256, 0, h->stream>>>(h->W[0], stage, h->ld, h->perm_e, (int)h->ne, 3 * h->ndof);
  CKL("k_rows_to_tiled");
  k_fill_bytes<<<grid_for(h->ld, 256), 256, 0, h->stream>>>(h->wet, 1, (int)h->ld);
  CKL("k_fill_bytes");
  if (h->prm.wetdry) {
    if (h->prm.p == 1) k_wetdry_only<1><<<grid_for(h->ne, 128), 128, 0, h->stream>>>(h->W[0], h->hv, h->wet, (int)h->ne, h->ld, h->prm.h0_dry);
    else if (h->prm.p == 3) k_wetdry_only<3><<<grid_for(h->ne, 128), 128, 0, h->stream>>>(h->W[0], h->hv, h->wet, (int)h->ne, h->ld, h->prm.h0_dry);
    else k_wetdry_only<2><<<grid_for(h->ne, 128), 128, 0, h->stream>>>(h->W[0], h->hv, h->wet, (int)h->ne, h->ld, h->prm.h0_dry);
    CKL("k_wetdry_only");
  }
  CK(cudaStreamSynchronize(h->stream));   // the caller's buffers may be reused after return
  h->t = t;
  h->step_dt = 0.0;
  h->last_out = h->W[0];
  return DGSWEM_OK;
}

int api_set_tide(Handle* h, double amp, double omega, double phase) {
  if (!h) return DGSWEM_E_ARG;
  h->tide_amp = amp; h->tide_omega = omega; h->tide_phase = phase;
  return DGSWEM_OK;
}

int api_set_wind_holland(Handle* h, const dgswem_holland* hol) {
  if (!h) return DGSWEM_E_ARG;
  drop_graphs(h);   // the vortex parameters are frozen arguments of a captured wind kernel
  if (hol) {
    if (!(hol->rmax > 0.0) || !(hol->rho_air > 0.0) || !(hol->rho_water > 0.0) || !(hol->B > 0.0))
      return h->fail(DGSWEM_E_ARG, "Holland parameters must be positive");
    h->hol = *hol; h->wind_on = true;
  } else {
    h->wind_on = false;
  }
  return DGSWEM_OK;
}

int api_set_wind_forcing(Handle* h, int stress_on, int pressure_on) {
  if (!h) return DGSWEM_E_ARG;
  drop_graphs(h);   // frozen kernel arguments
  h->stress_on = stress_on != 0; h->press_on = pressure_on != 0;
  return DGSWEM_OK;
}

int api_set_rain(Handle* h, double rate) {
  if (!h) return DGSWEM_E_ARG;
  if (!std::isfinite(rate)) return h->fail(DGSWEM_E_ARG, "rain rate must be finite");
  drop_graphs(h);
  h->rain = rate;
  return DGSWEM_OK;
}

int api_step(Handle* h, int64_t nsteps, double dt) {
  if (!h) return DGSWEM_E_ARG;
  if (nsteps < 0 || !(dt > 0.0)) return h->fail(DGSWEM_E_ARG, "need nsteps >= 0 and dt > 0");
  if (h->step_dt != 0.0) return h->fail(DGSWEM_E_ARG, "a stage-granular step is in progress (dgswem_end_step)");
  if (h->capturing) return h->fail(DGSWEM_E_ARG, "capture mode is on (dgswem_capture_mode(0) first)");
  CK(cudaSetDevice(h->prm.device));
  return h->prm.p == 1 ? run_steps<1>(h, nsteps, dt) : h->prm.p == 2 ? run_steps<2>(h, nsteps, dt) : run_steps<3>(h, nsteps, dt);
}

// ---- stage-granular stepping + halo lists: the building blocks of a domain-decomposed run
int api_begin_step(Handle* h, double dt) {
  if (!h) return DGSWEM_E_ARG;
  if (!(dt > 0.0)) return h->fail(DGSWEM_E_ARG, "need dt > 0");
  if (h->step_dt != 0.0) return h->fail(DGSWEM_E_ARG, "a step is already in progress");
  CK(cudaSetDevice(h->prm.device));
  if (h->wind_on) { int rc = launch_wind(h, h->t); if (rc) return rc; }
  h->step_dt = dt;
  h->last_out = h->W[0];
  return DGSWEM_OK;
}

int api_stage_rhs(Handle* h, int s, int part) {
  if (!h) return DGSWEM_E_ARG;
  if (h->step_dt == 0.0) return h->fail(DGSWEM_E_ARG, "no step in progress (dgswem_begin_step)");
  if (s < 0 || s >= h->nstage) return h->fail(DGSWEM_E_ARG, "stage index out of range");
  if (part < 0 || part > 2) return h->fail(DGSWEM_E_ARG, "part must be 0 (all), 1 (send-list elements) or 2 (the others)");
  CK(cudaSetDevice(h->prm.device));
  const StageBufs B = stage_bufs(h, s);
  const double ts = h->t + B.c * h->step_dt;
  const int rc = h->prm.p == 1 ? run_stage_rhs<1>(h, B.win, B.w0, B.wout, B.beta * h->step_dt, B.a, B.b, B.first, ts, s, part)
               : h->prm.p == 2 ? run_stage_rhs<2>(h, B.win, B.w0, B.wout, B.beta * h->step_dt, B.a, B.b, B.first, ts, s, part)
                               : run_stage_rhs<3>(h, B.win, B.w0, B.wout, B.beta * h->step_dt, B.a, B.b, B.first, ts, s, part);
  if (rc == 0) h->last_out = B.wout;
  return rc;
}

int api_stage_limit(Handle* h, int s) {
  if (!h) return DGSWEM_E_ARG;
  if (h->step_dt == 0.0) return h->fail(DGSWEM_E_ARG, "no step in progress (dgswem_begin_step)");
  if (s < 0 || s >= h->nstage) return h->fail(DGSWEM_E_ARG, "stage index out of range");
  if (h->prm.limiter == 0) return DGSWEM_OK;
  CK(cudaSetDevice(h->prm.device));
  const StageBufs B = stage_bufs(h, s);
  return h->prm.p == 1 ? launch_limwd<1>(h, B.wout) : h->prm.p == 2 ? launch_limwd<2>(h, B.wout) : launch_limwd<3>(h, B.wout);
}

int api_end_step(Handle* h) {
  if (!h) return DGSWEM_E_ARG;
  if (h->step_dt == 0.0) return h->fail(DGSWEM_E_ARG, "no step in progress (dgswem_begin_step)");
  if (h->capturing) {
    // being recorded into the caller's graph, not run: time does not move; the replayed step ends by moving to the next table row
    CK(cudaSetDevice(h->prm.device));
    k_advance<<<1, 1, 0, h->stream>>>(h->step_ctr);
    CKL("k_advance");
  } else {
    h->t = h->t + h->step_dt;
  }
  h->step_dt = 0.0;
  h->last_out = h->W[0];
  return DGSWEM_OK;
}

// ---- a stage-granular step recorded into the CALLER's CUDA graph (a decomposed run's whole step: all partitions + the exchange)
int api_capture_mode(Handle* h, int on) {
  if (!h) return DGSWEM_E_ARG;
  if (h->step_dt != 0.0) return h->fail(DGSWEM_E_ARG, "a stage-granular step is in progress");
  if (on && h->profiling) return h->fail(DGSWEM_E_ARG, "per-launch profiling events cannot be recorded into a graph (dgswem_profile(0) first)");
  if (on) { CK(cudaSetDevice(h->prm.device)); int rc = ensure_scalar_table(h); if (rc) return rc; }
  h->capturing = on != 0;
  return DGSWEM_OK;
}
int api_graph_steps(Handle* h, int64_t nsteps, double dt) {
  if (!h) return DGSWEM_E_ARG;
  if (nsteps < 0 || !(dt > 0.0)) return h->fail(DGSWEM_E_ARG, "need nsteps >= 0 and dt > 0");
  if (h->capturing || h->step_dt != 0.0) return h->fail(DGSWEM_E_ARG, "not while a step is being recorded or is in progress");
  CK(cudaSetDevice(h->prm.device));
  int rc = ensure_scalar_table(h);
  if (rc) return rc;
  if (nsteps > h->scal_cap) return h->fail(DGSWEM_E_ARG, "at most 4096 steps per call");
  if ((rc = upload_scalar_rows(h, nsteps, dt))) return rc;
  for (int64_t n = 0; n < nsteps; ++n) h->t = h->t + dt;
  return DGSWEM_OK;
}

int api_set_halo(Handle* h, int64_t n_send, const int32_t* send_ids, int64_t n_recv, const int32_t* recv_ids) {
  if (!h) return DGSWEM_E_ARG;
  if (n_send < 0 || n_recv < 0 || (n_send > 0 && !send_ids) || (n_recv > 0 && !recv_ids)) return h->fail(DGSWEM_E_ARG, "bad halo lists");
  CK(cudaSetDevice(h->prm.device));
  // caller numbering -> internal numbering (host copy of inv_e)
  std::vector<int> inv;
  if (h->inv_e) {
    inv.resize((size_t)h->ne);
    CK(cudaMemcpyAsync(inv.data(), h->inv_e, (size_t)h->ne * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
  }
  auto conv = [&](int64_t n, const int32_t* ids, std::vector<int>& out) -> bool {
    out.resize((size_t)std::max<int64_t>(n, 1));
    for (int64_t i = 0; i < n; ++i) {
      if (ids[i] < 0 || ids[i] >= h->ne) return false;
      out[(size_t)i] = inv.empty() ? ids[i] : inv[(size_t)ids[i]];
    }
    return true;
  };
  std::vector<int> snd, rcv;
  if (!conv(n_send, send_ids, snd) || !conv(n_recv, recv_ids, rcv)) return h->fail(DGSWEM_E_ARG, "halo element id out of range");
  int r;
  CK(cudaStreamSynchronize(h->stream));        // nothing in flight may still read the lists being replaced
  h->dfree(h->halo_send); h->dfree(h->halo_recv); h->dfree(h->halo_buf); h->dfree(h->send_uniq); h->dfree(h->send_mask);
  h->halo_send = nullptr; h->halo_recv = nullptr; h->halo_buf = nullptr; h->n_send = 0; h->n_recv = 0;
  h->send_uniq = nullptr; h->send_mask = nullptr; h->n_send_uniq = 0;
  {
    std::vector<unsigned char> mask((size_t)h->ld, 0);
    std::vector<int> uniq;
    for (int64_t i = 0; i < n_send; ++i)
      if (!mask[(size_t)snd[(size_t)i]]) { mask[(size_t)snd[(size_t)i]] = 1; uniq.push_back(snd[(size_t)i]); }
    std::sort(uniq.begin(), uniq.end());
    h->n_send_uniq = (long long)uniq.size();
    if (uniq.empty()) uniq.push_back(0);
    if ((r = upload(h, h->send_uniq, uniq))) return r;
    if ((r = upload(h, h->send_mask, mask))) return r;
  }
  if ((r = upload(h, h->halo_send, snd))) return r;
  if ((r = upload(h, h->halo_recv, rcv))) return r;
  h->n_send = n_send; h->n_recv = n_recv;
  h->halo_buf = (double*)h->dalloc((size_t)3 * h->ndof * (size_t)std::max<int64_t>(std::max(n_send, n_recv), 1) * sizeof(double));
  if (!h->halo_buf) return h->fail(DGSWEM_E_CUDA, "device allocation failed");
  return DGSWEM_OK;
}

static int halo_rows(const Handle* h, int what) { return what == 0 ? 3 * h->ndof : 3; }

int api_halo_pack(Handle* h, int what, double* buf, int buf_on_device) {
  if (!h) return DGSWEM_E_ARG;
  if ((what != 0 && what != 1) || (!buf && h->n_send > 0)) return h->fail(DGSWEM_E_ARG, "bad halo_pack arguments");
  if (!buf_on_device) NO_CAPTURE();   // the host-buffer form copies back and synchronises
  if (h->n_send == 0) return DGSWEM_OK;
  CK(cudaSetDevice(h->prm.device));
  const int rows = halo_rows(h, what);
  const real* src = what == 0 ? h->last_out : h->mean;
  double* dbuf = buf_on_device ? buf : h->halo_buf;
  k_halo_pack<<<grid_for(h->n_send, 256), 256, 0, h->stream>>>(dbuf, src, h->halo_send, (int)h->n_send, rows);
  CKL("k_halo_pack");
  if (!buf_on_device) {
    CK(cudaMemcpyAsync(buf, dbuf, (size_t)rows * h->n_send * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
  }
  return DGSWEM_OK;
}

int api_halo_unpack(Handle* h, int what, const double* buf, int buf_on_device) {
  if (!h) return DGSWEM_E_ARG;
  if ((what != 0 && what != 1) || (!buf && h->n_recv > 0)) return h->fail(DGSWEM_E_ARG, "bad halo_unpack arguments");
  if (!buf_on_device) NO_CAPTURE();   // the host-buffer form synchronises
  if (h->n_recv == 0) return DGSWEM_OK;
  CK(cudaSetDevice(h->prm.device));
  const int rows = halo_rows(h, what);
  real* dst = what == 0 ? h->last_out : h->mean;
  const double* dbuf = buf;
  if (!buf_on_device) {
    CK(cudaMemcpyAsync(h->halo_buf, buf, (size_t)rows * h->n_recv * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    dbuf = h->halo_buf;
  }
  if (what == 0) k_halo_unpack<<<grid_for(h->n_recv, 256), 256, 0, h->stream>>>(dst, dbuf, h->halo_recv, (int)h->n_recv, rows);
  else k_halo_unpack_means<<<grid_for(h->n_recv, 256), 256, 0, h->stream>>>(h->mean, h->last_out, dbuf, h->halo_recv, (int)h->n_recv, h->ndof);
  CKL("k_halo_unpack");
  if (!buf_on_device) CK(cudaStreamSynchronize(h->stream));
  return DGSWEM_OK;
}

int api_eval_rhs(Handle* h, double* rze, double* rqx, double* rqy) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (!rze || !rqx || !rqy) return h->fail(DGSWEM_E_ARG, "NULL output pointer");
  if (h->step_dt != 0.0) return h->fail(DGSWEM_E_ARG, "a stage-granular step is in progress: its stage buffer is the scratch of dgswem_eval_rhs");
  CK(cudaSetDevice(h->prm.device));
  int rc;
  if (h->wind_on && (rc = launch_wind(h, h->t))) return rc;
  real* rbuf = h->W[1];   // scratch: W[1] holds no live data between steps
  if (h->fused) {
    rc = h->prm.p == 1 ? launch_stage<1, MODE_RHS>(h, h->W[0], h->W[0], rbuf, 0.0, RL(0.0), RL(1.0), 1, false, false, scal(h, 0, tide_value(h, h->t)))
                       : launch_stage<2, MODE_RHS>(h, h->W[0], h->W[0], rbuf, 0.0, RL(0.0), RL(1.0), 1, false, false, scal(h, 0, tide_value(h, h->t)));
    if (rc) return rc;
  } else if (h->prm.p == 1) {
    if ((rc = launch_edge<1>(h, h->W[0], scal(h, 0, tide_value(h, h->t))))) return rc;
    if ((rc = launch_elem<1, MODE_RHS>(h, h->W[0], h->W[0], rbuf, 0.0, RL(0.0), RL(1.0), 1, false, false))) return rc;
  } else if (h->prm.p == 2) {
    if ((rc = launch_edge<2>(h, h->W[0], scal(h, 0, tide_value(h, h->t))))) return rc;
    if ((rc = launch_elem<2, MODE_RHS>(h, h->W[0], h->W[0], rbuf, 0.0, RL(0.0), RL(1.0), 1, false, false))) return rc;
  } else {
    if ((rc = launch_edge<3>(h, h->W[0], scal(h, 0, tide_value(h, h->t))))) return rc;
    if ((rc = launch_elem<3, MODE_RHS>(h, h->W[0], h->W[0], rbuf, 0.0, RL(0.0), RL(1.0), 1, false, false))) return rc;
  }
  k_tiled_to_rows<<<dim3(grid_for(h->ne, 256), 3 * h->ndof), 256, 0, h->stream>>>(h->stage_buf, h->ld, rbuf, h->inv_e, (int)h->ne, 3 * h->ndof);
  CKL("k_tiled_to_rows");
  const double* src = h->stage_buf;
  double* dst[3] = {rze, rqx, rqy};
  const size_t row = (size_t)h->ne * sizeof(double);
  for (int c = 0; c < 3; ++c)
    CK(cudaMemcpy2DAsync(dst[c], row, src + (size_t)c * h->ndof * h->ld, (size_t)h->ld * sizeof(double), row, h->ndof,
                         cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return DGSWEM_OK;
}

int api_get_flux(Handle* h, double* flux) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (!flux) return h->fail(DGSWEM_E_ARG, "NULL output pointer");
  if (h->fused && h->step_dt != 0.0) return h->fail(DGSWEM_E_ARG, "a stage-granular step is in progress");
  CK(cudaSetDevice(h->prm.device));
  if (h->fused) {   // the element-centric stage kernel keeps no flux buffer: evaluate A1 on the current state
    int rc = h->prm.p == 1 ? launch_edge<1>(h, h->W[0], scal(h, 0, tide_value(h, h->t))) : h->prm.p == 2 ? launch_edge<2>(h, h->W[0], scal(h, 0, tide_value(h, h->t)))
                           : launch_edge<3>(h, h->W[0], scal(h, 0, tide_value(h, h->t)));
    if (rc) return rc;
  }
  // internal edge order and working precision -> caller's order, binary64
  k_gather_rows<<<dim3(grid_for(h->nd, 256), 3 * h->nqe), 256, 0, h->stream>>>(h->stage_buf, h->ldd, h->flux, h->ldd, h->inv_d, (int)h->nd, 3 * h->nqe);
  CKL("k_gather_rows");
  const double* src = h->stage_buf;
  const size_t row = (size_t)h->nd * sizeof(double);
  CK(cudaMemcpy2DAsync(flux, row, src, (size_t)h->ldd * sizeof(double), row, 3 * h->nqe, cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return DGSWEM_OK;
}

int api_get_state(Handle* h, double* t, double* ze, double* qx, double* qy) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (!ze || !qx || !qy) return h->fail(DGSWEM_E_ARG, "NULL output pointer");
  CK(cudaSetDevice(h->prm.device));
  k_tiled_to_rows<<<dim3(grid_for(h->ne, 256), 3 * h->ndof), 256, 0, h->stream>>>(h->stage_buf, h->ld, h->W[0], h->inv_e, (int)h->ne, 3 * h->ndof);
  CKL("k_tiled_to_rows");
  const double* src = h->stage_buf;
  CK(cudaMemsetAsync(h->nf_flag, 0, sizeof(int), h->stream));
  k_check_finite<<<148 * 8, 256, 0, h->stream>>>(h->W[0], (long long)3 * h->ndof * h->ld, h->nf_flag);
  CKL("k_check_finite");
  double* dst[3] = {ze, qx, qy};
  const size_t row = (size_t)h->ne * sizeof(double);
  for (int c = 0; c < 3; ++c)
    CK(cudaMemcpy2DAsync(dst[c], row, src + (size_t)c * h->ndof * h->ld, (size_t)h->ld * sizeof(double), row, h->ndof,
                         cudaMemcpyDeviceToHost, h->stream));
  int flag = 0;
  CK(cudaMemcpyAsync(&flag, h->nf_flag, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  if (t) *t = h->t;
  if (flag) return h->fail(DGSWEM_E_NONFINITE, "non-finite value in the state at t=%g", h->t);
  return DGSWEM_OK;
}

int api_get_wetdry(Handle* h, uint8_t* wet) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (!wet) return h->fail(DGSWEM_E_ARG, "NULL output pointer");
  CK(cudaSetDevice(h->prm.device));
  const unsigned char* src = h->wet;
  if (h->inv_e) {
    k_gather_bytes<<<grid_for(h->ne, 256), 256, 0, h->stream>>>(h->wet_stage, h->wet, h->inv_e, (int)h->ne);
    CKL("k_gather_bytes");
    src = h->wet_stage;
  }
  CK(cudaMemcpyAsync(wet, src, (size_t)h->ne, cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return DGSWEM_OK;
}

int api_get_nodal(Handle* h, double* zn, double* qxn, double* qyn) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (!zn || !qxn || !qyn) return h->fail(DGSWEM_E_ARG, "NULL output pointer");
  CK(cudaSetDevice(h->prm.device));
  double* out = h->stage_buf;   // [3][ldn] (3 * ldn <= the state-sized staging buffer: n_nodes < n_elem + 3 for any triangulation with a boundary)
  if ((size_t)3 * h->ldn * sizeof(double) > h->stage_bytes) return h->fail(DGSWEM_E_ARG, "nodal output needs n_nodes <= ndof * n_elem");
  if (h->prm.p == 1) k_nodal<1><<<grid_for(h->nn, 256), 256, 0, h->stream>>>(out, h->ldn, h->W[0], h->node_ptr, h->node_ev, (int)h->nn);
  else if (h->prm.p == 3) k_nodal<3><<<grid_for(h->nn, 256), 256, 0, h->stream>>>(out, h->ldn, h->W[0], h->node_ptr, h->node_ev, (int)h->nn);
  else k_nodal<2><<<grid_for(h->nn, 256), 256, 0, h->stream>>>(out, h->ldn, h->W[0], h->node_ptr, h->node_ev, (int)h->nn);
  CKL("k_nodal");
  double* dst[3] = {zn, qxn, qyn};
  for (int c = 0; c < 3; ++c)
    CK(cudaMemcpyAsync(dst[c], out + (size_t)c * h->ldn, (size_t)h->nn * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return DGSWEM_OK;
}

int api_get_wind(Handle* h, double* tau) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (!tau) return h->fail(DGSWEM_E_ARG, "NULL output pointer");
  CK(cudaSetDevice(h->prm.device));
  k_gather_rows<<<dim3(grid_for(h->nn, 256), 2), 256, 0, h->stream>>>(h->stage_buf, h->ldn, h->tau, h->ldn, nullptr, (int)h->nn, 2);
  CKL("k_gather_rows");
  const size_t row = (size_t)h->nn * sizeof(double);
  CK(cudaMemcpy2DAsync(tau, row, h->stage_buf, (size_t)h->ldn * sizeof(double), row, 2, cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return DGSWEM_OK;
}

int api_get_pressure(Handle* h, double* etap) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (!etap) return h->fail(DGSWEM_E_ARG, "NULL output pointer");
  CK(cudaSetDevice(h->prm.device));
  k_gather_rows<<<dim3(grid_for(h->nn, 256), 1), 256, 0, h->stream>>>(h->stage_buf, h->ldn, h->etap, h->ldn, nullptr, (int)h->nn, 1);
  CKL("k_gather_rows");
  CK(cudaMemcpyAsync(etap, h->stage_buf, (size_t)h->nn * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return DGSWEM_OK;
}

int api_test_math(Handle* h, int64_t n, const double* x, double* out) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (n < 1 || !x || !out) return h->fail(DGSWEM_E_ARG, "need n >= 1 and non-NULL pointers");
  CK(cudaSetDevice(h->prm.device));
  double* dx = (double*)h->dalloc((size_t)n * sizeof(double));
  double* dout = (double*)h->dalloc((size_t)4 * n * sizeof(double));
  if (!dx || !dout) return h->fail(DGSWEM_E_CUDA, "device allocation failed");
  CK(cudaMemcpyAsync(dx, x, (size_t)n * sizeof(double), cudaMemcpyHostToDevice, h->stream));
  k_test_math<<<grid_for(n, 256), 256, 0, h->stream>>>(dx, (long long)n, dout);
  CKL("k_test_math");
  const cudaError_t e1 = cudaMemcpyAsync(out, dout, (size_t)4 * n * sizeof(double), cudaMemcpyDeviceToHost, h->stream);
  const cudaError_t e2 = cudaStreamSynchronize(h->stream);
  h->dfree(dx); h->dfree(dout);
  if (e1 != cudaSuccess) return h->cuda_fail(e1, "cudaMemcpyAsync");
  if (e2 != cudaSuccess) return h->cuda_fail(e2, "cudaStreamSynchronize");
  return DGSWEM_OK;
}

int api_fp64_peak(Handle* h, double* dfma_per_s) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (!dfma_per_s) return h->fail(DGSWEM_E_ARG, "NULL output pointer");
  CK(cudaSetDevice(h->prm.device));
  int sms = 0;
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->prm.device));
  const int grid = sms * 8, threads = 256, rounds = 20000;
  cudaEvent_t a, b;
  CK(cudaEventCreate(&a)); CK(cudaEventCreate(&b));
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {      // first repetition warms up
    CK(cudaEventRecord(a, h->stream));
    k_dfma_probe<<<grid, threads, 0, h->stream>>>(h->stage_buf, rounds, 0.999999, 1e-6);
    CKL("k_dfma_probe");
    CK(cudaEventRecord(b, h->stream));
    CK(cudaEventSynchronize(b));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, a, b));
    const double rate = (double)grid * threads * 8.0 * rounds / (ms * 1e-3);
    if (rep > 0 && rate > best) best = rate;
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  *dfma_per_s = best;
  return DGSWEM_OK;
}

int api_stage_form(const Handle* h) { return (h && h->fused) ? (h->staged ? 3 : h->tiled ? 2 : 1) : 0; }

int64_t api_launch_count(const Handle* h) { return h ? h->launches : 0; }

int api_profile(Handle* h, int enable) {
  if (!h) return DGSWEM_E_ARG;
  if (enable && h->capturing) return h->fail(DGSWEM_E_ARG, "capture mode is on: profiling events cannot be recorded into a graph");
  h->profiling = enable != 0;
  return DGSWEM_OK;
}

int api_profile_read(Handle* h, double* ms, int64_t* count) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  if (!ms || !count) return h->fail(DGSWEM_E_ARG, "NULL output pointer");
  CK(cudaSetDevice(h->prm.device));
  CK(cudaStreamSynchronize(h->stream));
  for (int k = 0; k < PK_COUNT; ++k) { ms[k] = 0.0; count[k] = 0; }
  for (auto& r : h->prof) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess) { ms[r.kind] += (double)t; count[r.kind]++; }
    cudaEventDestroy(r.a); cudaEventDestroy(r.b);
  }
  h->prof.clear();
  return DGSWEM_OK;
}

int api_sync(Handle* h) {
  if (!h) return DGSWEM_E_ARG;
  NO_CAPTURE();
  CK(cudaSetDevice(h->prm.device));
  CK(cudaStreamSynchronize(h->stream));
  return DGSWEM_OK;
}


}  // namespace DGK_IMPL_NS
