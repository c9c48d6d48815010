// dgswem_static.cu -- dgswem_nodal_static: the nodal output of PAPER.md:109 ("we convert the modal representation to a
// nodal representation by averaging the neighboring elements of each node") for callers that must not allocate.
//
// Who that is.  dgswem_get_nodal works on a handle, and a handle gets its node -> element incidence table (and every
// other buffer) from cudaMalloc or from the caller's allocation hooks inside dgswem_create.  Some programs cannot do
// either at the moment they want nodal fields: an output routine that runs while a stream capture is open in the
// process (cudaMalloc is not allowed during a capture and invalidates it); a solver embedded in a host application
// whose memory pool already owns the whole device, so that cudaMalloc fails; a time loop that must not stall, since
// cudaMalloc and cudaFree synchronise the device.  They hold the mesh connectivity and the modal state in device
// buffers of their own and only need the averaging done.
//
// What this file does about it.  The incidence table k_nodal reads is rebuilt on the device, per call, in ONE file-scope
// `static __device__` array of fixed size, so the entry point calls no cudaMalloc, no cudaFree and no library routine
// that allocates.  The price: a size limit (DGSWEM_STATIC_MAX_ELEM elements, DGSWEM_STATIC_MAX_NODES nodes), 20 MiB
// of device memory held by every GPU that loads libdgswem.so until the process exits, and one shared array: two calls
// that overlap on the same GPU (different streams, different host threads) race on it.
//
// The table is built without atomics (the library has none, tests/test_abi.py): the 3 n_elem (node, element, vertex)
// triples are sorted as 64-bit keys by a bitonic network, which leaves every node's incident elements contiguous and in
// ascending element id -- the summation order of k_nodal -- so the result has the same bits as dgswem_get_nodal on a
// binary64 handle.
#include "dgswem.h"

#include <mutex>
#include <string>

#include <cuda_runtime.h>

namespace {

constexpr long long kMaxElem = DGSWEM_STATIC_MAX_ELEM;
constexpr long long kMaxNodes = DGSWEM_STATIC_MAX_NODES;
constexpr long long kMaxKeys = 1LL << 21;   // 3 * kMaxElem = 1,572,864 triples, padded to the next power of two
static_assert(3 * kMaxElem <= kMaxKeys, "key array too small for DGSWEM_STATIC_MAX_ELEM");
constexpr int kLocal = 2048;                // keys one CTA sorts / merges in shared memory
constexpr unsigned long long kPad = ~0ULL;  // padding key: sorts behind every real triple

// The scratch.  Layout: kMaxKeys 64-bit keys (node << 32 | element * 4 + local vertex), then first[kMaxNodes] and
// last[kMaxNodes] (int32: each node's slice [first, last) of the sorted keys).  16 MiB + 2 MiB + 2 MiB.
// In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device address and must never be
// passed to a kernel; device code may use it directly, but the kernels below take the resolved pointer as an argument
// so that they read like every other kernel of the library.
constexpr size_t kScratchBytes = (size_t)kMaxKeys * 8 + (size_t)kMaxNodes * 4 * 2;
static_assert(kScratchBytes == DGSWEM_STATIC_SCRATCH_BYTES, "include/dgswem.h states the scratch size");
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_scratch_addr[kMaxDevices];   // device address of g_static_scratch on each device; nullptr = not resolved yet
thread_local std::string g_err;

int fail(int code, const std::string& msg) { g_err = msg; return code; }
int cuda_fail(cudaError_t e, const char* what) {
  g_err = std::string(what) + ": " + cudaGetErrorString(e);
  return DGSWEM_E_CUDA;
}

// Values of the Dubiner modes 00,01,10, 02,11,20, 03,12,21,30 (eq. (4)) at the three vertices of the
// reference triangle.  At a vertex the collapsed coordinates are (a, s, xi_2) = (-1, 1, -1), (1, 1, -1), (0, 0, 1), and
// phi_ij = A_i(a, s) B_j(xi_2) with A = 1, a, (3a^2 - s^2)/2, (5a^3 - 3 a s^2)/2 and the Jacobi factors
// B^(1) = 1, (3y+1)/2, (5y^2+2y-1)/2, (35y^3+15y^2-15y-3)/8; B^(3) = 1, (5y+3)/2, (21y^2+18y+1)/4; B^(5) = 1, (7y+5)/2:
// all small integers, exact in binary64.
struct VertexBasis { double v[3][10]; };
const VertexBasis kPhiV = {{{1, -1, -1, 1, 1, 1, -1, -1, -1, -1},
                            {1, -1, 1, 1, -1, 1, -1, 1, -1, 1},
                            {1, 2, 0, 3, 0, 0, 4, 0, 0, 0}}};

__device__ __forceinline__ void cmpswap(unsigned long long& a, unsigned long long& b, bool ascending) {
  if ((a > b) == ascending) { const unsigned long long t = a; a = b; b = t; }
}

// keys[i] for i < n_pad: the triple of (element i / 3, vertex i % 3), or the padding key behind the last triple and for a
// node id outside [0, nn) (such an entry is left out of every average; it cannot be reported without a
// synchronisation).  Also clears first / last, which must start at zero: a node that no element touches keeps the
// empty slice [0, 0) and gets the value 0, as in dgswem_get_nodal.
__global__ void __launch_bounds__(256) ks_fill(unsigned long long* __restrict__ keys, int* __restrict__ first, int* __restrict__ last,
                                               const int32_t* __restrict__ tri, long long ne, long long nn, long long n_pad) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < nn) { first[i] = 0; last[i] = 0; }
  if (i >= n_pad) return;
  unsigned long long key = kPad;
  if (i < 3 * ne) {
    const int node = tri[i];
    const long long e = i / 3;
    const int v = (int)(i - 3 * e);
    if (node >= 0 && node < nn) key = ((unsigned long long)(unsigned)node << 32) | (unsigned long long)(e * 4 + v);
  }
  keys[i] = key;
}

// bitonic network, stages k = 2 .. kLocal entirely inside one CTA's kLocal keys (direction from the GLOBAL index)
__global__ void __launch_bounds__(kLocal / 2) ks_sort_local(unsigned long long* __restrict__ keys) {
  __shared__ unsigned long long s[kLocal];
  const long long base = (long long)blockIdx.x * kLocal;
  const int t = threadIdx.x;
  s[t] = keys[base + t];
  s[t + kLocal / 2] = keys[base + t + kLocal / 2];
  __syncthreads();
  for (int k = 2; k <= kLocal; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      const int i = 2 * t - (t & (j - 1));
      cmpswap(s[i], s[i + j], ((base + i) & k) == 0);
      __syncthreads();
    }
  }
  keys[base + t] = s[t];
  keys[base + t + kLocal / 2] = s[t + kLocal / 2];
}

// one compare-exchange pass of stage k at distance j >= kLocal, in global memory
__global__ void __launch_bounds__(256) ks_merge_global(unsigned long long* __restrict__ keys, long long j, long long k, long long n_half) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_half) return;
  const long long i = 2 * t - (t & (j - 1));
  unsigned long long a = keys[i], b = keys[i + j];
  if ((a > b) == ((i & k) == 0)) { keys[i] = b; keys[i + j] = a; }
}

// the passes j = kLocal / 2 .. 1 of stage k > kLocal, inside one CTA's kLocal keys
__global__ void __launch_bounds__(kLocal / 2) ks_merge_local(unsigned long long* __restrict__ keys, long long k) {
  __shared__ unsigned long long s[kLocal];
  const long long base = (long long)blockIdx.x * kLocal;
  const int t = threadIdx.x;
  s[t] = keys[base + t];
  s[t + kLocal / 2] = keys[base + t + kLocal / 2];
  __syncthreads();
  const bool ascending = (base & k) == 0;   // k > kLocal: one direction for the whole CTA
  for (int j = kLocal / 2; j > 0; j >>= 1) {
    const int i = 2 * t - (t & (j - 1));
    cmpswap(s[i], s[i + j], ascending);
    __syncthreads();
  }
  keys[base + t] = s[t];
  keys[base + t + kLocal / 2] = s[t + kLocal / 2];
}

// slice [first, last) of the sorted keys per node; every slot has exactly one writer
__global__ void __launch_bounds__(256) ks_bounds(const unsigned long long* __restrict__ keys, int* __restrict__ first, int* __restrict__ last,
                                                 long long n_pad) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_pad) return;
  const unsigned long long key = keys[i];
  if (key == kPad) return;
  const unsigned node = (unsigned)(key >> 32);
  if (i == 0 || (unsigned)(keys[i - 1] >> 32) != node) first[node] = (int)i;
  if (i + 1 == n_pad || (unsigned)(keys[i + 1] >> 32) != node) last[node] = (int)(i + 1);
}

// k_nodal's arithmetic (dgswem_kernels.cuh) on the caller's [ndof][n_elem] binary64 arrays: per incident element, in
// ascending element id, the polynomial at the node (mode 0, then one fma per further mode), summed, divided by the count.
template <int ND>
__global__ void __launch_bounds__(256) ks_nodal(double* __restrict__ zn, double* __restrict__ qxn, double* __restrict__ qyn,
                                                const double* __restrict__ ze, const double* __restrict__ qx, const double* __restrict__ qy,
                                                const unsigned long long* __restrict__ keys, const int* __restrict__ first,
                                                const int* __restrict__ last, long long ne, long long nn, const VertexBasis B) {
  const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= nn) return;
  const int b = first[n], e1 = last[n];
  const double* w[3] = {ze, qx, qy};
  double s[3] = {0.0, 0.0, 0.0};
  for (int i = b; i < e1; ++i) {
    const unsigned ev = (unsigned)(keys[i] & 0xffffffffULL);
    const long long e = ev >> 2;
    const int v = ev & 3;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double val = w[c][e];
#pragma unroll
      for (int k = 1; k < ND; ++k) val = fma(w[c][(long long)k * ne + e], B.v[v][k], val);
      s[c] = s[c] + val;
    }
  }
  const int cnt = e1 - b;
  zn[n] = cnt > 0 ? s[0] / (double)cnt : 0.0;
  qxn[n] = cnt > 0 ? s[1] / (double)cnt : 0.0;
  qyn[n] = cnt > 0 ? s[2] / (double)cnt : 0.0;
}

inline unsigned grid_for(long long n, int block) { return (unsigned)((n + block - 1) / block); }

}  // namespace

extern "C" {

const char* dgswem_nodal_static_error(void) { return g_err.c_str(); }

int dgswem_nodal_static(int device, void* stream, int p, int64_t n_nodes, int64_t n_elem, const int32_t* tri,
                        const double* ze, const double* qx, const double* qy, double* zn, double* qxn, double* qyn) {
  if (p < 1 || p > 3) return fail(DGSWEM_E_ARG, "p must be 1, 2 or 3");
  if (n_elem < 1 || n_nodes < 1) return fail(DGSWEM_E_ARG, "need n_elem >= 1 and n_nodes >= 1");
  if (n_elem > kMaxElem)
    return fail(DGSWEM_E_ARG, "n_elem = " + std::to_string((long long)n_elem) + " is beyond DGSWEM_STATIC_MAX_ELEM = " + std::to_string(kMaxElem) +
                                  ": the fixed scratch array of dgswem_nodal_static cannot hold this mesh (use dgswem_get_nodal on a handle)");
  if (n_nodes > kMaxNodes)
    return fail(DGSWEM_E_ARG, "n_nodes = " + std::to_string((long long)n_nodes) + " is beyond DGSWEM_STATIC_MAX_NODES = " + std::to_string(kMaxNodes) +
                                  ": the fixed scratch array of dgswem_nodal_static cannot hold this mesh (use dgswem_get_nodal on a handle)");
  if (!tri || !ze || !qx || !qy || !zn || !qxn || !qyn) return fail(DGSWEM_E_ARG, "NULL device pointer");
  if (device < 0 || device >= kMaxDevices) return fail(DGSWEM_E_ARG, "device ordinal must be in 0..63");

  cudaError_t e = cudaSetDevice(device);
  if (e != cudaSuccess) return cuda_fail(e, "cudaSetDevice");
  unsigned char* scratch = nullptr;
  {
    // Set-up, once per device, with that device current: ask the runtime where THIS device keeps the array.  The
    // symbol's name is a host-side stand-in; only the address returned here may be given to a kernel.  This may load
    // the module, so the first call on a device belongs before any stream capture.
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[device]) {
      void* ptr = nullptr;
      e = cudaGetSymbolAddress(&ptr, g_static_scratch);
      if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_static_scratch)");
      if (!ptr) return fail(DGSWEM_E_CUDA, "cudaGetSymbolAddress returned a null address");
      g_scratch_addr[device] = ptr;
    }
    scratch = static_cast<unsigned char*>(g_scratch_addr[device]);
  }
  unsigned long long* keys = reinterpret_cast<unsigned long long*>(scratch);
  int* first = reinterpret_cast<int*>(scratch + (size_t)kMaxKeys * 8);
  int* last = first + kMaxNodes;
  cudaStream_t st = static_cast<cudaStream_t>(stream);

  long long n_pad = kLocal;
  while (n_pad < 3 * (long long)n_elem) n_pad <<= 1;

#define CKS(name)                                                  \
  do {                                                             \
    const cudaError_t e_ = cudaGetLastError();                     \
    if (e_ != cudaSuccess) return cuda_fail(e_, name " launch");   \
  } while (0)
  ks_fill<<<grid_for(n_pad > n_nodes ? n_pad : n_nodes, 256), 256, 0, st>>>(keys, first, last, tri, n_elem, n_nodes, n_pad);
  CKS("ks_fill");
  ks_sort_local<<<(unsigned)(n_pad / kLocal), kLocal / 2, 0, st>>>(keys);
  CKS("ks_sort_local");
  for (long long k = 2 * kLocal; k <= n_pad; k <<= 1) {
    for (long long j = k >> 1; j >= kLocal; j >>= 1) {
      ks_merge_global<<<grid_for(n_pad / 2, 256), 256, 0, st>>>(keys, j, k, n_pad / 2);
      CKS("ks_merge_global");
    }
    ks_merge_local<<<(unsigned)(n_pad / kLocal), kLocal / 2, 0, st>>>(keys, k);
    CKS("ks_merge_local");
  }
  ks_bounds<<<grid_for(n_pad, 256), 256, 0, st>>>(keys, first, last, n_pad);
  CKS("ks_bounds");
  const unsigned g = grid_for(n_nodes, 256);
  if (p == 1) ks_nodal<3><<<g, 256, 0, st>>>(zn, qxn, qyn, ze, qx, qy, keys, first, last, n_elem, n_nodes, kPhiV);
  else if (p == 2) ks_nodal<6><<<g, 256, 0, st>>>(zn, qxn, qyn, ze, qx, qy, keys, first, last, n_elem, n_nodes, kPhiV);
  else ks_nodal<10><<<g, 256, 0, st>>>(zn, qxn, qyn, ze, qx, qy, keys, first, last, n_elem, n_nodes, kPhiV);
  CKS("ks_nodal");
#undef CKS
  return DGSWEM_OK;
}

}  // extern "C"
