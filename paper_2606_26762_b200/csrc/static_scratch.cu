// protokv_query_attention_static: Alg. 4 (Eq. 4) with the split-context partials of the fp32 SIMT
// attention kernel (query_kernels.cu) in a file-scope device array instead of the caller's workspace, for callers that may
// not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Nothing here, nor anything it
// calls, allocates: no cudaMalloc / cudaFree / cudaMallocAsync, no tensor-map encode, no stream or event creation.
//
// The array (kStaticPartBytes = 8 MiB) is part of the library's device image: every GPU that loads the library holds it
// until the process exits.  It is shared by every state and every call on that GPU and keeps the last call's contents.
// Nothing in it has to start at zero: the attention kernel rewrites every partial (acc[d], m, l) the merge of the same
// call reads -- the launcher below sizes the grid so that (rows x splits) partials are written and exactly those are read.
// Two calls that overlap on one GPU (different streams, or two states with different streams) race on the array; calls on
// one stream are ordered by the stream.
#include <mutex>

#include "common.cuh"

namespace pkv {

constexpr size_t kStaticPartFloats = (size_t)2 << 20;                 // 8 MiB of fp32 partials
static __device__ __align__(256) float g_static_part[kStaticPartFloats];

size_t static_scratch_bytes() { return kStaticPartFloats * sizeof(float); }

// In host code `g_static_part` is a host-side stand-in of the symbol, not a device address.  The address is resolved once
// per device, with that device current, and cached.
constexpr int kMaxDevices = 64;
static std::mutex g_static_mu;
static float* g_static_ptr[kMaxDevices];

static cudaError_t static_part_ptr(float** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[dev]) {
    float* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_static_part);
    if (e != cudaSuccess) return e;
    if (!p || (uintptr_t)p % 256) return cudaErrorInvalidSymbol;
    g_static_ptr[dev] = p;
  }
  *out = g_static_ptr[dev];
  return cudaSuccess;
}

// Returns the number of kernels launched (>= 2), -1 if the query does not fit the array (*need_bytes = what one split
// would take), -2 on a CUDA error while resolving the array (*cuda_err).
int launch_attention_static(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, int sm_count, cudaStream_t s,
                            size_t* need_bytes, cudaError_t* cuda_err) {
  const int R = A.n_q * D.group;
  const long long nb = (long long)D.NS * A.layer_count * D.Hkv;
  const size_t per_split = (size_t)nb * R * (D.d + 2);                // floats of one split's partials
  *need_bytes = per_split * sizeof(float);
  if (per_split == 0 || per_split > kStaticPartFloats) return -1;
  float* part = nullptr;
  *cuda_err = static_part_ptr(&part);
  if (*cuda_err != cudaSuccess) return -2;
  // splits of the context: enough CTAs for four per SM (what attention_simt_splits does for the configured n_q), at most
  // what the array holds
  const long long ctas = nb * ((R + 3) / 4);
  long long ns = (4LL * sm_count + ctas - 1) / ctas;
  const long long room = (long long)(kStaticPartFloats / per_split);
  if (ns > 64) ns = 64;
  if (ns > room) ns = room;
  if (ns < 1) ns = 1;
  Dev Vs = V;
  Vs.part = part;                                                     // the only difference from the workspace path
  AttnArgs As = A;
  As.nsplit = (int)ns;
  int nl = 0;
  if (H.flags & PROTOKV_ROPE) nl += launch_rope_tables(D, H, Vs, As, s);
  nl += launch_attention_simt(D, H, Vs, As, s);
  return nl;
}

}  // namespace pkv
