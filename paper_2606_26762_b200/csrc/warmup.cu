// PQ codebook warm-up ("initialized via mini-batch k-means on a warm-up reservoir of residuals collected
// during the first T_warm streaming steps, run separately for each subspace and for key/value"; L478: T_warm is an
// implementation constant the paper does not print).  DESIGN.md readings 32-36.
//
//   reservoir_plan_kernel  per warm-up frame: which reservoir slot the residual of each absorbed token goes to.
//                          Algorithm R on the bank's running residual index i: slot i while i < R, else slot
//                          u = draw mod (i + 1) if u < R.  Two tokens of one frame may draw the same slot; the later
//                          one (larger i) must win, whatever order the update kernel's warps run in: every token posts
//                          i + 1 to a per-slot claim word with atomicMax, and keeps the slot only if its own value is
//                          what the word holds afterwards.  The update kernels then store r^K, r^V rows at those slots.
//   kmeans_kernel          CTA = (subspace, side, bank).  Sculley's mini-batch k-means: centres start at rows
//                          floor(z n / C); per iteration km_batch rows are drawn with replacement (same rows for every
//                          subspace and side), assigned with the centres frozen (thread = sample), then applied in
//                          batch order with rate 1 / v_z (thread = (centre, dim): the updates of different centres and
//                          dimensions are independent, so walking the batch in order per thread IS the sequential order).
// Both decisions (nearest centre) and updates are fp32, one rounding per operation, no fused multiply-add, in the order
// reading 35 states, so the codebooks are reproducible bit for bit from the reservoir.
#include "common.cuh"

namespace pkv {

__device__ __forceinline__ unsigned long long wu_mix64(unsigned long long x) {   // SplitMix64 output function
  unsigned long long z = x + 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
__device__ __forceinline__ unsigned long long wu_draw(unsigned long long seed, unsigned long long stream,
                                                      unsigned long long counter) {
  return wu_mix64(seed ^ wu_mix64(2ull * counter + stream));
}

__global__ void __launch_bounds__(256) reservoir_plan_kernel(Dims D, Hyper H, Dev V, FrameArgs F,
                                                             unsigned long long* __restrict__ claim) {
  const int b = blockIdx.x, tid = threadIdx.x;
  const unsigned long long seed = H.km_seed + (unsigned long long)b;
  const long long R = H.warm_reservoir;
  const int ntok = D.T - F.n_fill;
  unsigned long long* cl = claim + (size_t)b * R;
  for (int j = tid; j < F.n_fill; j += 256) V.rslot[(size_t)b * D.T + j] = -1;   // slot fills leave no residual (reading 8)
  for (int jj = tid; jj < ntok; jj += 256) {
    const long long i = F.res_base + jj;
    long long slot = i;
    if (i >= R) {
      const unsigned long long u = wu_draw(seed, 0ull, (unsigned long long)i) % (unsigned long long)(i + 1);
      slot = u < (unsigned long long)R ? (long long)u : -1;
    }
    if (slot >= 0) atomicMax(cl + slot, (unsigned long long)(i + 1));
  }
  __threadfence();
  __syncthreads();
  for (int jj = tid; jj < ntok; jj += 256) {
    const long long i = F.res_base + jj;
    long long slot = i;
    if (i >= R) {
      const unsigned long long u = wu_draw(seed, 0ull, (unsigned long long)i) % (unsigned long long)(i + 1);
      slot = u < (unsigned long long)R ? (long long)u : -1;
    }
    int out = -1;
    if (slot >= 0 && __ldcg(cl + slot) == (unsigned long long)(i + 1)) out = (int)slot;
    V.rslot[(size_t)b * D.T + F.n_fill + jj] = out;
  }
}

int launch_reservoir_plan(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, cudaStream_t s) {
  if (D.T - F.n_fill <= 0) return 0;
  // the claim words live behind the reservoirs (see carve()): [B][R] u64
  unsigned long long* claim = reinterpret_cast<unsigned long long*>(V.resV + (size_t)D.B * H.warm_reservoir * D.d);
  reservoir_plan_kernel<<<D.B, 256, 0, s>>>(D, H, V, F, claim);
  return 1;
}

constexpr int kKmThreads = 256;

__global__ void __launch_bounds__(kKmThreads) kmeans_kernel(Dims D, Hyper H, Dev V, float* __restrict__ cbk,
                                                            float* __restrict__ cbv, long long fill) {
  extern __shared__ __align__(16) unsigned char km_smem[];
  const int g = blockIdx.x, side = blockIdx.y, b = blockIdx.z, tid = threadIdx.x;
  const int sub = D.sub, Cn = D.C, nel = Cn * sub, batch = H.km_batch;
  float* cen = reinterpret_cast<float*>(km_smem);                    // [C][sub]
  int* cnt = reinterpret_cast<int*>(cen + nel);                     // [C]
  int* cnt2 = cnt + Cn;                                             // [C] counts after this iteration
  int* asg = cnt2 + Cn;                                             // [batch]
  int* rows = asg + batch;                                          // [batch]
  const float* X = (side ? V.resV : V.resK) + (size_t)b * H.warm_reservoir * D.d + (size_t)g * sub;
  const unsigned long long seed = H.km_seed + (unsigned long long)b;
  for (int e = tid; e < nel; e += kKmThreads) {
    const int z = e / sub, m = e - z * sub;
    const long long row = (long long)z * fill / Cn;
    cen[e] = X[(size_t)row * D.d + m];
  }
  for (int z = tid; z < Cn; z += kKmThreads) cnt[z] = 0;
  __syncthreads();
  for (int it = 0; it < H.km_iters; ++it) {
    for (int q = tid; q < batch; q += kKmThreads) {                 // assignment, centres frozen
      const int row = (int)(wu_draw(seed, 1ull, (unsigned long long)it * (unsigned long long)batch + (unsigned long long)q) %
                            (unsigned long long)fill);
      const float* x = X + (size_t)row * D.d;
      int zb = 0;
      float db = INFINITY;
      for (int z = 0; z < Cn; ++z) {
        float acc = 0.f;
        for (int m = 0; m < sub; ++m) {
          const float t = __fsub_rn(x[m], cen[z * sub + m]);
          acc = __fadd_rn(acc, __fmul_rn(t, t));
        }
        if (acc < db) { db = acc; zb = z; }                         // lowest index on ties
      }
      asg[q] = zb;
      rows[q] = row;
    }
    __syncthreads();
    for (int e = tid; e < nel; e += kKmThreads) {                   // updates, in batch order per (centre, dim)
      const int z = e / sub, m = e - z * sub;
      float c = cen[e];
      int v = cnt[z];
      for (int q = 0; q < batch; ++q) {
        if (asg[q] != z) continue;
        v += 1;
        const float eta = __fdiv_rn(1.0f, (float)v);
        const float keep = __fsub_rn(1.0f, eta);
        const float x = X[(size_t)rows[q] * D.d + m];
        c = __fadd_rn(__fmul_rn(keep, c), __fmul_rn(eta, x));
      }
      cen[e] = c;                                                   // nobody else reads cen[e] in this phase
      if (m == 0) cnt2[z] = v;
    }
    __syncthreads();
    for (int z = tid; z < Cn; z += kKmThreads) cnt[z] = cnt2[z];
    __syncthreads();
  }
  float* out = (side ? cbv : cbk) + ((size_t)b * D.G + g) * nel;
  for (int e = tid; e < nel; e += kKmThreads) out[e] = cen[e];
}

static size_t kmeans_smem(const Dims& D, const Hyper& H) {
  return (size_t)D.C * D.sub * 4 + 2 * (size_t)D.C * 4 + 2 * (size_t)H.km_batch * 4;
}

bool warmup_prepare(const Dims& D, const Hyper& H) { return kmeans_smem(D, H) <= 48 * 1024; }

int launch_kmeans(const Dims& D, const Hyper& H, const Dev& V, float* cbk, float* cbv, long long fill, cudaStream_t s) {
  dim3 grid(D.G, 2, D.B);
  kmeans_kernel<<<grid, kKmThreads, kmeans_smem(D, H), s>>>(D, H, V, cbk, cbv, fill);
  return 1;
}

}  // namespace pkv
