// Alg. 2 PrototypeMaintenance (Alg. 1 l.15), once per frame after the
// absorptions of the frame (frame-synchronous reading): aging -> pairwise merge -> recycling, one CTA per bank.
// Readings of what Alg. 2 leaves open: DESIGN.md readings 20, 24-27 (same as oracle/protokv_oracle.cpp Bank::maintain).
//
//   aging    n_k <- floor((1 - gamma) n_k) while t - tau_k > T_idle (fp64, like the definition reads)
//   merge    pairs i < j in lexicographic order, both with n >= 1: if |c_i - c_j| < eps_K and |p_i - p_j| < eps_V the
//            lower index absorbs the other (mass-weighted c, p, mu; n, H^K, H^V, n_res summed); later pairs (i, j') see
//            the UPDATED centres of i.  The K_max^2 pair scan of the definition is cut down exactly: a pair whose two
//            members have not changed since they were last compared cannot have become mergeable, so only pairs with a
//            member stamped for this pass are looked at (all pairs after create / import) -- stamped by this frame's
//            fill / update, or by the previous pass for what it changed after its own scan (survivors, recycled slots); a pair is dropped early on
//            |  |c_i| - |c_j|  | >= eps_K (norms come with the Eq. 1 records) and on the distance over the first 16
//            dimensions, both with a safety margin, and only the survivors get the full fp64 distances.  The (rare)
//            candidates are then processed in order by the whole CTA against the live state, with a rescan of the
//            survivor's row after each merge.
//   recycle  every slot emptied by decay or merging is re-initialised like a slot fill (Alg. 1 l.4) from the newest
//            near-window tokens: the r-th such slot, in slot order, takes token T-1-(r mod T) of the (r/T)-th newest
//            frame.  Never-used slots stay free for Alg. 1 l.3-4, so the active set remains the prefix [0, n_used).
#include "common.cuh"
#include "derived.cuh"

namespace pkv {

constexpr int kMtThreads = 256, kMtWarps = kMtThreads / 32;
constexpr int kMtMaxCand = 2048;

struct MtSmemLayout {   // dynamic shared memory, sizes depend on K
  float* norm;                 // [K]  |c_k|
  uint32_t* alive;             // [K/32 + 1] n_k >= 1
  uint32_t* chgbits;           // [K/32 + 1] c_k / p_k changed this frame
  uint16_t* list;              // [K] changed list, later the list of emptied slots
  unsigned long long* cand;    // [kMtMaxCand] (i << 32 | j)
};
// The first four coordinates of every key centre are kept in shared memory as a second exact-safe filter of the pair
// scan (a partial squared distance never exceeds the full one) while the bank is small enough for them to fit.
constexpr int kMtC4MaxK = 8192;
__host__ __device__ inline size_t mt_smem_bytes(int K) {
  const size_t words = (size_t)K / 32 + 1;
  return align_up((size_t)K * 4 + 2 * words * 4 + (size_t)K * 2, 16) + (size_t)kMtMaxCand * 8 +
         (K <= kMtC4MaxK ? (size_t)K * 16 : 0);
}

__device__ __forceinline__ bool mt_bit(const uint32_t* bits, int k) { return (bits[k >> 5] >> (k & 31)) & 1u; }

// Exact squared distances of Alg. 2 l.7 for one pair, by one thread, in the oracle's order (fp64, dims ascending).
__device__ __forceinline__ bool mt_pair_exact(const float* __restrict__ ci, const float* __restrict__ cj,
                                              const float* __restrict__ pi, const float* __restrict__ pj, int d,
                                              double ek2, double ev2) {
  double dk = 0.0;
  for (int e = 0; e < d; ++e) {
    const double a = (double)ci[e] - (double)cj[e];
    dk = __dadd_rn(dk, __dmul_rn(a, a));
  }
  if (!(dk < ek2)) return false;
  double dv = 0.0;
  for (int e = 0; e < d; ++e) {
    const double a = (double)pi[e] - (double)pj[e];
    dv = __dadd_rn(dv, __dmul_rn(a, a));
  }
  return dv < ev2;
}

// Cheap exact-safe rejections (margins cover fp32 rounding of the norms and of the partial sum).
__device__ __forceinline__ bool mt_maybe_close(const float* __restrict__ ci16, const float* __restrict__ cj, float ni,
                                               float nj, float eps_k, int d) {
  if (fabsf(ni - nj) > eps_k * 1.001f + 1e-4f * fmaxf(ni, nj)) return false;   // | |a| - |b| | <= |a - b|
  float s = 0.f;
  const int m = d < 16 ? d : 16;
  for (int e = 0; e < m; ++e) { const float a = ci16[e] - cj[e]; s = fmaf(a, a, s); }
  return s <= eps_k * eps_k * 1.001f;
}

struct MaintArgs {
  int t;          // stream time of this step
  int n_used;     // slots initialised so far (= active prefix)
  int slot;       // ring slot of the newest frame
  int held;       // frames in the near window
  int full;       // 1: treat every prototype as changed (first call, after an import)
  int epoch;      // synthesis epoch to stamp
  float gamma, eps_k, eps_v;
  int t_idle;
};

template <typename T>
__global__ void __launch_bounds__(kMtThreads) maintenance_kernel(Dims D, Hyper H, Dev V, MaintArgs A) {
  extern __shared__ __align__(16) unsigned char mt_smem[];
  const int K = D.K, d = D.d, words = K / 32 + 1;
  float* norm_s = reinterpret_cast<float*>(mt_smem);
  uint32_t* alive = reinterpret_cast<uint32_t*>(norm_s + K);
  uint32_t* chgbits = alive + words;
  uint16_t* list = reinterpret_cast<uint16_t*>(chgbits + words);
  unsigned long long* cand = reinterpret_cast<unsigned long long*>(mt_smem + align_up((size_t)K * 4 + 2 * (size_t)words * 4 + (size_t)K * 2, 16));
  float4* c4 = K <= kMtC4MaxK ? reinterpret_cast<float4*>(cand + kMtMaxCand) : nullptr;
  __shared__ int nlist, ncand, nsurv;
  __shared__ unsigned long long cur_key, min_key;
  __shared__ double red[2][kMtWarps];
  __shared__ int pass_flag;
  __shared__ uint16_t surv[256];

  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const size_t pk0 = (size_t)b * K;
  const int nu = A.n_used;
  if (tid == 0) { nlist = 0; ncand = 0; nsurv = 0; cur_key = 0ull; }
  for (int w = tid; w < words; w += kMtThreads) { alive[w] = 0u; chgbits[w] = 0u; }
  __syncthreads();

  // ---- aging (l.1-5), alive / changed bitmaps, norms ----
  for (int k0 = 0; k0 < nu; k0 += kMtThreads) {
    const int k = k0 + tid;
    bool al = false, ch = false;
    if (k < nu) {
      const size_t pk = pk0 + k;
      int n = V.n[pk];
      if ((long long)A.t - (long long)V.tau[pk] > (long long)A.t_idle && n > 0) {
        const int nn = (int)floor(__dmul_rn(__dsub_rn(1.0, (double)A.gamma), (double)n));
        if (nn != n) {
          atomicAdd(V.mcount + 0, (unsigned long long)(n - nn));
          V.n[pk] = nn;
          V.logn[pk] = log_mass(nn);
          n = nn;
        }
      }
      al = n >= 1;
      ch = A.full || V.mstamp[pk] == A.t;   // touched by this frame's fill / update, or left changed by the previous pass
      const float invc = reinterpret_cast<const float*>(V.rec)[rec_slot(pk, 6)];
      norm_s[k] = invc > 0.f ? 1.f / invc : 0.f;
      if (c4) c4[k] = *reinterpret_cast<const float4*>(V.c + pk * d);
    }
    const uint32_t ba = __ballot_sync(0xffffffffu, al), bc = __ballot_sync(0xffffffffu, ch && al);
    if (lane == 0 && (k0 >> 5) + warp < words) {
      alive[(k0 >> 5) + warp] = ba;
      chgbits[(k0 >> 5) + warp] = bc;
      if (bc) {
        const int off = atomicAdd(&nlist, __popc(bc));
        uint32_t m = bc;
        int o = off;
        while (m) { const int bit = __ffs(m) - 1; m &= m - 1; list[o++] = (uint16_t)(k0 + warp * 32 + bit); }
      }
    }
  }
  __syncthreads();

  // ---- merge candidates from the pre-merge state: pairs with a changed member ----
  const double ek2 = __dmul_rn((double)A.eps_k, (double)A.eps_k), ev2 = __dmul_rn((double)A.eps_v, (double)A.eps_v);
  const int nch = nlist;
  if (A.eps_k > 0.f && A.eps_v > 0.f) {
    for (int ci = warp; ci < nch; ci += kMtWarps) {
      const int a = (int)list[ci];
      const float* ca = V.c + (pk0 + a) * d;
      float ca16[16];
#pragma unroll
      for (int e = 0; e < 16; ++e) ca16[e] = e < d ? ca[e] : 0.f;
      const float na = norm_s[a];
      for (int b0 = 0; b0 < nu; b0 += 32) {
        const int bb = b0 + lane;
        if (bb >= nu || bb == a) continue;
        if (c4) {   // first four coordinates from shared memory, tested first: almost every pair of different clusters ends here
          const float4 q = c4[bb];
          const float e0 = ca16[0] - q.x, e1 = ca16[1] - q.y, e2 = ca16[2] - q.z, e3 = ca16[3] - q.w;
          if (fmaf(e0, e0, fmaf(e1, e1, fmaf(e2, e2, e3 * e3))) > A.eps_k * A.eps_k * 1.001f) continue;
        }
        if (!mt_bit(alive, bb)) continue;
        if (mt_bit(chgbits, bb) && bb < a) continue;          // both changed: the pair is taken from its lower member
        const float* cb = V.c + (pk0 + bb) * d;
        if (!mt_maybe_close(ca16, cb, na, norm_s[bb], A.eps_k, d)) continue;
        const int i = a < bb ? a : bb, j = a < bb ? bb : a;
        if (mt_pair_exact(V.c + (pk0 + i) * d, V.c + (pk0 + j) * d, V.p + (pk0 + i) * d, V.p + (pk0 + j) * d, d, ek2, ev2)) {
          const int o = atomicAdd(&ncand, 1);
          if (o < kMtMaxCand) cand[o] = ((unsigned long long)i << 32) | (unsigned)j;
          else atomicOr(V.err, PKV_ERR_MAINT_OVERFLOW);
        }
      }
    }
  }
  __syncthreads();

  // ---- merge (l.6-13): candidates in lexicographic order against the live state ----
  const int GC2 = 2 * D.G * D.C;
  while (true) {
    if (tid == 0) min_key = ~0ull;
    __syncthreads();
    const int nc = ncand < kMtMaxCand ? ncand : kMtMaxCand;
    unsigned long long mine = ~0ull;
    for (int e = tid; e < nc; e += kMtThreads) { const unsigned long long c = cand[e]; if (c > cur_key && c < mine) mine = c; }
    if (mine != ~0ull) atomicMin(&min_key, mine);
    __syncthreads();
    const unsigned long long key = min_key;
    if (key == ~0ull) break;
    const int i = (int)(key >> 32), j = (int)(uint32_t)key;
    const size_t pi = pk0 + i, pj = pk0 + j;
    bool go = mt_bit(alive, i) && mt_bit(alive, j);
    if (go) {   // the decision against the current centres (CTA-parallel fp64 sums)
      double dk = 0.0, dv = 0.0;
      for (int e = tid; e < d; e += kMtThreads) {
        const double a = (double)V.c[pi * d + e] - (double)V.c[pj * d + e], q = (double)V.p[pi * d + e] - (double)V.p[pj * d + e];
        dk += a * a; dv += q * q;
      }
      for (int o = 16; o > 0; o >>= 1) { dk += __shfl_xor_sync(0xffffffffu, dk, o); dv += __shfl_xor_sync(0xffffffffu, dv, o); }
      if (lane == 0) { red[0][warp] = dk; red[1][warp] = dv; }
      __syncthreads();
      if (tid == 0) {
        double sk = 0.0, sv = 0.0;
        for (int w = 0; w < kMtWarps; ++w) { sk += red[0][w]; sv += red[1][w]; }
        pass_flag = (sk < ek2 && sv < ev2) ? 1 : 0;
      }
      __syncthreads();
      go = pass_flag != 0;
    }
    if (go) {
      const double ni = (double)V.n[pi], nj = (double)V.n[pj], w = ni + nj;
      for (int e = tid; e < d; e += kMtThreads) {
        V.c[pi * d + e] = (float)__ddiv_rn(__dadd_rn(__dmul_rn(ni, (double)V.c[pi * d + e]), __dmul_rn(nj, (double)V.c[pj * d + e])), w);
        V.p[pi * d + e] = (float)__ddiv_rn(__dadd_rn(__dmul_rn(ni, (double)V.p[pi * d + e]), __dmul_rn(nj, (double)V.p[pj * d + e])), w);
      }
      if (tid < 2)
        V.mu[pi * 2 + tid] = (float)__ddiv_rn(__dadd_rn(__dmul_rn(ni, (double)V.mu[pi * 2 + tid]), __dmul_rn(nj, (double)V.mu[pj * 2 + tid])), w);
      for (int e = tid; e < GC2; e += kMtThreads) V.hist[pi * GC2 + e] += V.hist[pj * GC2 + e];
      __syncthreads();
      if (tid == 0) {
        V.n[pi] = (int)(ni + nj);
        V.nres[pi] += V.nres[pj];
        V.pos_first[pi] = V.pos_first[pi] < V.pos_first[pj] ? V.pos_first[pi] : V.pos_first[pj];   // reading 30
        V.pos_sum[pi] += V.pos_sum[pj];
        V.pos_cnt[pi] += V.pos_cnt[pj];
        V.n[pj] = 0;
        alive[j >> 5] &= ~(1u << (j & 31));
        atomicAdd(V.mcount + 1, 1ull);
        bool seen = false;
        for (int s = 0; s < nsurv; ++s) seen = seen || surv[s] == (uint16_t)i;
        if (!seen) {
          if (nsurv < 256) surv[nsurv++] = (uint16_t)i;
          else atomicOr(V.err, PKV_ERR_MAINT_OVERFLOW);
        }
      }
      // new norm of the survivor, then its row is rescanned for partners beyond j
      double cc = 0.0;
      for (int e = tid; e < d; e += kMtThreads) { const double x = (double)V.c[pi * d + e]; cc += x * x; }
      for (int o = 16; o > 0; o >>= 1) cc += __shfl_xor_sync(0xffffffffu, cc, o);
      if (lane == 0) red[0][warp] = cc;
      __syncthreads();
      if (tid == 0) {
        double s = 0.0;
        for (int w2 = 0; w2 < kMtWarps; ++w2) s += red[0][w2];
        norm_s[i] = (float)sqrt(s);
      }
      __syncthreads();
      const float* ci = V.c + pi * d;
      float ci16[16];
#pragma unroll
      for (int e = 0; e < 16; ++e) ci16[e] = e < d ? ci[e] : 0.f;
      const float nin = norm_s[i];
      for (int jj = j + 1 + tid; jj < nu; jj += kMtThreads) {
        if (!mt_bit(alive, jj)) continue;
        if (!mt_maybe_close(ci16, V.c + (pk0 + jj) * d, nin, norm_s[jj], A.eps_k, d)) continue;
        if (mt_pair_exact(ci, V.c + (pk0 + jj) * d, V.p + pi * d, V.p + (pk0 + jj) * d, d, ek2, ev2)) {
          const int o = atomicAdd(&ncand, 1);
          if (o < kMtMaxCand) cand[o] = ((unsigned long long)i << 32) | (unsigned)jj;
          else atomicOr(V.err, PKV_ERR_MAINT_OVERFLOW);
        }
      }
    }
    __syncthreads();
    if (tid == 0) cur_key = key;
    __syncthreads();
  }

  // ---- derived data of the merge survivors (centres, mass, histograms changed) ----
  const int st = b / (D.L * D.Hkv);
  const int vec = d / 32;
  for (int s = warp; s < nsurv; s += kMtWarps) {
    const int k = (int)surv[s];
    const size_t pk = pk0 + k;
    float cc = 0.f;
    for (int v = 0; v < vec; ++v) { const float x = V.c[pk * d + lane * vec + v]; cc = fmaf(x, x, cc); }
    cc = warp_sum(cc);
    if (V.c_bf)
      for (int e = lane; e < d; e += 32) {
        V.c_bf[pk * d + e] = __float2bfloat16_rn(V.c[pk * d + e]);
        V.p_bf[pk * d + e] = __float2bfloat16_rn(V.p[pk * d + e]);
      }
    if (V.c_hi) {
      const float invc = inv_norm(cc);
      for (int v = 0; v < vec; ++v) {
        const int e = lane * vec + v;
        __nv_bfloat16 hi, lo;
        split_bf16(V.c[pk * d + e] * invc, hi, lo);
        V.c_hi[pk * d + e] = hi; V.c_lo[pk * d + e] = lo;
      }
    }
    if (lane == 0) {
      store_rec(V.rec, pk, make_rec(cc, V.mu[pk * 2], V.mu[pk * 2 + 1], V.sigma[pk * 3], V.sigma[pk * 3 + 1],
                                    V.sigma[pk * 3 + 2], V.tau[pk], H));
      V.logn[pk] = log_mass(V.n[pk]);
      V.mstamp[pk] = A.t + 1;   // its pairs with lower-index rows are only looked at again by the next pass
      mark_dirty(D, V, b, k, A.epoch);
    }
  }
  __syncthreads();

  // ---- recycling (l.14-19): emptied slots in slot order ----
  if (tid == 0) {
    int r = 0;
    for (int w = 0; w < words; ++w) {
      const int base = w * 32;
      if (base >= nu) break;
      uint32_t m = ~alive[w];
      if (nu - base < 32) m &= (1u << (nu - base)) - 1u;
      while (m) { const int bit = __ffs(m) - 1; m &= m - 1; list[r++] = (uint16_t)(base + bit); }
    }
    nlist = r;
    if (r) atomicAdd(V.mcount + 2, (unsigned long long)r);
  }
  __syncthreads();
  const int nrec = nlist;
  const int ghc = 2 * D.G * D.C;
  for (int r = warp; r < nrec; r += kMtWarps) {
    const int k = (int)list[r];
    const size_t pk = pk0 + k;
    int back = r / D.T;
    if (back >= A.held) back = A.held - 1;
    const int j = D.T - 1 - (r % D.T);
    const int slot = ((A.slot - back) % D.Wf + D.Wf) % D.Wf;
    const T* Ke = (const T*)V.ringK + (((size_t)b * D.Wf + slot) * D.T + j) * d;
    const T* Ve = (const T*)V.ringV + (((size_t)b * D.Wf + slot) * D.T + j) * d;
    float cc = 0.f;
    for (int v = 0; v < vec; ++v) {
      const int e = lane * vec + v;
      const float kf = to_f32(Ke[e]), vf = to_f32(Ve[e]);
      V.c[pk * d + e] = kf;
      V.p[pk * d + e] = vf;
      if (V.c_bf) { V.c_bf[pk * d + e] = __float2bfloat16_rn(kf); V.p_bf[pk * d + e] = __float2bfloat16_rn(vf); }
      cc = fmaf(kf, kf, cc);
    }
    cc = warp_sum(cc);
    if (V.c_hi) {
      const float invc = inv_norm(cc);
      for (int v = 0; v < vec; ++v) {
        const int e = lane * vec + v;
        __nv_bfloat16 hi, lo;
        split_bf16(to_f32(Ke[e]) * invc, hi, lo);
        V.c_hi[pk * d + e] = hi; V.c_lo[pk * d + e] = lo;
      }
    }
    for (int e = lane; e < ghc; e += 32) V.hist[pk * ghc + e] = 0u;
    if (lane == 0) {
      const float* se = V.ringS + (((size_t)st * D.Wf + slot) * D.T + j) * 2;
      V.n[pk] = 1;
      V.mu[pk * 2] = se[0]; V.mu[pk * 2 + 1] = se[1];
      V.sigma[pk * 3] = 1.f; V.sigma[pk * 3 + 1] = 0.f; V.sigma[pk * 3 + 2] = 1.f;
      V.tau[pk] = A.t;
      const long long ps = H.pos0 + (long long)(A.t - back) * D.T + j;
      V.pos[pk] = ps; V.pos_first[pk] = ps; V.pos_sum[pk] = ps; V.pos_cnt[pk] = 1;
      V.nres[pk] = 0u;
      store_rec(V.rec, pk, make_rec(cc, se[0], se[1], 1.f, 0.f, 1.f, A.t, H));
      V.logn[pk] = 0.f;
      V.mstamp[pk] = A.t + 1;   // re-initialised after this pass's merge scan: compared by the next pass
      mark_dirty(D, V, b, k, A.epoch);
    }
  }
}

bool maintenance_prepare() {
  const int bytes = (int)mt_smem_bytes(kMaxKmax);
  bool ok = cudaFuncSetAttribute(maintenance_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess;
  ok = ok && cudaFuncSetAttribute(maintenance_kernel<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess;
  if (!ok) cudaGetLastError();
  return ok;
}

int launch_maintenance(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, int held, int full, float gamma,
                       float eps_k, float eps_v, cudaStream_t s) {
  if (F.n_act <= 0) return 0;
  MaintArgs A{};
  A.t = F.t; A.n_used = F.n_act; A.slot = F.slot; A.held = held; A.full = full; A.epoch = F.epoch;
  A.gamma = gamma; A.eps_k = eps_k; A.eps_v = eps_v; A.t_idle = H.t_idle;
  const size_t sm = mt_smem_bytes(D.K);
  if (D.bf16) maintenance_kernel<__nv_bfloat16><<<D.B, kMtThreads, sm, s>>>(D, H, V, A);
  else maintenance_kernel<float><<<D.B, kMtThreads, sm, s>>>(D, H, V, A);
  return 1;
}

}  // namespace pkv
