// D.3 dynamic pseudo-token allocation: S_k = S_tot Var(H_k) / sum_j Var(H_j) with the total fixed
// at S_tot = K_max S (L_context unchanged, L616), and the synthesis of a ragged number of modes per prototype.
// DESIGN.md readings 37-40.  Only with PROTOKV_VAR_ALLOC; the fixed-S path does not pass through this file.
//
//   allocation_kernel     CTA = bank.  (1) thread = prototype: Var(H_k) = total variance of the codewords its histograms
//                         count, both sides, in fp64 with every operation rounded separately in the order of reading 37,
//                         fixed to v_k = floor(Var 2^20 + 1/2); (2) integer shares: one each, the rest of the budget by
//                         floor(bud v_k / sum v), capped at s_cap; (3) what is left goes one unit at a time, round after
//                         round, to the prototypes below the cap in (remainder descending, index ascending) order -- whole
//                         rounds are plain increments, the last partial round ranks the eligible prototypes by counting;
//                         (4) exclusive prefix sum of S_k = row offsets of the bank's codes, kind[] of every slot.
//   synthesis_var_kernel  warp = (prototype, side): Alg. 3 with beam width S_k -- under the total
//                         order of reading 13 and additive scores a beam of width >= S_k returns exactly the global top
//                         S_k, the same tuples the width-B beam returns.  Lane i holds beam entry i; the candidates of a
//                         lane (its entry + the subspace's codes in (cost, code) order) form a sorted run, and the S_k
//                         smallest of the runs are taken by repeated warp-wide minima.
#include "common.cuh"

namespace pkv {

constexpr int kAlThreads = 256;

__global__ void __launch_bounds__(kAlThreads) allocation_kernel(Dims D, Hyper H, Dev V, int n_act) {
  extern __shared__ __align__(16) unsigned char al_smem[];
  float* cbk_s = reinterpret_cast<float*>(al_smem);                  // [G][C][sub]
  float* cbv_s = cbk_s + D.G * D.C * D.sub;
  __shared__ unsigned long long vsum_s, used_s;
  __shared__ int na_s, elig_s, wsum[kAlThreads / 32];
  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool has_cb = V.cbk != nullptr;
  const int K = D.K, ncb = D.G * D.C * D.sub;
  int* Sk = V.scount + (size_t)b * K;
  long long* vfx = V.varfx + (size_t)b * K;
  long long* rem = V.varfx + (size_t)D.B * K + (size_t)b * K;         // second half of the array: remainders
  if (has_cb)
    for (int e = tid; e < ncb; e += kAlThreads) { cbk_s[e] = V.cbk[(size_t)b * ncb + e]; cbv_s[e] = V.cbv[(size_t)b * ncb + e]; }
  if (tid == 0) { vsum_s = 0ull; used_s = 0ull; na_s = 0; }
  __syncthreads();
  // ---- (1) variances, kinds ----
  for (int k = tid; k < K; k += kAlThreads) {
    const size_t pk = (size_t)b * K + k;
    const bool present = k < n_act && V.n[pk] >= 1;
    const bool zero = !has_cb || V.nres[pk] == 0u;
    V.kind[pk] = present ? (zero ? 1 : 0) : 2;
    long long v = 0;
    if (present && !zero) {
      double total = 0.0;
      for (int kv = 0; kv < 2; ++kv) {
        const float* cb = kv ? cbv_s : cbk_s;
        for (int g = 0; g < D.G; ++g) {
          const uint32_t* h = V.hist + ((pk * 2 + kv) * D.G + g) * D.C;
          double tot = 0.0;
          for (int z = 0; z < D.C; ++z) tot = __dadd_rn(tot, (double)h[z]);
          if (tot == 0.0) continue;
          double dz[kMaxC];
#pragma unroll
          for (int z = 0; z < kMaxC; ++z) dz[z] = 0.0;
          for (int m = 0; m < D.sub; ++m) {
            double a = 0.0;
            for (int z = 0; z < D.C; ++z) a = __dadd_rn(a, __dmul_rn((double)h[z], (double)cb[(g * D.C + z) * D.sub + m]));
            const double mean = __ddiv_rn(a, tot);
#pragma unroll
            for (int z = 0; z < kMaxC; ++z) {
              if (z < D.C) {
                const double t = __dsub_rn((double)cb[(g * D.C + z) * D.sub + m], mean);
                dz[z] = __dadd_rn(dz[z], __dmul_rn(t, t));
              }
            }
          }
          double var = 0.0;
#pragma unroll
          for (int z = 0; z < kMaxC; ++z)
            if (z < D.C) var = __dadd_rn(var, __dmul_rn((double)h[z], dz[z]));
          total = __dadd_rn(total, __ddiv_rn(var, tot));
        }
      }
      v = (long long)floor(__dadd_rn(__dmul_rn(total, 1048576.0), 0.5));
    }
    vfx[k] = v;
    Sk[k] = present ? 1 : 0;
    if (present) { atomicAdd(&vsum_s, (unsigned long long)v); atomicAdd(&na_s, 1); }
  }
  __syncthreads();
  const long long vsum = (long long)vsum_s;
  const int na = na_s, cap = H.s_cap;
  const long long stot = (long long)K * D.S;
  // ---- (2) proportional shares ----
  if (na > 0) {
    if (vsum == 0) {
      const int s0 = D.S < cap ? D.S : cap;
      for (int k = tid; k < K; k += kAlThreads) if (Sk[k]) Sk[k] = s0;
    } else {
      const long long bud = stot - na;
      for (int k = tid; k < K; k += kAlThreads) {
        if (!Sk[k]) { rem[k] = -1; continue; }
        const long long prod = bud * vfx[k];
        const long long e = 1 + prod / vsum;
        const int s = (int)(e < cap ? e : cap);
        Sk[k] = s;
        rem[k] = prod % vsum;
        atomicAdd(&used_s, (unsigned long long)s);
      }
      __syncthreads();
      long long left = stot - (long long)used_s;
      // ---- (3) leftovers, round by round ----
      while (left > 0) {
        if (tid == 0) elig_s = 0;
        __syncthreads();
        int mine = 0;
        for (int k = tid; k < K; k += kAlThreads) mine += (Sk[k] > 0 && Sk[k] < cap) ? 1 : 0;
        if (mine) atomicAdd(&elig_s, mine);
        __syncthreads();
        const int elig = elig_s;
        __syncthreads();
        if (elig == 0) break;
        if (left >= elig) {
          for (int k = tid; k < K; k += kAlThreads) if (Sk[k] > 0 && Sk[k] < cap) Sk[k] += 1;
          left -= elig;
          __syncthreads();
        } else {   // the first `left` eligible prototypes in (remainder descending, index ascending) order
          int bump[kMaxKmax / kAlThreads];
          int cnt = 0;
          for (int k = tid; k < K; k += kAlThreads, ++cnt) {
            bump[cnt] = 0;
            if (!(Sk[k] > 0 && Sk[k] < cap)) continue;
            const long long rk = rem[k];
            long long rank = 0;
            for (int j = 0; j < K; ++j) {
              const int sj = Sk[j];
              if (!(sj > 0 && sj < cap)) continue;
              const long long rj = rem[j];
              rank += (rj > rk || (rj == rk && j < k)) ? 1 : 0;
            }
            bump[cnt] = rank < left ? 1 : 0;
          }
          __syncthreads();                                          // every rank was computed on the old counts
          cnt = 0;
          for (int k = tid; k < K; k += kAlThreads, ++cnt) if (bump[cnt]) Sk[k] += 1;
          left = 0;
          __syncthreads();
        }
      }
    }
  }
  __syncthreads();
  // ---- (4) exclusive prefix sum of S_k over the bank ----
  int* off = V.soff + (size_t)b * (K + 1);
  int base = 0;
  for (int k0 = 0; k0 < K; k0 += kAlThreads) {
    const int k = k0 + tid;
    const int s = k < K ? Sk[k] : 0;
    int incl = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    int woff = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < kAlThreads / 32; ++w) { const int c = wsum[w]; if (w < warp) woff += c; tot += c; }
    if (k < K) off[k] = base + woff + incl - s;
    base += tot;
    __syncthreads();
  }
  if (tid == 0) off[K] = base;
}

static size_t alloc_smem(const Dims& D) { return 2 * (size_t)D.G * D.C * D.sub * 4; }

bool alloc_prepare(const Dims& D) { return alloc_smem(D) <= 48 * 1024; }

int launch_allocation(const Dims& D, const Hyper& H, const Dev& V, int n_act, cudaStream_t s) {
  allocation_kernel<<<D.B, kAlThreads, alloc_smem(D), s>>>(D, H, V, n_act);
  return 1;
}

// ---------------------------------------------------------------------------------------------------------
// Ragged synthesis: warp = (prototype, side).  Keys as in query_kernels.cu: (cost << 32 | tuple), cost = -sum of the
// fixed-point log-probabilities (reading 13), tuple with z_1 in the most significant used nibble; smaller is better.
// ---------------------------------------------------------------------------------------------------------
constexpr int kSvWarps = 8;
typedef unsigned long long SvKey;
constexpr SvKey kSvNone = ~0ull;

__device__ __forceinline__ SvKey sv_min(SvKey a, SvKey b) { return a < b ? a : b; }

__global__ void __launch_bounds__(kSvWarps * 32) synthesis_var_kernel(Dims D, Hyper H, Dev V, int n_act) {
  __shared__ unsigned long long scost[kSvWarps][kMaxC];              // subspace codes in (cost, code) order: cost << 4 | z
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long task = (long long)blockIdx.x * kSvWarps + warp;
  const long long ntask = (long long)D.B * D.K * 2;
  if (task >= ntask) return;
  const int side = (int)(task & 1);
  const size_t pk = (size_t)(task >> 1);
  const int b = (int)(pk / D.K), k = (int)(pk % D.K);
  if (V.kind[pk] != 0) return;                                       // absent, or zero residuals: no tuples to decode
  const int W = V.scount[pk];                                        // beam width = modes wanted
  const int off = V.soff[(size_t)b * (D.K + 1) + k];
  const uint32_t* Hrow = V.hist + (pk * 2 + side) * D.G * D.C;
  SvKey beam = lane == 0 ? 0ull : kSvNone;
  int nbeam = 1;
  for (int g = 0; g < D.G; ++g) {
    // fixed-point costs of this subspace's codes, then their order by (cost, code)
    uint32_t h = 0u;
    if (lane < D.C) h = Hrow[g * D.C + lane];
    double tot = (double)h;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);   // integers below 2^53: exact in any order
    const double logden = log(tot + (double)D.C * H.pq_eps);
    unsigned long long ck = ~0ull;
    if (lane < D.C) {
      const double lognum = h < (uint32_t)PKV_SYN_LOGTAB ? V.logtab[h] : log((double)h + H.pq_eps);
      const long long q = -llround((lognum - logden) * 16777216.0);
      const unsigned long long c = (unsigned long long)(q < 0 ? 0 : (q < 0xfffffffell ? q : 0xfffffffell));
      ck = (c << 4) | (unsigned long long)lane;
    }
    int rank = 0;
#pragma unroll
    for (int j = 0; j < kMaxC; ++j) {
      const unsigned long long o = __shfl_sync(0xffffffffu, ck, j);
      rank += o < ck ? 1 : 0;
    }
    __syncwarp();
    if (lane < D.C) scost[warp][rank] = ck;
    __syncwarp();
    // S_k-way selection from the sorted runs (lane i: beam entry i + codes in order)
    int head = 0;
    SvKey out = kSvNone;
    const int want = W;
    int got = 0;
    for (; got < want; ++got) {
      SvKey cand = kSvNone;
      if (lane < nbeam && beam != kSvNone && head < D.C) {
        const unsigned long long e = scost[warp][head];
        unsigned long long c = (beam >> 32) + (e >> 4);
        c = c < 0xfffffffeull ? c : 0xfffffffeull;
        cand = (c << 32) | (uint32_t)(((uint32_t)beam << 4) | (uint32_t)(e & 15ull));
      }
      SvKey best = cand;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) best = sv_min(best, __shfl_xor_sync(0xffffffffu, best, o));
      if (best == kSvNone) break;                                    // fewer than S_k tuples exist so far
      if (cand == best) head += 1;                                   // keys are distinct (distinct tuples)
      if (lane == got) out = best;
    }
    beam = out;
    nbeam = got;
  }
  // result: lane s holds the s-th best tuple; repack z_g from nibble (G - 1 - g) to bits [4g, 4g + 4)
  if (lane < W) {
    uint32_t w = 0u;
    if (beam != kSvNone) {
      const uint32_t t = (uint32_t)beam;
      for (int g = 0; g < D.G; ++g) w |= ((t >> (4 * (D.G - 1 - g))) & 15u) << (4 * g);
    }
    (side ? V.codesV : V.codesK)[(size_t)b * D.K * D.S + off + lane] = w;
  }
}

int launch_synthesis_var(const Dims& D, const Hyper& H, const Dev& V, int n_act, cudaStream_t s) {
  const long long ntask = (long long)D.B * D.K * 2;
  const unsigned grid = (unsigned)((ntask + kSvWarps - 1) / kSvWarps);
  synthesis_var_kernel<<<grid, kSvWarps * 32, 0, s>>>(D, H, V, n_act);
  return 1;
}

}  // namespace pkv
