// ProtoKV query-time path (Alg. 3, Eq. 3, Alg. 4, Eq. 2/4 L130/L405):
// pseudo-token synthesis (top-S residual modes per prototype) and the fp32 SIMT fused attention over
// [near window || pseudo-tokens] with the log-mass bias inside the online softmax.  Pseudo-tokens are built in
// registers from (c_k, p_k, codes, codebooks) and never written to HBM.  See DESIGN.md "Kernels".
#include "common.cuh"

namespace pkv {

// ---------------------------------------------------------------------------------------------------------
// Q1 synthesis.  Task = (bank, prototype, K|V); sorting networks are fully unrolled and live in registers (no
// dynamically indexed arrays).
//
// Scores are the fixed-point log-probabilities of Eq. 3, q(g,z) = llround(2^24 log((H[g,z]+eps)/(sum+C eps)))
// (reading 13), tuples are ordered by (sum of q descending, tuple ascending lexicographically, z_1 most
// significant).  Beam search with width >= S over additive per-subspace scores under that total order returns
// exactly the global top-S, so this kernel keeps the 8 best partial tuples per step.  Of the products of the sorted
// beam with the sorted codes of the next subspace only the staircase (i+1)(j+1) <= 8 can survive (an entry (i, j)
// is preceded by every (i', j') <= (i, j)): 20 candidates, which arrive as five sorted runs
//   R0 = beam[0] + code[0..7],  R1 = beam[1] + code[0..3],  R2 = beam[2] + code[0..1],  R3 = beam[3] + code[0..1],
//   R4 = beam[4..7] + code[0]
// and are reduced to the 8 best by bitonic merges.
// ---------------------------------------------------------------------------------------------------------
constexpr int kSynThreads = 256;
constexpr int kSynLanes = 4;                        // preparing lanes per task (each takes G / 4 subspaces)
constexpr int kSynTasks = kSynThreads / kSynLanes;  // tasks per block and round
constexpr int kSynLogTab = PKV_SYN_LOGTAB;          // entries of Dev::logtab
constexpr int kSynWords = 9;                        // shared words per (task, subspace): 8 costs + 8 packed codes

// A candidate is ONE 64-bit key: cost = -sum q (>= 0, smaller is better) in the high word, the tuple (z_1 in the most
// significant used nibble; smaller is better on equal cost) in the low word -- the total order of reading 13 is the
// order of the keys.  ~0 = no candidate.  A per-subspace cost is below 2^29 for every P >= 1e-13 (-log P * 2^24), the
// sum over G = 8 subspaces is saturated at 2^32 - 2 (tuples that improbable never reach the top S).
typedef unsigned long long SynKey;
constexpr SynKey kSynNone = ~0ull;
constexpr uint32_t kSynCostNone = 0xffffffffu;

__device__ __forceinline__ void syn_ce(SynKey& a, SynKey& b) {   // afterwards a <= b
  const SynKey lo = a < b ? a : b, hi = a < b ? b : a;
  a = lo; b = hi;
}
template <int N>
__device__ __forceinline__ void syn_bitonic_merge(SynKey (&x)[N]) {   // bitonic input -> ascending
#pragma unroll
  for (int j = N >> 1; j > 0; j >>= 1) {
#pragma unroll
    for (int i = 0; i < N; ++i)
      if ((i & j) == 0) syn_ce(x[i], x[i | j]);
  }
}
__device__ __forceinline__ SynKey syn_add(SynKey b, uint32_t cost, uint32_t z) {
  if (b == kSynNone || cost == kSynCostNone) return kSynNone;
  unsigned long long c = (b >> 32) + cost;
  c = c < 0xfffffffeull ? c : 0xfffffffeull;
  return (c << 32) | (uint32_t)(((uint32_t)b << 4) | z);
}

// Subspace g of one task: the 8 most probable codes, best first, as fixed-point costs -q(g, z) (kSynCostNone if there
// is no such code) and the codes packed into nibbles (code i in bits [4i, 4i+4)).
// log P = log(h + eps) - log(tot + C eps): the first term comes from a host-built table (Dev::logtab, libm), the
// second is one fp64 log.
__device__ __forceinline__ void syn_prepare(const Dims& D, const Hyper& H, const Dev& V, const uint32_t* Hrow, int g,
                                            uint32_t (&cost)[8], uint32_t& zpack) {
  const int C = D.C;
  // keys of the C codes: (count + 1) in the high bits, 15 - z in the low nibble; 0 = no such code
  uint32_t key[16];
  double tot = 0.0;
  if (C == 16) {
    const uint4* h4 = reinterpret_cast<const uint4*>(Hrow + g * 16);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const uint4 v = h4[q];
      key[4 * q] = v.x; key[4 * q + 1] = v.y; key[4 * q + 2] = v.z; key[4 * q + 3] = v.w;
    }
#pragma unroll
    for (int z = 0; z < 16; ++z) { tot += (double)key[z]; key[z] = ((key[z] + 1u) << 4) | (uint32_t)(15 - z); }
  } else {
#pragma unroll
    for (int z = 0; z < 16; ++z) {
      key[z] = 0u;
      if (z < C) {
        const uint32_t h = Hrow[g * C + z];
        tot += (double)h;
        key[z] = ((h + 1u) << 4) | (uint32_t)(15 - z);
      }
    }
  }
  // descending bitonic sort of the 16 keys (the best 8 are needed, sorted)
#pragma unroll
  for (int kk = 2; kk <= 16; kk <<= 1) {
#pragma unroll
    for (int j = kk >> 1; j > 0; j >>= 1) {
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        const int l = i ^ j;
        if (l > i) {
          const uint32_t lo = min(key[i], key[l]), hi = max(key[i], key[l]);
          const bool desc = (i & kk) == 0;
          key[i] = desc ? hi : lo; key[l] = desc ? lo : hi;
        }
      }
    }
  }
  const double logden = log(tot + (double)C * H.pq_eps);
  zpack = 0u;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    zpack |= (15u - (key[i] & 15u)) << (4 * i);
    if (key[i] == 0u) cost[i] = kSynCostNone;
    else if (i > 0 && (key[i] >> 4) == (key[i - 1] >> 4)) cost[i] = cost[i - 1];
    else {
      const uint32_t h = (key[i] >> 4) - 1u;
      const double lognum = h < (uint32_t)kSynLogTab ? V.logtab[h] : log((double)h + H.pq_eps);
      const long long q = -llround((lognum - logden) * 16777216.0);
      cost[i] = (uint32_t)(q < 0 ? 0 : (q < 0xfffffffell ? q : 0xfffffffell));
    }
  }
}

// Work list: the prototypes stamped with the current epoch (Dev::dirty); the codes of the others are still valid.
// Every block of a bank compacts the bank's stamps into the same list in shared memory (ballot + prefix), then the
// blocks share the list entries by index.
//
// One task = (prototype, K or V side) = one run of Alg. 3 over its G histogram rows.  A block takes kSynTasks tasks per
// round in two phases: (1) lane (task, g mod 4) prepares subspaces g, g + 4 -- loads the 16 counts, sorts the keys, turns the 8
// best into fixed-point costs -- and parks them in shared memory ([g][word][task]: phase 2 reads are conflict-free);
// (2) one thread per task walks the beam recurrence over g = 0..G-1.  Phase 1 is the 8-wide part of the work; phase 2
// is the dependent chain that sets the kernel's duration, kept short by the single-key candidates.
__global__ void __launch_bounds__(kSynThreads) synthesis_kernel(Dims D, Hyper H, Dev V, int n_act, int epoch) {
  pdl_wait();      // launched when the ring append exits (it has no trigger of its own)
  pdl_trigger();   // the attention kernel sets up (barriers, TMEM) as SMs drain
  extern __shared__ uint16_t syn_list[];      // [K]
  __shared__ int wcnt[kSynThreads / 32];
  __shared__ uint32_t prep[8 * kSynWords * kSynTasks];
  __shared__ uint8_t tstate[kSynTasks];       // 0 decode, 1 zero residual / absent / no task
  const int b = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t* flags = V.dirty + (size_t)b * D.K;
  int base = 0;
  for (int kb = 0; kb < D.K; kb += 8 * kSynThreads) {          // 8 independent loads in flight per thread
    uint32_t fl[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int k = kb + u * kSynThreads + tid;
      fl[u] = k < D.K ? flags[k] : ~(uint32_t)epoch;
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int k0 = kb + u * kSynThreads;
      if (k0 >= D.K) break;                                    // block-uniform
      const bool hit = fl[u] == (uint32_t)epoch;
      const uint32_t bal = __ballot_sync(0xffffffffu, hit);
      if (lane == 0) wcnt[warp] = __popc(bal);
      __syncthreads();
      int off = base, tot = 0;
#pragma unroll
      for (int w = 0; w < kSynThreads / 32; ++w) { const int c = wcnt[w]; if (w < warp) off += c; tot += c; }
      if (hit) syn_list[off + __popc(bal & ((1u << lane) - 1u))] = (uint16_t)(k0 + tid);
      base += tot;
      __syncthreads();
    }
  }
  const int ntask = 2 * base;
  const bool has_cb = V.cbk != nullptr;
  for (int t0 = blockIdx.x * kSynTasks; t0 < ntask; t0 += gridDim.x * kSynTasks) {   // block-uniform
    {   // ---- phase 1: thread = (task, subspace) ----
      const int tl = tid / kSynLanes, g0 = tid % kSynLanes, task = t0 + tl;
      bool decode = false;
      size_t pk = 0;
      int kv = 0;
      if (task < ntask) {
        const int k = (int)syn_list[task >> 1];
        kv = task & 1;
        pk = (size_t)b * D.K + k;
        const bool present = k < n_act && V.n[pk] >= 1;
        const bool zero = !has_cb || !present || V.nres[pk] == 0;
        decode = !zero;
        if (g0 == 0) {
          tstate[tl] = zero ? 1 : 0;
          if (kv == 0) V.kind[pk] = present ? (zero ? 1 : 0) : 2;
        }
      } else if (g0 == 0) {
        tstate[tl] = 1;
      }
      if (decode) {
        for (int g = g0; g < D.G; g += kSynLanes) {
          uint32_t cost[8], zpack;
          syn_prepare(D, H, V, V.hist + (pk * 2 + kv) * D.G * D.C, g, cost, zpack);
#pragma unroll
          for (int i = 0; i < 8; ++i) prep[(g * kSynWords + i) * kSynTasks + tl] = cost[i];
          prep[(g * kSynWords + 8) * kSynTasks + tl] = zpack;
        }
      }
    }
    __syncthreads();
    if (tid < kSynTasks && t0 + tid < ntask) {   // ---- phase 2: thread = task ----
      const int task = t0 + tid;
      const int k = (int)syn_list[task >> 1];
      const size_t pk = (size_t)b * D.K + k;
      uint32_t* codes = ((task & 1) ? V.codesV : V.codesK) + pk * D.S;
      if (tstate[tid]) {
        for (int s = 0; s < D.S; ++s) codes[s] = 0u;
      } else {
        SynKey beam[8];
#pragma unroll
        for (int i = 1; i < 8; ++i) beam[i] = kSynNone;
        beam[0] = 0ull;
        for (int g = 0; g < D.G; ++g) {
          uint32_t cost[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) cost[i] = prep[(g * kSynWords + i) * kSynTasks + tid];
          const uint32_t zp = prep[(g * kSynWords + 8) * kSynTasks + tid];
          SynKey a[8], bb[8], c4[4];
#pragma unroll
          for (int j = 0; j < 8; ++j) a[j] = syn_add(beam[0], cost[j], (zp >> (4 * j)) & 15u);          // R0, ascending
#pragma unroll
          for (int j = 0; j < 4; ++j) bb[j] = syn_add(beam[1], cost[j], (zp >> (4 * j)) & 15u);         // R1
#pragma unroll
          for (int i = 0; i < 4; ++i) bb[7 - i] = syn_add(beam[4 + i], cost[0], zp & 15u);              // R4 reversed: [R1, rev R4] is bitonic
          syn_bitonic_merge<8>(bb);
#pragma unroll
          for (int j = 0; j < 2; ++j) c4[j] = syn_add(beam[2], cost[j], (zp >> (4 * j)) & 15u);         // R2
#pragma unroll
          for (int j = 0; j < 2; ++j) c4[3 - j] = syn_add(beam[3], cost[j], (zp >> (4 * j)) & 15u);     // R3 reversed
          syn_bitonic_merge<4>(c4);
#pragma unroll
          for (int i = 0; i < 8; ++i) a[i] = a[i] < bb[7 - i] ? a[i] : bb[7 - i];                       // 8 best of R0 u R1 u R4, bitonic
          syn_bitonic_merge<8>(a);
#pragma unroll
          for (int i = 0; i < 4; ++i) a[4 + i] = a[4 + i] < c4[3 - i] ? a[4 + i] : c4[3 - i];           // 8 best of all 20, bitonic
          syn_bitonic_merge<8>(a);
#pragma unroll
          for (int i = 0; i < 8; ++i) beam[i] = a[i];
        }
#pragma unroll
        for (int s = 0; s < 8; ++s) {
          if (s < D.S) {
            uint32_t packed = 0u;
            if (beam[s] != kSynNone) {
              const uint32_t t = (uint32_t)beam[s];
              for (int g = 0; g < D.G; ++g) packed |= ((t >> (4 * (D.G - 1 - g))) & 15u) << (4 * g);
            }
            codes[s] = packed;
          }
        }
      }
    }
    __syncthreads();
  }
}

bool query_kernels_prepare(const Dims&) {
  // function attributes are per device, not per state: size for the largest k_max protokv_create admits
  if (cudaFuncSetAttribute(synthesis_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxKmax * 2) == cudaSuccess) return true;
  cudaGetLastError();
  return false;
}

int launch_synthesis(const Dims& D, const Hyper& H, const Dev& V, int n_act, int epoch, int max_dirty, int sm_count,
                     cudaStream_t s) {
  // grid-stride over each bank's work list; its length is only known on the device, but the host knows a bound: at most
  // max_dirty prototypes per bank were stamped since the last synthesis (<= T per appended frame) -- blocks beyond that
  // would only run the list compaction and exit
  const int bound = max_dirty < D.K ? (max_dirty > 0 ? max_dirty : 1) : D.K;
  int per_bank = (2 * bound + kSynTasks - 1) / kSynTasks;
  const int cap = (8 * sm_count + D.B - 1) / D.B;
  if (per_bank > cap) per_bank = cap;
  if (per_bank < 1) per_bank = 1;
  launch_chain(synthesis_kernel, dim3(per_bank, D.B), kSynThreads, (size_t)D.K * 2, s, !(H.flags & PROTOKV_SERIAL_LAUNCH), D, H, V, n_act, epoch);
  return 1;
}

// ---------------------------------------------------------------------------------------------------------
// Q2 fused attention, fp32 SIMT variant (Alg. 4 l.8-15; Eq. 4).  One warp per query row (query token x query
// head), DH/32 dims per lane, split over the context (flash-decoding style) with a combine kernel.
// Context element e < n_near is ring row e of the bank; e >= n_near is pseudo-token (k, s) of prototype
// k = (e - n_near) / S:  k~ = c_k + concat_g CK_g[zK(k,s,g)],  v~ = p_k + concat_g CV_g[zV(k,s,g)],  bias log n_k.
// ---------------------------------------------------------------------------------------------------------
constexpr int kAttWarps = 4;

struct Softmax1 {   // running (max, sum) of one row; acc lives in the caller
  float m, l;
};

template <int VEC>
__device__ __forceinline__ void online_update(Softmax1& st, float (&acc)[VEC], float logit, const float (&v)[VEC]) {
  if (logit > st.m) {
    const float sc = __expf(st.m - logit);   // exp(-inf) = 0 on the first element
    st.l = fmaf(st.l, sc, 1.f);
#pragma unroll
    for (int i = 0; i < VEC; ++i) acc[i] = fmaf(acc[i], sc, v[i]);
    st.m = logit;
  } else {
    const float w = __expf(logit - st.m);
    st.l += w;
#pragma unroll
    for (int i = 0; i < VEC; ++i) acc[i] = fmaf(w, v[i], acc[i]);
  }
}

// ---- rotary position anchoring (PROTOKV_ROPE, D.1; readings 28-31) --------------------
// Rotate-half convention: pair (i, i + d/2) of a vector at position p turns by p * theta^(-2i/d).  A lane of the
// attention warp holds VEC consecutive dims, so its partner dims live in lane ^ 16 at the same v.  The angles are
// evaluated in fp64 by rope_tables_kernel (positions reach ~1e6, fp32 angles would be off by 0.05 rad) and kept as
// float2 (cos, sin): J[j] for the token offset inside a frame, F[slot] for the first position of the frame held in a
// ring slot (a near token's rotation is the product of the two), P[k] for the anchor of every prototype (all S
// pseudo-tokens of a prototype share it), Qc[i] for the query tokens.
template <int VEC>
__device__ __forceinline__ void rope_apply(float (&x)[VEC], const float2 (&cs)[VEC], int lane) {
  const float sgn = lane < 16 ? -1.f : 1.f;
#pragma unroll
  for (int v = 0; v < VEC; ++v) {
    const float partner = __shfl_xor_sync(0xffffffffu, x[v], 16);
    x[v] = fmaf(sgn * partner, cs[v].y, x[v] * cs[v].x);
  }
}
__device__ __forceinline__ float2 cis_mul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.y, b.x, a.x * b.y));
}

__global__ void rope_tables_kernel(Dims D, Hyper H, Dev V, AttnArgs A) {
  extern __shared__ double inv_freq[];                 // [d/2]
  const int h = D.d / 2;
  for (int i = threadIdx.x; i < h; i += blockDim.x) inv_freq[i] = pow(H.rope_theta, -2.0 * (double)i / (double)D.d);
  __syncthreads();
  const long long nJ = (long long)D.T * h, nF = (long long)D.Wf * h, nQ = (long long)A.n_q * h;
  const long long nP = (long long)D.B * D.K * h, nR = (long long)D.Wf * D.T * h, total = nJ + nF + nQ + nP + nR;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    double p;
    float2* dst;
    int i;
    if (e < nJ) { i = (int)(e % h); p = (double)(e / h); dst = V.ropeJ + e; }
    else if (e < nJ + nF) {
      const long long x = e - nJ;
      i = (int)(x % h);
      const long long slot = x / h, last = A.frames - 1;
      const long long f = last >= slot ? last - ((last - slot) % D.Wf) : 0;   // the frame the slot holds (0 if none yet)
      p = (double)(H.pos0 + f * D.T);
      dst = V.ropeF + x;
    } else if (e < nJ + nF + nQ) {
      const long long x = e - nJ - nF;
      i = (int)(x % h);
      p = (double)(A.q_pos0 + x / h);
      dst = V.ropeQ + x;
    } else if (e >= nJ + nF + nQ + nP) {     // ring row (slot, j) at the position of the frame the slot holds
      const long long x = e - nJ - nF - nQ - nP;
      i = (int)(x % h);
      const long long row = x / h, slot = row / D.T, last = A.frames - 1;
      const long long f = last >= slot ? last - ((last - slot) % D.Wf) : 0;
      p = (double)(H.pos0 + f * D.T + row % D.T);
      dst = V.ropeR + x;
    } else {
      const long long x = e - nJ - nF - nQ;
      i = (int)(x % h);
      const long long pk = x / h;
      if ((int)(pk % D.K) >= A.n_act) continue;
      if (H.rope_anchor == 1) p = (double)V.pos_first[pk];
      else if (H.rope_anchor == 2) p = (double)V.pos_sum[pk] / (double)max(V.pos_cnt[pk], 1);
      else p = (double)V.pos[pk];
      dst = V.ropeP + x;
    }
    double sn, cs;
    sincos(p * inv_freq[i], &sn, &cs);
    *dst = make_float2((float)cs, (float)sn);
  }
}

int launch_rope_tables(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, cudaStream_t s) {
  const int h = D.d / 2;
  const long long total = (long long)(D.T + D.Wf + A.n_q) * h + (long long)D.B * D.K * h + (long long)D.Wf * D.T * h;
  const unsigned grid = (unsigned)((total + 255) / 256 < 4096 ? (total + 255) / 256 : 4096);
  rope_tables_kernel<<<grid, 256, (size_t)h * 8, s>>>(D, H, V, A);
  return 1;
}

template <typename T, int DH, bool ROPE>
__global__ void __launch_bounds__(kAttWarps * 32) attention_simt_kernel(Dims D, Hyper H, Dev V, AttnArgs A) {
  constexpr int VEC = DH / 32;
  extern __shared__ __align__(16) float cb_s[];
  const int gstride = D.C * D.sub + kCbPad;
  float* cbk_s = cb_s;
  float* cbv_s = cb_s + D.G * gstride;

  const int R = A.n_q * D.group;
  const int rgroups = (R + kAttWarps - 1) / kAttWarps;
  const int bsel = blockIdx.x / rgroups, rg = blockIdx.x % rgroups;
  const int hd = bsel % D.Hkv, ll = (bsel / D.Hkv) % A.layer_count, st = bsel / (D.Hkv * A.layer_count);
  const int b = (st * D.L + A.layer_begin + ll) * D.Hkv + hd;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool has_cb = V.cbk != nullptr;
  if (has_cb) {
    const int per_g = D.C * D.sub;
    for (int e = tid; e < D.G * per_g; e += kAttWarps * 32) {
      const int g = e / per_g, r = e % per_g;
      cbk_s[g * gstride + r] = V.cbk[(size_t)b * D.G * per_g + e];
      cbv_s[g * gstride + r] = V.cbv[(size_t)b * D.G * per_g + e];
    }
  }
  __syncthreads();
  const int row = rg * kAttWarps + warp;
  if (row >= R) return;
  const int qi = row / D.group, h = hd * D.group + row % D.group;
  const size_t qoff = ((((size_t)st * A.layer_count + ll) * A.n_q + qi) * D.Hq + h) * DH;
  float q[VEC];
  load_vec<T, VEC>((const T*)A.Q + qoff + lane * VEC, q);
  constexpr int HH = DH / 2;
  const int ri = (lane & 15) * VEC;                    // pair index of this lane's first dim (ROPE)
  if (ROPE) {
    float2 cs[VEC];
#pragma unroll
    for (int v = 0; v < VEC; ++v) cs[v] = V.ropeQ[(size_t)qi * HH + ri + v];
    rope_apply<VEC>(q, cs, lane);
  }
  const float scale = 1.0f / sqrtf((float)DH);
#pragma unroll
  for (int v = 0; v < VEC; ++v) q[v] *= scale;

  const int near_cnt = (H.flags & PROTOKV_FAR_ONLY) ? 0 : A.n_near;
  const int* soff = V.soff ? V.soff + (size_t)b * (D.K + 1) : nullptr;   // D.3: ragged pseudo-token counts
  const int ps_cnt = (H.flags & PROTOKV_NEAR_ONLY) ? 0 : (soff ? soff[D.K] : A.n_act * D.S);
  const int Lc = near_cnt + ps_cnt;
  const int chunk = (Lc + A.nsplit - 1) / A.nsplit;
  const int lo = blockIdx.y * chunk, hi = min(Lc, lo + chunk);
  Softmax1 sm{-INFINITY, 0.f};
  float acc[VEC];
#pragma unroll
  for (int v = 0; v < VEC; ++v) acc[v] = 0.f;

  // near-window tokens
  const T* rK = (const T*)V.ringK + (size_t)b * D.Wf * D.T * DH;
  const T* rV = (const T*)V.ringV + (size_t)b * D.Wf * D.T * DH;
  int e = lo;
  const int near_hi = min(hi, near_cnt);
  for (; e + 4 <= near_hi; e += 4) {
    float kk[4][VEC], vv[4][VEC], dot[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      load_vec<T, VEC>(rK + (size_t)(e + u) * DH + lane * VEC, kk[u]);
      load_vec<T, VEC>(rV + (size_t)(e + u) * DH + lane * VEC, vv[u]);
    }
    if (ROPE) {
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int slot = (e + u) / D.T, j = (e + u) - slot * D.T;
        float2 cs[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) cs[v] = cis_mul(V.ropeF[slot * HH + ri + v], V.ropeJ[(size_t)j * HH + ri + v]);
        rope_apply<VEC>(kk[u], cs, lane);
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      dot[u] = 0.f;
#pragma unroll
      for (int v = 0; v < VEC; ++v) dot[u] = fmaf(q[v], kk[u][v], dot[u]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
      for (int u = 0; u < 4; ++u) dot[u] += __shfl_xor_sync(0xffffffffu, dot[u], o);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) online_update<VEC>(sm, acc, dot[u], vv[u]);
  }
  for (; e < near_hi; ++e) {
    float kk[VEC], vv[VEC];
    load_vec<T, VEC>(rK + (size_t)e * DH + lane * VEC, kk);
    load_vec<T, VEC>(rV + (size_t)e * DH + lane * VEC, vv);
    if (ROPE) {
      const int slot = e / D.T, j = e - slot * D.T;
      float2 cs[VEC];
#pragma unroll
      for (int v = 0; v < VEC; ++v) cs[v] = cis_mul(V.ropeF[slot * HH + ri + v], V.ropeJ[(size_t)j * HH + ri + v]);
      rope_apply<VEC>(kk, cs, lane);
    }
    float dot = 0.f;
#pragma unroll
    for (int v = 0; v < VEC; ++v) dot = fmaf(q[v], kk[v], dot);
    dot = warp_sum(dot);
    online_update<VEC>(sm, acc, dot, vv);
  }
  // pseudo-tokens
  if (hi > near_cnt) {
    const int p_lo = max(lo, near_cnt) - near_cnt, p_hi = hi - near_cnt;
    const int LPS = 32 / D.G, g = lane / LPS, li = lane % LPS;
    const bool use_bias = !(H.flags & PROTOKV_NO_MASS_BIAS);
    int k = p_lo / D.S;
    if (soff) {                              // first prototype whose rows reach beyond p_lo
      int lo2 = 0, hi2 = D.K;
      while (lo2 < hi2) { const int mid = (lo2 + hi2) >> 1; if (soff[mid + 1] > p_lo) hi2 = mid; else lo2 = mid + 1; }
      k = lo2;
    }
    for (; k < D.K && (soff ? soff[k] : k * D.S) < p_hi; ++k) {
      const size_t pk = (size_t)b * D.K + k;
      const int kind = V.kind[pk];
      if (kind == 2) continue;
      const int row0 = soff ? soff[k] : k * D.S, nrow = soff ? soff[k + 1] - soff[k] : D.S;
      const int s_lo = max(p_lo - row0, 0), s_hi = min(p_hi - row0, nrow);
      const size_t crow = (size_t)b * D.K * D.S + row0;   // this prototype's code rows
      float c[VEC], p[VEC];
      load_vec<float, VEC>(V.c + pk * DH + lane * VEC, c);
      load_vec<float, VEC>(V.p + pk * DH + lane * VEC, p);
      const float bias = use_bias ? V.logn[pk] : 0.f;
      float2 pcs[VEC];
      if (ROPE) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) pcs[v] = V.ropeP[pk * HH + ri + v];
      }
      if (kind == 1) {             // zero residuals: S identical pseudo-tokens (Alg. 4 l.3-4)
        float kc[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) kc[v] = c[v];
        if (ROPE) rope_apply<VEC>(kc, pcs, lane);
        float dot = 0.f;
#pragma unroll
        for (int v = 0; v < VEC; ++v) dot = fmaf(q[v], kc[v], dot);
        dot = warp_sum(dot) + bias;
        for (int s = s_lo; s < s_hi; ++s) online_update<VEC>(sm, acc, dot, p);
        continue;
      }
      for (int s = s_lo; s < s_hi; ++s) {
        const uint32_t zk = (V.codesK[crow + s] >> (4 * g)) & 15u;
        const uint32_t zv = (V.codesV[crow + s] >> (4 * g)) & 15u;
        float rk[VEC], rv[VEC];
        load_vec<float, VEC>(cbk_s + g * gstride + zk * D.sub + li * VEC, rk);
        load_vec<float, VEC>(cbv_s + g * gstride + zv * D.sub + li * VEC, rv);
        float dot = 0.f;
#pragma unroll
        for (int v = 0; v < VEC; ++v) { rk[v] += c[v]; rv[v] += p[v]; }
        if (ROPE) rope_apply<VEC>(rk, pcs, lane);
#pragma unroll
        for (int v = 0; v < VEC; ++v) dot = fmaf(q[v], rk[v], dot);
        dot = warp_sum(dot) + bias;
        online_update<VEC>(sm, acc, dot, rv);
      }
    }
  }
  float* part = V.part + (((size_t)bsel * R + row) * A.nsplit + blockIdx.y) * (DH + 2);
#pragma unroll
  for (int v = 0; v < VEC; ++v) part[lane * VEC + v] = acc[v];
  if (lane == 0) { part[DH] = sm.m; part[DH + 1] = sm.l; }
}

template <typename T, int DH>
__global__ void __launch_bounds__(128) attention_combine_kernel(Dims D, Dev V, AttnArgs A, int rows_total) {
  constexpr int VEC = DH / 32;
  const int gr = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  pdl_wait();
  pdl_trigger();   // the next query's kernel may set up while the rows are merged
  if (gr >= rows_total) return;
  const int R = A.n_q * D.group;
  const int bsel = gr / R, row = gr % R;
  const int hd = bsel % D.Hkv, ll = (bsel / D.Hkv) % A.layer_count, st = bsel / (D.Hkv * A.layer_count);
  const int qi = row / D.group, h = hd * D.group + row % D.group;
  const float* part = V.part + (size_t)gr * A.nsplit * (DH + 2);
  // online (max, sum) merge of the splits, eight splits' loads in flight at a time (a two-pass merge over a runtime split
  // count kept one load in flight per warp: 2 x nsplit dependent L2 round trips for a few hundred bytes per row)
  float M = -INFINITY, l = 0.f, acc[VEC];
  bool poisoned = false;   // a partial with a NaN maximum or row sum (non-finite logits): the row is NaN
#pragma unroll
  for (int v = 0; v < VEC; ++v) acc[v] = 0.f;
  for (int sp0 = 0; sp0 < A.nsplit; sp0 += 8) {
    float2 ml[8];
    float pv[8][VEC];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int sp = sp0 + u < A.nsplit ? sp0 + u : A.nsplit - 1;   // clamp: a repeated split is skipped below
      const float* ps = part + (size_t)sp * (DH + 2);
      ml[u] = *reinterpret_cast<const float2*>(ps + DH);
#pragma unroll
      for (int v = 0; v < VEC; v += 2) {                            // rows are (DH + 2) floats apart: 8-byte aligned, not 16
        const float2 t = *reinterpret_cast<const float2*>(ps + lane * VEC + v);
        pv[u][v] = t.x; pv[u][v + 1] = t.y;
      }
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      if (sp0 + u >= A.nsplit) continue;
      const float m = ml[u].x, ls = ml[u].y;
      poisoned = poisoned || m != m || ls != ls;
      if (!(m > -INFINITY)) continue;                                // empty split
      const float Mn = fmaxf(M, m);
      const float so = __expf(M - Mn), sn = __expf(m - Mn);          // M = -inf: so = 0
      l = fmaf(l, so, ls * sn);
#pragma unroll
      for (int v = 0; v < VEC; ++v) acc[v] = fmaf(acc[v], so, pv[u][v] * sn);
      M = Mn;
    }
  }
  float inv = l > 0.f ? 1.f / l : 0.f;
  if (poisoned) {
    inv = __int_as_float(0x7fc00000);
#pragma unroll
    for (int v = 0; v < VEC; ++v) acc[v] = 1.f;
  }
  const size_t ooff = ((((size_t)st * A.layer_count + ll) * A.n_q + qi) * D.Hq + h);
  T* out = (T*)A.out + ooff * DH + lane * VEC;
#pragma unroll
  for (int v = 0; v < VEC; ++v) out[v] = from_f32<T>(acc[v] * inv);
  if (A.lse && lane == 0) A.lse[ooff] = poisoned ? inv : (l > 0.f ? M + logf(l) : -INFINITY);
}

int attention_simt_splits(const Dims& D, int sm_count) {
  const int R = D.Nq * D.group;
  const long long ctas = (long long)D.B * ((R + kAttWarps - 1) / kAttWarps);
  long long ns = (4LL * sm_count + ctas - 1) / ctas;
  if (ns < 1) ns = 1;
  if (ns > 64) ns = 64;
  return (int)ns;
}

template <typename T, int DH>
static int attention_simt_launch(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, cudaStream_t s) {
  const int R = A.n_q * D.group;
  const int nb = D.NS * A.layer_count * D.Hkv;
  const int rgroups = (R + kAttWarps - 1) / kAttWarps;
  const size_t sm = V.cbk ? 2 * (size_t)D.G * (D.C * D.sub + kCbPad) * 4 : 0;
  dim3 grid(nb * rgroups, A.nsplit);
  if (H.flags & PROTOKV_ROPE) attention_simt_kernel<T, DH, true><<<grid, kAttWarps * 32, sm, s>>>(D, H, V, A);
  else attention_simt_kernel<T, DH, false><<<grid, kAttWarps * 32, sm, s>>>(D, H, V, A);
  const int rows_total = nb * R;
  attention_combine_kernel<T, DH><<<(rows_total + 3) / 4, 128, 0, s>>>(D, V, A, rows_total);
  return 2;
}

int launch_attention_combine_bf16_128(const Dims& D, const Dev& V, const AttnArgs& A, bool pdl, cudaStream_t s) {
  const int rows_total = D.NS * A.layer_count * D.Hkv * A.n_q * D.group;
  launch_chain(attention_combine_kernel<__nv_bfloat16, 128>, (rows_total + 3) / 4, 128, 0, s, pdl, D, V, A, rows_total);
  return 1;
}

int launch_attention_simt(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, cudaStream_t s) {
  if (D.bf16) return D.d == 128 ? attention_simt_launch<__nv_bfloat16, 128>(D, H, V, A, s)
                                : attention_simt_launch<__nv_bfloat16, 64>(D, H, V, A, s);
  return D.d == 128 ? attention_simt_launch<float, 128>(D, H, V, A, s)
                    : attention_simt_launch<float, 64>(D, H, V, A, s);
}

}  // namespace pkv
