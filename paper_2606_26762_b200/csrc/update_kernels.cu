// ProtoKV per-frame far-memory update (Alg. 1): ring append, slot fill, Eq. 1 scoring (fp32
// SIMT variant), segmenting and the segmented prototype update with PQ residual histograms.
// See DESIGN.md "Kernels".  All launchers are asynchronous on the caller's stream.
#include "common.cuh"
#include "derived.cuh"

namespace pkv {

// ---------------------------------------------------------------------------------------------------------
// U1 ring append (Alg. 1 l.1): frame f goes to slot f % Wf, transposed from the model-native
// [stream][layer][T][Hkv][d] to the bank-major ring [bank][Wf][T][d].  A group of vpr lanes (16-byte vectors of one
// row) copies kApRows rows of K and of V: all 2 * kApRows loads are in flight before the first store (the copy is
// latency-bound otherwise), row indices are 32-bit.  The first threads also copy grid_pos and reset the keys.
// ---------------------------------------------------------------------------------------------------------
constexpr int kApRows = 4;
template <bool BF16>
__global__ void __launch_bounds__(256) ring_append_kernel(Dims D, Dev V, int slot, const uint4* __restrict__ Kin,
                                                          const uint4* __restrict__ Vin,
                                                          const float* __restrict__ grid_pos, int vpr) {
  const uint32_t gtid = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t rows = (uint32_t)(D.B * D.T);
  const uint32_t grp = gtid / (uint32_t)vpr, v = gtid % (uint32_t)vpr;
  const uint32_t ngrp = gridDim.x * blockDim.x / (uint32_t)vpr;
  uint4 wk[kApRows], wv[kApRows];
  uint32_t orow[kApRows];
#pragma unroll
  for (int i = 0; i < kApRows; ++i) {
    const uint32_t r = grp + (uint32_t)i * ngrp;           // r = b * T + j
    const bool valid = r < rows;
    const uint32_t rr = valid ? r : 0u;
    const uint32_t b = rr / (uint32_t)D.T, j = rr - b * (uint32_t)D.T;
    const uint32_t sl = b / (uint32_t)D.Hkv, hd = b - sl * (uint32_t)D.Hkv;   // sl = stream * L + layer
    const size_t src = (((size_t)sl * D.T + j) * D.Hkv + hd) * vpr + v;
    orow[i] = valid ? (b * (uint32_t)D.Wf + (uint32_t)slot) * (uint32_t)D.T + j : 0xffffffffu;
    wk[i] = __ldcg(Kin + src);                             // read once, ahead of pdl_wait(): straight from L2
    wv[i] = __ldcg(Vin + src);
  }
  float gp = 0.f;
  const bool has_gp = gtid < (uint32_t)(D.NS * D.T * 2);
  if (has_gp) gp = __ldcg(grid_pos + gtid);
  // everything above reads the caller's buffers only; the slot is overwritten once the update kernel has completed
  pdl_wait();   // no pdl_trigger(): the next frame's score kernel (one CTA per SM) started under this kernel's stores made
                // C5 frames 9 % slower; launched at this kernel's exit it still skips the launch latency
  if (has_gp) {
    const int st = (int)(gtid / (uint32_t)(D.T * 2)), e = (int)(gtid % (uint32_t)(D.T * 2));
    V.ringS[((size_t)st * D.Wf + slot) * D.T * 2 + e] = gp;
  }
  for (uint32_t i = gtid; i < (uint32_t)(D.B * D.T); i += gridDim.x * blockDim.x)
    V.akey[i] = ~0ull;                                     // next frame's assignment keys (see tc_assign.cu)
  uint4* outK = (uint4*)V.ringK;
  uint4* outV = (uint4*)V.ringV;
#pragma unroll
  for (int i = 0; i < kApRows; ++i) {
    const bool valid = orow[i] != 0xffffffffu;
    if (valid) {
      outK[(size_t)orow[i] * vpr + v] = wk[i];
      outV[(size_t)orow[i] * vpr + v] = wv[i];
    }
    const uint32_t ww[4] = {wk[i].x, wk[i].y, wk[i].z, wk[i].w};   // |K_j|^2, reduced over the lanes of the row
    float kk = 0.f;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      if (BF16) {
        const float lo = __uint_as_float(ww[e] << 16), hi = __uint_as_float(ww[e] & 0xffff0000u);
        kk = fmaf(lo, lo, kk); kk = fmaf(hi, hi, kk);
      } else {
        const float x = __uint_as_float(ww[e]);
        kk = fmaf(x, x, kk);
      }
    }
    for (int o = vpr >> 1; o > 0; o >>= 1) kk += __shfl_xor_sync(0xffffffffu, kk, o);
    if (valid && v == 0) V.ringN[orow[i]] = kk;
  }
}

int launch_ring_append(const Dims& D, const Dev& V, const FrameArgs& F, const void* Kin, const void* Vin,
                       const float* grid_pos, cudaStream_t s) {
  const int vpr = D.d * (D.bf16 ? 2 : 4) / 16;             // 8, 16 or 32 lanes per row: groups never straddle a warp
  const size_t rows = (size_t)D.B * D.T;
  const size_t groups = (rows + kApRows - 1) / kApRows;
  size_t threads = groups * vpr;
  const size_t need = (size_t)D.NS * D.T * 2;              // grid_pos copy
  if (threads < need) threads = need;
  const unsigned grid = (unsigned)((threads + 255) / 256);
  if (D.bf16) launch_chain(ring_append_kernel<true>, grid, 256, 0, s, F.pdl != 0, D, V, F.slot, (const uint4*)Kin, (const uint4*)Vin, grid_pos, vpr);
  else launch_chain(ring_append_kernel<false>, grid, 256, 0, s, F.pdl != 0, D, V, F.slot, (const uint4*)Kin, (const uint4*)Vin, grid_pos, vpr);
  return 1;
}

// ---------------------------------------------------------------------------------------------------------
// U2 slot fill (Alg. 1 l.3-4; L83): evicted token j < n_fill opens slot n_act0 + j.
// One warp per (token, bank).
// ---------------------------------------------------------------------------------------------------------
template <typename T>
__global__ void fill_kernel(Dims D, Hyper H, Dev V, FrameArgs F) {
  const int j = blockIdx.x, b = blockIdx.y, lane = threadIdx.x;
  const int k = F.n_act0 + j;
  const int st = b / (D.L * D.Hkv);
  const T* Ke = (const T*)V.ringK + (((size_t)b * D.Wf + F.slot) * D.T + j) * D.d;
  const T* Ve = (const T*)V.ringV + (((size_t)b * D.Wf + F.slot) * D.T + j) * D.d;
  const size_t pk = (size_t)b * D.K + k;
  float cc = 0.f;
  const int vec = D.d / 32;   // same per-lane order as update_kernel / refresh_derived_kernel: derived values agree bit for bit
  for (int v = 0; v < vec; ++v) {
    const int i = lane * vec + v;
    float kf = to_f32(Ke[i]), vf = to_f32(Ve[i]);
    V.c[pk * D.d + i] = kf;
    V.p[pk * D.d + i] = vf;
    if (V.c_bf) { V.c_bf[pk * D.d + i] = __float2bfloat16_rn(kf); V.p_bf[pk * D.d + i] = __float2bfloat16_rn(vf); }
    cc = fmaf(kf, kf, cc);
  }
  cc = warp_sum(cc);
  if (V.c_hi) {
    const float invc = inv_norm(cc);
    for (int i = lane; i < D.d; i += 32) {
      __nv_bfloat16 hi, lo;
      split_bf16(to_f32(Ke[i]) * invc, hi, lo);
      V.c_hi[pk * D.d + i] = hi; V.c_lo[pk * D.d + i] = lo;
    }
  }
  const int ghc = 2 * D.G * D.C;
  for (int i = lane; i < ghc; i += 32) V.hist[pk * ghc + i] = 0u;
  if (lane == 0) {
    const float* se = V.ringS + (((size_t)st * D.Wf + F.slot) * D.T + j) * 2;
    V.n[pk] = 1;
    V.mu[pk * 2] = se[0]; V.mu[pk * 2 + 1] = se[1];
    V.sigma[pk * 3] = 1.f; V.sigma[pk * 3 + 1] = 0.f; V.sigma[pk * 3 + 2] = 1.f;
    V.tau[pk] = F.t;
    const long long ps = H.pos0 + (long long)F.ev_frame * D.T + j;
    V.pos[pk] = ps; V.pos_first[pk] = ps; V.pos_sum[pk] = ps; V.pos_cnt[pk] = 1;   // D.1 anchors
    V.nres[pk] = 0u;
    store_rec(V.rec, pk, make_rec(cc, se[0], se[1], 1.f, 0.f, 1.f, F.t, H));
    V.logn[pk] = 0.f;
    V.mstamp[pk] = F.t;
    mark_dirty(D, V, b, k, F.epoch);
    V.assign[(size_t)b * D.T + j] = k;
    V.best[(size_t)b * D.T + j] = 0.f;
  }
  for (int g = lane; g < D.G; g += 32) {
    V.tcodeK[((size_t)b * D.T + j) * D.G + g] = 255;
    V.tcodeV[((size_t)b * D.T + j) * D.G + g] = 255;
  }
}

int launch_fill(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, cudaStream_t s) {
  if (F.n_fill <= 0) return 0;
  dim3 grid(F.n_fill, D.B);
  if (D.bf16) fill_kernel<__nv_bfloat16><<<grid, 32, 0, s>>>(D, H, V, F);
  else fill_kernel<float><<<grid, 32, 0, s>>>(D, H, V, F);
  return 1;
}

// ---------------------------------------------------------------------------------------------------------
// U3 assignment, fp32 SIMT variant (Eq. 1; Alg. 1 l.6).  Used for fp32 inputs and as the
// cross-check of the tcgen05 kernel.  CTA = (bank, tile of 32 tokens); 256 threads = 32 tokens x 8 prototype
// lanes; prototypes are staged through shared memory 64 at a time.
// ---------------------------------------------------------------------------------------------------------
constexpr int kScoreTok = 32, kScoreKc = 64, kScoreThreads = 256;

template <typename T, int DH>
__global__ void __launch_bounds__(kScoreThreads) score_simt_kernel(Dims D, Hyper H, Dev V, FrameArgs F) {
  extern __shared__ float smem[];
  float* tokT = smem;                          // [DH][32]   token tile, transposed
  float* cs = tokT + DH * kScoreTok;           // [64][DH]   centre chunk
  ScoreRec* recs = (ScoreRec*)(cs + kScoreKc * DH);  // [64]
  float* bestv = (float*)(recs + kScoreKc);    // [8][32]
  int* besti = (int*)(bestv + 8 * kScoreTok);  // [8][32]

  const int b = blockIdx.y, j0 = F.n_fill + blockIdx.x * kScoreTok;
  const int tid = threadIdx.x, tl = tid & 31, kg = tid >> 5;
  const int st = b / (D.L * D.Hkv);
  const T* Ke = (const T*)V.ringK + ((size_t)b * D.Wf + F.slot) * D.T * DH;
  // token tile -> smem (transposed), zero beyond T
  for (int e = tid; e < kScoreTok * DH; e += kScoreThreads) {
    int tt = e / DH, i = e % DH;
    int j = j0 + tt;
    tokT[i * kScoreTok + tt] = j < D.T ? to_f32(Ke[(size_t)j * DH + i]) : 0.f;
  }
  __syncthreads();
  const int j = j0 + tl;
  float kk = 0.f;
  for (int i = 0; i < DH; ++i) { float x = tokT[i * kScoreTok + tl]; kk = fmaf(x, x, kk); }
  const float invk = kk > 0.f ? rsqrtf(kk) : 0.f;
  const float inv_cap = 1.f / H.cos_eps;       // cos = dot / max(|K||c|, cos_eps)  (reading 6)
  float sx = 0.f, sy = 0.f;
  if (j < D.T) {
    const float* se = V.ringS + (((size_t)st * D.Wf + F.slot) * D.T + j) * 2;
    sx = se[0]; sy = se[1];
  }
  float best = INFINITY;
  int bidx = 0x7fffffff;
  const bool squared = H.flags & PROTOKV_MAH_SQUARED;
  for (int k0 = 0; k0 < F.n_act; k0 += kScoreKc) {
    __syncthreads();
    const int nk = min(kScoreKc, F.n_act - k0);
    const float4* src = (const float4*)(V.c + ((size_t)b * D.K + k0) * DH);
    for (int e = tid; e < nk * DH / 4; e += kScoreThreads) ((float4*)cs)[e] = src[e];
    if (tid < nk) recs[tid] = load_rec(V.rec, (size_t)b * D.K + k0 + tid);
    __syncthreads();
    float acc[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = 0.f;
    for (int i = 0; i < DH; i += 4) {
      float x0 = tokT[(i + 0) * kScoreTok + tl], x1 = tokT[(i + 1) * kScoreTok + tl];
      float x2 = tokT[(i + 2) * kScoreTok + tl], x3 = tokT[(i + 3) * kScoreTok + tl];
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        float4 cv = *(const float4*)(cs + (kg * 8 + q) * DH + i);
        acc[q] = fmaf(x0, cv.x, acc[q]); acc[q] = fmaf(x1, cv.y, acc[q]);
        acc[q] = fmaf(x2, cv.z, acc[q]); acc[q] = fmaf(x3, cv.w, acc[q]);
      }
    }
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const int kl = kg * 8 + q;
      if (kl < nk) {
        const ScoreRec r = recs[kl];
        float dx = sx - r.mux, dy = sy - r.muy;
        float y1 = dx * r.u, y2 = fmaf(dy, r.v, -(dx * r.w));
        float qq = fmaf(y1, y1, y2 * y2);
        float sp = squared ? qq : sqrtf(qq);
        float idle = (F.t - r.tau > H.t_idle) ? H.lambda_idle : 0.f;
        float inv = fminf(r.invc * invk, inv_cap);
        float sc = fmaf(-acc[q], inv, sp + idle);
        if (sc < best) { best = sc; bidx = k0 + kl; }   // increasing k within a thread: lowest index on ties
      }
    }
  }
  bestv[kg * kScoreTok + tl] = best;
  besti[kg * kScoreTok + tl] = bidx;
  __syncthreads();
  if (kg == 0 && j < D.T) {
#pragma unroll
    for (int q = 1; q < 8; ++q) {
      float v = bestv[q * kScoreTok + tl];
      int ix = besti[q * kScoreTok + tl];
      if (v < best || (v == best && ix < bidx)) { best = v; bidx = ix; }
    }
    V.assign[(size_t)b * D.T + j] = bidx;
    V.best[(size_t)b * D.T + j] = best;
  }
}

static size_t score_simt_smem(int dh) {
  return (size_t)(dh * kScoreTok + kScoreKc * dh) * 4 + kScoreKc * sizeof(ScoreRec) + 8 * kScoreTok * 8;
}

template <typename T, int DH>
static void score_simt_launch(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, dim3 grid,
                              cudaStream_t s) {
  const size_t sm = score_simt_smem(DH);
  score_simt_kernel<T, DH><<<grid, kScoreThreads, sm, s>>>(D, H, V, F);
}

int launch_score_simt(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, cudaStream_t s) {
  const int ntok = D.T - F.n_fill;
  if (ntok <= 0) return 0;
  dim3 grid((ntok + kScoreTok - 1) / kScoreTok, D.B);
  if (D.bf16) {
    if (D.d == 128) score_simt_launch<__nv_bfloat16, 128>(D, H, V, F, grid, s);
    else score_simt_launch<__nv_bfloat16, 64>(D, H, V, F, grid, s);
  } else {
    if (D.d == 128) score_simt_launch<float, 128>(D, H, V, F, grid, s);
    else score_simt_launch<float, 64>(D, H, V, F, grid, s);
  }
  return 1;
}

// ---------------------------------------------------------------------------------------------------------
// U4 segmenting + U5 prototype update + U6 residual histograms (Alg. 1 l.8-13).
//
// CTA = (chunk, bank).  Every CTA of a bank sorts the bank's (k*, j) keys in shared memory (bitonic; stable in
// eviction order because j is the low part of the key), so that segments = runs of equal k*.  Warps then take
// segment heads round-robin over all CTAs of the bank; one warp owns one prototype: it holds c_k and p_k in
// registers (DH/32 dims per lane) and replays Alg. 1 l.8-13 over its tokens in eviction order.
//
// Arithmetic: the EMA / mean / covariance recurrences are evaluated like the definition reads, in fp64 from the
// fp32 state with one rounding back to fp32 per step (a handful of DFMA-class ops per token and dimension);
// the PQ distances |r_g - C_g[z]|^2 are fp32, reduced over the 32/G lanes that share a subspace.
// ---------------------------------------------------------------------------------------------------------
constexpr int kUpdThreads = 256, kUpdWarps = kUpdThreads / 32;

__device__ __forceinline__ float ema_step(double one_minus, double rate, float state, float x) {
  // (1 - a) * state + a * x with every product and the sum rounded separately (no contraction), then to fp32
  return (float)__dadd_rn(__dmul_rn(one_minus, (double)state), __dmul_rn(rate, (double)x));
}

template <typename T, int DH>
__global__ void __launch_bounds__(kUpdThreads) update_kernel(Dims D, Hyper H, Dev V, FrameArgs F, int P) {
  constexpr int VEC = DH / 32;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint32_t* keys = (uint32_t*)smem_raw;                      // [P]
  float* cbk_s = (float*)(keys + P);                         // [G][C*sub + pad]
  const int gstride = D.C * D.sub + kCbPad;
  float* cbv_s = cbk_s + D.G * gstride;

  const int b = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int ntok = D.T - F.n_fill;
  const bool has_cb = V.cbk != nullptr;
  for (int i = tid; i < P; i += kUpdThreads) {
    const int j = F.n_fill + i;
    uint32_t key = 0xffffffffu;
    if (i < ntok) {
      int a;
      if (F.keys) {   // tcgen05 assignment: (orderable(|K_j| * score) << 32 | k), see tc_assign.cu
        const unsigned long long ak = V.akey[(size_t)b * D.T + j];
        a = (int)(uint32_t)ak;
        if (blockIdx.x == 0) {
          const uint32_t o = (uint32_t)(ak >> 32);
          const float sc = __uint_as_float((o & 0x80000000u) ? (o ^ 0x80000000u) : ~o);
          const float kk = V.ringN[((size_t)b * D.Wf + F.slot) * D.T + j];
          V.assign[(size_t)b * D.T + j] = a;
          V.best[(size_t)b * D.T + j] = kk > 0.f ? sc / sqrtf(kk) : sc;
        }
      } else {
        a = V.assign[(size_t)b * D.T + j];
      }
      if ((uint32_t)a >= (uint32_t)F.n_act) {   // no finite score (non-finite key or bank): not absorbed, flagged
        a = kNoProto;
        if (blockIdx.x == 0) { V.assign[(size_t)b * D.T + j] = -2; atomicOr(V.err, PKV_ERR_UNASSIGNED); }
      }
      key = ((uint32_t)a << 12) | (uint32_t)j;
    }
    keys[i] = key;
  }
  if (has_cb) {
    const int per_g = D.C * D.sub;
    for (int e = tid; e < D.G * per_g; e += kUpdThreads) {
      const int g = e / per_g, r = e % per_g;
      cbk_s[g * gstride + r] = V.cbk[(size_t)b * D.G * per_g + e];
      cbv_s[g * gstride + r] = V.cbv[(size_t)b * D.G * per_g + e];
    }
  }
  __syncthreads();
  for (int size = 2; size <= P; size <<= 1) {
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = tid; i < P / 2; i += kUpdThreads) {
        const int lo = 2 * i - (i & (stride - 1)), hi = lo + stride;
        const bool up = (lo & size) == 0;
        const uint32_t a = keys[lo], c = keys[hi];
        if ((a > c) == up) { keys[lo] = c; keys[hi] = a; }
      }
      __syncthreads();
    }
  }

  const int st = b / (D.L * D.Hkv);
  const T* ringK = (const T*)V.ringK + ((size_t)b * D.Wf + F.slot) * D.T * DH;
  const T* ringV = (const T*)V.ringV + ((size_t)b * D.Wf + F.slot) * D.T * DH;
  const float* ringS = V.ringS + ((size_t)st * D.Wf + F.slot) * D.T * 2;
  const double al = (double)H.alpha, be = (double)H.beta, et = (double)H.eta;
  const double oma = 1.0 - al, omb = 1.0 - be, ome = 1.0 - et;
  const int LPS = 32 / D.G;                       // lanes per PQ subspace
  const int g = lane / LPS, li = lane % LPS;

  for (int i = blockIdx.x * kUpdWarps + warp; i < ntok; i += gridDim.x * kUpdWarps) {
    const uint32_t key = keys[i];
    const int k = (int)(key >> 12);
    if (k == kNoProto) break;                               // unassigned tokens sort last
    if (i > 0 && (int)(keys[i - 1] >> 12) == k) continue;   // not a segment head
    const size_t pk = (size_t)b * D.K + k;
    float c[VEC], p[VEC];
    load_vec<float, VEC>(V.c + pk * DH + lane * VEC, c);
    load_vec<float, VEC>(V.p + pk * DH + lane * VEC, p);
    float mu0 = V.mu[pk * 2], mu1 = V.mu[pk * 2 + 1];
    float sxx = V.sigma[pk * 3], sxy = V.sigma[pk * 3 + 1], syy = V.sigma[pk * 3 + 2];
    int n = V.n[pk];
    int m = 0, jlast = 0, jsum = 0;
    for (int ii = i; ii < ntok && (int)(keys[ii] >> 12) == k; ++ii) {
      const int j = (int)(keys[ii] & 0xfffu);
      float ke[VEC], ve[VEC];
      load_vec<T, VEC>(ringK + (size_t)j * DH + lane * VEC, ke);
      load_vec<T, VEC>(ringV + (size_t)j * DH + lane * VEC, ve);
      const float s0 = ringS[j * 2], s1 = ringS[j * 2 + 1];
#pragma unroll
      for (int v = 0; v < VEC; ++v) {
        c[v] = ema_step(oma, al, c[v], ke[v]);                       // l.8
        p[v] = ema_step(omb, be, p[v], ve[v]);                       // l.9
      }
      n += 1; ++m; jlast = j; jsum += j;                             // l.10
      mu0 = ema_step(ome, et, mu0, s0);                              // l.11
      mu1 = ema_step(ome, et, mu1, s1);
      const double dx = (double)s0 - (double)mu0, dy = (double)s1 - (double)mu1;   // new mu
      const double edx = __dmul_rn(et, dx), edy = __dmul_rn(et, dy);
      sxx = (float)__dadd_rn(__dmul_rn(ome, (double)sxx), __dmul_rn(edx, dx));     // l.12
      sxy = (float)__dadd_rn(__dmul_rn(ome, (double)sxy), __dmul_rn(edx, dy));
      syy = (float)__dadd_rn(__dmul_rn(ome, (double)syy), __dmul_rn(edy, dy));
      if (F.warm) {                                                  // L312: residual of a warm-up step -> reservoir
        const int slot = V.rslot[(size_t)b * D.T + j];
        if (slot >= 0) {
          float* rk = V.resK + ((size_t)b * H.warm_reservoir + slot) * DH + lane * VEC;
          float* rv = V.resV + ((size_t)b * H.warm_reservoir + slot) * DH + lane * VEC;
#pragma unroll
          for (int v = 0; v < VEC; ++v) { rk[v] = ke[v] - c[v]; rv[v] = ve[v] - p[v]; }
        }
      }
      if (has_cb) {                                                  // l.13, residual of the updated centres
#pragma unroll
        for (int kv = 0; kv < 2; ++kv) {
          const float* cb = (kv ? cbv_s : cbk_s) + g * gstride + li * VEC;
          float r[VEC];
#pragma unroll
          for (int v = 0; v < VEC; ++v) r[v] = kv ? ve[v] - p[v] : ke[v] - c[v];
          float bestd = INFINITY;
          int bz = 0;
          for (int z = 0; z < D.C; ++z) {
            float cw[VEC];
            load_vec<float, VEC>(cb + z * D.sub, cw);
            float dist = 0.f;
#pragma unroll
            for (int v = 0; v < VEC; ++v) { const float t = r[v] - cw[v]; dist = fmaf(t, t, dist); }
            for (int o = LPS >> 1; o > 0; o >>= 1) dist += __shfl_xor_sync(0xffffffffu, dist, o);
            if (dist < bestd) { bestd = dist; bz = z; }              // lowest z on ties
          }
          if (li == 0) {
            atomicAdd(V.hist + ((pk * 2 + kv) * D.G + g) * D.C + bz, 1u);
            (kv ? V.tcodeV : V.tcodeK)[((size_t)b * D.T + j) * D.G + g] = (uint8_t)bz;
          }
        }
      }
    }
    // write back the prototype and everything derived from it
    if (VEC == 4) {
      *(float4*)(V.c + pk * DH + lane * 4) = make_float4(c[0], c[1], c[2], c[VEC - 1]);
      *(float4*)(V.p + pk * DH + lane * 4) = make_float4(p[0], p[1], p[2], p[VEC - 1]);
    } else {
      *(float2*)(V.c + pk * DH + lane * 2) = make_float2(c[0], c[1]);
      *(float2*)(V.p + pk * DH + lane * 2) = make_float2(p[0], p[1]);
    }
    float cc = 0.f;
#pragma unroll
    for (int v = 0; v < VEC; ++v) cc = fmaf(c[v], c[v], cc);
    cc = warp_sum(cc);
    store_shadows<VEC>(V, pk * DH + lane * VEC, c, inv_norm(cc));
    store_bf16_copy<VEC>(V.c_bf, pk * DH + lane * VEC, c);
    store_bf16_copy<VEC>(V.p_bf, pk * DH + lane * VEC, p);
    if (lane == 0) {
      V.n[pk] = n;
      V.tau[pk] = F.t;
      const long long ps0 = H.pos0 + (long long)F.ev_frame * D.T;
      V.pos[pk] = ps0 + jlast;
      V.pos_sum[pk] += ps0 * m + jsum; V.pos_cnt[pk] += m;
      V.mu[pk * 2] = mu0; V.mu[pk * 2 + 1] = mu1;
      V.sigma[pk * 3] = sxx; V.sigma[pk * 3 + 1] = sxy; V.sigma[pk * 3 + 2] = syy;
      if (has_cb) V.nres[pk] += (uint32_t)m;
      store_rec(V.rec, pk, make_rec(cc, mu0, mu1, sxx, sxy, syy, F.t, H));
      V.logn[pk] = log_mass(n);
      V.mstamp[pk] = F.t;
      mark_dirty(D, V, b, k, F.epoch);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// U4-U6, specialised for the production shape (head_dim 128, G = 8, C = 16; bf16 or fp32 tokens).
//
// CTA = (split, bank), 8 warps.  Every CTA of a bank orders the bank's (k*, j) keys by rank counting (key distinct,
// rank = number of smaller keys: T^2 broadcast compares instead of a bitonic network), marks segment heads, scans
// them into a segment table, and the warps of all CTAs of the bank take segments round-robin.  A warp owns one
// prototype (4 dims per lane, so the 4 lanes [4g, 4g+4) hold PQ subspace g) and replays Alg. 1 l.8-13 over its tokens
// in eviction order with the next token's K/V prefetched.  PQ search: the residual is exchanged through a per-warp
// shared scratch so that every lane holds its subspace's 16 dims, lane (g, li) evaluates codewords li, li+4, li+8,
// li+12 in full (no shuffles inside the distance), and a 2-step lexicographic (distance, code) min over the 4 lanes
// picks the codeword.  Codebooks sit in shared memory as [g][q][z] float4 with a 4-unit pad per g: the 8 lanes of a
// quarter warp then read 8 distinct 16-byte bank groups.
// ---------------------------------------------------------------------------------------------------------
constexpr int kUfThreads = 256, kUfWarps = kUfThreads / 32;
constexpr int kCbG = 68;   // float4 units per subspace block: 4 q x 16 z + 4 pad

// packed fp32 pairs (sm_100 f32x2): one issue slot for two FMAs
__device__ __forceinline__ uint64_t uf_pack2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ uint64_t uf_fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}

// Nearest codeword of subspace g to the residual (reading 10: squared L2, lowest index on ties) in the expanded form
// argmin_z |C[z]|^2 - 2 r.C[z] (|r|^2 is common to all z): 8 packed FMAs per codeword instead of a subtract and an
// FMA per dimension.  Lane (g, li) evaluates codewords li, li+4, li+8, li+12; a 2-step lexicographic (score, code)
// min over the 4 lanes of the subspace picks the codeword.  cn = |C[z]|^2 per (g, z).
__device__ __forceinline__ void pq_pick(const float4* __restrict__ cb4, const float* __restrict__ cn,
                                        const float4* __restrict__ rsc, int g, int li, int& code) {
  uint64_t r2[8];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const float4 r = rsc[g * 4 + q];
    r2[2 * q] = uf_pack2(-2.f * r.x, -2.f * r.y);
    r2[2 * q + 1] = uf_pack2(-2.f * r.z, -2.f * r.w);
  }
  float bestd = INFINITY;
  int bz = 0;
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const int z = li + 4 * t;
    uint64_t acc = uf_pack2(cn[g * 16 + z], 0.f);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const float4 cw = cb4[g * kCbG + q * 16 + z];
      acc = uf_fma2(r2[2 * q], uf_pack2(cw.x, cw.y), acc);
      acc = uf_fma2(r2[2 * q + 1], uf_pack2(cw.z, cw.w), acc);
    }
    float a0, a1;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a0), "=f"(a1) : "l"(acc));
    const float dist = a0 + a1;
    if (dist < bestd) { bestd = dist; bz = z; }           // increasing z within the lane: lowest z on ties
  }
#pragma unroll
  for (int o = 1; o <= 2; o <<= 1) {
    const float od = __shfl_xor_sync(0xffffffffu, bestd, o);
    const int oz = __shfl_xor_sync(0xffffffffu, bz, o);
    if (od < bestd || (od == bestd && oz < bz)) { bestd = od; bz = oz; }
  }
  code = bz;
}

template <typename T>
__global__ void __launch_bounds__(kUfThreads, 4) update_fast_kernel(Dims D, Hyper H, Dev V, FrameArgs F, int Tpad) {
  constexpr int DH = 128;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* cbk4 = (float4*)smem_raw;                           // [8][68]
  float4* cbv4 = cbk4 + 8 * kCbG;
  float4* scratch = cbv4 + 8 * kCbG;                          // [warps][2][32]
  float* cnk = (float*)(scratch + kUfWarps * 64);             // [8][16] |C^K_g[z]|^2
  float* cnv = cnk + 128;
  uint32_t* keys = (uint32_t*)(cnv + 128);                    // [Tpad]
  uint32_t* sorted = keys + Tpad;                             // [Tpad]
  int* segstart = (int*)(sorted + Tpad);                      // [Tpad + 1]
  __shared__ int wtot[kUfWarps];
  __shared__ int nseg_s, nmine_s, next_task_s;

  const int b = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int ntok_all = D.T - F.n_fill;
  const bool has_cb = V.cbk != nullptr;
  const size_t bt = (size_t)b * D.T;
  const size_t rrow = ((size_t)b * D.Wf + F.slot) * D.T;      // ring row of evicted token 0
  if (tid == 0) { nmine_s = 0; next_task_s = 0; }
  if (has_cb) {   // codebooks: not written by any kernel of the frame chain, so loaded ahead of pdl_wait()
    const float4* sk = (const float4*)(V.cbk + (size_t)b * 2048);
    const float4* sv = (const float4*)(V.cbv + (size_t)b * 2048);
    for (int e = tid; e < 512; e += kUfThreads) {             // e = (g * 16 + z) * 4 + q
      const int q = e & 3, z = (e >> 2) & 15, g = e >> 6;
      cbk4[g * kCbG + q * 16 + z] = sk[e];
      cbv4[g * kCbG + q * 16 + z] = sv[e];
    }
  }
  pdl_wait();      // the assignment of this frame (score kernel) is complete and visible
  pdl_trigger();   // the ring append may fetch the new frame's rows while this kernel runs
  __syncthreads();
  // CTA x of the bank's gridDim.x CTAs owns the prototypes k with k mod gridDim.x == x: it keeps only the tokens
  // assigned to those, so that the sort below is over ~T / gridDim.x keys instead of T in every CTA
  for (int i = tid; i < ntok_all; i += kUfThreads) {
    const int j = F.n_fill + i;
    int a;
    if (F.keys) {   // tcgen05 assignment: (orderable(|K_j| * score) << 32 | k), see tc_assign.cu
      const unsigned long long ak = V.akey[bt + j];
      a = (int)(uint32_t)ak;
      if (blockIdx.x == 0) {
        const uint32_t o = (uint32_t)(ak >> 32);
        const float sc = __uint_as_float((o & 0x80000000u) ? (o ^ 0x80000000u) : ~o);
        const float kk = V.ringN[rrow + j];
        V.assign[bt + j] = a;
        V.best[bt + j] = kk > 0.f ? sc / sqrtf(kk) : sc;
      }
    } else {
      a = V.assign[bt + j];
    }
    if ((uint32_t)a >= (uint32_t)F.n_act) {   // no finite score (non-finite key or bank): not absorbed, flagged
      if (blockIdx.x == 0) { V.assign[bt + j] = -2; atomicOr(V.err, PKV_ERR_UNASSIGNED); }
    } else if ((uint32_t)a % gridDim.x == blockIdx.x) {
      keys[atomicAdd(&nmine_s, 1)] = ((uint32_t)a << 12) | (uint32_t)j;   // any order: the keys are distinct
    }
  }
  __syncthreads();
  if (has_cb) {                                               // codeword norms: thread = (side, g, z)
    const int side = tid >> 7, gz = tid & 127, gg = gz >> 4, z = gz & 15;
    const float4* cb = side ? cbv4 : cbk4;
    float n2 = 0.f;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const float4 cw = cb[gg * kCbG + q * 16 + z];
      n2 = fmaf(cw.x, cw.x, n2); n2 = fmaf(cw.y, cw.y, n2); n2 = fmaf(cw.z, cw.z, n2); n2 = fmaf(cw.w, cw.w, n2);
    }
    (side ? cnv : cnk)[gz] = n2;
  }
  // ---- U4: rank counting sort of this CTA's keys, segment heads, segment table ----
  const int ntok = nmine_s;
  for (int i = tid; i < ntok; i += kUfThreads) {
    const uint32_t my = keys[i];
    int r = 0;
    int i2 = 0;
    for (; i2 + 4 <= ntok; i2 += 4) {
      const uint4 kq = *(const uint4*)(keys + i2);
      r += (kq.x < my) + (kq.y < my) + (kq.z < my) + (kq.w < my);
    }
    for (; i2 < ntok; ++i2) r += keys[i2] < my;
    sorted[r] = my;
  }
  __syncthreads();
  int base = 0;
  for (int r0 = 0; r0 < ntok; r0 += kUfThreads) {
    const int r = r0 + tid;
    const bool head = r < ntok && (r == 0 || (sorted[r] >> 12) != (sorted[r - 1] >> 12));
    const uint32_t bal = __ballot_sync(0xffffffffu, head);
    if (lane == 0) wtot[warp] = __popc(bal);
    __syncthreads();
    int off = base, tot = 0;
#pragma unroll
    for (int w = 0; w < kUfWarps; ++w) { const int c = wtot[w]; if (w < warp) off += c; tot += c; }
    if (head) segstart[off + __popc(bal & ((1u << lane) - 1u))] = r;
    base += tot;
    __syncthreads();
  }
  if (tid == 0) { segstart[base] = ntok; nseg_s = base; }
  __syncthreads();
  const int nseg = nseg_s;

  // ---- U5 / U6 ----
  const int st = b / (D.L * D.Hkv);
  const T* ringK = (const T*)V.ringK + rrow * DH;
  const T* ringV = (const T*)V.ringV + rrow * DH;
  const float* ringS = V.ringS + ((size_t)st * D.Wf + F.slot) * D.T * 2;
  const double et = (double)H.eta, ome = 1.0 - et;
  const float alf = H.alpha, bef = H.beta;
  const int g = lane >> 2, li = lane & 3;
  float4* rsc = scratch + warp * 64;

  // A task = (segment, side): the key side replays c, mu, Sigma and the K histogram, the value side p and the V
  // histogram -- two independent dependency chains, so a segment's latency is that of the longer one
  // tasks are handed out dynamically (one shared counter per CTA): segments differ in length and the key side is the
  // heavier one, so a static round-robin leaves the CTA waiting for its unluckiest warp
  for (;;) {
    int task = 0;
    if (lane == 0) task = atomicAdd(&next_task_s, 1);
    task = __shfl_sync(0xffffffffu, task, 0);
    if (task >= 2 * nseg) break;
    const int seg = task >> 1, side = task & 1;
    const int r0 = segstart[seg], r1 = segstart[seg + 1];
    const int k = (int)(sorted[r0] >> 12);
    const size_t pk = (size_t)b * D.K + k;
    int jn = (int)(sorted[r0] & 0xfffu);
    if (side) {                                                        // ---- value side: l.9 and the V half of l.13
      float p[4], ven[4];
      load_vec<float, 4>(V.p + pk * DH + lane * 4, p);
      load_vec<T, 4>(ringV + (size_t)jn * DH + lane * 4, ven);
      for (int r = r0; r < r1; ++r) {
        const int j = jn;
        float ve[4];
#pragma unroll
        for (int v = 0; v < 4; ++v) ve[v] = ven[v];
        if (r + 1 < r1) {
          jn = (int)(sorted[r + 1] & 0xfffu);
          load_vec<T, 4>(ringV + (size_t)jn * DH + lane * 4, ven);
        }
#pragma unroll
        for (int v = 0; v < 4; ++v) p[v] = fmaf(bef, ve[v] - p[v], p[v]);              // l.9
        if (F.warm) {                                                // L312: residual of a warm-up step -> reservoir
          const int slot = V.rslot[bt + j];
          if (slot >= 0)
            *(float4*)(V.resV + ((size_t)b * H.warm_reservoir + slot) * DH + lane * 4) =
                make_float4(ve[0] - p[0], ve[1] - p[1], ve[2] - p[2], ve[3] - p[3]);
        }
        if (has_cb) {
          __syncwarp();
          rsc[lane] = make_float4(ve[0] - p[0], ve[1] - p[1], ve[2] - p[2], ve[3] - p[3]);
          __syncwarp();
          int zv;
          pq_pick(cbv4, cnv, rsc, g, li, zv);
          if (li == 0) {
            atomicAdd(V.hist + ((pk * 2 + 1) * 8 + g) * 16 + zv, 1u);
            V.tcodeV[(bt + j) * 8 + g] = (uint8_t)zv;
          }
        }
      }
      *(float4*)(V.p + pk * DH + lane * 4) = make_float4(p[0], p[1], p[2], p[3]);
      store_bf16_copy<4>(V.p_bf, pk * DH + lane * 4, p);
      continue;
    }
    // ---- key side: l.8, l.10-12, the K half of l.13 and everything derived from the prototype
    float c[4];
    load_vec<float, 4>(V.c + pk * DH + lane * 4, c);
    const float2 mu2 = *(const float2*)(V.mu + pk * 2);
    float mu0 = mu2.x, mu1 = mu2.y;
    float sxx = V.sigma[pk * 3], sxy = V.sigma[pk * 3 + 1], syy = V.sigma[pk * 3 + 2];
    const int n_old = V.n[pk];                                       // read now: the write-back must not wait for them
    const uint32_t nres_old = has_cb ? V.nres[pk] : 0u;
    const long long psum_old = V.pos_sum[pk];
    const int pcnt_old = V.pos_cnt[pk];
    int jsum = 0;
    float ken[4];
    load_vec<T, 4>(ringK + (size_t)jn * DH + lane * 4, ken);
    float2 sn = *(const float2*)(ringS + jn * 2);
    int j = jn;
    for (int r = r0; r < r1; ++r) {
      j = jn;
      jsum += j;
      float ke[4];
#pragma unroll
      for (int v = 0; v < 4; ++v) ke[v] = ken[v];
      const float s0 = sn.x, s1 = sn.y;
      if (r + 1 < r1) {                                              // prefetch the next token of the segment
        jn = (int)(sorted[r + 1] & 0xfffu);
        load_vec<T, 4>(ringK + (size_t)jn * DH + lane * 4, ken);
        sn = *(const float2*)(ringS + jn * 2);
      }
#pragma unroll
      for (int v = 0; v < 4; ++v) c[v] = fmaf(alf, ke[v] - c[v], c[v]);                // l.8  (1 - a) c + a K  =  c + a (K - c)
      mu0 = ema_step(ome, et, mu0, s0);                              // l.11
      mu1 = ema_step(ome, et, mu1, s1);
      const double dx = (double)s0 - (double)mu0, dy = (double)s1 - (double)mu1;   // new mu
      const double edx = __dmul_rn(et, dx), edy = __dmul_rn(et, dy);
      sxx = (float)__dadd_rn(__dmul_rn(ome, (double)sxx), __dmul_rn(edx, dx));     // l.12
      sxy = (float)__dadd_rn(__dmul_rn(ome, (double)sxy), __dmul_rn(edx, dy));
      syy = (float)__dadd_rn(__dmul_rn(ome, (double)syy), __dmul_rn(edy, dy));
      if (F.warm) {                                                  // L312: residual of a warm-up step -> reservoir
        const int slot = V.rslot[bt + j];
        if (slot >= 0)
          *(float4*)(V.resK + ((size_t)b * H.warm_reservoir + slot) * DH + lane * 4) =
              make_float4(ke[0] - c[0], ke[1] - c[1], ke[2] - c[2], ke[3] - c[3]);
      }
      if (has_cb) {                                                  // l.13, residual of the updated centre
        __syncwarp();
        rsc[lane] = make_float4(ke[0] - c[0], ke[1] - c[1], ke[2] - c[2], ke[3] - c[3]);
        __syncwarp();
        int zk;
        pq_pick(cbk4, cnk, rsc, g, li, zk);
        if (li == 0) {
          atomicAdd(V.hist + ((pk * 2 + 0) * 8 + g) * 16 + zk, 1u);
          V.tcodeK[(bt + j) * 8 + g] = (uint8_t)zk;
        }
      }
    }
    // write back the prototype and everything derived from it
    *(float4*)(V.c + pk * DH + lane * 4) = make_float4(c[0], c[1], c[2], c[3]);
    float cc = 0.f;
#pragma unroll
    for (int v = 0; v < 4; ++v) cc = fmaf(c[v], c[v], cc);
    cc = warp_sum(cc);
    store_shadows<4>(V, pk * DH + lane * 4, c, inv_norm(cc));
    store_bf16_copy<4>(V.c_bf, pk * DH + lane * 4, c);
    if (lane == 0) {
      const int m = r1 - r0;
      const int n = n_old + m;                                       // l.10
      V.n[pk] = n;
      V.tau[pk] = F.t;
      const long long ps0 = H.pos0 + (long long)F.ev_frame * D.T;
      V.pos[pk] = ps0 + j;
      V.pos_sum[pk] = psum_old + ps0 * m + jsum; V.pos_cnt[pk] = pcnt_old + m;       // D.1 anchors
      *(float2*)(V.mu + pk * 2) = make_float2(mu0, mu1);
      V.sigma[pk * 3] = sxx; V.sigma[pk * 3 + 1] = sxy; V.sigma[pk * 3 + 2] = syy;
      if (has_cb) V.nres[pk] = nres_old + (uint32_t)m;
      store_rec(V.rec, pk, make_rec(cc, mu0, mu1, sxx, sxy, syy, F.t, H));
      V.logn[pk] = log_mass(n);
      V.mstamp[pk] = F.t;
      mark_dirty(D, V, b, k, F.epoch);
    }
  }
}

static int next_pow2(int x) { int p = 2; while (p < x) p <<= 1; return p; }

static size_t update_fast_smem(int ntok) {
  const int Tpad = (ntok + 3) / 4 * 4;
  return (size_t)(2 * 8 * kCbG + kUfWarps * 64) * 16 + 256 * 4 + (size_t)(3 * Tpad + 1) * 4;
}
static size_t update_generic_smem(const Dims& D, int ntok) {
  return (size_t)next_pow2(ntok) * 4 + 2 * (size_t)D.G * (D.C * D.sub + kCbPad) * 4;
}

template <typename K> static bool set_smem(K kernel, size_t bytes) {
  if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) == cudaSuccess) return true;
  cudaGetLastError();
  return false;
}

bool update_kernels_prepare(const Dims& D0) {
  // function attributes are per device, not per state: size for the largest frame / PQ shape protokv_create admits
  Dims D = D0;
  D.T = kMaxT; D.G = kMaxG; D.C = kMaxC; D.sub = 128 / kMaxG;   // G (C sub + pad) is largest at G = 8
  bool ok = true;
  ok &= set_smem(score_simt_kernel<__nv_bfloat16, 128>, score_simt_smem(128));
  ok &= set_smem(score_simt_kernel<__nv_bfloat16, 64>, score_simt_smem(64));
  ok &= set_smem(score_simt_kernel<float, 128>, score_simt_smem(128));
  ok &= set_smem(score_simt_kernel<float, 64>, score_simt_smem(64));
  const size_t uf = update_fast_smem(D.T), ug = update_generic_smem(D, D.T);
  ok &= set_smem(update_fast_kernel<__nv_bfloat16>, uf);
  ok &= set_smem(update_fast_kernel<float>, uf);
  ok &= set_smem(update_kernel<__nv_bfloat16, 128>, ug);
  ok &= set_smem(update_kernel<__nv_bfloat16, 64>, ug);
  ok &= set_smem(update_kernel<float, 128>, ug);
  ok &= set_smem(update_kernel<float, 64>, ug);
  return ok;
}

int launch_update(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, int sm_count, cudaStream_t s) {
  const int ntok = D.T - F.n_fill;
  if (ntok <= 0) return 0;
  if (D.d == 128 && D.G == 8 && D.C == 16) {
    const int Tpad = (ntok + 3) / 4 * 4;
    const size_t sm = update_fast_smem(ntok);
    int nsplit = 4 * sm_count / D.B;
    const int max_split = (ntok + 2 * kUfWarps - 1) / (2 * kUfWarps);
    if (nsplit > max_split) nsplit = max_split;
    if (nsplit < 1) nsplit = 1;
    dim3 grid(nsplit, D.B);
    if (D.bf16) launch_chain(update_fast_kernel<__nv_bfloat16>, grid, kUfThreads, sm, s, F.pdl != 0, D, H, V, F, Tpad);
    else launch_chain(update_fast_kernel<float>, grid, kUfThreads, sm, s, F.pdl != 0, D, H, V, F, Tpad);
    return 1;
  }
  const int P = next_pow2(ntok);
  int nchunk = (2 * sm_count + D.B - 1) / D.B;
  nchunk = nchunk < 1 ? 1 : nchunk;
  const int max_chunk = (ntok + kUpdWarps - 1) / kUpdWarps;
  if (nchunk > max_chunk) nchunk = max_chunk;
  if (nchunk > 32) nchunk = 32;
  const size_t sm = update_generic_smem(D, ntok);
  dim3 grid(nchunk, D.B);
  if (D.bf16) {
    if (D.d == 128) update_kernel<__nv_bfloat16, 128><<<grid, kUpdThreads, sm, s>>>(D, H, V, F, P);
    else update_kernel<__nv_bfloat16, 64><<<grid, kUpdThreads, sm, s>>>(D, H, V, F, P);
  } else {
    if (D.d == 128) update_kernel<float, 128><<<grid, kUpdThreads, sm, s>>>(D, H, V, F, P);
    else update_kernel<float, 64><<<grid, kUpdThreads, sm, s>>>(D, H, V, F, P);
  }
  return 1;
}

// ---------------------------------------------------------------------------------------------------------
// Derived per-prototype data (scoring record, log-mass, bf16 shadows) recomputed from the primary state of one
// bank -- used after protokv_import_state.  One warp per prototype.
// ---------------------------------------------------------------------------------------------------------
__global__ void refresh_derived_kernel(Dims D, Hyper H, Dev V, int b, int epoch) {
  const int k = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (k >= D.K) return;
  const size_t pk = (size_t)b * D.K + k;
  float cc = 0.f;
  const int vec = D.d / 32;   // same per-lane order as update_kernel so that derived values are reproduced bit for bit
  for (int v = 0; v < vec; ++v) {
    const float x = V.c[pk * D.d + lane * vec + v];
    cc = fmaf(x, x, cc);
  }
  cc = warp_sum(cc);
  if (V.c_hi) {
    const float invc = inv_norm(cc);
    for (int v = 0; v < vec; ++v) {
      const int i = lane * vec + v;
      __nv_bfloat16 hi, lo;
      split_bf16(V.c[pk * D.d + i] * invc, hi, lo);
      V.c_hi[pk * D.d + i] = hi; V.c_lo[pk * D.d + i] = lo;
    }
  }
  if (V.c_bf)
    for (int i = lane; i < D.d; i += 32) {
      V.c_bf[pk * D.d + i] = __float2bfloat16_rn(V.c[pk * D.d + i]);
      V.p_bf[pk * D.d + i] = __float2bfloat16_rn(V.p[pk * D.d + i]);
    }
  if (lane == 0) {
    store_rec(V.rec, pk, make_rec(cc, V.mu[pk * 2], V.mu[pk * 2 + 1], V.sigma[pk * 3], V.sigma[pk * 3 + 1],
                         V.sigma[pk * 3 + 2], V.tau[pk], H));
    const int n = V.n[pk];
    V.logn[pk] = log_mass(n);
    mark_dirty(D, V, b, k, epoch);
  }
}

__global__ void fill_u32_kernel(uint32_t* dst, uint32_t value, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = value;
}
int launch_fill_u32(uint32_t* dst, uint32_t value, size_t n, cudaStream_t s) {
  if (n == 0) return 0;
  const unsigned grid = (unsigned)((n + 255) / 256 < 1024 ? (n + 255) / 256 : 1024);
  fill_u32_kernel<<<grid, 256, 0, s>>>(dst, value, n);
  return 1;
}

__global__ void codebook_copy_kernel(__nv_bfloat16* dst, const float* cbk, const float* cbv, size_t per_bank, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t b = i / (2 * per_bank), r = i % (2 * per_bank);
    dst[i] = __float2bfloat16_rn(r < per_bank ? cbk[b * per_bank + r] : cbv[b * per_bank + r - per_bank]);
  }
}
int launch_codebook_copy(const Dims& D, const Dev& V, const float* cbk, const float* cbv, cudaStream_t s) {
  if (!V.cb_bf || !cbk) return 0;
  const size_t per_bank = (size_t)D.G * D.C * D.sub, n = (size_t)D.B * 2 * per_bank;
  codebook_copy_kernel<<<(unsigned)((n + 255) / 256 < 1024 ? (n + 255) / 256 : 1024), 256, 0, s>>>(V.cb_bf, cbk, cbv, per_bank, n);
  return 1;
}

__global__ void or_u32_kernel(uint32_t* dst, uint32_t bits) { atomicOr(dst, bits); }
int launch_or_u32(uint32_t* dst, uint32_t bits, cudaStream_t s) {
  or_u32_kernel<<<1, 1, 0, s>>>(dst, bits);
  return 1;
}

int launch_refresh_derived(const Dims& D, const Hyper& H, const Dev& V, int bank, int epoch, cudaStream_t s) {
  refresh_derived_kernel<<<(D.K + 7) / 8, 256, 0, s>>>(D, H, V, bank, epoch);
  return 1;
}

}  // namespace pkv
