// Q2 fused attention for DECODE-STYLE queries, register-resident variant (bf16, d = 128, S = 8, G = 8, C = 16,
// n_q * group <= 16 query rows per bank): Alg. 4 l.8-15 / Eq. 4 (L574: the bounded attention
// over W + K_max S tokens is the only ProtoKV work on the latency of a query).  For a handful of rows that is ~2.7 MB per
// bank streamed once, i.e. HBM time; the kernel is built so that nothing but those bytes moves:
//
//   * every warp is its own flash-decoding worker over a strided share of the bank's context: it streams its units (16
//     ring rows, or 8 prototypes) through a private cp.async ring in shared memory -- no block barrier in the loop -- and
//     fills the mma.sync m16n8k16 operand fragments from there with plain 16-byte loads (chunks are XOR-swizzled at
//     staging so that these loads are bank-conflict free).  The contraction index of Q K^T may be permuted freely, so a
//     lane's four pieces of a key row are whole 16-byte chunks (chunk q = j + 4c holds dims [8q, 8q + 8) = k-steps 2c and
//     2c + 1); the query fragments use the same permutation.  For P V the output dims are permuted instead (a lane owns
//     dims [16 g, 16 g + 16) of its four value rows), and PRMTs pair two rows per operand register;
//   * pseudo-tokens k~ = c_k + concat_g CK_g[z], v~ = p_k + concat_g CV_g[z] (Alg. 4 l.5-9) exist only as B fragments:
//     the lane takes its chunks of bf16(c_k) / bf16(p_k) (copies kept by the update path), adds its 16-byte pieces of
//     the selected codewords from a 4 KB bf16 codebook in shared memory (add.rn.bf16x2 -- the same rounding as the
//     tcgen05 kernel's builders), and feeds the MMA.  With the value-side dim permutation a lane's dims [16 g, 16 g + 16) are exactly PQ subspace g;
//   * online softmax in the accumulator fragments (exp2 domain, log-mass bias log2 n_k on pseudo columns, Eq. 2/4), P
//     re-used from the accumulators as the A fragment of P V (FlashAttention-2 register reuse).
// A CTA's four warps merge their (m, l, O) through shared memory and write one unnormalised partial per query row;
// attention_combine_kernel (query_kernels.cu) merges the nsplit partials of a row.
// Two kernels: attention_decode2_kernel (9-16 rows: query rows = MMA M, padded to 16) and attention_decode8_kernel
// (<= 8 rows: context columns = MMA M, rows = N = 8; its ROPE / RAGGED variants serve PROTOKV_ROPE / PROTOKV_VAR_ALLOC
// states for queries of any length as 8-row blocks).  Measured history: profiles/r02_decode.md.
#include "common.cuh"

namespace pkv {

constexpr int kD2Threads = 128, kD2Warps = 4;
constexpr int kD2Rows = 16;
constexpr int kD2CtasPerSm = 2;
constexpr float kD2Log2e = 1.4426950408889634f;
constexpr float kD2Ln2 = 0.6931471805599453f;
constexpr float kD2Slack = 8.f;

struct D2Smem {
  static constexpr uint32_t CBK = 0;                     // [G][C][16] bf16 = 128 rows x 32 B
  static constexpr uint32_t CBV = 4096;                  // the same at a 48-byte pitch: a quarter warp gathers up to 8 different
                                                         // value codewords, which then fall into different bank groups
  static constexpr uint32_t O = 10240;                    // [4 warps][16 rows][128] fp32 (re-uses the operand ring)
  static constexpr uint32_t ML = O + 4 * 16 * 128 * 4;   // [4][16][2] fp32
  static constexpr uint32_t Total = ML + 4 * 16 * 2 * 4;
};

struct D2Args {
  const __nv_bfloat16* Q;
  float* part;              // [(bsel * R + row) * nsplit + split][130]
  int n_q, layer_begin, layer_count;
  int n_near, n_act;
  int use_bias;
  int nsplit;
  int R;                    // n_q * group
};

__device__ __forceinline__ void d2_mma(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
               "{%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t d2_pack(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ uint32_t d2_add2(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("add.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
__device__ __forceinline__ float d2_ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t d2_prmt(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t r;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(sel));
  return r;
}
__device__ __forceinline__ uint4 d2_ldg16(const void* p) { return __ldg(reinterpret_cast<const uint4*>(p)); }
__device__ __forceinline__ uint4 d2_add2x4(uint4 a, uint4 b) {
  return make_uint4(d2_add2(a.x, b.x), d2_add2(a.y, b.y), d2_add2(a.z, b.z), d2_add2(a.w, b.w));
}
// 8 consecutive fp32 -> 4 bf16x2
__device__ __forceinline__ uint4 d2_cvt8(const float* p) {
  const float4 f0 = __ldg(reinterpret_cast<const float4*>(p)), f1 = __ldg(reinterpret_cast<const float4*>(p) + 1);
  return make_uint4(d2_pack(f0.x, f0.y), d2_pack(f0.z, f0.w), d2_pack(f1.x, f1.y), d2_pack(f1.z, f1.w));
}

// Per-warp flash-decoding state: rows g and g + 8 of the 16-row MMA tile.
struct D2Soft {
  float m0, m1, l0, l1;
};

// One step over 16 context columns.  x0 / x1: logits (log2 domain, bias and mask applied) of column groups 0 / 1 in
// accumulator layout (c0, c1: row g; c2, c3: row g + 8).  Returns P as the A fragment of the P V MMAs.
__device__ __forceinline__ void d2_softmax(D2Soft& s, float (&o)[16][4], const float (&x0)[4], const float (&x1)[4],
                                           uint32_t (&pa)[4]) {
  float mx0 = fmaxf(fmaxf(x0[0], x0[1]), fmaxf(x1[0], x1[1]));
  float mx1 = fmaxf(fmaxf(x0[2], x0[3]), fmaxf(x1[2], x1[3]));
  mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1)); mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
  mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1)); mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
  // The reference maximum of a row moves only when a step's maximum exceeds it by more than kD2Slack (P <= 2^kD2Slack is
  // harmless in bf16 / fp32), so that the rescale of the 64 O accumulators is rare instead of once per early step.
  const float mn0 = mx0 > s.m0 + kD2Slack ? mx0 : s.m0, mn1 = mx1 > s.m1 + kD2Slack ? mx1 : s.m1;   // m = -inf: moves on any finite
  const float mu0 = mn0 == -INFINITY ? 0.f : mn0, mu1 = mn1 == -INFINITY ? 0.f : mn1;   // all masked so far
  const float a0 = d2_ex2(s.m0 - mu0), a1 = d2_ex2(s.m1 - mu1);   // m = -inf: 0
  s.m0 = mn0; s.m1 = mn1;
  const float p00 = d2_ex2(x0[0] - mu0), p01 = d2_ex2(x0[1] - mu0), p02 = d2_ex2(x0[2] - mu1), p03 = d2_ex2(x0[3] - mu1);
  const float p10 = d2_ex2(x1[0] - mu0), p11 = d2_ex2(x1[1] - mu0), p12 = d2_ex2(x1[2] - mu1), p13 = d2_ex2(x1[3] - mu1);
  s.l0 = fmaf(s.l0, a0, (p00 + p01) + (p10 + p11));
  s.l1 = fmaf(s.l1, a1, (p02 + p03) + (p12 + p13));
  if (__any_sync(0xffffffffu, a0 != 1.f || a1 != 1.f)) {
#pragma unroll
    for (int i = 0; i < 16; ++i) { o[i][0] *= a0; o[i][1] *= a0; o[i][2] *= a1; o[i][3] *= a1; }
  }
  pa[0] = d2_pack(p00, p01); pa[1] = d2_pack(p02, p03);
  pa[2] = d2_pack(p10, p11); pa[3] = d2_pack(p12, p13);
}

// O += P V for 16 context rows: v[t][0..7] = the lane's 16 dims [16 g, 16 g + 16) of value row t (t = 0, 1: columns
// 2j, 2j + 1 of group 0; t = 2, 3: of group 1) as bf16 pairs; MMA tile i pairs dim 16 g + i of two rows.
__device__ __forceinline__ void d2_pv(float (&o)[16][4], const uint32_t (&pa)[4], const uint32_t (&v)[4][8]) {
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const uint32_t sel = (i & 1) ? 0x7632u : 0x5410u;
    const uint32_t b0 = d2_prmt(v[0][i >> 1], v[1][i >> 1], sel);
    const uint32_t b1 = d2_prmt(v[2][i >> 1], v[3][i >> 1], sel);
    d2_mma(o[i], pa, b0, b1);
  }
}

// Per-warp operand ring: every warp streams its own units (16 ring rows, or 8 prototypes) through kD2Stages stages
// with cp.async -- two units in flight while one is consumed, no block barrier.
constexpr int kD2Stages = 3;
constexpr uint32_t kD2StageBytes = 8768;
struct D2Stage {   // byte offsets inside a stage
  static constexpr uint32_t K = 0, Vv = 4096;                                           // near unit: 16 rows x 256 B each
  static constexpr uint32_t C = 0, P = 4096, ZK = 8192, ZV = 8448, LN = 8704, KD = 8736;  // far unit: 8 prototypes
};
constexpr uint32_t kD2Ring = 10240;                                                      // after the two codebooks
constexpr uint32_t kD2SmemTotal = kD2Ring + kD2Warps * kD2Stages * kD2StageBytes;        // 113,408 B: two CTAs per SM
static_assert(kD2Warps * kD2Stages * kD2StageBytes >= D2Smem::Total - D2Smem::O, "merge buffer must fit in the ring");

__device__ __forceinline__ void d2_cp16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void d2_cp4(uint32_t dst, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void d2_cp8(uint32_t dst, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ uint4 d2_cvt8s(const unsigned char* p) {    // 8 fp32 in shared memory -> 4 bf16x2
  const float4 f0 = *reinterpret_cast<const float4*>(p), f1 = *reinterpret_cast<const float4*>(p + 16);
  return make_uint4(d2_pack(f0.x, f0.y), d2_pack(f0.z, f0.w), d2_pack(f1.x, f1.y), d2_pack(f1.z, f1.w));
}

__global__ void __launch_bounds__(kD2Threads, kD2CtasPerSm) attention_decode2_kernel(Dims D, Dev V, D2Args A) {
  extern __shared__ __align__(16) unsigned char sm[];
  pdl_wait();   // launched under the tail of the previous kernel of the stream (see common.cuh); no early trigger of its own
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, j = lane & 3;
  const int bsel = blockIdx.y, split = blockIdx.x;
  const int hd = bsel % D.Hkv, ll = (bsel / D.Hkv) % A.layer_count, st = bsel / (D.Hkv * A.layer_count);
  const int b = (st * D.L + A.layer_begin + ll) * D.Hkv + hd;
  const bool has_cb = V.cbk != nullptr;

  // ---- this warp's unit list and its first two units in flight ----
  const int wi = split * kD2Warps + warp, NW = A.nsplit * kD2Warps;
  const int NUn = (A.n_near + 15) >> 4, NUf = (A.n_act + 7) >> 3;
  const int nn = wi < NUn ? (NUn - wi + NW - 1) / NW : 0, nf = wi < NUf ? (NUf - wi + NW - 1) / NW : 0;
  const int ntot = nn + nf;
  const char* ringK = (const char*)V.ringK + (size_t)b * D.Wf * D.T * 256;
  const char* ringV = (const char*)V.ringV + (size_t)b * D.Wf * D.T * 256;
  unsigned char* ring = sm + kD2Ring + warp * kD2Stages * kD2StageBytes;
  const uint32_t ring_u32 = (uint32_t)__cvta_generic_to_shared(ring);
  auto issue = [&](int i) {
    if (i < ntot) {
      const uint32_t dst = ring_u32 + (uint32_t)(i % kD2Stages) * kD2StageBytes;
      if (i < nn) {
        const int base = (wi + i * NW) << 4, last = A.n_near - 1;
#pragma unroll
        for (int r = 0; r < 8; ++r) {                         // 256 16-byte pieces per operand: piece = r * 32 + lane
          const int piece = r * 32 + lane, row = piece >> 4, ch = piece & 15;
          const size_t src = (size_t)min(base + row, last) * 256 + ch * 16;   // ragged tail: clamp, masked by the consumer
          // 16-byte chunks are XOR-swizzled so that the fragment reads below are bank-conflict free: a quarter warp reads
          // key rows g, g + 1 at the same chunks, and value rows 2j (+1) at chunks 2g, 2g + 1
          d2_cp16(dst + D2Stage::K + row * 256 + ((ch ^ ((row & 1) << 2)) << 4), ringK + src);
          d2_cp16(dst + D2Stage::Vv + row * 256 + ((ch ^ (((row >> 2) & 1) << 2)) << 4), ringV + src);
        }
      } else {
        const size_t pk0 = (size_t)b * D.K + (size_t)(wi + (i - nn) * NW) * 8;
        const char* cs = (const char*)(V.c_bf + pk0 * 128);     // bf16 copies of the centres (Dev::c_bf / p_bf)
        const char* ps = (const char*)(V.p_bf + pk0 * 128);
#pragma unroll
        for (int r = 0; r < 4; ++r) {                           // 8 prototypes x 256 B = 128 pieces per side
          d2_cp16(dst + D2Stage::C + (r * 32 + lane) * 16, cs + (r * 32 + lane) * 16);
          d2_cp16(dst + D2Stage::P + (r * 32 + lane) * 16, ps + (r * 32 + lane) * 16);
        }
        if (lane < 16) d2_cp16(dst + D2Stage::ZK + lane * 16, (const char*)(V.codesK + pk0 * 8) + lane * 16);
        else d2_cp16(dst + D2Stage::ZV + (lane - 16) * 16, (const char*)(V.codesV + pk0 * 8) + (lane - 16) * 16);
        if (lane < 2) d2_cp16(dst + D2Stage::LN + lane * 16, (const char*)(V.logn + pk0) + lane * 16);
        else if (lane == 2) d2_cp8(dst + D2Stage::KD, V.kind + pk0);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  issue(0);
  issue(1);

  // ---- codebooks as bf16 [g][z][16] (32-byte rows) ----
  if (has_cb && A.n_act > 0) {
    const float4* srck = reinterpret_cast<const float4*>(V.cbk + (size_t)b * 2048);
    const float4* srcv = reinterpret_cast<const float4*>(V.cbv + (size_t)b * 2048);
    for (int e = tid; e < 512; e += kD2Threads) {               // float4 e = (g * 16 + z) * 4 + quarter
      const float4 a = srck[e], c = srcv[e];
      *reinterpret_cast<uint2*>(sm + D2Smem::CBK + e * 8) = make_uint2(d2_pack(a.x, a.y), d2_pack(a.z, a.w));
      *reinterpret_cast<uint2*>(sm + D2Smem::CBV + (e >> 2) * 48 + (e & 3) * 8) = make_uint2(d2_pack(c.x, c.y), d2_pack(c.z, c.w));
    }
  }

  // ---- Q as A fragments under the key-side permutation: k-steps 2c, 2c + 1 <- chunk q = j + 4c of rows g, g + 8 ----
  uint32_t qa[8][4];
  {
    uint4 t[4], u[4];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int r = g + 8 * h;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint4 val = make_uint4(0u, 0u, 0u, 0u);
        if (r < A.R) {
          const int qi = r / D.group, hh = r % D.group;
          const size_t off = ((((size_t)st * A.layer_count + ll) * A.n_q + qi) * D.Hq + hd * D.group + hh) * 128 + (j + 4 * c) * 8;
          val = d2_ldg16(A.Q + off);
        }
        if (h == 0) t[c] = val; else u[c] = val;
      }
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      qa[2 * c][0] = t[c].x; qa[2 * c][2] = t[c].y; qa[2 * c][1] = u[c].x; qa[2 * c][3] = u[c].y;
      qa[2 * c + 1][0] = t[c].z; qa[2 * c + 1][2] = t[c].w; qa[2 * c + 1][1] = u[c].z; qa[2 * c + 1][3] = u[c].w;
    }
  }
  __syncthreads();                                              // codebooks visible

  float o[16][4];
#pragma unroll
  for (int i = 0; i < 16; ++i) { o[i][0] = 0.f; o[i][1] = 0.f; o[i][2] = 0.f; o[i][3] = 0.f; }
  D2Soft S{-INFINITY, -INFINITY, 0.f, 0.f};
  const float sc2 = kD2Log2e * rsqrtf(128.f);
  const unsigned char* cbK = sm + D2Smem::CBK;
  const unsigned char* cbV = sm + D2Smem::CBV;

  for (int i = 0; i < ntot; ++i) {
    asm volatile("cp.async.wait_group 1;" ::: "memory");        // this lane's pieces of unit i have landed
    __syncwarp();                                               // ... every lane's; and unit i - 1 has been consumed
    issue(i + 2);
    const unsigned char* stg = ring + (i % kD2Stages) * kD2StageBytes;
    if (i < nn) {
      // ---- near window: 16 ring rows ----
      const int base = (wi + i * NW) << 4;
      uint4 k0[4], k1[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const int ch = (j + 4 * c) ^ ((g & 1) << 2);            // rows g and 8 + g have the same parity
        k0[c] = *reinterpret_cast<const uint4*>(stg + D2Stage::K + g * 256 + ch * 16);
        k1[c] = *reinterpret_cast<const uint4*>(stg + D2Stage::K + (8 + g) * 256 + ch * 16);
      }
      float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
      float s0b[4] = {0.f, 0.f, 0.f, 0.f}, s1b[4] = {0.f, 0.f, 0.f, 0.f};   // two accumulation chains per column group
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        d2_mma(s0, qa[2 * c], k0[c].x, k0[c].y);
        d2_mma(s0b, qa[2 * c + 1], k0[c].z, k0[c].w);
        d2_mma(s1, qa[2 * c], k1[c].x, k1[c].y);
        d2_mma(s1b, qa[2 * c + 1], k1[c].z, k1[c].w);
      }
#pragma unroll
      for (int e = 0; e < 4; ++e) { s0[e] += s0b[e]; s1[e] += s1b[e]; }
      const int c0 = base + 2 * j;                              // accumulator columns 2j, 2j + 1 of a group
      float x0[4], x1[4];
      x0[0] = c0 < A.n_near ? s0[0] * sc2 : -INFINITY; x0[1] = c0 + 1 < A.n_near ? s0[1] * sc2 : -INFINITY;
      x0[2] = c0 < A.n_near ? s0[2] * sc2 : -INFINITY; x0[3] = c0 + 1 < A.n_near ? s0[3] * sc2 : -INFINITY;
      x1[0] = c0 + 8 < A.n_near ? s1[0] * sc2 : -INFINITY; x1[1] = c0 + 9 < A.n_near ? s1[1] * sc2 : -INFINITY;
      x1[2] = c0 + 8 < A.n_near ? s1[2] * sc2 : -INFINITY; x1[3] = c0 + 9 < A.n_near ? s1[3] * sc2 : -INFINITY;
      uint32_t pa[4];
      d2_softmax(S, o, x0, x1, pa);
      uint32_t v[4][8];
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        const int row = (t >> 1) * 8 + 2 * j + (t & 1), sw = ((row >> 2) & 1) << 2;
        const unsigned char* src = stg + D2Stage::Vv + row * 256;
        // odd j reads its high half first: the eight lanes of a quarter warp then touch eight distinct 16-byte bank groups
        const uint4 first = *reinterpret_cast<const uint4*>(src + (((2 * g + (j & 1)) ^ sw) << 4));
        const uint4 second = *reinterpret_cast<const uint4*>(src + (((2 * g + 1 - (j & 1)) ^ sw) << 4));
        const uint4 lo = (j & 1) ? second : first, hi = (j & 1) ? first : second;
        v[t][0] = lo.x; v[t][1] = lo.y; v[t][2] = lo.z; v[t][3] = lo.w;
        v[t][4] = hi.x; v[t][5] = hi.y; v[t][6] = hi.z; v[t][7] = hi.w;
      }
      d2_pv(o, pa, v);
    } else {
      // ---- far bank: 8 prototypes = 4 steps of 2 prototypes = 16 pseudo-tokens (column group = prototype, column = mode) ----
      const int k0 = (wi + (i - nn) * NW) * 8;
      const float* lns = reinterpret_cast<const float*>(stg + D2Stage::LN);
      const uint32_t* zks = reinterpret_cast<const uint32_t*>(stg + D2Stage::ZK);
      const uint32_t* zvs = reinterpret_cast<const uint32_t*>(stg + D2Stage::ZV);
#pragma unroll 1
      for (int ss = 0; ss < 4; ++ss) {
        if (k0 + 2 * ss >= A.n_act) break;
        int kind[2];
        float bias[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int kl = 2 * ss + h;
          kind[h] = k0 + kl < A.n_act ? (int)stg[D2Stage::KD + kl] : 2;
          bias[h] = kind[h] == 2 ? -INFINITY : (A.use_bias ? lns[kl] * kD2Log2e : 0.f);
        }
        // key side: lane (s = g, j) builds chunks q = j + 4c of k~_{k, s}
        float s01[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int kl = 2 * ss + h;
          const uint32_t code = zks[kl * 8 + g];
          uint4 kr[4];
#pragma unroll
          for (int c = 0; c < 4; ++c) kr[c] = *reinterpret_cast<const uint4*>(stg + D2Stage::C + kl * 256 + (j + 4 * c) * 16);
          if (kind[h] == 0) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              const int gg = (j + 4 * c) >> 1;
              const uint32_t z = (code >> (4 * gg)) & 15u;
              kr[c] = d2_add2x4(kr[c], *reinterpret_cast<const uint4*>(cbK + (gg * 16 + z) * 32 + (j & 1) * 16));
            }
          }
          float sb[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            d2_mma(s01[h], qa[2 * c], kr[c].x, kr[c].y);
            d2_mma(sb, qa[2 * c + 1], kr[c].z, kr[c].w);
          }
#pragma unroll
          for (int e = 0; e < 4; ++e) s01[h][e] += sb[e];
        }
        float x0[4], x1[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) { x0[e] = fmaf(s01[0][e], sc2, bias[0]); x1[e] = fmaf(s01[1][e], sc2, bias[1]); }
        uint32_t pa[4];
        d2_softmax(S, o, x0, x1, pa);
        // value side: rows t = 0, 1: modes 2j, 2j + 1 of prototype A; t = 2, 3: of prototype B; dims [16 g, 16 g + 16) = subspace g
        uint32_t v[4][8];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int kl = 2 * ss + h;
          const uint4 plo = *reinterpret_cast<const uint4*>(stg + D2Stage::P + kl * 256 + g * 32);
          const uint4 phi = *reinterpret_cast<const uint4*>(stg + D2Stage::P + kl * 256 + g * 32 + 16);
          const uint2 zz = *reinterpret_cast<const uint2*>(zvs + kl * 8 + 2 * j);
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            uint4 lo = plo, hi = phi;
            if (kind[h] == 0) {
              const uint32_t z = ((e ? zz.y : zz.x) >> (4 * g)) & 15u;
              const uint4* cw = reinterpret_cast<const uint4*>(cbV + (g * 16 + z) * 48);
              lo = d2_add2x4(lo, cw[0]); hi = d2_add2x4(hi, cw[1]);
            }
            const int t = 2 * h + e;
            v[t][0] = lo.x; v[t][1] = lo.y; v[t][2] = lo.z; v[t][3] = lo.w;
            v[t][4] = hi.x; v[t][5] = hi.y; v[t][6] = hi.z; v[t][7] = hi.w;
          }
        }
        d2_pv(o, pa, v);
      }
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();                                              // every warp is done with its ring: reuse it for the merge

  // ---- merge the four warps' (m, l, O) and write this CTA's partial ----
  S.l0 += __shfl_xor_sync(0xffffffffu, S.l0, 1); S.l0 += __shfl_xor_sync(0xffffffffu, S.l0, 2);
  S.l1 += __shfl_xor_sync(0xffffffffu, S.l1, 1); S.l1 += __shfl_xor_sync(0xffffffffu, S.l1, 2);
  float* Om = reinterpret_cast<float*>(sm + D2Smem::O) + warp * 16 * 128;
  float* ml = reinterpret_cast<float*>(sm + D2Smem::ML) + warp * 32;
#pragma unroll
  for (int i = 0; i < 16; ++i) {            // tile i, accumulator column n = 2j (+1)  <->  dim 16 n + i
    Om[g * 128 + 16 * (2 * j) + i] = o[i][0];
    Om[g * 128 + 16 * (2 * j + 1) + i] = o[i][1];
    Om[(g + 8) * 128 + 16 * (2 * j) + i] = o[i][2];
    Om[(g + 8) * 128 + 16 * (2 * j + 1) + i] = o[i][3];
  }
  if (j == 0) { ml[g * 2] = S.m0; ml[g * 2 + 1] = S.l0; ml[(g + 8) * 2] = S.m1; ml[(g + 8) * 2 + 1] = S.l1; }
  __syncthreads();
  {
    const int r = tid >> 3, d0 = (tid & 7) * 16;          // 16 rows x 8 threads, 16 dims each
    if (r < A.R) {
      const float* mlb = reinterpret_cast<const float*>(sm + D2Smem::ML);
      float M = -INFINITY;
#pragma unroll
      for (int w = 0; w < kD2Warps; ++w) M = fmaxf(M, mlb[w * 32 + r * 2]);
      const float Mu = M == -INFINITY ? 0.f : M;
      float wgt[kD2Warps], l = 0.f;
#pragma unroll
      for (int w = 0; w < kD2Warps; ++w) {
        wgt[w] = d2_ex2(mlb[w * 32 + r * 2] - Mu);
        l = fmaf(mlb[w * 32 + r * 2 + 1], wgt[w], l);
      }
      float* dst = A.part + (((size_t)bsel * A.R + r) * A.nsplit + split) * 130;
      const float* Ob = reinterpret_cast<const float*>(sm + D2Smem::O);
#pragma unroll
      for (int e = 0; e < 16; e += 4) {
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int w = 0; w < kD2Warps; ++w) {
          const float4 x = *reinterpret_cast<const float4*>(Ob + (w * 16 + r) * 128 + d0 + e);
          acc.x = fmaf(x.x, wgt[w], acc.x); acc.y = fmaf(x.y, wgt[w], acc.y);
          acc.z = fmaf(x.z, wgt[w], acc.z); acc.w = fmaf(x.w, wgt[w], acc.w);
        }
        dst[d0 + e] = acc.x; dst[d0 + e + 1] = acc.y; dst[d0 + e + 2] = acc.z; dst[d0 + e + 3] = acc.w;
      }
      if ((tid & 7) == 0) {
        dst[128] = M == -INFINITY ? -INFINITY : M * kD2Ln2;
        dst[129] = l;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// The same kernel for <= 8 query rows per bank (one decoded token of a GQA group of up to 8 -- the common case), with
// the MMA roles swapped so that nothing is padded: the 16 context columns of a step are the M dimension and the query
// rows the N = 8 dimension.
//   S^T = K~ Q^T   A = key rows g, g + 8 (same chunk permutation as above), B = Q^T: 8 MMAs per 16 columns
//   softmax        thread (g, j) holds (ctx g | g + 8) x (rows 2j, 2j + 1); row maxima reduce over the g lanes
//   P^T            the PV B fragment wants (ctx 2j, 2j + 1; row g): an 8 x 8 transpose inside the warp -- movmatrix
//   O^T += V~^T P^T   A = V~^T (M = dims [16 g, 16 g + 16) in pairs, K = ctx), 8 MMAs per 16 columns, 32 accumulators
// Half the MMAs, half the accumulators and ~150 registers: three CTAs (12 warps) per SM instead of two.
// ---------------------------------------------------------------------------------------------------------
constexpr int kD8CtasPerSm = 3;
constexpr int kD8Stages = 2;
constexpr uint32_t kD8StageBytes = 8192;
constexpr uint32_t kD8CbV = 4128;                                                      // two bf16 codebooks: 128 rows x 32 B + one zero row
constexpr uint32_t kD8Ring = 8256;
constexpr uint32_t kD8SmemTotal = kD8Ring + kD2Warps * kD8Stages * kD8StageBytes;      // 73,728 B

__device__ __forceinline__ void d8_mma(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                       uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
               "{%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t d8_trans(uint32_t x) {     // 8 x 8 b16 transpose across the warp
  uint32_t r;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(r) : "r"(x));
  return r;
}

// x[0], x[1]: (ctx g; rows 2j, 2j + 1), x[2], x[3]: (ctx g + 8; rows 2j, 2j + 1).  Returns the PV B fragment (P^T).
__device__ __forceinline__ void d8_softmax(D2Soft& s, float (&o)[8][4], const float (&x)[4], uint32_t& b0, uint32_t& b1) {
  float mx0 = fmaxf(x[0], x[2]), mx1 = fmaxf(x[1], x[3]);
#pragma unroll
  for (int sh = 4; sh <= 16; sh <<= 1) {
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, sh));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, sh));
  }
  const float mn0 = mx0 > s.m0 + kD2Slack ? mx0 : s.m0, mn1 = mx1 > s.m1 + kD2Slack ? mx1 : s.m1;   // lazy reference maximum
  const float mu0 = mn0 == -INFINITY ? 0.f : mn0, mu1 = mn1 == -INFINITY ? 0.f : mn1;
  const float a0 = d2_ex2(s.m0 - mu0), a1 = d2_ex2(s.m1 - mu1);
  s.m0 = mn0; s.m1 = mn1;
  const float p0 = d2_ex2(x[0] - mu0), p1 = d2_ex2(x[1] - mu1), p2 = d2_ex2(x[2] - mu0), p3 = d2_ex2(x[3] - mu1);
  s.l0 = fmaf(s.l0, a0, p0 + p2);
  s.l1 = fmaf(s.l1, a1, p1 + p3);
  if (__any_sync(0xffffffffu, a0 != 1.f || a1 != 1.f)) {
#pragma unroll
    for (int i = 0; i < 8; ++i) { o[i][0] *= a0; o[i][1] *= a1; o[i][2] *= a0; o[i][3] *= a1; }
  }
  b0 = d8_trans(d2_pack(p0, p1));
  b1 = d8_trans(d2_pack(p2, p3));
}

// O^T += V~^T P^T: v[t][0..7] as in d2_pv; tile i holds dims 16 g + 2 i (M index g) and 16 g + 2 i + 1 (M index g + 8)
__device__ __forceinline__ void d8_pv(float (&o)[8][4], uint32_t b0, uint32_t b1, const uint32_t (&v)[4][8]) {
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const uint32_t a0 = d2_prmt(v[0][i], v[1][i], 0x5410u), a1 = d2_prmt(v[0][i], v[1][i], 0x7632u);
    const uint32_t a2 = d2_prmt(v[2][i], v[3][i], 0x5410u), a3 = d2_prmt(v[2][i], v[3][i], 0x7632u);
    d8_mma(o[i], a0, a1, a2, a3, b0, b1);
  }
}

// Rotary embedding (PROTOKV_ROPE, D.1; readings 28-31) of 8 rotation pairs held as two 16-byte chunks: x =
// dims [8q, 8q + 8) with q < 8, y = the partner dims [8q + 64, 8q + 72) -- the key-side chunk permutation keeps both in
// one lane (chunks c and c + 2).  tab: the 8 (cos, sin) pairs of pair indices 8q .. 8q + 7 at the row's position.
__device__ __forceinline__ void d8_rope8(uint4& x, uint4& y, const float2* __restrict__ tab) {
  uint32_t xs[4] = {x.x, x.y, x.z, x.w}, ys[4] = {y.x, y.y, y.z, y.w};
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const float4 cs = __ldg(reinterpret_cast<const float4*>(tab) + t);       // (cos, sin) of pairs 2t, 2t + 1
    const float xl = __uint_as_float(xs[t] << 16), xh = __uint_as_float(xs[t] & 0xffff0000u);
    const float yl = __uint_as_float(ys[t] << 16), yh = __uint_as_float(ys[t] & 0xffff0000u);
    xs[t] = d2_pack(fmaf(xl, cs.x, -yl * cs.y), fmaf(xh, cs.z, -yh * cs.w));
    ys[t] = d2_pack(fmaf(yl, cs.x, xl * cs.y), fmaf(yh, cs.z, xh * cs.w));
  }
  x = make_uint4(xs[0], xs[1], xs[2], xs[3]);
  y = make_uint4(ys[0], ys[1], ys[2], ys[3]);
}

// ROPE: keys and queries are rotated in registers on their way into the fragments.  blockIdx.z = block of 8 query rows: a
// query of more rows (the multi-token prefill of a PROTOKV_ROPE state) runs as independent 8-row blocks over the same bank.
// RAGGED: PROTOKV_VAR_ALLOC (D.3) -- prototype k owns S_k rows of the bank's code arrays from row
// soff[k]; a far unit is still 8 prototypes, but its pseudo-tokens are walked 16 rows at a time and every row looks up
// its own prototype among the unit's eight.
template <bool ROPE, bool RAGGED>
__global__ void __launch_bounds__(kD2Threads, (ROPE || RAGGED) ? 2 : kD8CtasPerSm) attention_decode8_kernel(Dims D, Dev V, D2Args A) {
  extern __shared__ __align__(16) unsigned char sm[];
  pdl_wait();   // launched under the tail of the previous kernel of the stream (see common.cuh); no early trigger of its own
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, j = lane & 3;
  const int bsel = blockIdx.y, split = blockIdx.x, r0 = blockIdx.z * 8;   // first query row of this block
  const int hd = bsel % D.Hkv, ll = (bsel / D.Hkv) % A.layer_count, st = bsel / (D.Hkv * A.layer_count);
  const int b = (st * D.L + A.layer_begin + ll) * D.Hkv + hd;
  const bool has_cb = V.cbk != nullptr;

  const int wi = split * kD2Warps + warp, NW = A.nsplit * kD2Warps;
  const int NUn = (A.n_near + 15) >> 4, NUf = (A.n_act + 7) >> 3;
  const int nn = wi < NUn ? (NUn - wi + NW - 1) / NW : 0, nf = wi < NUf ? (NUf - wi + NW - 1) / NW : 0;
  const int ntot = nn + nf;
  const char* ringK = (const char*)V.ringK + (size_t)b * D.Wf * D.T * 256;
  const char* ringV = (const char*)V.ringV + (size_t)b * D.Wf * D.T * 256;
  unsigned char* ring = sm + kD8Ring + warp * kD8Stages * kD8StageBytes;
  const uint32_t ring_u32 = (uint32_t)__cvta_generic_to_shared(ring);
  auto issue = [&](int i) {
    if (i < ntot) {
      const uint32_t dst = ring_u32 + (uint32_t)(i % kD8Stages) * kD8StageBytes;
      if (i < nn) {
        const int base = (wi + i * NW) << 4, last = A.n_near - 1;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
          const int piece = r * 32 + lane, row = piece >> 4, ch = piece & 15;
          const size_t src = (size_t)min(base + row, last) * 256 + ch * 16;
          d2_cp16(dst + D2Stage::K + row * 256 + ((ch ^ ((row & 1) << 2)) << 4), ringK + src);
          d2_cp16(dst + D2Stage::Vv + row * 256 + ((ch ^ (((row >> 2) & 1) << 2)) << 4), ringV + src);
        }
      } else {
        const size_t pk0 = (size_t)b * D.K + (size_t)(wi + (i - nn) * NW) * 8;
        const char* cs = (const char*)(V.c_bf + pk0 * 128);
        const char* ps = (const char*)(V.p_bf + pk0 * 128);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          d2_cp16(dst + D2Stage::C + (r * 32 + lane) * 16, cs + (r * 32 + lane) * 16);
          d2_cp16(dst + D2Stage::C + 2048 + (r * 32 + lane) * 16, ps + (r * 32 + lane) * 16);
        }
        if (RAGGED) {   // this unit's code rows [soff[k0], soff[k0 + 8)) (<= 256), its 9 offsets, masses and kinds
          const int* so = V.soff + (size_t)b * (D.K + 1) + (pk0 - (size_t)b * D.K);
          const int r0 = __ldg(so), nrows = __ldg(so + 8) - r0;
          const uint32_t* ck = V.codesK + (size_t)b * D.K * 8 + r0;
          const uint32_t* cv = V.codesV + (size_t)b * D.K * 8 + r0;
          for (int e = lane; e < nrows; e += 32) {
            d2_cp4(dst + 4096 + e * 4, ck + e);
            d2_cp4(dst + 5120 + e * 4, cv + e);
          }
          if (lane < 9) d2_cp4(dst + 6192 + lane * 4, so + lane);
          if (lane < 2) d2_cp16(dst + 6144 + lane * 16, (const char*)(V.logn + pk0) + lane * 16);
          else if (lane == 2) d2_cp8(dst + 6176, V.kind + pk0);
        } else {
          if (lane < 16) d2_cp16(dst + 4096 + lane * 16, (const char*)(V.codesK + pk0 * 8) + lane * 16);
          else d2_cp16(dst + 4352 + (lane - 16) * 16, (const char*)(V.codesV + pk0 * 8) + (lane - 16) * 16);
          if (lane < 2) d2_cp16(dst + 4608 + lane * 16, (const char*)(V.logn + pk0) + lane * 16);
          else if (lane == 2) d2_cp8(dst + 4640, V.kind + pk0);
        }
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  // the bank's bf16 codebooks (Dev::cb_bf) ride in the first cp.async group; they are needed from the first far unit on
  if (has_cb && A.n_act > 0) {
    const char* src = (const char*)(V.cb_bf + (size_t)b * 4096);
    const uint32_t s0 = (uint32_t)__cvta_generic_to_shared(sm);
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      d2_cp16(s0 + (r * 128 + tid) * 16, src + (r * 128 + tid) * 16);
      d2_cp16(s0 + kD8CbV + (r * 128 + tid) * 16, src + 4096 + (r * 128 + tid) * 16);
    }
  }
  // row 128 of either codebook is all zero: prototypes without decoded residuals (n_res = 0, Alg. 4 l.3-4) add it, so that
  // the fragment build of the fixed-S path is branch-free
  if (tid < 8) reinterpret_cast<uint32_t*>(sm + 4096)[tid] = 0u;
  else if (tid < 16) reinterpret_cast<uint32_t*>(sm + kD8CbV + 4096)[tid - 8] = 0u;
  issue(0);

  // Q^T as B fragments: column n = g is query row g; k-steps 2c, 2c + 1 <- chunk q = j + 4c
  uint32_t qb[8][2];
  uint4 qv[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    uint4 val = make_uint4(0u, 0u, 0u, 0u);
    if (r0 + g < A.R) {
      const int qi = (r0 + g) / D.group, hh = (r0 + g) % D.group;
      const size_t off = ((((size_t)st * A.layer_count + ll) * A.n_q + qi) * D.Hq + hd * D.group + hh) * 128 + (j + 4 * c) * 8;
      val = d2_ldg16(A.Q + off);
    }
    qv[c] = val;
  }
  if (ROPE && r0 + g < A.R) {                                    // query token qi sits at q_pos0 + qi (reading 29)
    const float2* tq = V.ropeQ + (size_t)((r0 + g) / D.group) * 64;
    d8_rope8(qv[0], qv[2], tq + 8 * j);
    d8_rope8(qv[1], qv[3], tq + 8 * (j + 4));
  }
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    qb[2 * c][0] = qv[c].x; qb[2 * c][1] = qv[c].y; qb[2 * c + 1][0] = qv[c].z; qb[2 * c + 1][1] = qv[c].w;
  }

  float o[8][4];
#pragma unroll
  for (int i = 0; i < 8; ++i) { o[i][0] = 0.f; o[i][1] = 0.f; o[i][2] = 0.f; o[i][3] = 0.f; }
  D2Soft S{-INFINITY, -INFINITY, 0.f, 0.f};                     // rows 2j (m0, l0) and 2j + 1 (m1, l1)
  const float sc2 = kD2Log2e * rsqrtf(128.f);
  const unsigned char* cbK = sm;
  const unsigned char* cbV = sm + kD8CbV;

  bool cb_ready = false;                                        // exactly one block barrier per warp: codebooks visible
  for (int i = 0; i < ntot; ++i) {
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (i == nn) { __syncthreads(); cb_ready = true; }          // first far unit of this warp (warp-uniform)
    __syncwarp();
    issue(i + 1);
    const unsigned char* stg = ring + (i % kD8Stages) * kD8StageBytes;
    if (i < nn) {
      const int base = (wi + i * NW) << 4;
      float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int cp = 0; cp < 2; ++cp) {                          // chunks cp and cp + 2 hold the two halves of 8 rotation pairs
        const int cha = (j + 4 * cp) ^ ((g & 1) << 2), chb = (j + 4 * cp + 8) ^ ((g & 1) << 2);
        uint4 ka = *reinterpret_cast<const uint4*>(stg + D2Stage::K + g * 256 + cha * 16);
        uint4 ka2 = *reinterpret_cast<const uint4*>(stg + D2Stage::K + g * 256 + chb * 16);
        uint4 kb = *reinterpret_cast<const uint4*>(stg + D2Stage::K + (8 + g) * 256 + cha * 16);
        uint4 kb2 = *reinterpret_cast<const uint4*>(stg + D2Stage::K + (8 + g) * 256 + chb * 16);
        if (ROPE) {                                             // near tokens keep their stream positions (L126)
          const int last = A.n_near - 1;
          d8_rope8(ka, ka2, V.ropeR + (size_t)min(base + g, last) * 64 + 8 * (j + 4 * cp));
          d8_rope8(kb, kb2, V.ropeR + (size_t)min(base + 8 + g, last) * 64 + 8 * (j + 4 * cp));
        }
        d8_mma(s0, ka.x, kb.x, ka.y, kb.y, qb[2 * cp][0], qb[2 * cp][1]);
        d8_mma(s1, ka.z, kb.z, ka.w, kb.w, qb[2 * cp + 1][0], qb[2 * cp + 1][1]);
        d8_mma(s0, ka2.x, kb2.x, ka2.y, kb2.y, qb[2 * cp + 4][0], qb[2 * cp + 4][1]);
        d8_mma(s1, ka2.z, kb2.z, ka2.w, kb2.w, qb[2 * cp + 5][0], qb[2 * cp + 5][1]);
      }
      float x[4];
      const bool in0 = base + g < A.n_near, in1 = base + 8 + g < A.n_near;
      x[0] = in0 ? (s0[0] + s1[0]) * sc2 : -INFINITY; x[1] = in0 ? (s0[1] + s1[1]) * sc2 : -INFINITY;
      x[2] = in1 ? (s0[2] + s1[2]) * sc2 : -INFINITY; x[3] = in1 ? (s0[3] + s1[3]) * sc2 : -INFINITY;
      uint32_t b0, b1;
      d8_softmax(S, o, x, b0, b1);
      uint32_t v[4][8];
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        const int row = (t >> 1) * 8 + 2 * j + (t & 1), sw = ((row >> 2) & 1) << 2;
        const unsigned char* src = stg + D2Stage::Vv + row * 256;
        const uint4 first = *reinterpret_cast<const uint4*>(src + (((2 * g + (j & 1)) ^ sw) << 4));
        const uint4 second = *reinterpret_cast<const uint4*>(src + (((2 * g + 1 - (j & 1)) ^ sw) << 4));
        const uint4 lo = (j & 1) ? second : first, hi = (j & 1) ? first : second;
        v[t][0] = lo.x; v[t][1] = lo.y; v[t][2] = lo.z; v[t][3] = lo.w;
        v[t][4] = hi.x; v[t][5] = hi.y; v[t][6] = hi.z; v[t][7] = hi.w;
      }
      d8_pv(o, b0, b1, v);
    } else if (RAGGED) {
      const int k0 = (wi + (i - nn) * NW) * 8;
      const float* lns = reinterpret_cast<const float*>(stg + 6144);
      const uint32_t* zks = reinterpret_cast<const uint32_t*>(stg + 4096);
      const uint32_t* zvs = reinterpret_cast<const uint32_t*>(stg + 5120);
      const int* offs = reinterpret_cast<const int*>(stg + 6192);
      int rel[8];                                               // first row of each of the unit's prototypes
#pragma unroll
      for (int q = 0; q < 8; ++q) rel[q] = offs[q] - offs[0];
      const int nrows = offs[8] - offs[0];
      auto owner = [&](int r) {                                 // prototype (0..7) that owns local row r
        int kl = 0;
#pragma unroll
        for (int q = 1; q < 8; ++q) kl += r >= rel[q] ? 1 : 0;
        return kl;
      };
#pragma unroll 1
      for (int t0 = 0; t0 < nrows; t0 += 16) {
        int kl[2], kind[2];
        float bias[2];
        uint4 kr[2][4];
#pragma unroll
        for (int h = 0; h < 2; ++h) {                           // key side: rows t0 + g and t0 + 8 + g
          const int r = t0 + 8 * h + g;
          const bool in = r < nrows;
          kl[h] = in ? owner(r) : 0;
          kind[h] = in ? (int)stg[6176 + kl[h]] : 2;
          bias[h] = kind[h] == 2 ? -INFINITY : (A.use_bias ? lns[kl[h]] * kD2Log2e : 0.f);
          const uint32_t code = in ? zks[r] : 0u;
#pragma unroll
          for (int c = 0; c < 4; ++c) kr[h][c] = *reinterpret_cast<const uint4*>(stg + D2Stage::C + kl[h] * 256 + (j + 4 * c) * 16);
          if (kind[h] == 0) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              const int gg = (j + 4 * c) >> 1;
              const uint32_t z = (code >> (4 * gg)) & 15u;
              kr[h][c] = d2_add2x4(kr[h][c], *reinterpret_cast<const uint4*>(cbK + (gg * 16 + z) * 32 + (j & 1) * 16));
            }
          }
          if (ROPE) {
            const float2* tp = V.ropeP + ((size_t)b * D.K + min(k0 + kl[h], D.K - 1)) * 64;
            d8_rope8(kr[h][0], kr[h][2], tp + 8 * j);
            d8_rope8(kr[h][1], kr[h][3], tp + 8 * (j + 4));
          }
        }
        float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          d8_mma(s0, kr[0][c].x, kr[1][c].x, kr[0][c].y, kr[1][c].y, qb[2 * c][0], qb[2 * c][1]);
          d8_mma(s1, kr[0][c].z, kr[1][c].z, kr[0][c].w, kr[1][c].w, qb[2 * c + 1][0], qb[2 * c + 1][1]);
        }
        float x[4];
        x[0] = fmaf(s0[0] + s1[0], sc2, bias[0]); x[1] = fmaf(s0[1] + s1[1], sc2, bias[0]);
        x[2] = fmaf(s0[2] + s1[2], sc2, bias[1]); x[3] = fmaf(s0[3] + s1[3], sc2, bias[1]);
        uint32_t b0, b1;
        d8_softmax(S, o, x, b0, b1);
        uint32_t v[4][8];
#pragma unroll
        for (int tt = 0; tt < 4; ++tt) {                        // value side: rows t0 + 2j (+1) and t0 + 8 + 2j (+1)
          const int r = t0 + (tt >> 1) * 8 + 2 * j + (tt & 1);
          const bool in = r < nrows;
          const int kv = in ? owner(r) : 0;
          uint4 lo = *reinterpret_cast<const uint4*>(stg + D2Stage::C + 2048 + kv * 256 + g * 32);
          uint4 hi = *reinterpret_cast<const uint4*>(stg + D2Stage::C + 2048 + kv * 256 + g * 32 + 16);
          if (in && stg[6176 + kv] == 0) {
            const uint32_t z = (zvs[r] >> (4 * g)) & 15u;
            const uint4* cw = reinterpret_cast<const uint4*>(cbV + (g * 16 + z) * 32);
            lo = d2_add2x4(lo, cw[0]); hi = d2_add2x4(hi, cw[1]);
          }
          v[tt][0] = lo.x; v[tt][1] = lo.y; v[tt][2] = lo.z; v[tt][3] = lo.w;
          v[tt][4] = hi.x; v[tt][5] = hi.y; v[tt][6] = hi.z; v[tt][7] = hi.w;
        }
        d8_pv(o, b0, b1, v);
      }
    } else {
      const int k0 = (wi + (i - nn) * NW) * 8;
      const float* lns = reinterpret_cast<const float*>(stg + 4608);
      const uint32_t* zks = reinterpret_cast<const uint32_t*>(stg + 4096);
      const uint32_t* zvs = reinterpret_cast<const uint32_t*>(stg + 4352);
#pragma unroll
      for (int ss = 0; ss < 4; ++ss) {
        if (k0 + 2 * ss >= A.n_act) break;
        int kind[2];
        float bias[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int kl = 2 * ss + h;
          kind[h] = k0 + kl < A.n_act ? (int)stg[4640 + kl] : 2;
          bias[h] = kind[h] == 2 ? -INFINITY : (A.use_bias ? lns[kl] * kD2Log2e : 0.f);
        }
        // key side: rows g (prototype A, mode g) and g + 8 (prototype B, mode g) of the 16-column step
        uint4 kr[2][4];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int kl = 2 * ss + h;
          const uint32_t code = zks[kl * 8 + g];
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            const int gg = (j + 4 * c) >> 1;
            const uint32_t row = kind[h] == 0 ? (uint32_t)(gg * 16) + ((code >> (4 * gg)) & 15u) : 128u;
            kr[h][c] = d2_add2x4(*reinterpret_cast<const uint4*>(stg + D2Stage::C + kl * 256 + (j + 4 * c) * 16),
                                 *reinterpret_cast<const uint4*>(cbK + row * 32 + (j & 1) * 16));
          }
        }
        if (ROPE) {                                             // the S pseudo-tokens of a prototype sit at its anchor (L126, D.1)
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const float2* tp = V.ropeP + ((size_t)b * D.K + min(k0 + 2 * ss + h, D.K - 1)) * 64;
            d8_rope8(kr[h][0], kr[h][2], tp + 8 * j);
            d8_rope8(kr[h][1], kr[h][3], tp + 8 * (j + 4));
          }
        }
        float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          d8_mma(s0, kr[0][c].x, kr[1][c].x, kr[0][c].y, kr[1][c].y, qb[2 * c][0], qb[2 * c][1]);
          d8_mma(s1, kr[0][c].z, kr[1][c].z, kr[0][c].w, kr[1][c].w, qb[2 * c + 1][0], qb[2 * c + 1][1]);
        }
        float x[4];
        x[0] = fmaf(s0[0] + s1[0], sc2, bias[0]); x[1] = fmaf(s0[1] + s1[1], sc2, bias[0]);
        x[2] = fmaf(s0[2] + s1[2], sc2, bias[1]); x[3] = fmaf(s0[3] + s1[3], sc2, bias[1]);
        uint32_t b0, b1;
        d8_softmax(S, o, x, b0, b1);
        uint32_t v[4][8];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int kl = 2 * ss + h;
          const uint4 plo = *reinterpret_cast<const uint4*>(stg + D2Stage::C + 2048 + kl * 256 + g * 32);
          const uint4 phi = *reinterpret_cast<const uint4*>(stg + D2Stage::C + 2048 + kl * 256 + g * 32 + 16);
          const uint2 zz = *reinterpret_cast<const uint2*>(zvs + kl * 8 + 2 * j);
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const uint32_t row = kind[h] == 0 ? (uint32_t)(g * 16) + (((e ? zz.y : zz.x) >> (4 * g)) & 15u) : 128u;
            const uint4* cw = reinterpret_cast<const uint4*>(cbV + row * 32);
            const uint4 lo = d2_add2x4(plo, cw[0]), hi = d2_add2x4(phi, cw[1]);
            const int t = 2 * h + e;
            v[t][0] = lo.x; v[t][1] = lo.y; v[t][2] = lo.z; v[t][3] = lo.w;
            v[t][4] = hi.x; v[t][5] = hi.y; v[t][6] = hi.z; v[t][7] = hi.w;
          }
        }
        d8_pv(o, b0, b1, v);
      }
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  if (!cb_ready) __syncthreads();                               // a warp without far units still owes the codebook barrier
  __syncthreads();

  // ---- merge the four warps' (m, l, O^T) and write this CTA's partial ----
#pragma unroll
  for (int sh = 4; sh <= 16; sh <<= 1) {
    S.l0 += __shfl_xor_sync(0xffffffffu, S.l0, sh);
    S.l1 += __shfl_xor_sync(0xffffffffu, S.l1, sh);
  }
  float* Om = reinterpret_cast<float*>(sm + kD8Ring) + warp * 8 * 128;      // [4 warps][8 rows][128]
  float* ml = reinterpret_cast<float*>(sm + kD8Ring + 4 * 8 * 128 * 4) + warp * 16;
#pragma unroll
  for (int i = 0; i < 8; ++i) {             // tile i: M index g -> dim 16 g + 2 i, M index g + 8 -> dim 16 g + 2 i + 1
    Om[(2 * j) * 128 + 16 * g + 2 * i] = o[i][0];
    Om[(2 * j + 1) * 128 + 16 * g + 2 * i] = o[i][1];
    Om[(2 * j) * 128 + 16 * g + 2 * i + 1] = o[i][2];
    Om[(2 * j + 1) * 128 + 16 * g + 2 * i + 1] = o[i][3];
  }
  if (g == 0) { ml[(2 * j) * 2] = S.m0; ml[(2 * j) * 2 + 1] = S.l0; ml[(2 * j + 1) * 2] = S.m1; ml[(2 * j + 1) * 2 + 1] = S.l1; }
  __syncthreads();
  {
    const int r = tid >> 4, d0 = (tid & 15) * 8;          // 8 rows x 16 threads, 8 dims each
    if (r0 + r < A.R) {
      const float* mlb = reinterpret_cast<const float*>(sm + kD8Ring + 4 * 8 * 128 * 4);
      float M = -INFINITY;
#pragma unroll
      for (int w = 0; w < kD2Warps; ++w) M = fmaxf(M, mlb[w * 16 + r * 2]);
      const float Mu = M == -INFINITY ? 0.f : M;
      float wgt[kD2Warps], l = 0.f;
#pragma unroll
      for (int w = 0; w < kD2Warps; ++w) {
        wgt[w] = d2_ex2(mlb[w * 16 + r * 2] - Mu);
        l = fmaf(mlb[w * 16 + r * 2 + 1], wgt[w], l);
      }
      float* dst = A.part + (((size_t)bsel * A.R + r0 + r) * A.nsplit + split) * 130;
      const float* Ob = reinterpret_cast<const float*>(sm + kD8Ring);
#pragma unroll
      for (int e = 0; e < 8; e += 4) {
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int w = 0; w < kD2Warps; ++w) {
          const float4 xx = *reinterpret_cast<const float4*>(Ob + (w * 8 + r) * 128 + d0 + e);
          acc.x = fmaf(xx.x, wgt[w], acc.x); acc.y = fmaf(xx.y, wgt[w], acc.y);
          acc.z = fmaf(xx.z, wgt[w], acc.z); acc.w = fmaf(xx.w, wgt[w], acc.w);
        }
        dst[d0 + e] = acc.x; dst[d0 + e + 1] = acc.y; dst[d0 + e + 2] = acc.z; dst[d0 + e + 3] = acc.w;
      }
      if ((tid & 15) == 0) {
        dst[128] = M == -INFINITY ? -INFINITY : M * kD2Ln2;
        dst[129] = l;
      }
    }
  }
}

// PROTOKV_ROPE states: any number of query rows (8-row blocks)
bool decode2_rope_supported(const Dims& D) {
  return D.bf16 && D.d == 128 && D.S == 8 && D.G == 8 && D.C == 16 && D.K % 8 == 0;
}

bool decode2_attention_supported(const Dims& D, int n_q) {
  return D.bf16 && D.d == 128 && D.S == 8 && D.G == 8 && D.C == 16 && n_q * D.group <= kD2Rows && D.K % 8 == 0;   // (Dev::c_bf exists for exactly these shapes)
}

bool decode2_attention_prepare() {
  if (cudaFuncSetAttribute(attention_decode2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kD2SmemTotal) !=
      cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  if (cudaFuncSetAttribute(attention_decode8_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kD8SmemTotal) !=
          cudaSuccess ||
      cudaFuncSetAttribute(attention_decode8_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kD8SmemTotal) !=
          cudaSuccess ||
      cudaFuncSetAttribute(attention_decode8_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kD8SmemTotal) !=
          cudaSuccess ||
      cudaFuncSetAttribute(attention_decode8_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kD8SmemTotal) !=
          cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return true;
}

// Partials per row the launch below writes at most (part buffer sizing in carve()).
int decode2_max_splits() { return 16; }

int launch_attention_decode2(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, int sm_count, cudaStream_t s,
                             int* nsplit_out) {
  D2Args a{};
  a.Q = (const __nv_bfloat16*)A.Q;
  a.part = V.part;
  a.n_q = A.n_q; a.layer_begin = A.layer_begin; a.layer_count = A.layer_count;
  a.n_near = (H.flags & PROTOKV_FAR_ONLY) ? 0 : A.n_near;
  a.n_act = (H.flags & PROTOKV_NEAR_ONLY) ? 0 : A.n_act;
  a.use_bias = !(H.flags & PROTOKV_NO_MASS_BIAS);
  a.R = A.n_q * D.group;
  const int nb = D.NS * A.layer_count * D.Hkv;
  // splits per bank: the kernel's time goes like waves / ns with waves = ceil(nb ns / resident CTAs) -- take the smallest
  // ns within 3 % of the best, so that the last wave is nearly full
  const int units = (a.n_near + 15) / 16 + (a.n_act + 7) / 8;
  int cap = (units + kD2Warps - 1) / kD2Warps;
  if (cap > decode2_max_splits()) cap = decode2_max_splits();
  if (cap < 1) cap = 1;
  const bool rope = (H.flags & PROTOKV_ROPE) != 0, ragged = V.soff != nullptr;
  const bool rows8 = rope || ragged || a.R <= 8;               // the N = 8 variant; ROPE / VAR_ALLOC queries run as 8-row blocks
  const int nrb = rows8 ? (a.R + 7) / 8 : 1;
  const int slots = ((rope || ragged) ? 2 : (rows8 ? kD8CtasPerSm : kD2CtasPerSm)) * sm_count;
  const long long room = ((long long)D.B * 16 * decode2_max_splits()) / ((long long)nb * a.R);   // partials the buffer holds per row
  if (cap > room) cap = room < 1 ? 1 : (int)room;
  int ns = 1;
  double best = 1e30;
  for (int c = 1; c <= cap; ++c) {
    const double cost = (double)(((long long)nb * nrb * c + slots - 1) / slots) / c * (1.0 + 0.02 * c);   // + per-CTA fixed work
    if (cost < best * 0.97) { best = cost; ns = c; }
  }
  a.nsplit = ns;
  *nsplit_out = ns;
  const bool pdl = !(H.flags & PROTOKV_SERIAL_LAUNCH);
  if (rope && ragged) launch_chain(attention_decode8_kernel<true, true>, dim3(ns, nb, nrb), kD2Threads, kD8SmemTotal, s, pdl, D, V, a);
  else if (rope) launch_chain(attention_decode8_kernel<true, false>, dim3(ns, nb, nrb), kD2Threads, kD8SmemTotal, s, pdl, D, V, a);
  else if (ragged) launch_chain(attention_decode8_kernel<false, true>, dim3(ns, nb, nrb), kD2Threads, kD8SmemTotal, s, pdl, D, V, a);
  else if (rows8) launch_chain(attention_decode8_kernel<false, false>, dim3(ns, nb, 1), kD2Threads, kD8SmemTotal, s, pdl, D, V, a);
  else launch_chain(attention_decode2_kernel, dim3(ns, nb), kD2Threads, kD2SmemTotal, s, pdl, D, V, a);
  return 1;
}

}  // namespace pkv
