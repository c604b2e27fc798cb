// Q2 fused attention for DECODE-STYLE queries (bf16, d = 128, S = 8, G = 8, C = 16, n_q * group <= 16 query rows per
// bank): Alg. 4 l.8-15 / Eq. 4 as a split-KV kernel that is bound by streaming the bank, not
// by the tensor pipe.  PAPER.md:L574 (§C.3): the only ProtoKV work on the latency of a query is the bounded attention
// over W + K_max S tokens -- for a one-token query that is ~2.7 MB per bank read once for a handful of rows, i.e. pure
// HBM time (SURVEY.md 8(d) "a decode-style query would be pure HBM").
//
// The 128-row tcgen05 kernel of tc_attention.cu pays a 128 x 128 MMA tile, a TMEM round trip and a five-role pipeline
// per 128 context columns whatever the number of valid rows; here every warp is its own flash-decoding worker:
//   grid = (split, bank selection): a CTA owns a contiguous range of 64-column context tiles of one bank,
//   near tiles    64 ring rows of K and V, cp.async into a double-buffered shared stage,
//   pseudo tiles  8 prototypes x S = 64 pseudo-tokens k~ = c_k + concat_g CK_g[zK], v~ = p_k + concat_g CV_g[zV] built
//                 in shared memory by all 128 threads from operands prefetched into registers one tile ahead
//                 (pseudo-tokens never exist in HBM),
//   S = Q K~^T    mma.sync m16n8k16 (rows padded to 16), warp w owns columns [16 w, 16 w + 16) of the tile,
//   softmax       online (running row maximum, FA2 style) in the accumulator fragments, log-mass bias log n_k added
//                 to the pseudo columns (Eq. 2/4), exp2 domain,
//   O += P V~     mma.sync with P re-used from the accumulator registers as the A fragment.
// Warps w and w + 4 share a column group: both evaluate its S and softmax (cheap), each accumulates one half of the
// head dimension of O -- twice the warps per SM for the same shared-memory footprint.  Every column group keeps its own
// (m, l, O) and writes one unnormalised partial per query row; attention_combine_kernel (query_kernels.cu) merges the
// 4 x nsplit partials of a row.
#include "common.cuh"

namespace pkv {

constexpr int kDcThreads = 256, kDcWarps = 8;   // warp = (column group of 16, half of the head dim for O)
constexpr int kDcGroups = 4;                   // column groups per tile = partials per CTA and row
constexpr int kDcCols = 64;              // context columns per tile (16 per warp)
constexpr int kDcProto = 8;              // prototypes per pseudo tile (x S = 8)
constexpr int kDcStride = 272;           // bytes per staged row: 256 B of bf16 + 16 B pad (ldmatrix conflict-free)
constexpr int kDcRows = 16;              // query rows (MMA M)
constexpr int kDcCtasPerSm = 2;          // 113.4 KB of shared memory per CTA
constexpr float kDcLog2e = 1.4426950408889634f;
constexpr float kDcLn2 = 0.6931471805599453f;

constexpr int kDcStages = 3;             // operand ring: tiles t + 1 and t + 2 are in flight while tile t is consumed
constexpr uint32_t kDcStageBytes = kDcCols * kDcStride;   // one operand (K~ or V~) of one tile: 17,408 B
struct DcSmem {
  static constexpr uint32_t K = 0;                                   // [stages][64][272]
  static constexpr uint32_t V = K + kDcStages * kDcStageBytes;       // [stages][64][272]; a pseudo tile's RAW operands
                                                                     // land at the start of its V stage (see DcRaw)
  static constexpr uint32_t CBK = V + kDcStages * kDcStageBytes;     // [C][G][16] bf16
  static constexpr uint32_t CBV = CBK + 4096;
  static constexpr uint32_t Bias = CBV + 4096;                       // [stages][64] fp32, log2 domain
  static constexpr uint32_t Total = Bias + kDcStages * kDcCols * 4;  // 113,408 B: two CTAs per SM
  static constexpr uint32_t Q = K;                                   // [16][272], staged in stage 0 before the pipeline starts
};
struct DcRaw {   // byte offsets of a pseudo tile's raw operands inside its V stage
  static constexpr uint32_t C = 0, P = 4096, ZK = 8192, ZV = 8448, Ln = 8704, Kd = 8736;
};

struct DcArgs {
  const __nv_bfloat16* Q;
  float* part;              // [(bsel * R + row) * NS + split * 4 + column group][130]
  int n_q, layer_begin, layer_count;
  int n_near, n_act;
  int use_bias;
  int nt_near, nt_ps, ntile, nsplit;
  int R;                    // n_q * group
};

__device__ __forceinline__ uint32_t dc_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void dc_cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void dc_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void dc_cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void dc_ldsm_x4(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void dc_ldsm_x4_trans(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
// D (16x8 fp32) += A (16x16 bf16, row) * B (16x8 bf16, col)
__device__ __forceinline__ void dc_mma(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
               "{%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t dc_pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ uint32_t dc_add_bf16x2(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("add.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
__device__ __forceinline__ float dc_ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// Raw operands of one pseudo tile held by thread (side, kk, ch): 16-byte chunk ch (8 dims of subspace ch / 2) of the key
// (side 0) or value (side 1) centre of prototype kk, and that side's packed codes.
struct DcProtoRegs {
  float4 x0, x1;     // centre chunk (fp32)
  uint4 z0, z1;      // packed codes of the S modes
  int kind;          // 0 decoded, 1 zero residual, 2 absent
  float logn;
};

__device__ __forceinline__ void dc_read_staged(DcProtoRegs& r, const unsigned char* raw, int side, int kk, int ch, bool in_range) {
  const float4* xp = reinterpret_cast<const float4*>(raw + (side ? DcRaw::P : DcRaw::C) + kk * 512 + ch * 32);
  r.x0 = xp[0]; r.x1 = xp[1];
  const uint4* zp = reinterpret_cast<const uint4*>(raw + (side ? DcRaw::ZV : DcRaw::ZK) + kk * 32);
  r.z0 = zp[0]; r.z1 = zp[1];
  r.kind = in_range ? (int)raw[DcRaw::Kd + kk] : 2;
  r.logn = reinterpret_cast<const float*>(raw + DcRaw::Ln)[kk];
}

// Writes the 8 pseudo rows (kk * 8 + s) of this thread's chunk into one operand stage.
__device__ __forceinline__ void dc_build(unsigned char* dst, const unsigned char* cb, const DcProtoRegs& r, int kk, int ch) {
  const int sh = (ch >> 1) * 4;
  uint4 x = make_uint4(dc_pack_bf16(r.x0.x, r.x0.y), dc_pack_bf16(r.x0.z, r.x0.w), dc_pack_bf16(r.x1.x, r.x1.y),
                       dc_pack_bf16(r.x1.z, r.x1.w));
  if (r.kind == 2) x = make_uint4(0u, 0u, 0u, 0u);
  const uint32_t z[8] = {r.z0.x, r.z0.y, r.z0.z, r.z0.w, r.z1.x, r.z1.y, r.z1.z, r.z1.w};
  unsigned char* row = dst + kk * 8 * kDcStride + ch * 16;
  const unsigned char* cbt = cb + ch * 16;
#pragma unroll
  for (int s = 0; s < 8; ++s) {
    uint4 o = x;
    if (r.kind == 0) {
      const uint4 e = *reinterpret_cast<const uint4*>(cbt + ((z[s] >> sh) & 15u) * 256);
      o.x = dc_add_bf16x2(x.x, e.x); o.y = dc_add_bf16x2(x.y, e.y); o.z = dc_add_bf16x2(x.z, e.z); o.w = dc_add_bf16x2(x.w, e.w);
    }
    *reinterpret_cast<uint4*>(row + s * kDcStride) = o;
  }
}

__global__ void __launch_bounds__(kDcThreads, kDcCtasPerSm) attention_decode_kernel(Dims D, Dev V, DcArgs A) {
  extern __shared__ __align__(128) unsigned char sm[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int gid = lane >> 2, tig = lane & 3;
  const int bsel = blockIdx.y, split = blockIdx.x;
  const int hd = bsel % D.Hkv, ll = (bsel / D.Hkv) % A.layer_count, st = bsel / (D.Hkv * A.layer_count);
  const int b = (st * D.L + A.layer_begin + ll) * D.Hkv + hd;
  const int t0 = (int)(((long long)split * A.ntile) / A.nsplit), t1 = (int)(((long long)(split + 1) * A.ntile) / A.nsplit);

  // ---- one-time staging: Q rows (zero padded to 16), codebooks as bf16 [z][g][16] ----
  for (int e = tid; e < kDcRows * 16; e += kDcThreads) {
    const int r = e >> 4, chunk = e & 15;
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (r < A.R) {
      const int qi = r / D.group, hh = r % D.group;
      const size_t off = ((((size_t)st * A.layer_count + ll) * A.n_q + qi) * D.Hq + hd * D.group + hh) * 128 + chunk * 8;
      v = *reinterpret_cast<const uint4*>(A.Q + off);
    }
    *reinterpret_cast<uint4*>(sm + DcSmem::Q + r * kDcStride + chunk * 16) = v;
  }
  if (V.cbk && A.nt_ps > 0) {
    const float4* srck = reinterpret_cast<const float4*>(V.cbk + (size_t)b * 2048);
    const float4* srcv = reinterpret_cast<const float4*>(V.cbv + (size_t)b * 2048);
    for (int e = tid; e < 512; e += kDcThreads) {              // float4 e = (g, z, quarter)
      const int gg = e >> 6, z = (e >> 2) & 15, qd = e & 3;
      const float4 a = srck[e], c = srcv[e];
      const uint32_t off = (uint32_t)(z * 256 + gg * 32 + qd * 8);
      *reinterpret_cast<uint2*>(sm + DcSmem::CBK + off) = make_uint2(dc_pack_bf16(a.x, a.y), dc_pack_bf16(a.z, a.w));
      *reinterpret_cast<uint2*>(sm + DcSmem::CBV + off) = make_uint2(dc_pack_bf16(c.x, c.y), dc_pack_bf16(c.z, c.w));
    }
  }
  __syncthreads();
  uint32_t qa[8][4];                                            // A fragments of Q for the 8 k-chunks
  {
    const int mi = lane >> 3;
    const uint32_t base = dc_smem_u32(sm + DcSmem::Q) + ((lane & 7) + (mi & 1) * 8) * kDcStride + (mi >> 1) * 16;
#pragma unroll
    for (int kc = 0; kc < 8; ++kc) dc_ldsm_x4(base + kc * 32, qa[kc]);
  }

  const int side = tid >> 7, kk = (tid >> 4) & 7, ch = tid & 15;   // builder coordinates
  const int cgp = warp & 3, half = warp >> 2;                   // column group of the tile, half of the head dim
  const char* ringK = (const char*)V.ringK + (size_t)b * D.Wf * D.T * 256;
  const char* ringV = (const char*)V.ringV + (size_t)b * D.Wf * D.T * 256;
  float* bias_s = reinterpret_cast<float*>(sm + DcSmem::Bias);

  // issue the loads of tile t into stage `buf` (one cp.async group per tile): near rows straight into the operand
  // stages, a pseudo tile's raw operands (contiguous in the bank arrays) into the start of its V stage
  auto issue = [&](int t, int buf) {
    const uint32_t ks = dc_smem_u32(sm + DcSmem::K) + buf * kDcStageBytes, vs = dc_smem_u32(sm + DcSmem::V) + buf * kDcStageBytes;
    if (t < A.nt_near) {
      const int row0 = t * kDcCols;
#pragma unroll
      for (int i = 0; i < 4; ++i) {                             // 64 rows x 16 chunks = 1024 16-byte pieces per operand
        const int e = i * kDcThreads + tid, r = e >> 4, chunk = e & 15;
        const int rr = row0 + r < A.n_near ? row0 + r : A.n_near - 1;        // ragged tail: clamp (masked by the bias)
        const uint32_t dst = (uint32_t)(r * kDcStride + chunk * 16);
        dc_cp_async16(ks + dst, ringK + (size_t)rr * 256 + chunk * 16);
        dc_cp_async16(vs + dst, ringV + (size_t)rr * 256 + chunk * 16);
      }
    } else {
      const size_t pk0 = (size_t)b * D.K + (size_t)(t - A.nt_near) * kDcProto;
      const char* cs = (const char*)(V.c + pk0 * 128);
      const char* ps = (const char*)(V.p + pk0 * 128);
      dc_cp_async16(vs + DcRaw::C + tid * 16, cs + tid * 16);   // 8 prototypes x 512 B = 256 pieces per operand
      dc_cp_async16(vs + DcRaw::P + tid * 16, ps + tid * 16);
      if (tid < 16) dc_cp_async16(vs + DcRaw::ZK + tid * 16, (const char*)(V.codesK + pk0 * 8) + tid * 16);
      else if (tid < 32) dc_cp_async16(vs + DcRaw::ZV + (tid - 16) * 16, (const char*)(V.codesV + pk0 * 8) + (tid - 16) * 16);
      else if (tid < 34) dc_cp_async16(vs + DcRaw::Ln + (tid - 32) * 16, (const char*)(V.logn + pk0) + (tid - 32) * 16);
      else if (tid == 34)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(vs + DcRaw::Kd), "l"(V.kind + pk0) : "memory");
    }
  };

  float o[8][4];                                                // this warp's half of the head dim
#pragma unroll
  for (int i = 0; i < 8; ++i) { o[i][0] = 0.f; o[i][1] = 0.f; o[i][2] = 0.f; o[i][3] = 0.f; }
  float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;    // rows gid and gid + 8 (per-lane partial sums)
  const float sc2 = kDcLog2e * rsqrtf(128.f);

  __syncthreads();                                              // every warp holds its Q fragments: stage 0 is free
  if (t0 < t1) issue(t0, 0);
  dc_cp_async_commit();
  if (t0 + 1 < t1) issue(t0 + 1, 1);
  dc_cp_async_commit();
  for (int t = t0; t < t1; ++t) {
    const int buf = (t - t0) % kDcStages;
    asm volatile("cp.async.wait_group 1;" ::: "memory");        // this thread's pieces of tile t have landed
    __syncthreads();                                            // ... everybody's; and tile t - 1 has been consumed
    if (t + 2 < t1) issue(t + 2, (t - t0 + 2) % kDcStages);
    dc_cp_async_commit();
    unsigned char* kst = sm + DcSmem::K + buf * kDcStageBytes;
    unsigned char* vst = sm + DcSmem::V + buf * kDcStageBytes;
    if (t < A.nt_near) {
      if (tid < kDcCols) bias_s[buf * kDcCols + tid] = t * kDcCols + tid < A.n_near ? 0.f : -INFINITY;
      __syncthreads();
    } else {
      DcProtoRegs pr;
      const int k = (t - A.nt_near) * kDcProto + kk;
      dc_read_staged(pr, vst, side, kk, ch, k < A.n_act);
      __syncthreads();                                          // raw operands are in registers: V~ may overwrite them
      dc_build(side ? vst : kst, sm + (side ? DcSmem::CBV : DcSmem::CBK), pr, kk, ch);
      if (side == 0 && ch < 8) bias_s[buf * kDcCols + kk * 8 + ch] = pr.kind == 2 ? -INFINITY : (A.use_bias ? pr.logn * kDcLog2e : 0.f);
      __syncthreads();
    }
    // ---- S = Q K~^T for this warp's 16 columns ----
    float s[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
    {
      const int mi = lane >> 3;
      const uint32_t kbase = dc_smem_u32(kst) + (uint32_t)((cgp * 16 + (mi >> 1) * 8 + (lane & 7)) * kDcStride + (mi & 1) * 16);
#pragma unroll
      for (int kc = 0; kc < 8; ++kc) {
        uint32_t kb[4];
        dc_ldsm_x4(kbase + kc * 32, kb);
        dc_mma(s[0], qa[kc], kb[0], kb[1]);
        dc_mma(s[1], qa[kc], kb[2], kb[3]);
      }
    }
    // ---- online softmax on the fragments: lane holds rows gid (c0, c1) and gid + 8 (c2, c3) ----
    const float* bs = bias_s + buf * kDcCols + cgp * 16 + tig * 2;
    const float b00 = bs[0], b01 = bs[1], b10 = bs[8], b11 = bs[9];
    float x[2][4];
    x[0][0] = fmaf(s[0][0], sc2, b00); x[0][1] = fmaf(s[0][1], sc2, b01);
    x[0][2] = fmaf(s[0][2], sc2, b00); x[0][3] = fmaf(s[0][3], sc2, b01);
    x[1][0] = fmaf(s[1][0], sc2, b10); x[1][1] = fmaf(s[1][1], sc2, b11);
    x[1][2] = fmaf(s[1][2], sc2, b10); x[1][3] = fmaf(s[1][3], sc2, b11);
    float mx0 = fmaxf(fmaxf(x[0][0], x[0][1]), fmaxf(x[1][0], x[1][1]));
    float mx1 = fmaxf(fmaxf(x[0][2], x[0][3]), fmaxf(x[1][2], x[1][3]));
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1)); mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1)); mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
    const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
    const float mu0 = mn0 == -INFINITY ? 0.f : mn0, mu1 = mn1 == -INFINITY ? 0.f : mn1;   // all masked so far
    const float a0 = dc_ex2(m0 - mu0), a1 = dc_ex2(m1 - mu1);   // m = -inf: 0
    m0 = mn0; m1 = mn1;
    float p[2][4];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      p[nt][0] = dc_ex2(x[nt][0] - mu0); p[nt][1] = dc_ex2(x[nt][1] - mu0);
      p[nt][2] = dc_ex2(x[nt][2] - mu1); p[nt][3] = dc_ex2(x[nt][3] - mu1);
    }
    l0 = fmaf(l0, a0, (p[0][0] + p[0][1]) + (p[1][0] + p[1][1]));
    l1 = fmaf(l1, a1, (p[0][2] + p[0][3]) + (p[1][2] + p[1][3]));
    if (__any_sync(0xffffffffu, a0 != 1.f || a1 != 1.f)) {
#pragma unroll
      for (int i = 0; i < 8; ++i) { o[i][0] *= a0; o[i][1] *= a0; o[i][2] *= a1; o[i][3] *= a1; }
    }
    // ---- O += P V~: P (accumulator layout of two n-tiles) is the A fragment of a k = 16 step ----
    uint32_t pa[4];
    pa[0] = dc_pack_bf16(p[0][0], p[0][1]); pa[1] = dc_pack_bf16(p[0][2], p[0][3]);
    pa[2] = dc_pack_bf16(p[1][0], p[1][1]); pa[3] = dc_pack_bf16(p[1][2], p[1][3]);
    {
      const int mi = lane >> 3;
      const uint32_t vbase = dc_smem_u32(vst) + (uint32_t)((cgp * 16 + (mi & 1) * 8 + (lane & 7)) * kDcStride + (mi >> 1) * 16) +
                             half * 128;
#pragma unroll
      for (int dn = 0; dn < 8; dn += 2) {
        uint32_t vb[4];
        dc_ldsm_x4_trans(vbase + dn * 16, vb);
        dc_mma(o[dn], pa, vb[0], vb[1]);
        dc_mma(o[dn + 1], pa, vb[2], vb[3]);
      }
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");

  // ---- partial result of this warp: unnormalised O, m (natural log units), l ----
  l0 += __shfl_xor_sync(0xffffffffu, l0, 1); l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
  l1 += __shfl_xor_sync(0xffffffffu, l1, 1); l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
  const int NS = A.nsplit * kDcGroups;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int r = gid + 8 * h;
    if (r >= A.R) continue;
    float* dst = A.part + (((size_t)bsel * A.R + r) * NS + split * kDcGroups + cgp) * 130;
#pragma unroll
    for (int dn = 0; dn < 8; ++dn)
      *reinterpret_cast<float2*>(dst + half * 64 + dn * 8 + tig * 2) = make_float2(o[dn][2 * h], o[dn][2 * h + 1]);
    if (tig == 0 && half == 0) {
      const float m = h ? m1 : m0, l = h ? l1 : l0;
      dst[128] = m == -INFINITY ? -INFINITY : m * kDcLn2;
      dst[129] = l;
    }
  }
}

bool decode_attention_supported(const Dims& D, int n_q) {
  return D.bf16 && D.d == 128 && D.S == 8 && D.G == 8 && D.C == 16 && n_q * D.group <= kDcRows && D.K % kDcProto == 0;
}

size_t decode_attention_part_bytes(const Dims& D) {
  // at most (kDcCtasPerSm * 148 + B) CTAs x 4 warps x 16 rows partial rows of 130 floats
  return (size_t)(kDcCtasPerSm * 148 + D.B) * kDcGroups * kDcRows * 130 * sizeof(float);
}

bool decode_attention_prepare() {
  if (cudaFuncSetAttribute(attention_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DcSmem::Total) !=
      cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return true;
}

// Launches the decode kernel and fills `nsplit_out` with the number of partials per row the combine kernel must merge.
int launch_attention_decode(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, int sm_count, cudaStream_t s,
                            int* nsplit_out) {
  DcArgs a{};
  a.Q = (const __nv_bfloat16*)A.Q;
  a.part = V.part;
  a.n_q = A.n_q; a.layer_begin = A.layer_begin; a.layer_count = A.layer_count;
  a.n_near = (H.flags & PROTOKV_FAR_ONLY) ? 0 : A.n_near;
  a.n_act = (H.flags & PROTOKV_NEAR_ONLY) ? 0 : A.n_act;
  a.use_bias = !(H.flags & PROTOKV_NO_MASS_BIAS);
  a.nt_near = (a.n_near + kDcCols - 1) / kDcCols;
  a.nt_ps = (a.n_act + kDcProto - 1) / kDcProto;
  a.ntile = a.nt_near + a.nt_ps;
  a.R = A.n_q * D.group;
  const int nb = D.NS * A.layer_count * D.Hkv;
  int ns = (kDcCtasPerSm * sm_count + nb - 1) / nb;          // one wave of resident CTAs
  if (ns > a.ntile) ns = a.ntile;
  if (ns < 1) ns = 1;
  while (ns > 1 && (long long)ns * nb > (long long)kDcCtasPerSm * 148 + D.B) --ns;         // partial buffer bound (decode_attention_part_bytes)
  a.nsplit = ns;
  *nsplit_out = ns * kDcGroups;
  attention_decode_kernel<<<dim3(ns, nb), kDcThreads, DcSmem::Total, s>>>(D, V, a);
  return 1;
}

}  // namespace pkv
