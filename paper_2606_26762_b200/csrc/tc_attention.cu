// Q2 fused attention on the 5th-gen tensor cores (bf16, d = 128, S = 8, G = 8, C = 16): Alg. 4 l.8-15 / Eq. 4
// as a flash-style kernel over [near window || pseudo-tokens].
//
//   near tiles    128 ring rows of K and V, loaded by TMA (128-byte swizzle)
//   pseudo tiles  16 prototypes x S = 128 pseudo-tokens k~ = c_k + concat_g CK_g[zK(k,s,g)], v~ = p_k + concat_g CV_g[zV]
//                 (Alg. 4 l.5-9) built in shared memory by the builder warpgroup: the tile's centres, codes, kinds and
//                 log-masses arrive in a staging buffer by bulk copies issued one tile ahead, the codebooks sit in
//                 shared memory as bf16 -- pseudo-tokens never exist in HBM
//   S = Q K~^T    tcgen05.mma, Q tile (M = 128 query rows) and K~ tile from shared memory, fp32 accumulator in TMEM
//   softmax       one thread per query row drains S with tcgen05.ld (double-buffered 32-column chunks), adds the
//                 log-mass bias log n_k (Eq. 2/4, 0 on near tokens), exponentiates against a lazily updated reference
//                 maximum (packed f32x2 arithmetic), writes P as bf16 back into the columns S occupied (tcgen05.st)
//   O += P V~     tcgen05.mma with A = P from TMEM, B = V~ tile (MN-major) from shared memory
//
// One CTA works on two M tiles of a bank (256 query rows = n_q x GQA group) in ping-pong, so the tensor pipe runs the
// MMAs of one tile while the softmax warps of the other drain theirs.  The grid is persistent: the (item, tile) space
// -- item = (bank, block of <= 256 query rows) -- is cut into gridDim.x equal contiguous spans, so a CTA's span may
// cover the tail of one item and the head of the next; every (item, span) piece writes an unnormalised partial
// (O, m, l) and attention_tc_combine_kernel merges the pieces of an item.
//
// Warp roles (16 warps, warpgroup-aligned so that setmaxnreg can move registers to the softmax threads):
//   warps 0-3 / 4-7   softmax of M tile 0 / 1 (warp % 4 = TMEM lane quarter)
//   warps 8-11        builders of the pseudo tiles
//   warp 12           MMA issuer + TMEM owner;  warp 13: loader (TMA for Q and near tiles, bulk copies into the staging
//                     buffer);  warps 14-15 idle
#include "common.cuh"
#include "tc_common.cuh"

namespace pkv {

using namespace tc;

constexpr int kAtThreads = 512;
constexpr int kAtCols = 128;            // context columns per tile
constexpr int kAtProto = 16;            // prototypes per pseudo tile (x S = 8)
constexpr int kAtRows = 256;            // query rows per item (two M tiles)
constexpr uint32_t kAtHalf = 128 * 128; // one [128 rows][64 bf16] swizzled box = 16 KB
constexpr int kAtBiasRing = 4;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
// P is packed to bf16 by TRUNCATION (one PRMT per pair on the ALU pipe; cvt.rn.bf16x2 runs on the 4-lane XU pipe next
// to MUFU.EX2, the pipe that bounds the softmax).  Truncation alone is biased by -2^-9 relative, so the exponent
// carries +log2(1 + 2^-9): P^ = (1 + 2^-9) P truncated has zero mean error and the spread of round-to-nearest; the
// row sum is accumulated from P^ and scaled back by 1 / (1 + 2^-9) once per tile.
constexpr float kTruncBiasLog2 = 0.0028151f;
constexpr float kTruncBiasInv = 0.99805068f;
constexpr float kRescaleSum = 256.f;    // a tile's row sum of P above this moves the reference maximum (P <= 2^8 in bf16)
constexpr int kRegsSoftmax = 184, kRegsBuilder = 104, kRegsAux = 40;  // 2 * 184 + 104 + 40 = 512 = 4 * 128

struct AtSmem {   // byte offsets from a 1024-byte aligned base
  static constexpr uint32_t Q = 0;                          // 2 d-halves x [256 rows][128 B]
  static constexpr uint32_t K = Q + 4 * kAtHalf;            // 2 stages x (2 d-halves x 16 KB)
  static constexpr uint32_t V = K + 4 * kAtHalf;            // 2 stages x (2 d-halves x 16 KB)
  static constexpr uint32_t CBK = V + 4 * kAtHalf;          // [C][G][16] bf16: code z at z * 256 B, chunk ch at ch * 16 B
  static constexpr uint32_t CBV = CBK + 4096;
  static constexpr uint32_t StgC = CBV + 4096;              // staging of one pseudo tile: c [16][128] fp32
  static constexpr uint32_t StgP = StgC + 8192;             //   p [16][128] fp32
  static constexpr uint32_t StgZK = StgP + 8192;            //   codesK [16][8] u32
  static constexpr uint32_t StgZV = StgZK + 512;            //   codesV
  static constexpr uint32_t StgLn = StgZV + 512;            //   log n [16] fp32
  static constexpr uint32_t StgKd = StgLn + 64;             //   kind [16] u8
  static constexpr uint32_t Bias = StgKd + 64;              // [ring][16] fp32, log2 domain
  static constexpr uint32_t Bar = Bias + kAtBiasRing * kAtProto * 4;
  static constexpr uint32_t Total = Bar + 256;
};
constexpr uint32_t kStgBytes = 8192 + 8192 + 512 + 512 + 64 + 16;

// Partition of the tile space shared by the kernel, the combine kernel and the host.
struct AtPlan {
  int items;        // (bank selection, row block) pairs
  int nrb;          // row blocks per bank
  int tb;           // query tokens per row block (tb * group <= 256)
  int nt_near;      // near tiles per item
  int nt_ps;        // pseudo tiles per item
  int ntile;        // nt_near + nt_ps
  int grid;
  int nsplit;       // max pieces per item (partial buffer stride)
  long long ttot;   // items * ntile
};

__host__ __device__ inline long long at_span_begin(const AtPlan& P, int cta) { return ((long long)cta * P.ttot) / P.grid; }
// CTA whose span contains global tile x.
__host__ __device__ inline int at_cta_of(const AtPlan& P, long long x) {
  if ((P.ttot + 1) * P.grid < (1ll << 31))   // the usual case: 32-bit division (the 64-bit one is a ~100-instruction routine)
    return (int)(((uint32_t)(x + 1) * (uint32_t)P.grid + (uint32_t)P.ttot - 1u) / (uint32_t)P.ttot) - 1;
  return (int)(((x + 1) * P.grid + P.ttot - 1) / P.ttot - 1);
}

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ uint32_t add_bf16x2(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("add.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
// packed fp32 pairs (sm_100 f32x2 arithmetic): one issue slot for two elements
__device__ __forceinline__ uint64_t pack_f32x2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack_f32x2(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t fma_f32x2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ uint64_t add_f32x2(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }

struct AtArgs {
  const void* Q;   // unused by the kernel (the tensor map addresses it); kept for the combine kernel's layout maths
  int n_q, layer_begin, layer_count;
  int n_near, n_act;
  int use_bias;
};

// One contiguous piece of an item inside this CTA's span.
struct AtSeg {
  int item, t0, t1;       // tiles [t0, t1) of the item
  int b;                  // bank
  int st, ll, hd, rb;     // stream, layer (relative to layer_begin), KV head, row block
  int R;                  // valid query rows of the block (<= 256)
  int ntm;                // M tiles in use (1 or 2)
  int piece;              // index of this piece among the item's pieces
};

__device__ __forceinline__ AtSeg at_segment(const AtPlan& P, const Dims& D, const AtArgs& A, long long g, long long g1) {
  AtSeg s;
  s.item = (int)(g / P.ntile);
  s.t0 = (int)(g - (long long)s.item * P.ntile);
  const long long room = g1 - g;
  s.t1 = (int)((long long)(P.ntile - s.t0) < room ? P.ntile : s.t0 + room);
  const int bsel = s.item / P.nrb;
  s.rb = s.item % P.nrb;
  s.hd = bsel % D.Hkv;
  s.ll = (bsel / D.Hkv) % A.layer_count;
  s.st = bsel / (D.Hkv * A.layer_count);
  s.b = (s.st * D.L + A.layer_begin + s.ll) * D.Hkv + s.hd;
  const int tok0 = s.rb * P.tb;
  const int ntok = min(P.tb, A.n_q - tok0);
  s.R = ntok * D.group;
  s.ntm = s.R > 128 ? 2 : 1;
  s.piece = (int)blockIdx.x - at_cta_of(P, (long long)s.item * P.ntile);
  return s;
}

// x'_i = S_i * sc2 + bm[i / 8]  (log2 domain, relative to the reference maximum); returns max_i x'_i of the row.
template <bool RAGGED>
__device__ __forceinline__ float at_row_max(uint32_t s_addr, float sc2, const float (&bm)[16], int nvalid) {
  float mx = -INFINITY;
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    uint32_t a[32];
    tmem_ld_32x32(s_addr + c * 32, a);
    tmem_ld_wait();
#pragma unroll
    for (int i = 0; i < 32; ++i) {
      float x = fmaf(__uint_as_float(a[i]), sc2, bm[(c * 32 + i) >> 3]);
      if (RAGGED && c * 32 + i >= nvalid) x = -INFINITY;
      mx = fmaxf(mx, x);
    }
  }
  return mx;
}

// One pass over the S tile of this row: P = exp2(x') packed to bf16 pairs and the row sum of P.  The 32-column chunks
// are double-buffered: chunk c + 1 is in flight from TMEM while chunk c is exponentiated.
template <bool RAGGED>
__device__ __forceinline__ void at_row_pass(uint32_t s_addr, float sc2, const float (&bm)[16], int nvalid,
                                            uint32_t (&pk)[64], float& lsum) {
  const uint64_t sc22 = pack_f32x2(sc2, sc2);
  uint64_t l2 = pack_f32x2(0.f, 0.f);
  uint32_t a[2][32];
  tmem_ld_32x32(s_addr, a[0]);
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    tmem_ld_wait();
    if (c < 3) tmem_ld_32x32(s_addr + (c + 1) * 32, a[(c + 1) & 1]);
#pragma unroll
    for (int i = 0; i < 32; i += 2) {
      const float b = bm[(c * 32 + i) >> 3] + kTruncBiasLog2;
      const uint64_t x2 = fma_f32x2(pack_f32x2(__uint_as_float(a[c & 1][i]), __uint_as_float(a[c & 1][i + 1])), sc22,
                                    pack_f32x2(b, b));
      float x0, x1;
      unpack_f32x2(x2, x0, x1);
      if (RAGGED) {
        if (c * 32 + i >= nvalid) x0 = -INFINITY;
        if (c * 32 + i + 1 >= nvalid) x1 = -INFINITY;
      }
      const float p0 = ex2_approx(x0), p1 = ex2_approx(x1);
      l2 = add_f32x2(l2, pack_f32x2(p0, p1));
      pk[c * 16 + (i >> 1)] = __byte_perm(__float_as_uint(p0), __float_as_uint(p1), 0x7632);
    }
  }
  float l0, l1;
  unpack_f32x2(l2, l0, l1);
  lsum = (l0 + l1) * kTruncBiasInv;
}

struct AtBars {
  uint64_t *q_full, *q_empty, *k_full, *k_empty, *v_full, *v_empty, *s_full, *p_full, *pv_done, *o_empty, *stg_full,
      *stg_empty;
  __device__ explicit AtBars(uint64_t* b)
      : q_full(b), q_empty(b + 1), k_full(b + 2), k_empty(b + 4), v_full(b + 6), v_empty(b + 8), s_full(b + 10),
        p_full(b + 12), pv_done(b + 14), o_empty(b + 16), stg_full(b + 18), stg_empty(b + 19) {}
};
constexpr int kAtNumBars = 20;

// ---- warp 12: MMA issuer ------------------------------------------------------------------------------------
// The whole warp runs the role converged (every lane observes every barrier phase); the tcgen05 instructions of a
// block are issued by one elected lane, so the compiler emits no per-instruction election loop.  Descriptors are a
// precomputed 64-bit base plus a small constant (the 14-bit address field never carries).
__device__ __forceinline__ void at_issue_s(uint32_t d_tmem, uint64_t qd, uint64_t kd) {
  constexpr uint32_t idesc = idesc_bf16(128, 128, 0, 0);
#pragma unroll
  for (int half = 0; half < 2; ++half) {
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) {
      const uint64_t ad = qd + (uint64_t)((half * 2 * kAtHalf + kk * 32) >> 4);
      const uint64_t bd = kd + (uint64_t)((half * kAtHalf + kk * 32) >> 4);
      umma_bf16(d_tmem, ad, bd, idesc, (half | kk) != 0);
    }
  }
}
__device__ __forceinline__ void at_issue_pv(uint32_t o_tmem, uint32_t p_tmem, uint64_t vd, bool acc) {
  constexpr uint32_t idesc = idesc_bf16(128, 128, 0, 1);   // B = V~ tile, MN-major (d contiguous)
#pragma unroll
  for (int kk = 0; kk < 8; ++kk)                           // 16 context columns (= MMA K) per instruction
    umma_bf16_ts(o_tmem, p_tmem + kk * 8, vd + (uint64_t)((kk * 2048) >> 4), idesc, acc || kk != 0);
}

__device__ void at_mma_role(unsigned char* sm, const AtBars& B, uint32_t tmem_base, const Dims& D, const AtArgs& A,
                            const AtPlan& P) {
  const uint64_t qd0 = desc_kmajor_sw128(smem_u32(sm + AtSmem::Q));
  const uint64_t kd0 = desc_kmajor_sw128(smem_u32(sm + AtSmem::K));
  const uint64_t vd0 = desc_mnmajor_sw128(smem_u32(sm + AtSmem::V), kAtHalf);
  constexpr uint64_t kStage = (2 * kAtHalf) >> 4, kQTile = kAtHalf >> 4;
  uint32_t kc = 0, vc = 0, ic = 0, pc[2] = {0, 0}, oc[2] = {0, 0};
  const long long g1 = at_span_begin(P, blockIdx.x + 1);
  for (long long g = at_span_begin(P, blockIdx.x); g < g1;) {
    const AtSeg sg = at_segment(P, D, A, g, g1);
    const int n = sg.t1 - sg.t0;
    g += n;
    mbar_wait(B.q_full, ic & 1);
    mbar_wait(B.k_full + (kc & 1), (kc >> 1) & 1);
    tc_fence_after_sync();
    if (elect_one_sync()) {
      for (int w = 0; w < sg.ntm; ++w) {
        at_issue_s(tmem_base + w * 128, qd0 + w * kQTile, kd0 + (kc & 1) * kStage);
        umma_commit(B.s_full + w);
      }
      umma_commit(B.k_empty + (kc & 1));
    }
    __syncwarp();
    ++kc;
    for (int jj = 0; jj < n; ++jj) {
      const bool more = jj + 1 < n;
      const uint32_t sv = vc & 1;
      mbar_wait(B.v_full + sv, (vc >> 1) & 1);
      for (int w = 0; w < sg.ntm; ++w) {
        mbar_wait(B.p_full + w, pc[w] & 1);
        ++pc[w];
        if (jj == 0) {             // the first PV of an item overwrites O: the previous item's epilogue must have read it
          mbar_wait(B.o_empty + w, (oc[w] & 1) ^ 1);
          ++oc[w];
        }
        if (more && w == 0) mbar_wait(B.k_full + (kc & 1), (kc >> 1) & 1);
        tc_fence_after_sync();
        if (elect_one_sync()) {
          at_issue_pv(tmem_base + 256 + w * 128, tmem_base + w * 128, vd0 + sv * kStage, jj > 0);
          umma_commit(B.pv_done + w);
          if (more) {              // S of the next tile goes after PV_w: P_w aliases S_w
            at_issue_s(tmem_base + w * 128, qd0 + w * kQTile, kd0 + (kc & 1) * kStage);
            umma_commit(B.s_full + w);
          }
          if (w + 1 == sg.ntm) {
            umma_commit(B.v_empty + sv);
            if (more) umma_commit(B.k_empty + (kc & 1));
          }
        }
        __syncwarp();
      }
      ++vc;
      if (more) ++kc;
    }
    if (elect_one_sync()) umma_commit(B.q_empty);
    __syncwarp();
    ++ic;
  }
}

// ---- warp 13: loader (one lane) -------------------------------------------------------------------------------
// Q boxes and near tiles by TMA straight into the operand stages; for pseudo tiles the raw operands of the tile
// (centres, codes, kinds, log-masses of its 16 prototypes, all contiguous in the bank arrays) by bulk copies into the
// single staging buffer, which the builders empty into registers before they build -- so the copies of tile j + 1
// overlap the build of tile j.
__device__ void at_loader_role(unsigned char* sm, const AtBars& B, const CUtensorMap* tmQ, const CUtensorMap* tmRK,
                               const CUtensorMap* tmRV, const Dims& D, const Dev& V, const AtArgs& A, const AtPlan& P) {
  const uint32_t qbytes = 256u * (uint32_t)D.group * (uint32_t)P.tb;   // two boxes {64 bf16, group, tb}
  uint32_t tcnt = 0, pcnt = 0, ic = 0;
  const long long g1 = at_span_begin(P, blockIdx.x + 1);
  for (long long g = at_span_begin(P, blockIdx.x); g < g1;) {
    const AtSeg sg = at_segment(P, D, A, g, g1);
    g += sg.t1 - sg.t0;
    mbar_wait(B.q_empty, (ic & 1) ^ 1);
    mbar_arrive_expect_tx(B.q_full, qbytes);
    const int tok = (sg.st * A.layer_count + sg.ll) * A.n_q + sg.rb * P.tb;
    tma_load_3d(sm + AtSmem::Q, tmQ, 0, sg.hd * D.group, tok, B.q_full);
    tma_load_3d(sm + AtSmem::Q + 2 * kAtHalf, tmQ, 64, sg.hd * D.group, tok, B.q_full);
    ++ic;
    for (int j = sg.t0; j < sg.t1; ++j, ++tcnt) {
      const uint32_t stg = tcnt & 1, par = ((tcnt >> 1) & 1) ^ 1;
      if (j < P.nt_near) {
        unsigned char* ks = sm + AtSmem::K + stg * 2 * kAtHalf;
        unsigned char* vs = sm + AtSmem::V + stg * 2 * kAtHalf;
        const int row0 = sg.b * D.Wf * D.T + j * kAtCols;
        mbar_wait(B.k_empty + stg, par);
        mbar_arrive_expect_tx(B.k_full + stg, 2 * kAtHalf);
        tma_load_2d(ks, tmRK, 0, row0, B.k_full + stg);
        tma_load_2d(ks + kAtHalf, tmRK, 64, row0, B.k_full + stg);
        mbar_wait(B.v_empty + stg, par);
        mbar_arrive_expect_tx(B.v_full + stg, 2 * kAtHalf);
        tma_load_2d(vs, tmRV, 0, row0, B.v_full + stg);
        tma_load_2d(vs + kAtHalf, tmRV, 64, row0, B.v_full + stg);
      } else {
        const size_t pk0 = (size_t)sg.b * D.K + (size_t)(j - P.nt_near) * kAtProto;
        mbar_wait(B.stg_empty, (pcnt & 1) ^ 1);
        mbar_arrive_expect_tx(B.stg_full, kStgBytes);
        bulk_load_1d(sm + AtSmem::StgC, V.c + pk0 * 128, 8192, B.stg_full);
        bulk_load_1d(sm + AtSmem::StgP, V.p + pk0 * 128, 8192, B.stg_full);
        bulk_load_1d(sm + AtSmem::StgZK, V.codesK + pk0 * 8, 512, B.stg_full);
        bulk_load_1d(sm + AtSmem::StgZV, V.codesV + pk0 * 8, 512, B.stg_full);
        bulk_load_1d(sm + AtSmem::StgLn, V.logn + pk0, 64, B.stg_full);
        bulk_load_1d(sm + AtSmem::StgKd, V.kind + pk0, 16, B.stg_full);
        ++pcnt;
      }
    }
  }
  if (ic > 0) mbar_wait(B.q_empty, (ic & 1) ^ 1);   // every MMA of this CTA has completed
}

// ---- warps 8-11: builders of the pseudo tiles ------------------------------------------------------------------
// Thread (kk, ch) owns the 16-byte chunk ch (8 dims of subspace ch / 2) of prototypes kk and kk + 8 of the tile, for
// all S pseudo-tokens of each.
struct AtProtoRegs {
  uint32_t x[2][4];     // centre chunk (c_k or p_k) as bf16 pairs
  uint32_t code[2][8];  // packed codes of the S modes (subspace g in bits [4g, 4g+4))
};

__device__ __forceinline__ void at_read_staged(AtProtoRegs& r, const unsigned char* centres, const unsigned char* codes,
                                               int kk, int ch) {
#pragma unroll
  for (int u = 0; u < 2; ++u) {
    const int kl = kk + 8 * u;
    const float4 a = *reinterpret_cast<const float4*>(centres + kl * 512 + ch * 32);
    const float4 b = *reinterpret_cast<const float4*>(centres + kl * 512 + ch * 32 + 16);
    r.x[u][0] = pack_bf16(a.x, a.y); r.x[u][1] = pack_bf16(a.z, a.w);
    r.x[u][2] = pack_bf16(b.x, b.y); r.x[u][3] = pack_bf16(b.z, b.w);
    const uint4 c0 = *reinterpret_cast<const uint4*>(codes + kl * 32);
    const uint4 c1 = *reinterpret_cast<const uint4*>(codes + kl * 32 + 16);
    r.code[u][0] = c0.x; r.code[u][1] = c0.y; r.code[u][2] = c0.z; r.code[u][3] = c0.w;
    r.code[u][4] = c1.x; r.code[u][5] = c1.y; r.code[u][6] = c1.z; r.code[u][7] = c1.w;
  }
}

// Writes rows (kl * 8 + s) of the tile (K-major, 128-byte swizzle, two d-halves) for this thread's two prototypes.
// kd: 0 decoded (centre + codeword), 1 zero residual (centre), 2 absent (zeros; its bias is -inf).
__device__ __forceinline__ void at_build_tile(unsigned char* tile, const unsigned char* cb, const AtProtoRegs& r,
                                              const int (&kd)[2], int kk, int ch) {
  const int sh = (ch >> 1) * 4;
  const unsigned char* cbt = cb + ch * 16;                 // + z * 256
  unsigned char* base = tile + (ch >> 3) * kAtHalf;
#pragma unroll
  for (int u = 0; u < 2; ++u) {
    uint4 x = make_uint4(r.x[u][0], r.x[u][1], r.x[u][2], r.x[u][3]);
    if (kd[u] == 2) x = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
    for (int s = 0; s < 8; ++s) {
      uint4 o = x;
      if (kd[u] == 0) {
        const uint32_t z = (r.code[u][s] >> sh) & 15u;
        const uint4 e = *reinterpret_cast<const uint4*>(cbt + z * 256);
        o.x = add_bf16x2(x.x, e.x); o.y = add_bf16x2(x.y, e.y); o.z = add_bf16x2(x.z, e.z); o.w = add_bf16x2(x.w, e.w);
      }
      const int row = (kk + 8 * u) * 8 + s;                // row & 7 == s
      *reinterpret_cast<uint4*>(base + row * 128 + (((ch & 7) ^ s) << 4)) = o;
    }
  }
}

__device__ void at_builder_role(unsigned char* sm, const AtBars& B, const Dims& D, const Dev& V, const AtArgs& A,
                                const AtPlan& P, int ptid) {
  const int kk = ptid >> 4, ch = ptid & 15;
  unsigned char* cbk_s = sm + AtSmem::CBK;
  unsigned char* cbv_s = sm + AtSmem::CBV;
  float* bias_s = reinterpret_cast<float*>(sm + AtSmem::Bias);
  uint32_t tcnt = 0, pcnt = 0;
  int cur_bank = -1;
  const long long g1 = at_span_begin(P, blockIdx.x + 1);
  for (long long g = at_span_begin(P, blockIdx.x); g < g1;) {
    const AtSeg sg = at_segment(P, D, A, g, g1);
    g += sg.t1 - sg.t0;
    if (sg.t1 <= P.nt_near) { tcnt += sg.t1 - sg.t0; continue; }
    if (sg.b != cur_bank && V.cbk) {   // codebooks of this bank -> bf16, [z][g][16]
      asm volatile("bar.sync 1, 128;" ::: "memory");      // nobody still builds with the previous bank's codebooks
      const float4* srck = reinterpret_cast<const float4*>(V.cbk + (size_t)sg.b * 2048);
      const float4* srcv = reinterpret_cast<const float4*>(V.cbv + (size_t)sg.b * 2048);
      for (int e = ptid; e < 512; e += 128) {              // float4 e = (g, z, quarter)
        const int gg = e >> 6, z = (e >> 2) & 15, qd = e & 3;
        const float4 a = srck[e], b = srcv[e];
        const uint32_t off = (uint32_t)(z * 256 + gg * 32 + qd * 8);
        *reinterpret_cast<uint2*>(cbk_s + off) = make_uint2(pack_bf16(a.x, a.y), pack_bf16(a.z, a.w));
        *reinterpret_cast<uint2*>(cbv_s + off) = make_uint2(pack_bf16(b.x, b.y), pack_bf16(b.z, b.w));
      }
      cur_bank = sg.b;
      asm volatile("bar.sync 1, 128;" ::: "memory");
    }
    const int jb = sg.t0 > P.nt_near ? sg.t0 : P.nt_near;
    tcnt += jb - sg.t0;
    for (int j = jb; j < sg.t1; ++j, ++tcnt, ++pcnt) {
      const uint32_t stg = tcnt & 1, par = ((tcnt >> 1) & 1) ^ 1;
      unsigned char* ks = sm + AtSmem::K + stg * 2 * kAtHalf;
      unsigned char* vs = sm + AtSmem::V + stg * 2 * kAtHalf;
      const int k0 = (j - P.nt_near) * kAtProto;
      mbar_wait(B.stg_full, pcnt & 1);
      AtProtoRegs r;
      at_read_staged(r, sm + AtSmem::StgC, sm + AtSmem::StgZK, kk, ch);
      int kd[2];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int kl = kk + 8 * u;
        kd[u] = k0 + kl < A.n_act ? (int)sm[AtSmem::StgKd + kl] : 2;
      }
      if (ptid < kAtProto) {
        float bias = -INFINITY;
        if (k0 + ptid < A.n_act && sm[AtSmem::StgKd + ptid] != 2)
          bias = A.use_bias ? reinterpret_cast<const float*>(sm + AtSmem::StgLn)[ptid] * kLog2e : 0.f;
        bias_s[(tcnt & (kAtBiasRing - 1)) * kAtProto + ptid] = bias;
      }
      mbar_wait(B.k_empty + stg, par);
      at_build_tile(ks, cbk_s, r, kd, kk, ch);
      fence_proxy_async_smem();
      asm volatile("bar.sync 1, 128;" ::: "memory");
      if (ptid == 0) mbar_arrive(B.k_full + stg);
      at_read_staged(r, sm + AtSmem::StgP, sm + AtSmem::StgZV, kk, ch);
      mbar_arrive(B.stg_empty);                            // staged operands are in registers: next tile may land
      mbar_wait(B.v_empty + stg, par);
      at_build_tile(vs, cbv_s, r, kd, kk, ch);
      fence_proxy_async_smem();
      asm volatile("bar.sync 1, 128;" ::: "memory");
      if (ptid == 0) mbar_arrive(B.v_full + stg);
    }
  }
}

// ---- warps 0-7: softmax (thread = query row of M tile w) ------------------------------------------------------
constexpr int kPartStride = 132;   // floats per partial row: O[128], m (natural log units), l, 2 pad (16-byte rows)

__device__ void at_softmax_role(unsigned char* sm, const AtBars& B, uint32_t tmem_base, const Dims& D, const AtArgs& A,
                                const AtPlan& P, float* part, int w, int q, int lane) {
  const int row = q * 32 + lane;
  const uint32_t lane_off = (uint32_t)(q * 32) << 16;
  const uint32_t s_addr = tmem_base + lane_off + w * 128;
  const uint32_t o_addr = tmem_base + lane_off + 256 + w * 128;
  const float sc2 = kLog2e * rsqrtf(128.f);
  const float* bias_s = reinterpret_cast<const float*>(sm + AtSmem::Bias);
  uint32_t cnt = 0, gt = 0;     // tiles this warpgroup has finished; tiles the CTA has been through
  const long long g1 = at_span_begin(P, blockIdx.x + 1);
  for (long long g = at_span_begin(P, blockIdx.x); g < g1;) {
    const AtSeg sg = at_segment(P, D, A, g, g1);
    const int n = sg.t1 - sg.t0;
    g += n;
    if (w >= sg.ntm) { gt += n; continue; }
    float m_ref = 0.f, l_run = 0.f;
    for (int jj = 0; jj < n; ++jj, ++cnt, ++gt) {
      const int j = sg.t0 + jj;
      const bool pseudo = j >= P.nt_near;
      const int nvalid = pseudo ? kAtCols : min(kAtCols, A.n_near - j * kAtCols);
      mbar_wait(B.s_full + w, cnt & 1);
      tc_fence_after_sync();
      float bm[16];
      auto load_bm = [&](float m) {
        if (pseudo) {
          const float4* bp = reinterpret_cast<const float4*>(bias_s + (gt & (kAtBiasRing - 1)) * kAtProto);
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const float4 v = bp[i];
            bm[4 * i] = v.x - m; bm[4 * i + 1] = v.y - m; bm[4 * i + 2] = v.z - m; bm[4 * i + 3] = v.w - m;
          }
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i) bm[i] = -m;
        }
      };
      if (jj == 0) {              // first tile of the piece: the reference maximum is this tile's row maximum
        load_bm(0.f);
        const float mx = nvalid < kAtCols ? at_row_max<true>(s_addr, sc2, bm, nvalid)
                                          : at_row_max<false>(s_addr, sc2, bm, nvalid);
        m_ref = mx == -INFINITY ? 0.f : mx;
      }
      load_bm(m_ref);
      uint32_t pk[64];
      float lsum;
      // At most one retry: after re-referencing to the true row maximum a tile's row sum is <= 128, so a second
      // failure can only come from non-finite logits (NaN / Inf in Q, K or a centre) -- those rows then produce NaN
      // like the SIMT path does, instead of spinning a persistent CTA forever.
      for (int attempt = 0;; ++attempt) {
        if (nvalid < kAtCols) at_row_pass<true>(s_addr, sc2, bm, nvalid, pk, lsum);
        else at_row_pass<false>(s_addr, sc2, bm, nvalid, pk, lsum);
        if (attempt == 1 || !__any_sync(0xffffffffu, !(lsum <= kRescaleSum))) break;
        // some row of this warp ran past its reference maximum (an element above 2^8 makes the sum exceed it): find
        // the row maxima, move the references up and rescale l and O (rare)
        const float mx = nvalid < kAtCols ? at_row_max<true>(s_addr, sc2, bm, nvalid)
                                          : at_row_max<false>(s_addr, sc2, bm, nvalid);
        float alpha = 1.f;
        if (mx > 0.f) {
          alpha = ex2_approx(-mx);
          m_ref += mx;
          l_run *= alpha;
#pragma unroll
          for (int i = 0; i < 16; ++i) bm[i] -= mx;
        }
        if (jj > 0) {
          mbar_wait(B.pv_done + w, (cnt - 1) & 1);
          tc_fence_after_sync();
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            uint32_t o[32];
            tmem_ld_32x32(o_addr + c * 32, o);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
            tmem_st_32x32(o_addr + c * 32, o);
          }
          tmem_st_wait();
        }
      }
      l_run += lsum;
#pragma unroll
      for (int c = 0; c < 4; ++c) tmem_st_32x16<64>(s_addr + c * 16, pk, c * 16);
      tmem_st_wait();
      tc_fence_before_sync();
      mbar_arrive(B.p_full + w);
    }
    // partial result of this piece: unnormalised O, reference maximum, row sum
    mbar_wait(B.pv_done + w, (cnt - 1) & 1);
    tc_fence_after_sync();
    const int r = w * 128 + row;
    float* dst = part + (((size_t)sg.item * P.nsplit + sg.piece) * kAtRows + r) * kPartStride;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      uint32_t o[32];
      tmem_ld_32x32(o_addr + c * 32, o);
      tmem_ld_wait();
      if (r < sg.R) {
#pragma unroll
        for (int i = 0; i < 32; i += 4)
          *reinterpret_cast<uint4*>(dst + c * 32 + i) = make_uint4(o[i], o[i + 1], o[i + 2], o[i + 3]);
      }
    }
    if (r < sg.R) *reinterpret_cast<float2*>(dst + 128) = make_float2(m_ref * kLn2, l_run);
    tc_fence_before_sync();
    mbar_arrive(B.o_empty + w);
  }
}

__global__ void __launch_bounds__(kAtThreads, 1)
attention_tc_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmRK,
                    const __grid_constant__ CUtensorMap tmRV, Dims D, Dev V, AtArgs A, AtPlan P, float* part) {
  extern __shared__ unsigned char smem_dyn[];
  unsigned char* sm = (unsigned char*)(((uintptr_t)smem_dyn + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + AtSmem::Bar);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + kAtNumBars);
  const AtBars B(bars);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    prefetch_tmap(&tmQ); prefetch_tmap(&tmRK); prefetch_tmap(&tmRV);
    mbar_init(B.q_full, 1); mbar_init(B.q_empty, 1);
    for (int i = 0; i < 2; ++i) {
      mbar_init(B.k_full + i, 1); mbar_init(B.k_empty + i, 1);
      mbar_init(B.v_full + i, 1); mbar_init(B.v_empty + i, 1);
      mbar_init(B.s_full + i, 1); mbar_init(B.p_full + i, 128);
      mbar_init(B.pv_done + i, 1); mbar_init(B.o_empty + i, 128);
    }
    mbar_init(B.stg_full, 1); mbar_init(B.stg_empty, 128);
    fence_barrier_init();
  }
  // rows of the Q staging area that no Q box ever writes must hold finite values
  for (uint32_t e = threadIdx.x; e < 4 * kAtHalf / 16; e += kAtThreads)
    reinterpret_cast<uint4*>(sm + AtSmem::Q)[e] = make_uint4(0u, 0u, 0u, 0u);
  fence_proxy_async_smem();
  if (warp == 12) tmem_alloc(tmem_slot, 512);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem_base = *tmem_slot;
  // barriers, TMEM and the zeroed Q rows are set up under the tail of the previous kernel of the stream (synthesis, or the
  // combine of the previous per-layer call).  No pdl_trigger(): a combine grid made pending under this persistent kernel
  // cost 7 % on the per-layer calls; launched at this kernel's exit it still skips the launch latency
  pdl_wait();

  if (warp < 8) {
    reg_inc<kRegsSoftmax>();
    at_softmax_role(sm, B, tmem_base, D, A, P, part, warp >> 2, warp & 3, lane);
  } else if (warp < 12) {
    reg_dec<kRegsBuilder>();
    at_builder_role(sm, B, D, V, A, P, (int)threadIdx.x - 256);
  } else {
    reg_dec<kRegsAux>();
    if (warp == 12) at_mma_role(sm, B, tmem_base, D, A, P);
    if (warp == 13 && lane == 0) at_loader_role(sm, B, &tmQ, &tmRK, &tmRV, D, V, A, P);
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 12) {
    __syncwarp();
    tc_fence_after_sync();
    tmem_dealloc(tmem_base, 512);
  }
}

// Merges the pieces of every item: one warp per output row, 4 dims per lane.
// WIDE = false: one warp per query row (superseded by attention_tc_combine4_kernel below, not launched).  WIDE = true: one CTA per row, the four
// warps take every fourth piece and merge through shared memory (few items cut into many pieces: a per-layer call, where
// a single warp walking 37 pieces with four loads in flight was a 17 us latency chain).
template <bool WIDE>
__global__ void __launch_bounds__(128) attention_tc_combine_kernel(Dims D, AtArgs A, AtPlan P, const float* part,
                                                                   __nv_bfloat16* out, float* lse, int rows_total) {
  const int wq = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int gr = WIDE ? (int)blockIdx.x : (int)blockIdx.x * 4 + wq;
  pdl_wait();
  pdl_trigger();   // the next call's kernel may set up while the rows are merged
  if (gr >= rows_total) return;
  const int Rb = A.n_q * D.group;
  const int bsel = gr / Rb, rr = gr % Rb;
  const int qi = rr / D.group, hh = rr % D.group;
  const int hd = bsel % D.Hkv, ll = (bsel / D.Hkv) % A.layer_count, st = bsel / (D.Hkv * A.layer_count);
  const int rb = qi / P.tb;
  const int rin = (qi - rb * P.tb) * D.group + hh;
  const int item = bsel * P.nrb + rb;
  int np = 0, cf = 0;
  if (P.ntile > 0) {
    cf = at_cta_of(P, (long long)item * P.ntile);
    np = at_cta_of(P, (long long)(item + 1) * P.ntile - 1) - cf + 1;
  }
  const float* base = part + ((size_t)item * P.nsplit * kAtRows + rin) * kPartStride;
  const size_t pstride = (size_t)kAtRows * kPartStride;
  // online merge, four pieces' loads in flight at a time (eight were slower on the per-layer calls: 786 vs 772 us)
  constexpr int U = 4;
  float M = -INFINITY, l = 0.f;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  bool poisoned = false;   // a piece with a NaN row sum (non-finite logits): the row is NaN, like the SIMT path returns it
  const int pstep = WIDE ? 4 : 1, pfirst = WIDE ? wq : 0;    // this warp's pieces: pfirst, pfirst + pstep, ...
  for (int sp0 = 0; pfirst + sp0 * pstep < np; sp0 += U) {
    float2 ml[U];
    float4 v[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int want = pfirst + (sp0 + u) * pstep;
      const int sp = want < np ? want : np - 1;              // clamp: a repeated piece is skipped below
      const float* ps = base + sp * pstride;
      ml[u] = *reinterpret_cast<const float2*>(ps + 128);
      v[u] = *reinterpret_cast<const float4*>(ps + lane * 4);
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const bool have = pfirst + (sp0 + u) * pstep < np;
      if (have && ml[u].y != ml[u].y) poisoned = true;
      if (!have || !(ml[u].y > 0.f)) continue;
      const float Mn = fmaxf(M, ml[u].x);
      const float so = __expf(M - Mn), sn = __expf(ml[u].x - Mn);   // M = -inf: so = 0
      l = fmaf(l, so, ml[u].y * sn);
      acc.x = fmaf(acc.x, so, v[u].x * sn); acc.y = fmaf(acc.y, so, v[u].y * sn);
      acc.z = fmaf(acc.z, so, v[u].z * sn); acc.w = fmaf(acc.w, so, v[u].w * sn);
      M = Mn;
    }
  }
  if (WIDE) {                                                 // merge the four warps' running (M, l, acc)
    __shared__ float4 sacc[4][32];
    __shared__ float sml[4][2];
    __shared__ int spois[4];
    sacc[wq][lane] = acc;
    if (lane == 0) { sml[wq][0] = M; sml[wq][1] = l; spois[wq] = poisoned ? 1 : 0; }
    __syncthreads();
    if (wq != 0) return;
    M = fmaxf(fmaxf(sml[0][0], sml[1][0]), fmaxf(sml[2][0], sml[3][0]));
    l = 0.f; acc = make_float4(0.f, 0.f, 0.f, 0.f); poisoned = false;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      poisoned = poisoned || spois[w] != 0;
      if (!(sml[w][1] > 0.f)) continue;
      const float sn = __expf(sml[w][0] - M);
      const float4 x = sacc[w][lane];
      l = fmaf(sml[w][1], sn, l);
      acc.x = fmaf(x.x, sn, acc.x); acc.y = fmaf(x.y, sn, acc.y); acc.z = fmaf(x.z, sn, acc.z); acc.w = fmaf(x.w, sn, acc.w);
    }
  }
  float inv = l > 0.f ? 1.f / l : 0.f;
  if (poisoned) { inv = __int_as_float(0x7fc00000); acc = make_float4(1.f, 1.f, 1.f, 1.f); l = inv; }
  const size_t ooff = (((size_t)st * A.layer_count + ll) * A.n_q + qi) * D.Hq + hd * D.group + hh;
  uint2 o;
  o.x = pack_bf16(acc.x * inv, acc.y * inv);
  o.y = pack_bf16(acc.z * inv, acc.w * inv);
  *reinterpret_cast<uint2*>(out + ooff * 128 + lane * 4) = o;
  if (lse && lane == 0) lse[ooff] = poisoned ? inv : (l > 0.f ? M + logf(l) : -INFINITY);
}

// The merge for items with few pieces (the batched query: <= 8 pieces per item, usually 1-3).  One warp merges FOUR
// consecutive rows of one item: the item-level index arithmetic (seven unsigned divisions: the one-row-per-warp form spent
// two thirds of its ~470 instructions per row on eleven signed ones) is done once per warp, and the loads of the four rows
// of a piece are in flight together.  Same arithmetic per row as attention_tc_combine_kernel.
__global__ void __launch_bounds__(128) attention_tc_combine4_kernel(Dims D, AtArgs A, AtPlan P, const float* part,
                                                                    __nv_bfloat16* out, float* lse, uint32_t nq4,
                                                                    uint32_t nwarps) {
  const uint32_t wq = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t gw = blockIdx.x * 4 + wq;
  pdl_wait();
  pdl_trigger();   // the next call's kernel may set up while the rows are merged
  if (gw >= nwarps) return;
  const uint32_t item = gw / nq4, quad = gw - item * nq4;
  const uint32_t bsel = item / (uint32_t)P.nrb, rb = item - bsel * (uint32_t)P.nrb;
  const uint32_t t1 = bsel / (uint32_t)D.Hkv, hd = bsel - t1 * (uint32_t)D.Hkv;          // t1 = st * layer_count + ll
  const uint32_t ntok = min((uint32_t)P.tb, (uint32_t)A.n_q - rb * (uint32_t)P.tb);
  const uint32_t R = ntok * (uint32_t)D.group;                                             // valid rows of the item
  const uint32_t rin0 = quad * 4;
  if (rin0 >= R) return;
  uint32_t np = 0;
  if (P.ntile > 0) {
    const int cf = at_cta_of(P, (long long)item * P.ntile);
    np = (uint32_t)(at_cta_of(P, (long long)(item + 1) * P.ntile - 1) - cf + 1);
  }
  const float* base = part + ((size_t)item * P.nsplit * kAtRows + rin0) * kPartStride;
  const size_t pstride = (size_t)kAtRows * kPartStride;
  float M[4], l[4];
  float4 acc[4];
  bool poisoned[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) { M[i] = -INFINITY; l[i] = 0.f; acc[i] = make_float4(0.f, 0.f, 0.f, 0.f); poisoned[i] = false; }
  for (uint32_t sp = 0; sp < np; ++sp) {
    const float* ps = base + sp * pstride;
    float2 ml[4];
    float4 v[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const uint32_t ri = rin0 + i < R ? i : 0;                  // clamp: rows past the item's end repeat row 0, never stored
      ml[i] = *reinterpret_cast<const float2*>(ps + ri * kPartStride + 128);
      v[i] = *reinterpret_cast<const float4*>(ps + ri * kPartStride + lane * 4);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      if (ml[i].y != ml[i].y) poisoned[i] = true;
      if (!(ml[i].y > 0.f)) continue;
      const float Mn = fmaxf(M[i], ml[i].x);
      const float so = __expf(M[i] - Mn), sn = __expf(ml[i].x - Mn);   // M = -inf: so = 0
      l[i] = fmaf(l[i], so, ml[i].y * sn);
      acc[i].x = fmaf(acc[i].x, so, v[i].x * sn); acc[i].y = fmaf(acc[i].y, so, v[i].y * sn);
      acc[i].z = fmaf(acc[i].z, so, v[i].z * sn); acc[i].w = fmaf(acc[i].w, so, v[i].w * sn);
      M[i] = Mn;
    }
  }
  uint32_t ql = rin0 / (uint32_t)D.group, hh = rin0 - ql * (uint32_t)D.group;             // token within the block, head
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (rin0 + i < R) {
      float inv = l[i] > 0.f ? 1.f / l[i] : 0.f;
      float4 a = acc[i];
      float li = l[i];
      if (poisoned[i]) { inv = __int_as_float(0x7fc00000); a = make_float4(1.f, 1.f, 1.f, 1.f); li = inv; }
      const size_t ooff = ((size_t)t1 * A.n_q + rb * (uint32_t)P.tb + ql) * D.Hq + hd * (uint32_t)D.group + hh;
      uint2 o;
      o.x = pack_bf16(a.x * inv, a.y * inv);
      o.y = pack_bf16(a.z * inv, a.w * inv);
      *reinterpret_cast<uint2*>(out + ooff * 128 + lane * 4) = o;
      if (lse && lane == 0) lse[ooff] = poisoned[i] ? inv : (li > 0.f ? M[i] + logf(li) : -INFINITY);
    }
    if (++hh == (uint32_t)D.group) { hh = 0; ++ql; }
  }
}

// ---------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------
bool tc_attention_supported(const Dims& D) {
  return D.bf16 && D.d == 128 && D.S == 8 && D.G == 8 && D.C == 16 && D.group <= kAtRows && D.K % kAtProto == 0;
}

static int at_rows_tb(const Dims& D, int n_q) {
  const int tb = kAtRows / D.group;
  return n_q < tb ? n_q : tb;
}

size_t tc_attention_part_bytes(const Dims& D) {
  // a call with I items on G <= 148 CTAs writes at most G + 2 I pieces (every item has <= ceil(G / I) + 1 of them)
  const int tb = at_rows_tb(D, D.Nq);
  const size_t items = (size_t)D.NS * D.L * D.Hkv * ((D.Nq + tb - 1) / tb);
  return (148 + 2 * items) * kAtRows * kPartStride * sizeof(float);
}

bool tc_attention_prepare() {
  const cudaError_t e = cudaFuncSetAttribute(attention_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)AtSmem::Total + 1024);
  if (e != cudaSuccess) { cudaGetLastError(); return false; }
  return true;
}

int launch_attention_tc(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, const TcMaps& maps,
                        int sm_count, cudaStream_t s) {
  AtArgs a{};
  a.Q = A.Q; a.n_q = A.n_q; a.layer_begin = A.layer_begin; a.layer_count = A.layer_count;
  a.n_near = (H.flags & PROTOKV_FAR_ONLY) ? 0 : A.n_near;
  a.n_act = (H.flags & PROTOKV_NEAR_ONLY) ? 0 : A.n_act;
  a.use_bias = !(H.flags & PROTOKV_NO_MASS_BIAS);
  const bool pdl = !(H.flags & PROTOKV_SERIAL_LAUNCH);
  AtPlan P{};
  P.tb = at_rows_tb(D, A.n_q);
  P.nrb = (A.n_q + P.tb - 1) / P.tb;
  P.items = D.NS * A.layer_count * D.Hkv * P.nrb;
  P.nt_near = (a.n_near + kAtCols - 1) / kAtCols;
  P.nt_ps = (a.n_act + kAtProto - 1) / kAtProto;
  P.ntile = P.nt_near + P.nt_ps;
  P.ttot = (long long)P.items * P.ntile;
  int grid = sm_count < 148 ? sm_count : 148;
  if ((long long)grid > P.ttot) grid = (int)P.ttot;
  P.grid = grid > 0 ? grid : 1;
  P.nsplit = 1;
  int launched = 0;
  if (P.ttot > 0) {
    for (int i = 0; i < P.items; ++i) {
      const int np = at_cta_of(P, (long long)(i + 1) * P.ntile - 1) - at_cta_of(P, (long long)i * P.ntile) + 1;
      if (np > P.nsplit) P.nsplit = np;
    }
    CUtensorMap tmQ;
    const uint64_t ntok = (uint64_t)D.NS * A.layer_count * A.n_q;
    if (!make_tmap_3d_bf16(&tmQ, A.Q, 128, (uint64_t)D.Hq, ntok, 64, (uint32_t)D.group, (uint32_t)P.tb)) return -1;
    launch_chain(attention_tc_kernel, P.grid, kAtThreads, AtSmem::Total + 1024, s, pdl, tmQ, maps.ringK, maps.ringV, D, V, a, P, V.part);
    ++launched;
  }
  const int rows_total = D.NS * A.layer_count * D.Hkv * A.n_q * D.group;
  if (P.nsplit > 8) {
    launch_chain(attention_tc_combine_kernel<true>, rows_total, 128, 0, s, pdl, D, a, P, (const float*)V.part, (__nv_bfloat16*)A.out, A.lse, rows_total);
  } else {
    const uint32_t nq4 = (uint32_t)(P.tb * D.group + 3) / 4, nwarps = (uint32_t)P.items * nq4;
    launch_chain(attention_tc_combine4_kernel, (nwarps + 3) / 4, 128, 0, s, pdl, D, a, P, (const float*)V.part, (__nv_bfloat16*)A.out, A.lse, nq4, nwarps);
  }
  return launched + 1;
}

}  // namespace pkv
