// U3 assignment on the 5th-gen tensor cores (bf16 inputs, d = 128): the tokens x prototypes x head_dim contraction of
// Eq. 1 as tcgen05.mma tiles fed by TMA, with the rest of Eq. 1 (Mahalanobis spatial term, idle
// penalty) and the argmin fused into the epilogue that drains TMEM.  See DESIGN.md "Kernels".
//
// Exactness: the evicted keys are bf16 already; the fp32 centres are normalised and split c/|c| = hi + lo (two bf16
// terms, kept as shadows by the update kernel); both products accumulate into the same fp32 TMEM tile, so the
// accumulator is |K_j| cos(K_j, c_k) with ~2^-17 relative error instead of bf16's 2^-9 -- below north_star's 1e-5 gap
// rule.  The epilogue minimises |K_j| * score = |K_j| (lambda_sp d_Mah + lambda_idle [idle]) - acc, which has the same
// argmin as Eq. 1 (|K_j| > 0 is constant along a row) and needs no per-column normalisation.
//
// Persistent kernel, one CTA per SM.  Work unit = (bank, pair of 128-token M tiles, chunk of 64 prototypes); the unit
// list is cut into gridDim.x contiguous spans, so consecutive units of a CTA share the token tiles (A operand, loaded
// once per (bank, pair)).  18 warps: warp 0 = TMA producer, warp 1 = TMEM owner + MMA issuer, warps 2-17 = epilogue in
// two groups of 8 (group = unit parity; warp = (M tile, TMEM lane quarter); thread <-> token row).  Prototype chunks
// (hi and lo, 32 KB) and their Eq. 1 records (2 KB) stream through 4-stage rings; accumulators rotate through
// 4 x 128 TMEM columns, so the MMAs run up to 4 units ahead of the epilogue.  Each thread keeps the running argmin of
// its row over the units it sees and merges it into akey[bank][token] with a 64-bit atomicMin on
// (orderable(score) << 32 | k): lowest score first, lowest index on ties, whatever CTA / group saw the chunk.
#include "common.cuh"
#include "tc_common.cuh"

namespace pkv {

using namespace tc;

constexpr int kUN = 64;                                  // prototypes per unit (UMMA N)
constexpr int kRing = 4;                                 // B stages = TMEM buffers
constexpr int kRecRing = 8;                              // record slots (deeper: a slot is held until the epilogue is done)
constexpr int kAsThreads = 18 * 32;
constexpr uint32_t kAHalf = 128 * 128;                   // [128 rows][64 bf16] swizzled box = 16 KB
constexpr uint32_t kBHalf = kUN * 128;                   // [64 rows][64 bf16] = 8 KB
constexpr uint32_t kBStage = 4 * kBHalf;                 // hi (2 K-halves) + lo (2 K-halves) = 32 KB
constexpr uint32_t kRecBytes = kUN * sizeof(ScoreRec);   // 2 KB

struct AsSmem {   // byte offsets from a 1024-byte aligned base
  static constexpr uint32_t A = 0;                                  // 2 tiles x 2 K-halves x 16 KB
  static constexpr uint32_t Bst = A + 4 * kAHalf;                   // kRing x 32 KB
  static constexpr uint32_t Rec = Bst + kRing * kBStage;            // kRecRing x 2 KB
  static constexpr uint32_t Bar = Rec + kRecRing * kRecBytes;
  static constexpr uint32_t Total = Bar + 256;
};

struct AsPlan {
  int NP;        // token-tile pairs per bank
  int NC;        // prototype chunks per bank
  int units;     // B * NP * NC
  int ntok;      // scored tokens per bank (T - n_fill)
};

struct AsUnit { int b, mp, nc, akey, ntiles; };

__device__ __forceinline__ AsUnit as_unit(const AsPlan& P, int u) {
  AsUnit x;
  x.nc = u % P.NC;
  x.akey = u / P.NC;
  x.mp = x.akey % P.NP;
  x.b = x.akey / P.NP;
  x.ntiles = (P.ntok - x.mp * 256) > 128 ? 2 : 1;
  return x;
}

__device__ __forceinline__ uint32_t orderable(float f) {
  const uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// packed fp32 pairs (sm_100 f32x2 arithmetic): one issue slot for the two prototypes of a record pair
__device__ __forceinline__ uint64_t as_pack2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void as_unpack2(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t as_fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ uint64_t as_mul2(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}

// One row's scan over the (up to) 64 accumulator columns of a unit: rest of Eq. 1 + running argmin, two prototypes
// per step.  The records arrive pair-interleaved (common.cuh rec_slot): {mux0, mux1, muy0, muy1}, {u0, u1, -w0, -w1},
// {v0, v1, tauf0, tauf1}.  The scan maximises  acc - |K_j| (lambda_sp d_Mah + lambda_idle [idle])  = -|K_j| score.
template <bool SQUARED, bool RAGGED>
__device__ __forceinline__ void as_scan(uint32_t taddr, uint32_t rc, int ncol, float sx, float sy, float nk,
                                        float thr, float lam_idle, float& ub, int& ucol) {
  const uint64_t sx2 = as_pack2(sx, sx), sy2 = as_pack2(sy, sy), m1 = as_pack2(-1.f, -1.f);
  const uint64_t nnk2 = as_pack2(-nk, -nk), li2 = as_pack2(lam_idle, lam_idle);
  float best = -ub;                                      // running maximum of -|K_j| score
#pragma unroll
  for (int c0 = 0; c0 < kUN; c0 += 32) {
    if (!RAGGED || c0 < ncol) {
      uint32_t acc[32];
      tmem_ld_32x32(taddr + c0, acc);
      tmem_ld_wait();
#pragma unroll
      for (int c = 0; c < 32; c += 2) {
        uint64_t mu_x, mu_y, u2, wn2, v2, tf2;
        const uint32_t ra = rc + ((c0 + c) >> 1) * 64;
        asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(mu_x), "=l"(mu_y) : "r"(ra) : "memory");
        asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(u2), "=l"(wn2) : "r"(ra + 16) : "memory");
        asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(v2), "=l"(tf2) : "r"(ra + 32) : "memory");
        const uint64_t dx = as_fma2(mu_x, m1, sx2), dy = as_fma2(mu_y, m1, sy2);     // s - mu
        const uint64_t y1 = as_mul2(dx, u2);
        const uint64_t y2 = as_fma2(dx, wn2, as_mul2(dy, v2));                       // dy v - dx w
        const uint64_t qq = as_fma2(y1, y1, as_mul2(y2, y2));
        float q0, q1, t0, t1;
        as_unpack2(qq, q0, q1);
        as_unpack2(tf2, t0, t1);
        float s0, s1;
        if (SQUARED) { s0 = q0; s1 = q1; }
        else {
          asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s0) : "f"(q0));
          asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s1) : "f"(q1));
        }
        const uint64_t ee = as_fma2(li2, as_pack2(__saturatef(thr - t0), __saturatef(thr - t1)), as_pack2(s0, s1));
        const uint64_t sc2 = as_fma2(nnk2, ee, as_pack2(__uint_as_float(acc[c]), __uint_as_float(acc[c + 1])));
        float n0, n1;
        as_unpack2(sc2, n0, n1);
        if (RAGGED) {
          if (c0 + c >= ncol) n0 = -INFINITY;
          if (c0 + c + 1 >= ncol) n1 = -INFINITY;
        }
        if (n0 > best) { best = n0; ucol = c0 + c; }     // increasing k: lowest index on ties
        if (n1 > best) { best = n1; ucol = c0 + c + 1; }
      }
    }
  }
  ub = -best;
}

template <bool SQUARED>
__global__ void __launch_bounds__(kAsThreads, 1)
score_tc_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmChi,
                const __grid_constant__ CUtensorMap tmClo, Dims D, Hyper H, Dev V, FrameArgs F, AsPlan P) {
  extern __shared__ unsigned char smem_dyn[];
  unsigned char* sm = (unsigned char*)(((uintptr_t)smem_dyn + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = (uint64_t*)(sm + AsSmem::Bar);
  uint64_t* a_full = bars + 0;
  uint64_t* a_empty = bars + 1;
  uint64_t* b_full = bars + 2;                 // [kRing]
  uint64_t* b_empty = b_full + kRing;
  uint64_t* t_full = b_empty + kRing;
  uint64_t* t_empty = t_full + kRing;
  uint64_t* r_full = t_empty + kRing;          // [kRecRing]
  uint64_t* r_empty = r_full + kRecRing;
  uint32_t* tmem_slot = (uint32_t*)(r_empty + kRecRing);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int u0 = (int)(((long long)blockIdx.x * P.units) / gridDim.x);
  const int u1 = (int)(((long long)(blockIdx.x + 1) * P.units) / gridDim.x);

  if (threadIdx.x == 0) {
    prefetch_tmap(&tmK); prefetch_tmap(&tmChi); prefetch_tmap(&tmClo);
    mbar_init(a_full, 1); mbar_init(a_empty, 1);
    for (int s = 0; s < kRing; ++s) {
      mbar_init(b_full + s, 1); mbar_init(b_empty + s, 1);
      mbar_init(t_full + s, 1); mbar_init(t_empty + s, 8);
    }
    for (int s = 0; s < kRecRing; ++s) { mbar_init(r_full + s, 1); mbar_init(r_empty + s, 8); }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, 512);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem_base = *tmem_slot;
  pdl_wait();        // barriers, TMEM and descriptors are set up under the tail of the previous frame's ring append
  pdl_trigger();     // the update kernel may load its codebooks as soon as an SM frees

  if (warp == 0) {
    // ===== TMA producer =====
    if (lane == 0) {
      int prev = -1, acnt = 0;
      for (int u = u0; u < u1; ++u) {
        const AsUnit x = as_unit(P, u);
        const int i = u - u0, s = i % kRing;
        const uint32_t par = ((i / kRing) & 1) ^ 1;
        if (x.akey != prev) {
          mbar_wait(a_empty, (acnt & 1) ^ 1);
          const int row0 = (x.b * D.Wf + F.slot) * D.T + F.n_fill + x.mp * 256;
          mbar_arrive_expect_tx(a_full, (uint32_t)x.ntiles * 2 * kAHalf);
          for (int t = 0; t < x.ntiles; ++t) {
            tma_load_2d(sm + AsSmem::A + (t * 2) * kAHalf, &tmK, 0, row0 + t * 128, a_full);
            tma_load_2d(sm + AsSmem::A + (t * 2 + 1) * kAHalf, &tmK, 64, row0 + t * 128, a_full);
          }
          prev = x.akey; ++acnt;
        }
        const int prow = x.b * D.K + x.nc * kUN;
        unsigned char* dst = sm + AsSmem::Bst + s * kBStage;
        mbar_wait(b_empty + s, par);
        mbar_arrive_expect_tx(b_full + s, kBStage);
        tma_load_2d(dst, &tmChi, 0, prow, b_full + s);
        tma_load_2d(dst + kBHalf, &tmChi, 64, prow, b_full + s);
        tma_load_2d(dst + 2 * kBHalf, &tmClo, 0, prow, b_full + s);
        tma_load_2d(dst + 3 * kBHalf, &tmClo, 64, prow, b_full + s);
        const int rs = i % kRecRing;
        mbar_wait(r_empty + rs, ((i / kRecRing) & 1) ^ 1);   // the epilogue of unit i - kRecRing has read this slot
        const int nrec = (min(kUN, D.K - x.nc * kUN) + 1) & ~1;   // whole record pairs (prow is even: K % 64 == 0 here)
        mbar_arrive_expect_tx(r_full + rs, (uint32_t)nrec * sizeof(ScoreRec));
        bulk_load_1d(sm + AsSmem::Rec + rs * kRecBytes, V.rec + (size_t)prow, (uint32_t)nrec * sizeof(ScoreRec), r_full + rs);
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: the whole warp walks the unit list (uniform control flow), one elected lane issues =====
    constexpr uint32_t idesc = idesc_bf16(128, kUN, 0, 0);
    const uint64_t a_desc0 = desc_kmajor_sw128(smem_u32(sm + AsSmem::A));
    const uint64_t b_desc0 = desc_kmajor_sw128(smem_u32(sm + AsSmem::Bst));
    int nc = u0 % P.NC, akey = u0 / P.NC, acnt = 0;
    bool fresh = true;                               // first unit on this (bank, pair): wait for its token tiles
    for (int u = u0; u < u1; ++u) {
      const int i = u - u0, s = i % kRing;
      const uint32_t par = (i / kRing) & 1;
      const int ntiles = (P.ntok - (akey % P.NP) * 256) > 128 ? 2 : 1;
      if (fresh) { mbar_wait(a_full, acnt & 1); ++acnt; fresh = false; }
      mbar_wait(t_empty + s, par ^ 1);
      mbar_wait(b_full + s, par);
      tc_fence_after_sync();
      const bool last = (nc + 1 == P.NC) || (u + 1 == u1);
      if (elect_one_sync()) {
        const uint64_t bs = b_desc0 + (uint64_t)(s * (kBStage >> 4));
        for (int t = 0; t < ntiles; ++t) {
          const uint32_t d_tmem = tmem_base + s * 128 + t * kUN;
          const uint64_t at = a_desc0 + (uint64_t)(t * (2 * kAHalf >> 4));
#pragma unroll
          for (int part = 0; part < 2; ++part) {        // hi, lo
#pragma unroll
            for (int half = 0; half < 2; ++half) {      // d 0..63, 64..127
#pragma unroll
              for (int kk = 0; kk < 4; ++kk) {          // 4 x K=16 inside the 128-byte swizzle atom
                const uint64_t ad = at + (uint64_t)((half * kAHalf + kk * 32) >> 4);
                const uint64_t bd = bs + (uint64_t)(((part * 2 + half) * kBHalf + kk * 32) >> 4);
                umma_bf16(d_tmem, ad, bd, idesc, (part | half | kk) != 0);
              }
            }
          }
        }
        umma_commit(b_empty + s);       // smem stage reusable once these MMAs have read it
        umma_commit(t_full + s);        // accumulators complete
        if (last) umma_commit(a_empty); // last unit on these token tiles
      }
      __syncwarp();
      if (++nc == P.NC) { nc = 0; ++akey; fresh = true; }
    }
  } else {
    // ===== epilogue: 16 warps; group = unit parity, tile = M tile of the pair, q = TMEM lane quarter =====
    const int e = warp - 2;
    const int grp = e >> 3, tile = (e >> 2) & 1, q = warp & 3;
    const int row = tile * 128 + q * 32 + lane;             // token row within the pair
    const float thr = (float)(F.t - H.t_idle);               // idle <=> tau < t - T_idle  (Eq. 1, reading 2)
    const float lam_idle = H.lambda_idle;
    float sx = 0.f, sy = 0.f, nk = 1.f, best = INFINITY;
    int bidx = 0x7fffffff, j = -1, cur_b = 0, prev = -1;
    bool valid = false;
    auto flush = [&]() {
      if (valid && best < INFINITY)
        atomicMin(V.akey + (size_t)cur_b * D.T + j, ((unsigned long long)orderable(best) << 32) | (uint32_t)bidx);
    };
    for (int u = u0 + grp; u < u1; u += 2) {
      const AsUnit x = as_unit(P, u);
      const int i = u - u0, s = i % kRing;
      const uint32_t par = (i / kRing) & 1;
      if (x.akey != prev) {
        flush();
        prev = x.akey; cur_b = x.b;
        j = F.n_fill + x.mp * 256 + row;
        valid = j < D.T;
        best = INFINITY; bidx = 0x7fffffff;
        if (valid) {
          const int st = x.b / (D.L * D.Hkv);
          const float2 se = *reinterpret_cast<const float2*>(V.ringS + (((size_t)st * D.Wf + F.slot) * D.T + j) * 2);
          sx = se.x; sy = se.y;
          const float kk = V.ringN[((size_t)x.b * D.Wf + F.slot) * D.T + j];
          nk = kk > 0.f ? sqrtf(kk) : 1.f;                   // |K_j| = 0: acc = 0 and Eq. 1 reduces to its other terms
        }
      }
      const int rs = i % kRecRing;
      mbar_wait(r_full + rs, (i / kRecRing) & 1);
      mbar_wait(t_full + s, par);
      tc_fence_after_sync();
      if (__any_sync(0xffffffffu, valid)) {
        const int ncol = min(kUN, F.n_act - x.nc * kUN);
        const uint32_t rc = smem_u32(sm + AsSmem::Rec + rs * kRecBytes);
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + s * 128 + tile * kUN;
        float ub = INFINITY;
        int ucol = 0;
        if (ncol == kUN) as_scan<SQUARED, false>(taddr, rc, ncol, sx, sy, nk, thr, lam_idle, ub, ucol);
        else as_scan<SQUARED, true>(taddr, rc, ncol, sx, sy, nk, thr, lam_idle, ub, ucol);
        if (ub < best) { best = ub; bidx = x.nc * kUN + ucol; }
      }
      tc_fence_before_sync();
      __syncwarp();
      if (lane == 0) { mbar_arrive(t_empty + s); mbar_arrive(r_empty + rs); }
    }
    flush();
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after_sync();
    tmem_dealloc(tmem_base, 512);
  }
}

// ---------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn lookup_encode_fn() {
  void* p = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
      qres == cudaDriverEntryPointSuccess)
    return (EncodeTiledFn)p;
  cudaGetLastError();
  return nullptr;
}
static EncodeTiledFn encode_fn() {
  static const EncodeTiledFn fn = lookup_encode_fn();   // initialised once, thread-safe (states may be created concurrently)
  return fn;
}

bool make_tmap_2d_bf16(CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint32_t box_rows,
                       uint32_t box_cols) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {cols * 2};
  const cuuint32_t box[2] = {box_cols, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  CUtensorMap m;
  const CUresult r = fn(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  *out = m;
  return true;
}

bool make_tmap_3d_bf16(CUtensorMap* out, const void* base, uint64_t n0, uint64_t n1, uint64_t n2, uint32_t b0,
                       uint32_t b1, uint32_t b2) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[3] = {n0, n1, n2};
  const cuuint64_t strides[2] = {n0 * 2, n0 * n1 * 2};
  const cuuint32_t box[3] = {b0, b1, b2};
  const cuuint32_t estr[3] = {1, 1, 1};
  CUtensorMap m;
  const CUresult r = fn(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  *out = m;
  return true;
}

bool tc_assign_supported(const Dims& D, const Hyper&) { return D.bf16 && D.d == 128 && D.K % 2 == 0; }   // record pairs

bool tc_build_maps(const Dims& D, const Dev& V, TcMaps* maps) {
  const uint64_t ring_rows = (uint64_t)D.B * D.Wf * D.T, bank_rows = (uint64_t)D.B * D.K;
  maps->ok = make_tmap_2d_bf16(&maps->ringK, V.ringK, ring_rows, 128, 128, 64) &&
             make_tmap_2d_bf16(&maps->ringV, V.ringV, ring_rows, 128, 128, 64) &&
             make_tmap_2d_bf16(&maps->c_hi, V.c_hi, bank_rows, 128, kUN, 64) &&
             make_tmap_2d_bf16(&maps->c_lo, V.c_lo, bank_rows, 128, kUN, 64);
  if (maps->ok) {
    cudaError_t e = cudaFuncSetAttribute(score_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)AsSmem::Total + 1024);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(score_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AsSmem::Total + 1024);
    if (e != cudaSuccess) { cudaGetLastError(); maps->ok = false; }
  }
  return maps->ok;
}

int launch_score_tc(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, const TcMaps& maps,
                    int sm_count, cudaStream_t s) {
  AsPlan P{};
  P.ntok = D.T - F.n_fill;
  if (P.ntok <= 0 || F.n_act <= 0) return 0;
  P.NP = (P.ntok + 255) / 256;
  P.NC = (F.n_act + kUN - 1) / kUN;
  P.units = D.B * P.NP * P.NC;
  const int grid = P.units < sm_count ? P.units : sm_count;
  if (H.flags & PROTOKV_MAH_SQUARED)
    launch_chain(score_tc_kernel<true>, grid, kAsThreads, AsSmem::Total + 1024, s, F.pdl != 0, maps.ringK, maps.c_hi, maps.c_lo, D, H, V, F, P);
  else
    launch_chain(score_tc_kernel<false>, grid, kAsThreads, AsSmem::Total + 1024, s, F.pdl != 0, maps.ringK, maps.c_hi, maps.c_lo, D, H, V, F, P);
  return 1;
}

}  // namespace pkv
