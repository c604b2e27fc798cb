// U3 assignment on the 5th-gen tensor cores (bf16 inputs, d = 128): the tokens x prototypes x head_dim contraction of
// Eq. 1 as tcgen05.mma tiles fed by TMA, with the rest of Eq. 1 (cosine normalisation, Mahalanobis
// spatial term, idle penalty) and the argmin fused into the epilogue that drains TMEM.  See DESIGN.md "Kernels".
//
// Exactness: the evicted keys are bf16 already; the fp32 centres are split c = c_hi + c_lo (two bf16 terms, kept as
// shadows by the update kernel), and both products accumulate into the same fp32 TMEM tile, so the dot product
// carries ~2^-17 relative error of |c| instead of bf16's 2^-9 -- below north_star's 1e-5 gap rule.
//
// CTA = (token tile of 128, bank); 6 warps: warp 0 = TMA producer, warp 1 = TMEM allocator + MMA issuer,
// warps 2-5 = epilogue (one TMEM lane quarter each; thread <-> token row).  Prototypes stream through shared
// memory in chunks of 128 (hi and lo, 64 KB per stage, 2 stages); accumulators are double-buffered in TMEM
// (2 x 128 columns) so the MMAs of chunk i+1 overlap the epilogue of chunk i.
#include "common.cuh"
#include "tc_common.cuh"

namespace pkv {

using namespace tc;

constexpr int kTcM = 128;        // tokens per CTA tile (UMMA M)
constexpr int kTcN = 128;        // prototypes per chunk (UMMA N)
constexpr int kTcStages = 2;
constexpr int kTcThreads = 192;
constexpr uint32_t kHalfTile = 128 * 64 * 2;           // one [128 rows][64 bf16] swizzled box = 16 KB
constexpr uint32_t kStageBytes = 4 * kHalfTile;        // c_hi (2 K-halves) + c_lo (2 K-halves)

struct __align__(16) EpiRec {   // transformed ScoreRec, 32 bytes: two LDS.128 per prototype column
  float ninvc, mux, muy, u;
  float v, w, idle, pad;
};

struct TcAssignSmem {
  // offsets from a 1024-byte aligned base
  static constexpr uint32_t A = 0;                                   // 2 x 16 KB token tile (K-halves)
  static constexpr uint32_t Bst = A + 2 * kHalfTile;                 // stages x 64 KB
  static constexpr uint32_t Rec = Bst + kTcStages * kStageBytes;     // 2 x 128 x 32 B
  static constexpr uint32_t Bar = Rec + 2 * kTcN * sizeof(EpiRec);   // barriers
  static constexpr uint32_t Total = Bar + 128;
};

__global__ void __launch_bounds__(kTcThreads, 1)
score_tc_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmChi,
                const __grid_constant__ CUtensorMap tmClo, Dims D, Hyper H, Dev V, FrameArgs F) {
  extern __shared__ unsigned char smem_dyn[];
  unsigned char* sm = (unsigned char*)(((uintptr_t)smem_dyn + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = (uint64_t*)(sm + TcAssignSmem::Bar);
  uint64_t* a_full = bars + 0;
  uint64_t* full = bars + 1;                  // [stages]
  uint64_t* empty = full + kTcStages;         // [stages]
  uint64_t* tfull = empty + kTcStages;        // [2]
  uint64_t* tempty = tfull + 2;               // [2]
  uint32_t* tmem_slot = (uint32_t*)(tempty + 2);
  EpiRec* recs = (EpiRec*)(sm + TcAssignSmem::Rec);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int b = blockIdx.y;
  const int j0 = F.n_fill + blockIdx.x * kTcM;          // first token of this tile
  const int nchunks = (F.n_act + kTcN - 1) / kTcN;

  if (threadIdx.x == 0) {
    prefetch_tmap(&tmK); prefetch_tmap(&tmChi); prefetch_tmap(&tmClo);
    mbar_init(a_full, 1);
    for (int s = 0; s < kTcStages; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(tfull + i, 1); mbar_init(tempty + i, 128); }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, 256);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer =====
    if (lane == 0) {
      const int row0 = (b * D.Wf + F.slot) * D.T + j0;
      mbar_arrive_expect_tx(a_full, 2 * kHalfTile);
      tma_load_2d(sm + TcAssignSmem::A, &tmK, 0, row0, a_full);
      tma_load_2d(sm + TcAssignSmem::A + kHalfTile, &tmK, 64, row0, a_full);
      for (int c = 0; c < nchunks; ++c) {
        const int s = c % kTcStages, ph = (c / kTcStages) & 1;
        mbar_wait(empty + s, ph ^ 1);
        unsigned char* dst = sm + TcAssignSmem::Bst + s * kStageBytes;
        const int prow = b * D.K + c * kTcN;
        mbar_arrive_expect_tx(full + s, kStageBytes);
        tma_load_2d(dst, &tmChi, 0, prow, full + s);
        tma_load_2d(dst + kHalfTile, &tmChi, 64, prow, full + s);
        tma_load_2d(dst + 2 * kHalfTile, &tmClo, 0, prow, full + s);
        tma_load_2d(dst + 3 * kHalfTile, &tmClo, 64, prow, full + s);
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer =====
    if (lane == 0) {
      constexpr uint32_t idesc = idesc_bf16(kTcM, kTcN, 0, 0);
      const uint32_t a_addr = smem_u32(sm + TcAssignSmem::A);
      mbar_wait(a_full, 0);
      for (int c = 0; c < nchunks; ++c) {
        const int s = c % kTcStages, ph = (c / kTcStages) & 1;
        const int buf = c & 1, bph = (c >> 1) & 1;
        mbar_wait(tempty + buf, bph ^ 1);
        mbar_wait(full + s, ph);
        tc_fence_after_sync();
        const uint32_t b_addr = smem_u32(sm + TcAssignSmem::Bst + s * kStageBytes);
        const uint32_t d_tmem = tmem_base + buf * kTcN;
        bool acc = false;
#pragma unroll
        for (int part = 0; part < 2; ++part) {        // c_hi, c_lo
#pragma unroll
          for (int half = 0; half < 2; ++half) {      // d 0..63, 64..127
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {          // 4 x K=16 inside the 128-byte swizzle atom
              const uint64_t ad = desc_kmajor_sw128(a_addr + half * kHalfTile + kk * 32);
              const uint64_t bd = desc_kmajor_sw128(b_addr + (part * 2 + half) * kHalfTile + kk * 32);
              umma_bf16(d_tmem, ad, bd, idesc, acc);
              acc = true;
            }
          }
        }
        umma_commit(empty + s);       // smem stage reusable once these MMAs have read it
        umma_commit(tfull + buf);     // accumulator complete
      }
    }
  } else {
    // ===== epilogue: warps 2..5, TMEM lane quarter = warp % 4 =====
    const int q = warp & 3;
    const int row = q * 32 + lane;                 // token row in the tile = TMEM lane
    const int et = (warp - 2) * 32 + lane;         // 0..127 index among the epilogue threads (rec staging)
    const int j = j0 + row;
    const int st = b / (D.L * D.Hkv);
    float sx = 0.f, sy = 0.f;
    if (j < D.T) {
      const float* se = V.ringS + (((size_t)st * D.Wf + F.slot) * D.T + j) * 2;
      sx = se[0]; sy = se[1];
    }
    auto load_rec = [&](int c) -> EpiRec {
      EpiRec e{0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      const int k = c * kTcN + et;
      if (c < nchunks && k < F.n_act) {
        const ScoreRec r = V.rec[(size_t)b * D.K + k];
        e.ninvc = -r.invc; e.mux = r.mux; e.muy = r.muy; e.u = r.u; e.v = r.v; e.w = r.w;
        e.idle = (F.t - r.tau > H.t_idle) ? H.lambda_idle : 0.f;
      }
      return e;
    };
    EpiRec next = load_rec(0);
    // |K_j|^2 from the swizzled A tile: row r, 16-byte chunk c lives at r*128 + ((c ^ (r & 7)) << 4) in each K-half
    mbar_wait(a_full, 0);
    float kk2 = 0.f;
#pragma unroll
    for (int half = 0; half < 2; ++half) {
      const unsigned char* base = sm + TcAssignSmem::A + half * kHalfTile + row * 128;
#pragma unroll
      for (int ch = 0; ch < 8; ++ch) {
        const uint4 w = *(const uint4*)(base + ((ch ^ (row & 7)) << 4));
        const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float lo = __uint_as_float(ww[e] << 16), hi = __uint_as_float(ww[e] & 0xffff0000u);
          kk2 = fmaf(lo, lo, kk2); kk2 = fmaf(hi, hi, kk2);
        }
      }
    }
    const float invk = kk2 > 0.f ? rsqrtf(kk2) : 0.f;
    const float ninv_cap = -1.f / H.cos_eps;       // cos = dot / max(|K||c|, cos_eps)  (reading 6)
    const bool squared = H.flags & PROTOKV_MAH_SQUARED;
    float best = INFINITY;
    int bidx = 0x7fffffff;
    for (int c = 0; c < nchunks; ++c) {
      const int buf = c & 1, bph = (c >> 1) & 1;
      recs[buf * kTcN + et] = next;
      next = load_rec(c + 1);
      asm volatile("bar.sync 1, 128;" ::: "memory");
      mbar_wait(tfull + buf, bph);
      tc_fence_after_sync();
      const int nk = min(kTcN, F.n_act - c * kTcN);
      const EpiRec* rc = recs + buf * kTcN;
      for (int col0 = 0; col0 < nk; col0 += 32) {
        uint32_t acc[32];
        tmem_ld_32x32(tmem_base + ((uint32_t)(q * 32) << 16) + buf * kTcN + col0, acc);
        tmem_ld_wait();
        const int lim = min(32, nk - col0);
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          if (i < lim) {
            const float4 r0 = *(const float4*)&rc[col0 + i].ninvc;
            const float4 r1 = *(const float4*)&rc[col0 + i].v;
            const float dx = sx - r0.y, dy = sy - r0.z;
            const float y1 = dx * r0.w, y2 = fmaf(dy, r1.x, -(dx * r1.y));
            const float qq = fmaf(y1, y1, y2 * y2);
            const float sp = squared ? qq : sqrtf(qq);
            const float ninv = fmaxf(r0.x * invk, ninv_cap);
            const float sc = fmaf(__uint_as_float(acc[i]), ninv, sp + r1.z);
            if (sc < best) { best = sc; bidx = c * kTcN + col0 + i; }   // increasing k: lowest index on ties
          }
        }
      }
      tc_fence_before_sync();
      mbar_arrive(tempty + buf);
    }
    if (j < D.T) {
      V.assign[(size_t)b * D.T + j] = bidx;
      V.best[(size_t)b * D.T + j] = best;
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after_sync();
    tmem_dealloc(tmem_base, 256);
  }
}

// ---------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
    else
      cudaGetLastError();
  }
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

bool tc_assign_supported(const Dims& D, const Hyper&) { return D.bf16 && D.d == 128; }

bool tc_build_maps(const Dims& D, const Dev& V, TcMaps* maps) {
  const uint64_t ring_rows = (uint64_t)D.B * D.Wf * D.T, bank_rows = (uint64_t)D.B * D.K;
  maps->ok = make_tmap_2d_bf16(&maps->ringK, V.ringK, ring_rows, 128, 128, 64) &&
             make_tmap_2d_bf16(&maps->ringV, V.ringV, ring_rows, 128, 128, 64) &&
             make_tmap_2d_bf16(&maps->c_hi, V.c_hi, bank_rows, 128, 128, 64) &&
             make_tmap_2d_bf16(&maps->c_lo, V.c_lo, bank_rows, 128, 128, 64);
  if (maps->ok) {
    const cudaError_t e = cudaFuncSetAttribute(score_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                               (int)TcAssignSmem::Total + 1024);
    if (e != cudaSuccess) { cudaGetLastError(); maps->ok = false; }
  }
  return maps->ok;
}

int launch_score_tc(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, const TcMaps& maps,
                    cudaStream_t s) {
  const int ntok = D.T - F.n_fill;
  if (ntok <= 0) return 0;
  dim3 grid((ntok + kTcM - 1) / kTcM, D.B);
  score_tc_kernel<<<grid, kTcThreads, TcAssignSmem::Total + 1024, s>>>(maps.ringK, maps.c_hi, maps.c_lo, D, H, V, F);
  return 1;
}

}  // namespace pkv
