// Internal definitions shared by the ProtoKV CUDA kernels and the C-ABI host code (not part of the ABI).
// Layout of the device state is documented in DESIGN.md "Data layout in HBM".
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/protokv.h"

namespace pkv {

constexpr int kMaxS = 8, kMaxG = 8, kMaxC = 16;
constexpr int kMaxT = 4096, kMaxKmax = 16384;   // limits protokv_create admits (sort keys hold 12 bits of token index)
#define PKV_SYN_LOGTAB 4096
constexpr int kCbPad = 16;
// Device-side error bits (Dev::err).  UNASSIGNED: an evicted token had no finite Eq. 1 score against any prototype (a
// NaN / Inf in its key row or in the bank); it is NOT absorbed (trace assign = -2) and the bit is raised.
constexpr uint32_t PKV_ERR_UNASSIGNED = 1u;
constexpr uint32_t PKV_ERR_MAINT_OVERFLOW = 2u;
constexpr uint32_t PKV_ERR_WARMUP_SHORT = 4u;     // warm-up ended with fewer than C residuals in a reservoir: no codebooks
constexpr int kMaxReservoir = 65536, kMaxKmBatch = 1024, kMaxSCap = 32;   // Alg. 2: more merge candidates in one frame than the kernel's list holds
constexpr int kNoProto = 0xfffff;   // sort-key prototype field of such a token (k_max <= 16384 < kNoProto)  // floats of padding after each subspace's [C][sub] block in shared memory

// Shapes, fixed at create.
struct Dims {
  int B;       // banks = NS * L * Hkv
  int NS, L, Hq, Hkv, group;
  int d, sub;  // head_dim, d / G
  int T, Wf;   // tokens per frame, near frames (= ring slots; frame f lives in slot f % Wf)
  int K;       // k_max
  int S, G, C;
  int Nq;
  int bf16;    // 1: K/V/Q/out are bf16, 0: fp32
};

struct Hyper {
  float lambda_sp, lambda_idle;
  int t_idle;
  float alpha, beta, eta, sigma_eps, cos_eps;
  double pq_eps;
  uint32_t flags;
  double rope_theta;     // PROTOKV_ROPE
  int rope_anchor;
  long long pos0;        // stream position of token 0 of frame 0
  int warm_reservoir, km_iters, km_batch;   // PROTOKV_WARMUP
  unsigned long long km_seed;
  int s_cap;             // PROTOKV_VAR_ALLOC
};

// Per-prototype scoring record (Eq. 1 terms that do not depend on the token), 32 bytes.
//   invc = 1/|c_k|;  (mux, muy) = mu_k;  (u, v, w) = lambda-scaled inverse Cholesky factor of Sigma_k + eps I:
//   lambda_sp * d_Mah = sqrt((dx u)^2 + (dy v - dx w)^2);  tau = frame index of the last absorption (tauf = the same
//   as a float, exact below 2^24 frames: the tcgen05 epilogue evaluates the idle test with one saturating add).
//   Field order = the two broadcast loads of the tcgen05 epilogue: {mux, muy, u, w} and {v, tauf}.
struct __align__(16) ScoreRec {
  float mux, muy, u, w;
  float v, tauf, invc;
  int tau;
};
// Storage of the records (Dev::rec): PAIRS of prototypes interleaved field by field, 16 floats per pair in the order
// mux, muy, u, -w | v, tauf, invc, tau -- the tcgen05 epilogue scores two prototypes at a time with packed f32x2
// arithmetic and wants each field of the pair as one aligned 64-bit operand (three 16-byte shared loads per pair).
// w is stored negated so that y2 = dy v - dx w is one multiply and one fused multiply-add without a negation.
__host__ __device__ inline size_t rec_slot(size_t pk, int field) { return (pk >> 1) * 16 + (size_t)field * 2 + (pk & 1); }
__device__ __forceinline__ void store_rec(ScoreRec* base, size_t pk, const ScoreRec& r) {
  float* f = reinterpret_cast<float*>(base);
  f[rec_slot(pk, 0)] = r.mux; f[rec_slot(pk, 1)] = r.muy; f[rec_slot(pk, 2)] = r.u; f[rec_slot(pk, 3)] = -r.w;
  f[rec_slot(pk, 4)] = r.v; f[rec_slot(pk, 5)] = r.tauf; f[rec_slot(pk, 6)] = r.invc;
  f[rec_slot(pk, 7)] = __int_as_float(r.tau);
}
__device__ __forceinline__ ScoreRec load_rec(const ScoreRec* base, size_t pk) {
  const float* f = reinterpret_cast<const float*>(base);
  ScoreRec r;
  r.mux = f[rec_slot(pk, 0)]; r.muy = f[rec_slot(pk, 1)]; r.u = f[rec_slot(pk, 2)]; r.w = -f[rec_slot(pk, 3)];
  r.v = f[rec_slot(pk, 4)]; r.tauf = f[rec_slot(pk, 5)]; r.invc = f[rec_slot(pk, 6)];
  r.tau = __float_as_int(f[rec_slot(pk, 7)]);
  return r;
}

// Device pointers into the workspace.
struct Dev {
  // near window
  void* ringK;   // [B][Wf][T][d] elt
  void* ringV;
  float* ringS;  // [NS][Wf][T][2]
  float* ringN;  // [B][Wf][T]  |K_j|^2 of the ring rows (written by the append; the tcgen05 assignment scales by |K_j|)
  // far bank
  float* c;      // [B][K][d]
  float* p;
  __nv_bfloat16* c_hi;  // [B][K][d] bf16 shadows (bf16 mode): c = c_hi + c_lo + O(2^-17 |c|)
  __nv_bfloat16* c_lo;
  __nv_bfloat16* c_bf;  // [B][K][d] bf16(c), bf16(p): what the decode-style attention streams (bf16, d = 128 states);
  __nv_bfloat16* p_bf;  // rewritten by whoever rewrites c / p
  int* n;        // [B][K]
  float* mu;     // [B][K][2]
  float* sigma;  // [B][K][3]
  int* tau;      // [B][K]
  long long* pos;  // [B][K]  stream position of the most recently absorbed token (D.1 default anchor)
  long long* pos_first;  // [B][K] ... of the initialising token
  long long* pos_sum;    // [B][K] sum over all absorbed tokens
  int* pos_cnt;          // [B][K]
  // rotary tables (PROTOKV_ROPE only), rebuilt by every query: cis(angle) as float2 from fp64 sincos
  float2* ropeJ;         // [T][d/2]        token offset j inside a frame
  float2* ropeF;         // [Wf][d/2]       first position of the frame held in each ring slot
  float2* ropeP;         // [B][K][d/2]     anchor of every prototype
  float2* ropeQ;         // [Nq][d/2]       query tokens
  float2* ropeR;         // [Wf * T][d/2]   every ring row at its stream position (what the decode-style kernel reads)
  uint32_t* nres;  // [B][K]
  ScoreRec* rec;   // [B * K / 2] pairs, see rec_slot()
  float* logn;     // [B][K]  log n_k (Eq. 4 bias)
  uint32_t* hist;  // [B][K][2][G][C]
  const double* logtab;  // [PKV_SYN_LOGTAB] log(h + pq_eps), h = 0, 1, ...: built on the host at create (synthesis, Eq. 3)
  float* cbk;      // [B][G][C][sub]  (NULL when the state has no residual statistics)
  float* cbv;
  __nv_bfloat16* cb_bf;  // [B][2][G * C][sub] bf16 copies of cbk, cbv (decode-style attention), written when the codebooks are
  // synthesis result
  uint32_t* codesK;  // [B][K][S], code of subspace g in bits [4g, 4g+4)
  uint32_t* codesV;
  uint8_t* kind;     // [B][K] 0 decoded, 1 zero residual, 2 absent
  // dirty[pk] = id of the synthesis epoch in which the prototype's histograms / mass last changed (0 = never).  The
  // host counts epochs (one per synthesis); the synthesis of epoch e re-decodes exactly the prototypes stamped e and
  // leaves the codes of the others, which are still valid, alone.  Plain stores, no atomics, nothing to clear.
  uint32_t* dirty;       // [B][K]
  // per-frame scratch / trace
  int* assign;       // [B][T]
  float* best;       // [B][T]
  unsigned long long* akey;  // [B][T] packed (orderable(|K_j| * score) << 32 | k): atomicMin target of the tcgen05
                             // assignment; all-ones between frames (reset by the append kernel)
  uint8_t* tcodeK;   // [B][T][G]
  uint8_t* tcodeV;
  // err[0]: sticky device-side error bits (PKV_ERR_*), read by protokv_error_flags
  uint32_t* err;
  // Alg. 2 maintenance: mstamp[pk] = stream time of the last change of c_k / p_k (fill, update, merge, recycle);
  // mcount = {mass decayed, prototypes merged away, slots recycled} since create
  int* mstamp;                   // [B][K]
  unsigned long long* mcount;    // [3]
  // PQ codebook warm-up (PROTOKV_WARMUP): reservoirs of residual pairs and this frame's write plan
  float* resK;   // [B][R][d]
  float* resV;
  int* rslot;    // [B][T] reservoir slot the residual of evicted token j goes to, -1 = none (written by reservoir_plan_kernel)
  // D.3 allocation (PROTOKV_VAR_ALLOC): counts, exclusive prefix offsets into the bank's [K * S] code rows, variances
  int* scount;   // [B][K]
  int* soff;     // [B][K + 1]
  long long* varfx;  // [B][K]
  // attention scratch
  float* part;   // [rows_total][nsplit][d + 2]
  // host-variant staging
  void* stageK; void* stageV; float* stageS; void* stageQ; void* stageO;
};

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

template <typename T> __device__ __forceinline__ float to_f32(T x);
template <> __device__ __forceinline__ float to_f32<float>(float x) { return x; }
template <> __device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 x) { return __bfloat162float(x); }
template <typename T> __device__ __forceinline__ T from_f32(float x);
template <> __device__ __forceinline__ float from_f32<float>(float x) { return x; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float x) { return __float2bfloat16_rn(x); }

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Load VEC consecutive elements starting at ptr[i0] as floats (VEC in {2, 4}; 4-/8-/16-byte aligned accesses).
template <typename T, int VEC> __device__ __forceinline__ void load_vec(const T* ptr, float (&out)[VEC]);
template <> __device__ __forceinline__ void load_vec<float, 4>(const float* ptr, float (&o)[4]) {
  float4 v = *reinterpret_cast<const float4*>(ptr); o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
}
template <> __device__ __forceinline__ void load_vec<float, 2>(const float* ptr, float (&o)[2]) {
  float2 v = *reinterpret_cast<const float2*>(ptr); o[0] = v.x; o[1] = v.y;
}
template <> __device__ __forceinline__ void load_vec<__nv_bfloat16, 4>(const __nv_bfloat16* ptr, float (&o)[4]) {
  uint2 v = *reinterpret_cast<const uint2*>(ptr);
  o[0] = __uint_as_float(v.x << 16); o[1] = __uint_as_float(v.x & 0xffff0000u);
  o[2] = __uint_as_float(v.y << 16); o[3] = __uint_as_float(v.y & 0xffff0000u);
}
template <> __device__ __forceinline__ void load_vec<__nv_bfloat16, 2>(const __nv_bfloat16* ptr, float (&o)[2]) {
  uint32_t v = *reinterpret_cast<const uint32_t*>(ptr);
  o[0] = __uint_as_float(v << 16); o[1] = __uint_as_float(v & 0xffff0000u);
}

// ---- launchers implemented in the .cu files (all asynchronous on `stream`) -------------------------------
struct FrameArgs {
  int t;         // stream time of this step = index of the appended frame (reading 2)
  int slot;      // ring slot of the appended frame = slot of the evicted frame (f % Wf)
  int evicted;   // 1 if a frame leaves the window in this step
  int ev_frame;  // index of the evicted frame
  int n_act0;    // active prototypes before this step's slot fill
  int n_fill;    // evicted tokens that open a new slot (Alg. 1 l.3-4)
  int n_act;     // active prototypes after the fill = what Eq. 1 scans
  int epoch;     // id of the current synthesis epoch (>= 1), see Dev::dirty
  int keys;      // 1: the assignment of this frame is in Dev::akey (tcgen05 path), 0: in Dev::assign / best (SIMT)
  int warm;      // 1: warm-up step -- residuals go to the reservoir slots of Dev::rslot, no histogram update
  long long res_base;  // residuals offered to each bank's reservoir before this frame
  int pdl;       // host side only: the frame's kernels are launched with programmatic stream serialisation (see pdl_wait)
};

// Programmatic dependent launch along the library's kernel chains (score -> update -> ring append; synthesis ->
// attention -> combine -> the next call's attention; decode kernel -> combine): a kernel launched with the attribute may
// start once every CTA of its predecessor has executed pdl_trigger() or exited; before pdl_wait() returns (= the
// predecessor has completed and its writes are visible) it touches nothing that a kernel of the library writes or that the
// caller passes in, with one exception, the ring append (see protokv_api.cu).  A kernel triggers only AFTER its own wait,
// so "the predecessor of my predecessor has completed" holds by induction.  Kernels whose successor is a persistent
// one-CTA-per-SM kernel (ring append, attention) do not trigger: measured, such a successor pending under their tail
// slows them down; it then starts at their exit and still skips the launch latency.  Without the attribute (and under
// PROTOKV_SERIAL_LAUNCH) both instructions are no-ops.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_chain(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, bool pdl,
                                Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// Every launcher returns the number of kernels it launched (0 if there was nothing to do).
int launch_ring_append(const Dims& D, const Dev& V, const FrameArgs& F, const void* Kin, const void* Vin,
                       const float* grid_pos, cudaStream_t s);
int launch_fill(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, cudaStream_t s);
int launch_score_simt(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, cudaStream_t s);
int launch_update(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, int sm_count, cudaStream_t s);
int launch_refresh_derived(const Dims& D, const Hyper& H, const Dev& V, int bank, int epoch, cudaStream_t s);
int launch_fill_u32(uint32_t* dst, uint32_t value, size_t n, cudaStream_t s);
int launch_or_u32(uint32_t* dst, uint32_t bits, cudaStream_t s);
int launch_codebook_copy(const Dims& D, const Dev& V, const float* cbk, const float* cbv, cudaStream_t s);   // fills Dev::cb_bf
// One-time (per device) function attributes of every kernel that needs more than 48 KB of shared memory for some
// admissible shape; returns false if the device refuses one of them.
bool update_kernels_prepare(const Dims& D);
bool query_kernels_prepare(const Dims& D);
int launch_synthesis(const Dims& D, const Hyper& H, const Dev& V, int n_act, int epoch, int max_dirty, int sm_count,
                     cudaStream_t s);

__device__ __forceinline__ void mark_dirty(const Dims& D, const Dev& V, int b, int k, int epoch) {
  V.dirty[(size_t)b * D.K + k] = (uint32_t)epoch;
}

struct AttnArgs {
  long long q_pos0;    // stream position of query token 0 (PROTOKV_ROPE)
  long long frames;    // frames appended so far (ring slot s holds frame ... see launch_rope_tables)
  const void* Q; void* out; float* lse;
  int n_q, layer_begin, layer_count;
  int n_near;          // near-window tokens currently held (frames held * T): ring rows [0, n_near) of each bank
  int n_act;
  int nsplit;
};
int attention_simt_splits(const Dims& D, int sm_count);   // nsplit the SIMT kernel uses (part buffer sizing)
int launch_attention_simt(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, cudaStream_t s);
int launch_rope_tables(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, cudaStream_t s);
// static_scratch.cu: the SIMT attention with its partials in the library's file-scope device array (no allocation)
size_t static_scratch_bytes();
int launch_attention_static(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, int sm_count, cudaStream_t s,
                            size_t* need_bytes, cudaError_t* cuda_err);

// PQ codebook warm-up (warmup.cu)
int launch_reservoir_plan(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, cudaStream_t s);
// cbk / cbv: where the trained codebooks go ([B][G][C][sub]); fill = rows every reservoir holds
int launch_kmeans(const Dims& D, const Hyper& H, const Dev& V, float* cbk, float* cbv, long long fill, cudaStream_t s);
bool warmup_prepare(const Dims& D, const Hyper& H);
// D.3 allocation + ragged synthesis (alloc.cu)
bool alloc_prepare(const Dims& D);
int launch_allocation(const Dims& D, const Hyper& H, const Dev& V, int n_act, cudaStream_t s);
int launch_synthesis_var(const Dims& D, const Hyper& H, const Dev& V, int n_act, cudaStream_t s);

// Alg. 2 maintenance (maintenance.cu)
bool maintenance_prepare();
int launch_maintenance(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, int held, int full, float gamma,
                       float eps_k, float eps_v, cudaStream_t s);

// decode-style attention (decode_attention.cu): bf16, d = 128, n_q * group <= 16 rows per bank
bool decode_attention_supported(const Dims& D, int n_q);
size_t decode_attention_part_bytes(const Dims& D);
bool decode_attention_prepare();
int launch_attention_decode(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, int sm_count, cudaStream_t s,
                            int* nsplit_out);
// register-resident decode kernel (decode_attention2.cu): the default for n_q * group <= 16 rows per bank
bool decode2_attention_supported(const Dims& D, int n_q);
bool decode2_rope_supported(const Dims& D);
bool decode2_attention_prepare();
int decode2_max_splits();
int launch_attention_decode2(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, int sm_count, cudaStream_t s,
                             int* nsplit_out);
// merges A.nsplit partials per row ([rows][nsplit][d + 2] in Dev::part) into out / lse (bf16, d = 128)
int launch_attention_combine_bf16_128(const Dims& D, const Dev& V, const AttnArgs& A, bool pdl, cudaStream_t s);

// tcgen05 paths (bf16, d = 128).  The TMA tensor maps are built once per state.
struct TcMaps {
  CUtensorMap ringK, ringV;   // [B*Wf*T][128] bf16, box {64 cols, 128 rows}, 128-byte swizzle
  CUtensorMap c_hi, c_lo;     // [B*K][128] bf16, same box
  bool ok;
};
bool tc_assign_supported(const Dims& D, const Hyper& H);
bool tc_build_maps(const Dims& D, const Dev& V, TcMaps* maps);
int launch_score_tc(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, const TcMaps& maps,
                    int sm_count, cudaStream_t s);
bool tc_attention_supported(const Dims& D);
size_t tc_attention_part_bytes(const Dims& D);   // partial-result buffer the tcgen05 attention needs at most
bool tc_attention_prepare();                     // one-time function attributes; false if the device refuses them
// Returns the number of kernels launched, or -1 if the Q tensor map could not be encoded.
int launch_attention_tc(const Dims& D, const Hyper& H, const Dev& V, const AttnArgs& A, const TcMaps& maps,
                        int sm_count, cudaStream_t s);

}  // namespace pkv
