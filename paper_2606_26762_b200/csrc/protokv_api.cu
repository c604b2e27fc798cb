// C ABI of the ProtoKV hot path (include/protokv.h): host-side state, workspace carving, argument checks and
// kernel sequencing.  No arithmetic of the method happens here; every step runs in the kernels of
// update_kernels.cu / query_kernels.cu / tc_*.cu.
#include <cstdarg>
#include <cstdio>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "common.cuh"

using namespace pkv;

struct protokv_state {
  protokv_config cfg;
  Dims D;
  Hyper H;
  Dev V;
  cudaStream_t stream;
  int device;         // ordinal the state was created on; every entry point runs with it current (DeviceGuard)
  bool poisoned;      // a launch failed half-way through a call: device and host counters may disagree
  bool maint_full;    // the next Alg. 2 pass must look at every pair (first pass, after an import)
  int sm_count;
  int64_t frames;     // frames appended so far = stream time of the next frame
  int n_act;          // active prototypes per bank (identical in every bank: slot fill is data-independent)
  int64_t launches;
  int last_ev_frame;  // index of the frame evicted by the last append, -1 if none
  int last_n_fill;
  // PQ codebook warm-up (PROTOKV_WARMUP): the codebook arrays are carved but stay hidden (Dev::cbk == NULL: no
  // histogram updates, zero residuals) until the training has written them
  bool warm;          // the state was created with PROTOKV_WARMUP
  bool trained;       // warm-up over (training ran or was skipped for lack of residuals)
  float *cb_store_k, *cb_store_v;
  int64_t res_seen;   // residuals offered to every bank's reservoir so far (identical in every bank)
  bool codes_valid;   // codes/kind describe the current histograms
  std::vector<double> logtab;   // host copy of Dev::logtab (source of an asynchronous copy: must outlive it)
  int epoch;          // synthesis epoch (see Dev::dirty_cnt)
  int dirty_bound;    // upper bound of the prototypes per bank stamped dirty since the last synthesis (sizes its grid)
  bool use_tc_assign;
  bool use_tc_attn;
  bool use_decode_attn;   // the split-KV mma.sync kernel serves queries of <= 16 rows per bank
  bool use_decode2;       // the register-resident decode kernel serves them (default where supported)
  // host-buffer variants: the H2D copies of a frame run on a copy stream of the library's own, next to the scoring and
  // update kernels (which only need the evicted frame that is already in the ring); the ring append waits for them
  cudaStream_t copy_stream;
  cudaEvent_t ev_copied, ev_appended;
  bool appended_pending;  // ev_appended has been recorded: the staging buffers are in use until it completes
  bool use_decode_rope;   // PROTOKV_ROPE / PROTOKV_VAR_ALLOC state served by the rotating / ragged variants of that kernel
                          // (any number of query rows)
  TcMaps maps;
  int nsplit;
  // stage timing (protokv_profile_*)
  bool profiling;
  std::vector<cudaEvent_t> ev_free;
  struct Span { int stage; cudaEvent_t a, b; };
  std::vector<Span> spans;
  double prof_ms[PROTOKV_N_STAGES];
  int64_t prof_n[PROTOKV_N_STAGES];
};

// Brackets one launcher call with events when profiling is on.
struct StageTimer {
  protokv_state* st;
  int stage;
  cudaEvent_t a = nullptr, b = nullptr;
  static cudaEvent_t get(protokv_state* st) {
    if (!st->ev_free.empty()) { cudaEvent_t e = st->ev_free.back(); st->ev_free.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
  }
  StageTimer(protokv_state* s, int stg) : st(s), stage(stg) {
    if (!st->profiling) return;
    a = get(st); b = get(st);
    cudaEventRecord(a, st->stream);
  }
  ~StageTimer();
};

static int drain_spans(protokv_state* st) {
  for (auto& sp : st->spans) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, sp.a, sp.b) == cudaSuccess) { st->prof_ms[sp.stage] += ms; st->prof_n[sp.stage] += 1; }
    st->ev_free.push_back(sp.a); st->ev_free.push_back(sp.b);
  }
  st->spans.clear();
  return 0;
}

StageTimer::~StageTimer() {
  if (!a) return;
  cudaEventRecord(b, st->stream);
  st->spans.push_back({stage, a, b});
  if (st->spans.size() >= 4096) {      // nobody reads the profile: fold the finished spans so the events are recycled
    cudaEventSynchronize(b);
    drain_spans(st);
  }
}

static thread_local char g_err[512] = "";

// Makes the state's device current for the duration of an entry point and restores the caller's device afterwards.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(const protokv_state* st) {
    if (!st) return;
    if (cudaGetDevice(&prev) == cudaSuccess && prev != st->device) switched = cudaSetDevice(st->device) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

static int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

#define PKV_CUDA(call)                                                                       \
  do {                                                                                       \
    cudaError_t e_ = (call);                                                                 \
    if (e_ != cudaSuccess) return fail(PROTOKV_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

static bool is_pow2(int x) { return x > 0 && (x & (x - 1)) == 0; }

// Validates everything that does not need a device.  Returns PROTOKV_OK or sets the error text.
static int validate(const protokv_config* c) {
  if (!c) return fail(PROTOKV_EINVAL, "cfg is NULL");
  if (c->struct_size != sizeof(protokv_config))
    return fail(PROTOKV_EINVAL, "struct_size %u != %zu", c->struct_size, sizeof(protokv_config));
  if (c->n_streams < 1 || c->n_layers < 1 || c->n_q_heads < 1 || c->n_kv_heads < 1 || c->tokens_per_frame < 1 ||
      c->near_frames < 1 || c->k_max < 1 || c->n_query_tokens < 1)
    return fail(PROTOKV_EINVAL, "shape fields must be >= 1");
  if (c->n_q_heads % c->n_kv_heads) return fail(PROTOKV_EINVAL, "n_q_heads %% n_kv_heads != 0");
  if (c->dtype != PROTOKV_F32 && c->dtype != PROTOKV_BF16) return fail(PROTOKV_EINVAL, "unknown dtype");
  if (c->head_dim != 64 && c->head_dim != 128) return fail(PROTOKV_EUNSUPPORTED, "head_dim must be 64 or 128");
  if (c->S < 1 || c->G < 1 || c->C < 1 || c->beam < c->S) return fail(PROTOKV_EINVAL, "need S,G,C >= 1, beam >= S");
  if (c->S > kMaxS || c->C > kMaxC || c->G > kMaxG || !is_pow2(c->G))
    return fail(PROTOKV_EUNSUPPORTED, "need S <= 8, C <= 16, G in {1,2,4,8}");
  if (c->head_dim % c->G) return fail(PROTOKV_EINVAL, "head_dim %% G != 0");
  {
    double tuples = 1;
    for (int g = 0; g < c->G; ++g) tuples *= c->C;
    if (tuples < c->S) return fail(PROTOKV_EINVAL, "C^G < S");
  }
  if (c->tokens_per_frame > kMaxT) return fail(PROTOKV_EUNSUPPORTED, "tokens_per_frame > 4096");
  if (c->k_max > kMaxKmax) return fail(PROTOKV_EUNSUPPORTED, "k_max > 16384");
  if (!(c->alpha >= 0.f && c->alpha <= 1.f && c->beta >= 0.f && c->beta <= 1.f && c->eta >= 0.f && c->eta <= 1.f))
    return fail(PROTOKV_EINVAL, "alpha, beta, eta must lie in [0, 1]");
  if (!(c->sigma_eps >= 0.f) || !(c->cos_eps > 0.f) || !(c->pq_eps > 0.0))
    return fail(PROTOKV_EINVAL, "need sigma_eps >= 0, cos_eps > 0, pq_eps > 0");
  if (c->flags & PROTOKV_MAINTENANCE) {
    if (!(c->gamma >= 0.f && c->gamma <= 1.f) || !(c->eps_k >= 0.f) || !(c->eps_v >= 0.f))
      return fail(PROTOKV_EINVAL, "maintenance needs gamma in [0, 1], eps_k >= 0, eps_v >= 0");
  }
  if (c->flags & PROTOKV_ROPE) {
    if (!(c->rope_theta > 1.0) || c->rope_anchor < 0 || c->rope_anchor > 2)
      return fail(PROTOKV_EINVAL, "rope needs rope_theta > 1 and rope_anchor in {0, 1, 2}");
  }
  if (c->flags & PROTOKV_WARMUP) {
    if (c->t_warm < 1 || c->warm_reservoir < 1 || c->warm_reservoir > kMaxReservoir || c->km_iters < 0 || c->km_batch < 1 ||
        c->km_batch > kMaxKmBatch)
      return fail(PROTOKV_EINVAL, "warm-up needs t_warm >= 1, 1 <= warm_reservoir <= 65536, km_iters >= 0, 1 <= km_batch <= 1024");
  } else if (c->flags & PROTOKV_WARMUP_MANUAL) {
    return fail(PROTOKV_EINVAL, "WARMUP_MANUAL without WARMUP");
  }
  if (c->flags & PROTOKV_VAR_ALLOC) {
    if (c->s_cap < 1 || c->s_cap > c->beam || c->s_cap > kMaxSCap) return fail(PROTOKV_EINVAL, "need 1 <= s_cap <= min(beam, 32)");
    double tuples = 1;
    for (int g = 0; g < c->G; ++g) tuples *= c->C;
    if (tuples < c->s_cap) return fail(PROTOKV_EINVAL, "C^G < s_cap");
    if (c->flags & PROTOKV_DECODE_SPLITKV) return fail(PROTOKV_EUNSUPPORTED, "VAR_ALLOC is served by the SIMT attention kernel only");
  }
  if (!(c->lambda_sp >= 0.f) || !(c->lambda_idle >= 0.f))   // Eq. 1's penalties are penalties (the score kernel prunes on it)
    return fail(PROTOKV_EINVAL, "need lambda_sp >= 0 and lambda_idle >= 0");
  if ((c->flags & PROTOKV_NEAR_ONLY) && (c->flags & PROTOKV_FAR_ONLY))
    return fail(PROTOKV_EINVAL, "NEAR_ONLY and FAR_ONLY are exclusive");
  return PROTOKV_OK;
}

static void fill_dims(const protokv_config* c, Dims* D, Hyper* H) {
  D->NS = c->n_streams; D->L = c->n_layers; D->Hq = c->n_q_heads; D->Hkv = c->n_kv_heads;
  D->group = c->n_q_heads / c->n_kv_heads;
  D->B = c->n_streams * c->n_layers * c->n_kv_heads;
  D->d = c->head_dim; D->sub = c->head_dim / c->G;
  D->T = c->tokens_per_frame; D->Wf = c->near_frames; D->K = c->k_max;
  D->S = c->S; D->G = c->G; D->C = c->C; D->Nq = c->n_query_tokens;
  D->bf16 = c->dtype == PROTOKV_BF16;
  H->lambda_sp = c->lambda_sp; H->lambda_idle = c->lambda_idle; H->t_idle = c->t_idle;
  H->alpha = c->alpha; H->beta = c->beta; H->eta = c->eta;
  H->sigma_eps = c->sigma_eps; H->cos_eps = c->cos_eps; H->pq_eps = c->pq_eps; H->flags = c->flags;
  H->rope_theta = c->rope_theta; H->rope_anchor = c->rope_anchor; H->pos0 = (long long)c->pos0;
  H->warm_reservoir = c->warm_reservoir; H->km_iters = c->km_iters; H->km_batch = c->km_batch;
  H->km_seed = (unsigned long long)c->km_seed; H->s_cap = c->s_cap;
}

// Lays the state out in the workspace (base may be NULL to only measure).  Every array is 256-byte aligned.
static size_t carve(const Dims& D, const Hyper& H, bool has_cb, bool rope, int nsplit, char* base, Dev* V) {
  size_t off = 0;
  auto take = [&](size_t bytes) -> void* {
    off = align_up(off, 256);
    void* p = base ? base + off : nullptr;
    off += bytes;
    return p;
  };
  const size_t elt = D.bf16 ? 2 : 4;
  const size_t BK = (size_t)D.B * D.K, BT = (size_t)D.B * D.T;
  const size_t ring = (size_t)D.B * D.Wf * D.T * D.d * elt;
  Dev v{};
  v.ringK = take(ring); v.ringV = take(ring);
  v.ringS = (float*)take((size_t)D.NS * D.Wf * D.T * 2 * 4);
  v.ringN = (float*)take((size_t)D.B * D.Wf * D.T * 4);
  v.c = (float*)take(BK * D.d * 4); v.p = (float*)take(BK * D.d * 4);
  if (D.bf16) {
    v.c_hi = (__nv_bfloat16*)take(BK * D.d * 2);
    v.c_lo = (__nv_bfloat16*)take(BK * D.d * 2);
    if (decode2_rope_supported(D)) {
      v.c_bf = (__nv_bfloat16*)take(BK * D.d * 2);
      v.p_bf = (__nv_bfloat16*)take(BK * D.d * 2);
      if (has_cb) v.cb_bf = (__nv_bfloat16*)take((size_t)D.B * 2 * D.G * D.C * D.sub * 2);
    }
  }
  v.n = (int*)take(BK * 4); v.mu = (float*)take(BK * 8); v.sigma = (float*)take(BK * 12);
  v.tau = (int*)take(BK * 4); v.pos = (long long*)take(BK * 8); v.nres = (uint32_t*)take(BK * 4);
  v.pos_first = (long long*)take(BK * 8); v.pos_sum = (long long*)take(BK * 8); v.pos_cnt = (int*)take(BK * 4);
  if (rope) {
    const size_t h = (size_t)D.d / 2;
    v.ropeJ = (float2*)take((size_t)D.T * h * 8); v.ropeF = (float2*)take((size_t)D.Wf * h * 8);
    v.ropeP = (float2*)take(BK * h * 8); v.ropeQ = (float2*)take((size_t)D.Nq * h * 8);
    v.ropeR = (float2*)take((size_t)D.Wf * D.T * h * 8);
  }
  v.rec = (ScoreRec*)take((BK + 1) * sizeof(ScoreRec)); v.logn = (float*)take(BK * 4);
  v.hist = (uint32_t*)take(BK * 2 * D.G * D.C * 4);
  v.logtab = (const double*)take((size_t)PKV_SYN_LOGTAB * 8);
  if (has_cb) {
    v.cbk = (float*)take((size_t)D.B * D.G * D.C * D.sub * 4);
    v.cbv = (float*)take((size_t)D.B * D.G * D.C * D.sub * 4);
  }
  v.codesK = (uint32_t*)take(BK * D.S * 4); v.codesV = (uint32_t*)take(BK * D.S * 4);
  v.kind = (uint8_t*)take(BK);
  v.dirty = (uint32_t*)take(BK * 4);
  v.assign = (int*)take(BT * 4); v.best = (float*)take(BT * 4);
  v.akey = (unsigned long long*)take(BT * 8);
  v.tcodeK = (uint8_t*)take(BT * D.G); v.tcodeV = (uint8_t*)take(BT * D.G);
  v.err = (uint32_t*)take(256);
  v.mcount = (unsigned long long*)take(256);
  v.mstamp = (int*)take(BK * 4);
  if ((H.flags & PROTOKV_WARMUP) && !(H.flags & PROTOKV_NO_RESIDUAL)) {
    const size_t res = (size_t)D.B * H.warm_reservoir * D.d * 4;
    v.resK = (float*)take(res);
    v.resV = (float*)take(res + (size_t)D.B * H.warm_reservoir * 8);   // + the claim words of reservoir_plan_kernel
    v.rslot = (int*)take(BT * 4);
  }
  if (H.flags & PROTOKV_VAR_ALLOC) {
    v.scount = (int*)take(BK * 4);
    v.soff = (int*)take((size_t)D.B * (D.K + 1) * 4);
    v.varfx = (long long*)take(BK * 8);
  }
  const size_t rows = (size_t)D.B * D.Nq * D.group;
  size_t part_bytes = rows * nsplit * (D.d + 2) * 4;
  if (tc_attention_supported(D) && tc_attention_part_bytes(D) > part_bytes) part_bytes = tc_attention_part_bytes(D);
  if (decode_attention_supported(D, 1) && decode_attention_part_bytes(D) > part_bytes) part_bytes = decode_attention_part_bytes(D);
  if (decode2_rope_supported(D)) {
    const size_t need = (size_t)D.B * 16 * decode2_max_splits() * 130 * 4;
    if (need > part_bytes) part_bytes = need;
  }
  v.part = (float*)take(part_bytes);
  const size_t frame = (size_t)D.NS * D.L * D.T * D.Hkv * D.d * elt;
  const size_t qbytes = (size_t)D.NS * D.L * D.Nq * D.Hq * D.d * elt;
  v.stageK = take(frame); v.stageV = take(frame);
  v.stageS = (float*)take((size_t)D.NS * D.T * 2 * 4);
  v.stageQ = take(qbytes); v.stageO = take(qbytes);
  if (V) *V = v;
  return align_up(off, 256);
}

// nsplit must be known without a device for protokv_workspace_bytes: size for the B200's 148 SMs.
static int plan_nsplit(const Dims& D) { return attention_simt_splits(D, 148); }

extern "C" {

const char* protokv_last_error(void) { return g_err; }

size_t protokv_workspace_bytes(const protokv_config* cfg) {
  if (validate(cfg) != PROTOKV_OK) return 0;
  Dims D; Hyper H;
  fill_dims(cfg, &D, &H);
  const bool has_cb = !(cfg->flags & PROTOKV_NO_RESIDUAL);   // sized as if codebooks were given
  return carve(D, H, has_cb, (cfg->flags & PROTOKV_ROPE) != 0, plan_nsplit(D), nullptr, nullptr);
}

protokv_state* protokv_create(const protokv_config* cfg) {
  g_err[0] = 0;
  if (validate(cfg) != PROTOKV_OK) return nullptr;
  if (!cfg->workspace) { fail(PROTOKV_EINVAL, "workspace is NULL"); return nullptr; }
  if ((uintptr_t)cfg->workspace % 256) { fail(PROTOKV_EINVAL, "workspace must be 256-byte aligned"); return nullptr; }
  if ((cfg->codebook_k == nullptr) != (cfg->codebook_v == nullptr)) {
    fail(PROTOKV_EINVAL, "codebook_k and codebook_v must both be given or both be NULL");
    return nullptr;
  }
  int dev = 0, major = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
    cudaGetLastError();
    fail(PROTOKV_EUNSUPPORTED, "no CUDA device: this library has no CPU fallback");
    return nullptr;
  }
  if (major != 10) { fail(PROTOKV_EUNSUPPORTED, "device is sm_%d0, this build is sm_100a only", major); return nullptr; }
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);

  protokv_state* st = new (std::nothrow) protokv_state();
  if (!st) { fail(PROTOKV_ENOMEM, "host allocation failed"); return nullptr; }
  st->cfg = *cfg;
  fill_dims(cfg, &st->D, &st->H);
  st->stream = (cudaStream_t)cfg->cuda_stream;
  st->device = dev;
  st->poisoned = false;
  st->maint_full = true;
  st->sm_count = sms;
  st->nsplit = plan_nsplit(st->D);
  st->warm = (cfg->flags & PROTOKV_WARMUP) && !(cfg->flags & PROTOKV_NO_RESIDUAL);
  st->trained = false; st->res_seen = 0;
  const bool carve_cb = (cfg->codebook_k || st->warm) && !(cfg->flags & PROTOKV_NO_RESIDUAL);
  const bool has_cb = carve_cb && !st->warm;                  // codebooks to copy now (warm-up states train their own)
  const size_t need = carve(st->D, st->H, carve_cb, (cfg->flags & PROTOKV_ROPE) != 0, st->nsplit, (char*)cfg->workspace, &st->V);
  st->cb_store_k = st->V.cbk; st->cb_store_v = st->V.cbv;
  if (st->warm) { st->V.cbk = nullptr; st->V.cbv = nullptr; }
  if (need > cfg->workspace_bytes) {
    fail(PROTOKV_ENOMEM, "workspace too small: need %zu bytes, got %zu", need, cfg->workspace_bytes);
    delete st;
    return nullptr;
  }
  cudaError_t e = cudaMemsetAsync(cfg->workspace, 0, need, st->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(st->V.akey, 0xff, (size_t)st->D.B * st->D.T * 8, st->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(st->V.kind, 2, (size_t)st->D.B * st->D.K, st->stream);   // every slot absent
  if (e == cudaSuccess && has_cb) {
    const size_t cb = (size_t)st->D.B * st->D.G * st->D.C * st->D.sub * 4;
    e = cudaMemcpyAsync(st->V.cbk, cfg->codebook_k, cb, cudaMemcpyDeviceToDevice, st->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(st->V.cbv, cfg->codebook_v, cb, cudaMemcpyDeviceToDevice, st->stream);
    if (e == cudaSuccess) { st->launches += launch_codebook_copy(st->D, st->V, st->V.cbk, st->V.cbv, st->stream); e = cudaGetLastError(); }
  }
  if (e == cudaSuccess) {   // numerators of Eq. 3 in log form (the host's libm, like the definition reads)
    st->logtab.resize(PKV_SYN_LOGTAB);
    for (int h = 0; h < PKV_SYN_LOGTAB; ++h) st->logtab[h] = log((double)h + cfg->pq_eps);
    e = cudaMemcpyAsync((void*)st->V.logtab, st->logtab.data(), (size_t)PKV_SYN_LOGTAB * 8, cudaMemcpyHostToDevice, st->stream);
  }
  if (e != cudaSuccess) {
    fail(PROTOKV_ECUDA, "state initialisation: %s", cudaGetErrorString(e));
    delete st;
    return nullptr;
  }
  st->copy_stream = nullptr; st->ev_copied = nullptr; st->ev_appended = nullptr; st->appended_pending = false;
  st->frames = 0; st->n_act = 0; st->launches = 0; st->last_ev_frame = -1; st->last_n_fill = 0;
  st->codes_valid = false;
  st->epoch = 1;
  st->dirty_bound = st->D.K;
  st->profiling = false;
  for (int i = 0; i < PROTOKV_N_STAGES; ++i) { st->prof_ms[i] = 0.0; st->prof_n[i] = 0; }
  st->maps.ok = false;
  if (!update_kernels_prepare(st->D) || !query_kernels_prepare(st->D) ||
      ((cfg->flags & PROTOKV_MAINTENANCE) && !maintenance_prepare()) || (st->warm && !warmup_prepare(st->D, st->H)) ||
      ((cfg->flags & PROTOKV_VAR_ALLOC) && !alloc_prepare(st->D))) {   // capability error: before any launch
    fail(PROTOKV_EUNSUPPORTED, "the device refused the shared-memory opt-in this shape needs");
    delete st;
    return nullptr;
  }
  const bool want_tc = !(cfg->flags & PROTOKV_FORCE_SIMT);
  if (want_tc && (tc_assign_supported(st->D, st->H) || tc_attention_supported(st->D))) tc_build_maps(st->D, st->V, &st->maps);
  st->use_tc_assign = want_tc && tc_assign_supported(st->D, st->H) && st->maps.ok;
  // the rotation stage and ragged pseudo-token counts exist in the SIMT attention kernel only
  const bool rope = (cfg->flags & (PROTOKV_ROPE | PROTOKV_VAR_ALLOC)) != 0;
  st->use_tc_attn = want_tc && !rope && tc_attention_supported(st->D) && st->maps.ok && tc_attention_prepare();
  st->use_decode_attn = want_tc && !rope && (cfg->flags & PROTOKV_DECODE_SPLITKV) && decode_attention_supported(st->D, 1) &&
                        decode_attention_prepare();
  st->use_decode2 = want_tc && !rope && !st->use_decode_attn && !(cfg->flags & PROTOKV_NO_DECODE_KERNEL) &&
                    decode2_attention_supported(st->D, 1) && decode2_attention_prepare();
  // PROTOKV_ROPE and / or PROTOKV_VAR_ALLOC states: the rotating / ragged variants of that kernel, 8-row blocks
  st->use_decode_rope = want_tc && (cfg->flags & (PROTOKV_ROPE | PROTOKV_VAR_ALLOC)) && !(cfg->flags & PROTOKV_NO_DECODE_KERNEL) &&
                        decode2_rope_supported(st->D) && decode2_attention_prepare();
  return st;
}

void protokv_destroy(protokv_state* st) {
  if (!st) return;
  DeviceGuard dg(st);
  for (auto& sp : st->spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
  for (auto e : st->ev_free) cudaEventDestroy(e);
  if (st->ev_copied) cudaEventDestroy(st->ev_copied);
  if (st->ev_appended) cudaEventDestroy(st->ev_appended);
  if (st->copy_stream) cudaStreamDestroy(st->copy_stream);
  delete st;
}

int protokv_profile_enable(protokv_state* st, int32_t on) {
  if (!st) return fail(PROTOKV_EINVAL, "NULL state");
  DeviceGuard dg(st);
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  drain_spans(st);
  for (int i = 0; i < PROTOKV_N_STAGES; ++i) { st->prof_ms[i] = 0.0; st->prof_n[i] = 0; }
  st->profiling = on != 0;
  return PROTOKV_OK;
}

int protokv_profile_read(protokv_state* st, double* ms_sum, int64_t* launches) {
  if (!st || !ms_sum || !launches) return fail(PROTOKV_EINVAL, "NULL argument");
  DeviceGuard dg(st);
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  drain_spans(st);
  for (int i = 0; i < PROTOKV_N_STAGES; ++i) {
    ms_sum[i] = st->prof_ms[i]; launches[i] = st->prof_n[i];
    st->prof_ms[i] = 0.0; st->prof_n[i] = 0;
  }
  return PROTOKV_OK;
}

// before_append: an event the ring append (the only consumer of K, V, grid_pos) waits for, or NULL
static int append_frame_impl(protokv_state* st, const void* K, const void* V, const float* grid_pos, cudaEvent_t before_append) {
  if (!st || !K || !V || !grid_pos) return fail(PROTOKV_EINVAL, "NULL argument");
  if (st->poisoned) return fail(PROTOKV_ESTATE, "an earlier launch failure left this state inconsistent; destroy it");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  FrameArgs F{};
  F.t = (int)st->frames;
  F.slot = (int)(st->frames % D.Wf);
  F.evicted = st->frames >= D.Wf;
  F.ev_frame = F.evicted ? (int)(st->frames - D.Wf) : -1;
  F.n_act0 = st->n_act;
  F.n_fill = F.evicted ? (D.K - st->n_act < D.T ? D.K - st->n_act : D.T) : 0;
  F.n_act = st->n_act + F.n_fill;
  F.keys = st->use_tc_assign ? 1 : 0;
  F.epoch = st->epoch;
  F.warm = st->warm && !st->trained && st->frames < st->cfg.t_warm;
  F.res_base = st->res_seen;
  F.pdl = (st->cfg.flags & PROTOKV_SERIAL_LAUNCH) ? 0 : 1;   // score and update touch nothing of the chain before pdl_wait()
  bool after_update = false;
  int nl = 0;
  if (F.evicted) {
    if (F.n_fill > 0) {
      StageTimer tm(st, PROTOKV_STAGE_FILL);
      nl += launch_fill(D, st->H, st->V, F, st->stream);                                // U2
    }
    if (D.T - F.n_fill > 0) {
      {
        StageTimer tm(st, PROTOKV_STAGE_SCORE);
        nl += st->use_tc_assign ? launch_score_tc(D, st->H, st->V, F, st->maps, st->sm_count, st->stream)      // U3
                                : launch_score_simt(D, st->H, st->V, F, st->stream);
      }
      StageTimer tm(st, PROTOKV_STAGE_UPDATE);
      if (F.warm) nl += launch_reservoir_plan(D, st->H, st->V, F, st->stream);          // L312: where this frame's residuals go
      nl += launch_update(D, st->H, st->V, F, st->sm_count, st->stream);                // U4-U6
      after_update = true;
    }
  }
  if (before_append) PKV_CUDA(cudaStreamWaitEvent(st->stream, before_append, 0));
  // the append reads the caller's K / V ahead of its pdl_wait(): only directly behind the update kernel, whose own wait
  // has then returned, i.e. everything the caller enqueued before this call has completed (common.cuh, pdl_wait)
  if (!after_update || before_append) F.pdl = 0;
  {
    StageTimer tm(st, PROTOKV_STAGE_APPEND);
    nl += launch_ring_append(D, st->V, F, K, V, grid_pos, st->stream);                  // U1 (overwrites the slot)
  }
  if ((st->H.flags & PROTOKV_MAINTENANCE) && F.evicted) {                               // Alg. 1 l.15 -> Alg. 2
    const int held = (int)(st->frames + 1 < D.Wf ? st->frames + 1 : D.Wf);
    nl += launch_maintenance(D, st->H, st->V, F, held, st->maint_full ? 1 : 0, st->cfg.gamma, st->cfg.eps_k, st->cfg.eps_v,
                             st->stream);
    st->maint_full = false;
  }
  {
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {   // some kernels of this frame may have run: the bank no longer matches the host counters
      st->poisoned = true;
      return fail(PROTOKV_ECUDA, "append_frame launch: %s", cudaGetErrorString(e));
    }
  }
  st->launches += nl;
  st->n_act = F.n_act;
  st->last_ev_frame = F.ev_frame;
  st->last_n_fill = F.n_fill;
  if (F.evicted) {
    st->codes_valid = false;   // fills and absorptions stamp at most T prototypes per bank; Alg. 2 may stamp any
    st->dirty_bound = (st->H.flags & PROTOKV_MAINTENANCE) ? D.K : (st->dirty_bound + D.T < D.K ? st->dirty_bound + D.T : D.K);
  }
  if (F.warm && F.evicted) st->res_seen += D.T - F.n_fill;
  st->frames += 1;
  if (st->warm && !st->trained && !(st->cfg.flags & PROTOKV_WARMUP_MANUAL) && st->frames == st->cfg.t_warm)
    return protokv_train_codebooks(st);                                                 // end of the warm-up (reading 33)
  return PROTOKV_OK;
}

int protokv_append_frame(protokv_state* st, const void* K, const void* V, const float* grid_pos) {
  return append_frame_impl(st, K, V, grid_pos, nullptr);
}

int protokv_train_codebooks(protokv_state* st) {
  if (!st) return fail(PROTOKV_EINVAL, "NULL state");
  if (st->poisoned) return fail(PROTOKV_ESTATE, "an earlier launch failure left this state inconsistent; destroy it");
  if (!st->warm || st->trained) return fail(PROTOKV_ESTATE, "the state has no warm-up in progress");
  DeviceGuard dg(st);
  st->trained = true;
  const int64_t fill = st->res_seen < st->cfg.warm_reservoir ? st->res_seen : st->cfg.warm_reservoir;
  if (fill < st->D.C) {   // fewer residuals than codewords: no codebooks, the state runs on without residual statistics
    st->launches += launch_or_u32(st->V.err, PKV_ERR_WARMUP_SHORT, st->stream);
    PKV_CUDA(cudaGetLastError());
    return PROTOKV_OK;
  }
  st->launches += launch_kmeans(st->D, st->H, st->V, st->cb_store_k, st->cb_store_v, (long long)fill, st->stream);
  st->launches += launch_codebook_copy(st->D, st->V, st->cb_store_k, st->cb_store_v, st->stream);
  PKV_CUDA(cudaGetLastError());
  st->V.cbk = st->cb_store_k; st->V.cbv = st->cb_store_v;     // from now on Alg. 1 l.13 updates the histograms
  st->codes_valid = false;
  return PROTOKV_OK;
}

int protokv_synthesize(protokv_state* st) {
  if (!st) return fail(PROTOKV_EINVAL, "NULL state");
  if (st->poisoned) return fail(PROTOKV_ESTATE, "an earlier launch failure left this state inconsistent; destroy it");
  DeviceGuard dg(st);
  {
    StageTimer tm(st, PROTOKV_STAGE_SYNTH);
    if (st->H.flags & PROTOKV_VAR_ALLOC) {   // D.3: shares S_k first (they move the code rows), then every prototype's modes
      st->launches += launch_allocation(st->D, st->H, st->V, st->n_act, st->stream);
      st->launches += launch_synthesis_var(st->D, st->H, st->V, st->n_act, st->stream);
    } else {
      st->launches += launch_synthesis(st->D, st->H, st->V, st->n_act, st->epoch, st->dirty_bound, st->sm_count, st->stream);
    }
  }
  PKV_CUDA(cudaGetLastError());
  st->epoch += 1;
  st->dirty_bound = 0;
  st->codes_valid = true;
  return PROTOKV_OK;
}

int protokv_query_attention_ex(protokv_state* st, const void* Q, int32_t n_q, int32_t layer_begin,
                               int32_t layer_count, void* out, float* lse, int32_t run_synthesis) {
  if (!st) return fail(PROTOKV_EINVAL, "NULL argument");
  return protokv_query_attention_at(st, Q, n_q, layer_begin, layer_count, out, lse, run_synthesis,
                                    (int64_t)st->H.pos0 + st->frames * st->D.T);
}

int protokv_query_attention_at(protokv_state* st, const void* Q, int32_t n_q, int32_t layer_begin, int32_t layer_count,
                               void* out, float* lse, int32_t run_synthesis, int64_t q_pos0) {
  if (!st || !Q || !out) return fail(PROTOKV_EINVAL, "NULL argument");
  if (st->poisoned) return fail(PROTOKV_ESTATE, "an earlier launch failure left this state inconsistent; destroy it");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  if (n_q < 1 || n_q > D.Nq) return fail(PROTOKV_EINVAL, "n_q %d outside [1, %d]", n_q, D.Nq);
  if (layer_begin < 0 || layer_count < 1 || layer_begin + layer_count > D.L)
    return fail(PROTOKV_EINVAL, "layer range [%d, %d) outside [0, %d)", layer_begin, layer_begin + layer_count, D.L);
  const bool far = !(st->H.flags & PROTOKV_NEAR_ONLY);
  if (far) {
    if (run_synthesis) {
      if (!st->codes_valid) {       // nothing changed since the last synthesis otherwise
        const int rc = protokv_synthesize(st);
        if (rc != PROTOKV_OK) return rc;
      }
    } else if (!st->codes_valid) {
      return fail(PROTOKV_ESTATE, "run_synthesis = 0 but no synthesis result is valid for the current state");
    }
  }
  AttnArgs A{};
  A.Q = Q; A.out = out; A.lse = lse;
  A.q_pos0 = (long long)q_pos0; A.frames = st->frames;
  A.n_q = n_q; A.layer_begin = layer_begin; A.layer_count = layer_count;
  const int64_t held = st->frames < D.Wf ? st->frames : D.Wf;
  A.n_near = (int)(held * D.T);
  A.n_act = st->n_act;
  A.nsplit = st->nsplit;
  {
    StageTimer tm(st, PROTOKV_STAGE_ATTN);
    if (st->use_decode_attn && decode_attention_supported(D, n_q) && (uintptr_t)Q % 16 == 0) {
      int ns = 1;
      st->launches += launch_attention_decode(D, st->H, st->V, A, st->sm_count, st->stream, &ns);
      A.nsplit = ns;
      st->launches += launch_attention_combine_bf16_128(D, st->V, A, !(st->cfg.flags & PROTOKV_SERIAL_LAUNCH), st->stream);
    } else if (st->use_decode_rope && (uintptr_t)Q % 16 == 0) {
      int ns = 1;
      if (st->H.flags & PROTOKV_ROPE) st->launches += launch_rope_tables(D, st->H, st->V, A, st->stream);
      st->launches += launch_attention_decode2(D, st->H, st->V, A, st->sm_count, st->stream, &ns);
      A.nsplit = ns;
      st->launches += launch_attention_combine_bf16_128(D, st->V, A, !(st->cfg.flags & PROTOKV_SERIAL_LAUNCH), st->stream);
    } else if (st->use_decode2 && decode2_attention_supported(D, n_q) && (uintptr_t)Q % 16 == 0) {
      int ns = 1;
      st->launches += launch_attention_decode2(D, st->H, st->V, A, st->sm_count, st->stream, &ns);
      A.nsplit = ns;
      st->launches += launch_attention_combine_bf16_128(D, st->V, A, !(st->cfg.flags & PROTOKV_SERIAL_LAUNCH), st->stream);
    } else if (st->use_tc_attn && (uintptr_t)Q % 16 == 0 && (uintptr_t)out % 8 == 0) {
      const int nl = launch_attention_tc(D, st->H, st->V, A, st->maps, st->sm_count, st->stream);
      if (nl < 0) return fail(PROTOKV_ECUDA, "cuTensorMapEncodeTiled failed for Q");
      st->launches += nl;
    } else {
      if (st->H.flags & PROTOKV_ROPE) st->launches += launch_rope_tables(D, st->H, st->V, A, st->stream);
      st->launches += launch_attention_simt(D, st->H, st->V, A, st->stream);
    }
  }
  PKV_CUDA(cudaGetLastError());
  return PROTOKV_OK;
}

size_t protokv_static_scratch_bytes(void) { return static_scratch_bytes(); }

int protokv_query_attention_static(protokv_state* st, const void* Q, int32_t n_q, int32_t layer_begin, int32_t layer_count,
                                   void* out, float* lse, int32_t run_synthesis) {
  if (!st || !Q || !out) return fail(PROTOKV_EINVAL, "NULL argument");
  if (st->poisoned) return fail(PROTOKV_ESTATE, "an earlier launch failure left this state inconsistent; destroy it");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  if (n_q < 1 || n_q > D.Nq) return fail(PROTOKV_EINVAL, "n_q %d outside [1, %d]", n_q, D.Nq);
  if (layer_begin < 0 || layer_count < 1 || layer_begin + layer_count > D.L)
    return fail(PROTOKV_EINVAL, "layer range [%d, %d) outside [0, %d)", layer_begin, layer_begin + layer_count, D.L);
  // the size check comes first: a query that does not fit leaves the state (codes, epoch) untouched
  const size_t need = (size_t)D.NS * layer_count * D.Hkv * n_q * D.group * (D.d + 2) * sizeof(float);
  if (need > static_scratch_bytes())
    return fail(PROTOKV_EUNSUPPORTED, "query of %d tokens x %d layers needs %zu bytes of partials; the static scratch holds "
                "%zu (use protokv_query_attention_ex, whose partials live in the workspace)", n_q, layer_count, need,
                static_scratch_bytes());
  if (!(st->H.flags & PROTOKV_NEAR_ONLY)) {
    if (run_synthesis) {
      if (!st->codes_valid) {
        const int rc = protokv_synthesize(st);
        if (rc != PROTOKV_OK) return rc;
      }
    } else if (!st->codes_valid) {
      return fail(PROTOKV_ESTATE, "run_synthesis = 0 but no synthesis result is valid for the current state");
    }
  }
  AttnArgs A{};
  A.Q = Q; A.out = out; A.lse = lse;
  A.q_pos0 = (long long)st->H.pos0 + st->frames * D.T; A.frames = st->frames;
  A.n_q = n_q; A.layer_begin = layer_begin; A.layer_count = layer_count;
  const int64_t held = st->frames < D.Wf ? st->frames : D.Wf;
  A.n_near = (int)(held * D.T);
  A.n_act = st->n_act;
  size_t nb = 0;
  cudaError_t ce = cudaSuccess;
  int nl;
  {
    StageTimer tm(st, PROTOKV_STAGE_ATTN);
    nl = launch_attention_static(D, st->H, st->V, A, st->sm_count, st->stream, &nb, &ce);
  }
  if (nl == -1) return fail(PROTOKV_EUNSUPPORTED, "query needs %zu bytes of partials; the static scratch holds %zu", nb, static_scratch_bytes());
  if (nl == -2) return fail(PROTOKV_ECUDA, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(ce));
  st->launches += nl;
  PKV_CUDA(cudaGetLastError());
  return PROTOKV_OK;
}

int protokv_query_attention(protokv_state* st, const void* Q, void* out) {
  if (!st) return fail(PROTOKV_EINVAL, "NULL state");
  return protokv_query_attention_ex(st, Q, st->D.Nq, 0, st->D.L, out, nullptr, 1);
}

static int ensure_copy_stream(protokv_state* st);

int protokv_append_frame_host(protokv_state* st, const void* K, const void* V, const float* grid_pos) {
  if (!st || !K || !V || !grid_pos) return fail(PROTOKV_EINVAL, "NULL argument");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  const size_t frame = (size_t)D.NS * D.L * D.T * D.Hkv * D.d * (D.bf16 ? 2 : 4);
  {
    const int rc0 = ensure_copy_stream(st);
    if (rc0 != PROTOKV_OK) return rc0;
  }
  // the staging buffers are free once the previous host-variant append has consumed them
  if (st->appended_pending) PKV_CUDA(cudaStreamWaitEvent(st->copy_stream, st->ev_appended, 0));
  PKV_CUDA(cudaMemcpyAsync(st->V.stageK, K, frame, cudaMemcpyHostToDevice, st->copy_stream));
  PKV_CUDA(cudaMemcpyAsync(st->V.stageV, V, frame, cudaMemcpyHostToDevice, st->copy_stream));
  PKV_CUDA(cudaMemcpyAsync(st->V.stageS, grid_pos, (size_t)D.NS * D.T * 8, cudaMemcpyHostToDevice, st->copy_stream));
  PKV_CUDA(cudaEventRecord(st->ev_copied, st->copy_stream));
  const int rc = append_frame_impl(st, st->V.stageK, st->V.stageV, st->V.stageS, st->ev_copied);
  if (rc != PROTOKV_OK) return rc;
  PKV_CUDA(cudaEventRecord(st->ev_appended, st->stream));
  st->appended_pending = true;
  return PROTOKV_OK;
}

static int ensure_copy_stream(protokv_state* st) {
  if (st->copy_stream) return PROTOKV_OK;
  PKV_CUDA(cudaStreamCreateWithFlags(&st->copy_stream, cudaStreamNonBlocking));
  PKV_CUDA(cudaEventCreateWithFlags(&st->ev_copied, cudaEventDisableTiming));
  PKV_CUDA(cudaEventCreateWithFlags(&st->ev_appended, cudaEventDisableTiming));
  return PROTOKV_OK;
}

int protokv_query_attention_host(protokv_state* st, const void* Q, void* out) {
  if (!st || !Q || !out) return fail(PROTOKV_EINVAL, "NULL argument");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  const size_t qbytes = (size_t)D.NS * D.L * D.Nq * D.Hq * D.d * (D.bf16 ? 2 : 4);
  int rc = ensure_copy_stream(st);
  if (rc != PROTOKV_OK) return rc;
  // Q travels on the copy stream while the synthesis (which does not need it) runs; the previous query's attention has
  // finished with the staging buffer (this call synchronises before it returns)
  PKV_CUDA(cudaMemcpyAsync(st->V.stageQ, Q, qbytes, cudaMemcpyHostToDevice, st->copy_stream));
  PKV_CUDA(cudaEventRecord(st->ev_copied, st->copy_stream));
  if (!(st->H.flags & PROTOKV_NEAR_ONLY) && !st->codes_valid) {
    rc = protokv_synthesize(st);
    if (rc != PROTOKV_OK) return rc;
  }
  PKV_CUDA(cudaStreamWaitEvent(st->stream, st->ev_copied, 0));
  rc = protokv_query_attention(st, st->V.stageQ, st->V.stageO);
  if (rc != PROTOKV_OK) return rc;
  PKV_CUDA(cudaMemcpyAsync(out, st->V.stageO, qbytes, cudaMemcpyDeviceToHost, st->stream));
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  return PROTOKV_OK;
}

int64_t protokv_frames_seen(const protokv_state* st) { return st ? st->frames : -1; }
int64_t protokv_kernel_launches(const protokv_state* st) { return st ? st->launches : -1; }

int protokv_maintenance_counters(protokv_state* st, int64_t* counts) {
  if (!st || !counts) return fail(PROTOKV_EINVAL, "NULL argument");
  DeviceGuard dg(st);
  PKV_CUDA(cudaMemcpyAsync(counts, st->V.mcount, 3 * sizeof(int64_t), cudaMemcpyDeviceToHost, st->stream));
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  return PROTOKV_OK;
}

int protokv_error_flags(protokv_state* st, uint32_t* flags, int32_t clear) {
  if (!st || !flags) return fail(PROTOKV_EINVAL, "NULL argument");
  DeviceGuard dg(st);
  PKV_CUDA(cudaMemcpyAsync(flags, st->V.err, 4, cudaMemcpyDeviceToHost, st->stream));
  if (clear) PKV_CUDA(cudaMemsetAsync(st->V.err, 0, 4, st->stream));
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  return PROTOKV_OK;
}

const char* protokv_stage_impl(const protokv_state* st, int32_t stage) {
  if (!st) return "none";
  if (stage == 0) return st->use_tc_assign ? "tcgen05" : "simt";
  if (stage == 1) return st->use_tc_attn ? "tcgen05" : (st->use_decode_rope ? "mma.sync register-resident (blocks)" : "simt");
  if (stage == 2)
    return st->use_decode_attn ? "mma.sync split-KV"
           : (st->use_decode2 ? "mma.sync register-resident"
              : (st->use_decode_rope ? "mma.sync register-resident (blocks)" : (st->use_tc_attn ? "tcgen05" : "simt")));
  return "none";
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------
// Parity / debug surface (not on the timed path): host views of the state.  All of these synchronise.
// ---------------------------------------------------------------------------------------------------------
static int check_bank(const protokv_state* st, int32_t bank) {
  if (!st) return fail(PROTOKV_EINVAL, "NULL state");
  if (bank < 0 || bank >= st->D.B) return fail(PROTOKV_EINVAL, "bank %d outside [0, %d)", bank, st->D.B);
  return PROTOKV_OK;
}

static inline float bf16_to_f32(uint16_t h) {
  uint32_t u = (uint32_t)h << 16;
  float f;
  memcpy(&f, &u, 4);
  return f;
}

extern "C" {

int protokv_export_state(protokv_state* st, int32_t bank, const protokv_bank_view* v) {
  int rc = check_bank(st, bank);
  if (rc) return rc;
  if (!v) return fail(PROTOKV_EINVAL, "NULL view");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  const Dev& V = st->V;
  const size_t K = D.K, o = (size_t)bank * K;
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  if (v->c) PKV_CUDA(cudaMemcpy(v->c, V.c + o * D.d, K * D.d * 4, cudaMemcpyDeviceToHost));
  if (v->p) PKV_CUDA(cudaMemcpy(v->p, V.p + o * D.d, K * D.d * 4, cudaMemcpyDeviceToHost));
  if (v->n) PKV_CUDA(cudaMemcpy(v->n, V.n + o, K * 4, cudaMemcpyDeviceToHost));
  if (v->mu) PKV_CUDA(cudaMemcpy(v->mu, V.mu + o * 2, K * 8, cudaMemcpyDeviceToHost));
  if (v->sigma) PKV_CUDA(cudaMemcpy(v->sigma, V.sigma + o * 3, K * 12, cudaMemcpyDeviceToHost));
  if (v->tau) PKV_CUDA(cudaMemcpy(v->tau, V.tau + o, K * 4, cudaMemcpyDeviceToHost));
  if (v->pos) PKV_CUDA(cudaMemcpy(v->pos, V.pos + o, K * 8, cudaMemcpyDeviceToHost));
  if (v->nres) PKV_CUDA(cudaMemcpy(v->nres, V.nres + o, K * 4, cudaMemcpyDeviceToHost));
  if (v->pos_first) PKV_CUDA(cudaMemcpy(v->pos_first, V.pos_first + o, K * 8, cudaMemcpyDeviceToHost));
  if (v->pos_sum) PKV_CUDA(cudaMemcpy(v->pos_sum, V.pos_sum + o, K * 8, cudaMemcpyDeviceToHost));
  if (v->pos_cnt) PKV_CUDA(cudaMemcpy(v->pos_cnt, V.pos_cnt + o, K * 4, cudaMemcpyDeviceToHost));
  const size_t gc = (size_t)D.G * D.C * 4;
  if (v->hist_k) PKV_CUDA(cudaMemcpy2D(v->hist_k, gc, V.hist + o * 2 * D.G * D.C, 2 * gc, gc, K, cudaMemcpyDeviceToHost));
  if (v->hist_v)
    PKV_CUDA(cudaMemcpy2D(v->hist_v, gc, V.hist + o * 2 * D.G * D.C + D.G * D.C, 2 * gc, gc, K, cudaMemcpyDeviceToHost));
  if (v->active)
    for (int k = 0; k < D.K; ++k) v->active[k] = k < st->n_act ? 1 : 0;
  return PROTOKV_OK;
}

int protokv_import_state(protokv_state* st, int32_t bank, const protokv_bank_view* v) {
  int rc = check_bank(st, bank);
  if (rc) return rc;
  if (!v) return fail(PROTOKV_EINVAL, "NULL view");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  const Dev& V = st->V;
  const size_t K = D.K, o = (size_t)bank * K;
  if (v->active) {   // the active set must be the prefix this state already has (slot fill is data-independent)
    int na = 0;
    while (na < D.K && v->active[na]) ++na;
    for (int k = na; k < D.K; ++k)
      if (v->active[k]) return fail(PROTOKV_EINVAL, "active set is not a prefix");
    if (na != st->n_act) return fail(PROTOKV_EINVAL, "imported active count %d != state's %d", na, st->n_act);
  }
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  if (v->c) PKV_CUDA(cudaMemcpy(V.c + o * D.d, v->c, K * D.d * 4, cudaMemcpyHostToDevice));
  if (v->p) PKV_CUDA(cudaMemcpy(V.p + o * D.d, v->p, K * D.d * 4, cudaMemcpyHostToDevice));
  if (v->n) PKV_CUDA(cudaMemcpy(V.n + o, v->n, K * 4, cudaMemcpyHostToDevice));
  if (v->mu) PKV_CUDA(cudaMemcpy(V.mu + o * 2, v->mu, K * 8, cudaMemcpyHostToDevice));
  if (v->sigma) PKV_CUDA(cudaMemcpy(V.sigma + o * 3, v->sigma, K * 12, cudaMemcpyHostToDevice));
  if (v->tau) PKV_CUDA(cudaMemcpy(V.tau + o, v->tau, K * 4, cudaMemcpyHostToDevice));
  if (v->pos) PKV_CUDA(cudaMemcpy(V.pos + o, v->pos, K * 8, cudaMemcpyHostToDevice));
  if (v->nres) PKV_CUDA(cudaMemcpy(V.nres + o, v->nres, K * 4, cudaMemcpyHostToDevice));
  if (v->pos_first) PKV_CUDA(cudaMemcpy(V.pos_first + o, v->pos_first, K * 8, cudaMemcpyHostToDevice));
  if (v->pos_sum) PKV_CUDA(cudaMemcpy(V.pos_sum + o, v->pos_sum, K * 8, cudaMemcpyHostToDevice));
  if (v->pos_cnt) PKV_CUDA(cudaMemcpy(V.pos_cnt + o, v->pos_cnt, K * 4, cudaMemcpyHostToDevice));
  const size_t gc = (size_t)D.G * D.C * 4;
  if (v->hist_k) PKV_CUDA(cudaMemcpy2D(V.hist + o * 2 * D.G * D.C, 2 * gc, v->hist_k, gc, gc, K, cudaMemcpyHostToDevice));
  if (v->hist_v)
    PKV_CUDA(cudaMemcpy2D(V.hist + o * 2 * D.G * D.C + D.G * D.C, 2 * gc, v->hist_v, gc, gc, K, cudaMemcpyHostToDevice));
  st->launches += launch_refresh_derived(D, st->H, V, bank, st->epoch, st->stream);
  PKV_CUDA(cudaGetLastError());
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  st->codes_valid = false;
  st->dirty_bound = D.K;
  st->maint_full = true;
  return PROTOKV_OK;
}

int protokv_export_ring(protokv_state* st, int32_t bank, float* K, float* Vv, float* s, int32_t* frame_index,
                        int32_t* n_frames) {
  int rc = check_bank(st, bank);
  if (rc) return rc;
  DeviceGuard dg(st);
  const Dims& D = st->D;
  const int held = (int)(st->frames < D.Wf ? st->frames : D.Wf);
  if (n_frames) *n_frames = held;
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  const size_t fe = (size_t)D.T * D.d, elt = D.bf16 ? 2 : 4;
  const int stream_idx = bank / (D.L * D.Hkv);
  std::vector<unsigned char> tmp(fe * elt);
  for (int i = 0; i < held; ++i) {
    const int64_t f = st->frames - held + i;
    const int slot = (int)(f % D.Wf);
    if (frame_index) frame_index[i] = (int32_t)f;
    for (int kv = 0; kv < 2; ++kv) {
      float* dst = kv ? Vv : K;
      if (!dst) continue;
      const char* src = (const char*)(kv ? st->V.ringV : st->V.ringK) + (((size_t)bank * D.Wf + slot) * fe) * elt;
      if (D.bf16) {
        PKV_CUDA(cudaMemcpy(tmp.data(), src, fe * 2, cudaMemcpyDeviceToHost));
        const uint16_t* h = (const uint16_t*)tmp.data();
        for (size_t e = 0; e < fe; ++e) dst[i * fe + e] = bf16_to_f32(h[e]);
      } else {
        PKV_CUDA(cudaMemcpy(dst + i * fe, src, fe * 4, cudaMemcpyDeviceToHost));
      }
    }
    if (s)
      PKV_CUDA(cudaMemcpy(s + (size_t)i * D.T * 2, st->V.ringS + ((size_t)stream_idx * D.Wf + slot) * D.T * 2,
                          (size_t)D.T * 8, cudaMemcpyDeviceToHost));
  }
  return PROTOKV_OK;
}

int protokv_export_codes(protokv_state* st, int32_t bank, uint8_t* codes_k, uint8_t* codes_v, uint8_t* kind) {
  int rc = check_bank(st, bank);
  if (rc) return rc;
  if (!st->codes_valid) return fail(PROTOKV_ESTATE, "no synthesis result for the current state");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  std::vector<uint32_t> tmp((size_t)D.K * D.S);
  const bool var = st->V.scount != nullptr;                 // D.3: ragged rows, exported as [k_max][s_cap][G]
  const int smax = var ? st->H.s_cap : D.S;
  std::vector<int> cnt, off;
  if (var) {
    cnt.resize(D.K); off.resize(D.K + 1);
    PKV_CUDA(cudaMemcpy(cnt.data(), st->V.scount + (size_t)bank * D.K, (size_t)D.K * 4, cudaMemcpyDeviceToHost));
    PKV_CUDA(cudaMemcpy(off.data(), st->V.soff + (size_t)bank * (D.K + 1), (size_t)(D.K + 1) * 4, cudaMemcpyDeviceToHost));
  }
  for (int kv = 0; kv < 2; ++kv) {
    uint8_t* dst = kv ? codes_v : codes_k;
    if (!dst) continue;
    PKV_CUDA(cudaMemcpy(tmp.data(), (kv ? st->V.codesV : st->V.codesK) + (size_t)bank * D.K * D.S, tmp.size() * 4,
                        cudaMemcpyDeviceToHost));
    if (var) {
      memset(dst, 0, (size_t)D.K * smax * D.G);
      for (int k = 0; k < D.K; ++k)
        for (int s2 = 0; s2 < cnt[k]; ++s2)
          for (int g = 0; g < D.G; ++g)
            dst[((size_t)k * smax + s2) * D.G + g] = (uint8_t)((tmp[(size_t)off[k] + s2] >> (4 * g)) & 15u);
      continue;
    }
    for (size_t e = 0; e < tmp.size(); ++e)
      for (int g = 0; g < D.G; ++g) dst[e * D.G + g] = (uint8_t)((tmp[e] >> (4 * g)) & 15u);
  }
  if (kind) PKV_CUDA(cudaMemcpy(kind, st->V.kind + (size_t)bank * D.K, D.K, cudaMemcpyDeviceToHost));
  return PROTOKV_OK;
}

int protokv_import_codes(protokv_state* st, int32_t bank, const uint8_t* codes_k, const uint8_t* codes_v) {
  int rc = check_bank(st, bank);
  if (rc) return rc;
  if (!st->codes_valid) return fail(PROTOKV_ESTATE, "run protokv_synthesize first (kind[] comes from it)");
  if (st->V.scount) return fail(PROTOKV_EUNSUPPORTED, "import_codes is not available with PROTOKV_VAR_ALLOC");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  std::vector<uint32_t> tmp((size_t)D.K * D.S);
  for (int kv = 0; kv < 2; ++kv) {
    const uint8_t* src = kv ? codes_v : codes_k;
    if (!src) continue;
    for (size_t e = 0; e < tmp.size(); ++e) {
      uint32_t w = 0;
      for (int g = 0; g < D.G; ++g) {
        if (src[e * D.G + g] >= D.C) return fail(PROTOKV_EINVAL, "code out of range");
        w |= (uint32_t)src[e * D.G + g] << (4 * g);
      }
      tmp[e] = w;
    }
    PKV_CUDA(cudaMemcpy((kv ? st->V.codesV : st->V.codesK) + (size_t)bank * D.K * D.S, tmp.data(), tmp.size() * 4,
                        cudaMemcpyHostToDevice));
  }
  // Forced codes last until the next synthesis: the whole bank is stamped with the epoch the next synthesis decodes,
  // so that it re-derives every tuple from the histograms instead of keeping forced ones on untouched prototypes.
  st->launches += launch_fill_u32(st->V.dirty + (size_t)bank * D.K, (uint32_t)st->epoch, (size_t)D.K, st->stream);
  st->dirty_bound = D.K;
  PKV_CUDA(cudaGetLastError());
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  return PROTOKV_OK;
}

int protokv_last_frame_trace(protokv_state* st, int32_t* assign, float* best, uint8_t* codes_k, uint8_t* codes_v,
                             int32_t* n_fill, int32_t* evicted_frame) {
  if (!st) return fail(PROTOKV_EINVAL, "NULL state");
  if (st->frames == 0) return fail(PROTOKV_ESTATE, "no frame appended yet");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  if (n_fill) *n_fill = st->last_n_fill;
  if (evicted_frame) *evicted_frame = st->last_ev_frame;
  const size_t BT = (size_t)D.B * D.T;
  if (st->last_ev_frame < 0) {
    if (assign) for (size_t i = 0; i < BT; ++i) assign[i] = -1;
    if (best) memset(best, 0, BT * 4);
    if (codes_k) memset(codes_k, 255, BT * D.G);
    if (codes_v) memset(codes_v, 255, BT * D.G);
    return PROTOKV_OK;
  }
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  if (assign) PKV_CUDA(cudaMemcpy(assign, st->V.assign, BT * 4, cudaMemcpyDeviceToHost));
  if (best) PKV_CUDA(cudaMemcpy(best, st->V.best, BT * 4, cudaMemcpyDeviceToHost));
  if (st->V.cbk) {
    if (codes_k) PKV_CUDA(cudaMemcpy(codes_k, st->V.tcodeK, BT * D.G, cudaMemcpyDeviceToHost));
    if (codes_v) PKV_CUDA(cudaMemcpy(codes_v, st->V.tcodeV, BT * D.G, cudaMemcpyDeviceToHost));
  } else {
    if (codes_k) memset(codes_k, 255, BT * D.G);
    if (codes_v) memset(codes_v, 255, BT * D.G);
  }
  return PROTOKV_OK;
}

int protokv_export_reservoir(protokv_state* st, int32_t bank, float* res_k, float* res_v, int64_t* fill, int64_t* seen) {
  int rc = check_bank(st, bank);
  if (rc) return rc;
  if (!st->warm) return fail(PROTOKV_ESTATE, "the state was created without PROTOKV_WARMUP");
  DeviceGuard dg(st);
  const int64_t n = st->res_seen < st->cfg.warm_reservoir ? st->res_seen : st->cfg.warm_reservoir;
  if (fill) *fill = n;
  if (seen) *seen = st->res_seen;
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  const size_t off = (size_t)bank * st->cfg.warm_reservoir * st->D.d, bytes = (size_t)n * st->D.d * 4;
  if (res_k && n) PKV_CUDA(cudaMemcpy(res_k, st->V.resK + off, bytes, cudaMemcpyDeviceToHost));
  if (res_v && n) PKV_CUDA(cudaMemcpy(res_v, st->V.resV + off, bytes, cudaMemcpyDeviceToHost));
  return PROTOKV_OK;
}

int protokv_import_reservoir(protokv_state* st, int32_t bank, const float* res_k, const float* res_v, int64_t n) {
  int rc = check_bank(st, bank);
  if (rc) return rc;
  if (!st->warm || st->trained) return fail(PROTOKV_ESTATE, "the state has no warm-up in progress");
  if (!res_k || !res_v || n < 0 || n > st->cfg.warm_reservoir) return fail(PROTOKV_EINVAL, "bad reservoir rows");
  DeviceGuard dg(st);
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  const size_t R = (size_t)st->cfg.warm_reservoir, off = (size_t)bank * R * st->D.d, bytes = (size_t)n * st->D.d * 4;
  if (n) {
    PKV_CUDA(cudaMemcpy(st->V.resK + off, res_k, bytes, cudaMemcpyHostToDevice));
    PKV_CUDA(cudaMemcpy(st->V.resV + off, res_v, bytes, cudaMemcpyHostToDevice));
  }
  // the claim words order residual indices; the count restarts at n for every bank
  PKV_CUDA(cudaMemset(st->V.resV + (size_t)st->D.B * R * st->D.d, 0, (size_t)st->D.B * R * 8));
  st->res_seen = n;
  return PROTOKV_OK;
}

int protokv_export_codebooks(protokv_state* st, int32_t bank, float* codebook_k, float* codebook_v) {
  int rc = check_bank(st, bank);
  if (rc) return rc;
  if (!st->V.cbk) return fail(PROTOKV_ESTATE, "the state has no codebooks (none given, or the warm-up has not ended)");
  DeviceGuard dg(st);
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  const size_t n = (size_t)st->D.G * st->D.C * st->D.sub;
  if (codebook_k) PKV_CUDA(cudaMemcpy(codebook_k, st->V.cbk + (size_t)bank * n, n * 4, cudaMemcpyDeviceToHost));
  if (codebook_v) PKV_CUDA(cudaMemcpy(codebook_v, st->V.cbv + (size_t)bank * n, n * 4, cudaMemcpyDeviceToHost));
  return PROTOKV_OK;
}

int protokv_export_allocation(protokv_state* st, int32_t bank, int32_t* s_count, int64_t* variance_fx) {
  int rc = check_bank(st, bank);
  if (rc) return rc;
  if (!s_count) return fail(PROTOKV_EINVAL, "NULL s_count");
  if (!st->codes_valid) return fail(PROTOKV_ESTATE, "no synthesis result for the current state");
  DeviceGuard dg(st);
  const Dims& D = st->D;
  PKV_CUDA(cudaStreamSynchronize(st->stream));
  if (st->V.scount) {
    PKV_CUDA(cudaMemcpy(s_count, st->V.scount + (size_t)bank * D.K, (size_t)D.K * 4, cudaMemcpyDeviceToHost));
    if (variance_fx) PKV_CUDA(cudaMemcpy(variance_fx, st->V.varfx + (size_t)bank * D.K, (size_t)D.K * 8, cudaMemcpyDeviceToHost));
  } else {
    std::vector<uint8_t> kind(D.K);
    PKV_CUDA(cudaMemcpy(kind.data(), st->V.kind + (size_t)bank * D.K, D.K, cudaMemcpyDeviceToHost));
    for (int k = 0; k < D.K; ++k) { s_count[k] = kind[k] == 2 ? 0 : D.S; if (variance_fx) variance_fx[k] = 0; }
  }
  return PROTOKV_OK;
}

}  // extern "C"
