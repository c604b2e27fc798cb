/*
 * protokv.h -- C ABI of the B200-native (sm_100a) ProtoKV two-tier KV memory hot path.
 *
 * Paper: arxiv 2606.26762 ("PAPER.md" below = the extracted text of that paper).  One *bank* is the memory
 * of one (stream, layer, KV head): an exact near-window ring buffer B_near of the last W = near_frames * T
 * visual tokens and a fixed-capacity far prototype bank B_far = {Pi_k}, k < K_max,
 * Pi_k = (c_k, p_k, n_k, R_k, mu_k, Sigma_k, tau_k).  Banks are independent
 * (PAPER.md:L312); one state object holds n_streams * n_layers * n_kv_heads of them and every call processes
 * all of them in batched kernel launches.
 *
 * Every step of Alg. 1 / 3 / 4 runs in hand-written CUDA kernels on the caller's stream.  The one piece of the
 * method's arithmetic evaluated on the host is a constant table: protokv_create fills the 4,096 numerators
 * log(h + pq_eps), h = 0..4095, of Eq. 3 with the host's libm and copies them to the device, where the
 * synthesis kernel looks them up (larger counts are evaluated by the kernel itself).  There is no CPU fallback: on a
 * machine without an sm_100 device protokv_create fails with PROTOKV_EUNSUPPORTED.
 *
 * Conventions
 *   - "device"/"host" says where a pointer must live.  Tensor arguments are caller-owned and contiguous.
 *   - Calls enqueue work on cfg.cuda_stream and return without synchronising unless stated otherwise.
 *     Arguments must stay valid until the stream has passed the call's work.
 *   - Every function returns a protokv_status (0 = OK) unless stated otherwise; argument, shape and capability
 *     errors are detected before any launch and leave the state unchanged.  protokv_last_error() returns a
 *     thread-local message for the last failing call.  Nothing throws or aborts across this boundary.
 *   - A state is not thread-safe; distinct states are independent.
 *
 * Layouts (row-major, last index fastest), bank = (stream * n_layers + layer) * n_kv_heads + kv_head:
 *   K, V      [n_streams][n_layers][T][n_kv_heads][head_dim]     dtype cfg.dtype
 *   grid_pos  [n_streams][T][2]  fp32 normalised (x, y) of each token's cell in its frame
 *   Q, out    [n_streams][n_layers][n_query_tokens][n_q_heads][head_dim]   dtype cfg.dtype
 *   query head h reads the bank of KV head h / (n_q_heads / n_kv_heads)    (GQA)
 *   codebooks [n_streams][n_layers][n_kv_heads][G][C][head_dim / G]  fp32
 */
#ifndef PROTOKV_H_
#define PROTOKV_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct protokv_state protokv_state; /* opaque; owned by the library until protokv_destroy */

typedef enum {
  PROTOKV_OK = 0,
  PROTOKV_EINVAL = 1,       /* NULL pointer, bad shape, bad struct_size, index out of range */
  PROTOKV_EUNSUPPORTED = 2, /* valid request this build cannot run (head_dim, C > 16, no sm_100 device, ...) */
  PROTOKV_ENOMEM = 3,       /* workspace too small */
  PROTOKV_ECUDA = 4,        /* a CUDA call failed; text in protokv_last_error() */
  PROTOKV_ESTATE = 5        /* call not valid in the current state (e.g. trace before any eviction) */
} protokv_status;

typedef enum { PROTOKV_F32 = 0, PROTOKV_BF16 = 1 } protokv_dtype;

/* cfg.flags */
enum {
  PROTOKV_MAH_SQUARED = 1u,  /* use d_Mah^2 in Eq. 1 (alternative reading of PAPER.md:L93)              */
  PROTOKV_NO_MASS_BIAS = 2u, /* b_k = 0              (Table 2 "w/o mass bias", L180)            */
  PROTOKV_NO_RESIDUAL = 4u,  /* never update histograms => zero residuals (Table 2)               */
  PROTOKV_NEAR_ONLY = 8u,    /* attention over the near window only (L176)                              */
  PROTOKV_FAR_ONLY = 16u,    /* attention over pseudo-tokens only   (L177)                              */
  PROTOKV_FORCE_SIMT = 32u,  /* use the fp32 SIMT kernels even where a tcgen05 kernel exists (cross-check) */
  PROTOKV_DECODE_SPLITKV = 128u, /* serve queries of <= 16 rows per bank with the shared-memory split-KV mma.sync kernel
                                (csrc/decode_attention.cu): the first decode kernel, kept as a cross-check (167-183 us
                                on the C3 one-token query).  The default route for such queries is the register-resident
                                kernel of csrc/decode_attention2.cu (86 us); the 128-row tcgen05 kernel takes 161 us */
  PROTOKV_ROPE = 256u,       /* rotary position anchoring (D.1 L578-596; readings 28-31): K and Q
                                are given UN-ROTATED; the attention rotates near tokens at their stream positions, the S
                                pseudo-tokens of prototype k at its anchor and the query tokens at q_pos0 + i.  bf16 states
                                with head_dim 128 are served by the rotating variant of the register-resident kernel
                                (csrc/decode_attention2.cu; queries of any length run as 8-row blocks), other shapes by
                                the fp32 SIMT kernel; the tcgen05 prefill kernel has no rotation stage */
  PROTOKV_NO_DECODE_KERNEL = 4096u, /* serve queries of <= 16 rows per bank with the 128-row tcgen05 kernel instead of
                                the register-resident decode kernel (csrc/decode_attention2.cu, the default): cross-check */
  PROTOKV_WARMUP = 512u,     /* PQ codebook warm-up (readings 32-36): cfg.codebook_k/v are
                                ignored; the residuals (r^K, r^V) of the tokens absorbed during the first t_warm steps go
                                into a per-bank reservoir (Algorithm R, capacity warm_reservoir), no histogram is updated
                                meanwhile, and the append of frame t_warm - 1 ends with mini-batch k-means per subspace and
                                side (km_iters x km_batch samples) that writes the bank's codebooks, fixed thereafter */
  PROTOKV_WARMUP_MANUAL = 1024u, /* with PROTOKV_WARMUP: the training is started by protokv_train_codebooks instead */
  PROTOKV_VAR_ALLOC = 2048u, /* D.3 (readings 37-40): variance-aware pseudo-token counts
                                S_k = S_tot Var(H_k) / sum_j Var(H_j) under S_tot = k_max S, 1 <= S_k <= s_cap, recomputed by
                                every synthesis; bf16 states with head_dim 128 are served by the ragged variant of the
                                register-resident kernel (8-row blocks), other shapes by the fp32 SIMT kernel */
  PROTOKV_SERIAL_LAUNCH = 8192u, /* launch every kernel fully serialised.  By default the kernels of a call are chained
                                with programmatic dependent launch (score -> update -> ring append; synthesis -> attention
                                -> combine; decode kernel -> combine): each kernel's set-up and the loads of data that no
                                kernel of the chain writes run under its predecessor's tail.  Results are bit-identical;
                                the flag exists for measurement and as a cross-check */
  PROTOKV_MAINTENANCE = 64u  /* run Alg. 2 at the end of every append_frame that evicted a frame
                                (Alg. 1 l.15); off by default: north_star's path and its invariant "total mass = tokens
                                absorbed" exclude it (reading 19) */
};

typedef struct {
  uint32_t struct_size;   /* = sizeof(protokv_config); ABI versioning */
  int32_t n_streams, n_layers, n_q_heads, n_kv_heads, head_dim; /* head_dim in {64, 128}; n_q % n_kv == 0 */
  int32_t dtype;          /* protokv_dtype of K, V, Q, out */
  int32_t tokens_per_frame; /* T  */
  int32_t near_frames;    /* W_f: the near window holds W_f whole frames, W = W_f * T tokens */
  int32_t k_max;          /* prototype capacity per bank */
  int32_t n_query_tokens; /* N_q of protokv_query_attention */
  int32_t S, G, C, beam;  /* Table 5: 8, 8, 16, 32.  S <= 8, G <= 8, C <= 16, C^G >= S, beam >= S */
  float lambda_sp, lambda_idle; /* Eq. 1 weights: 0.1, 0.01 */
  int32_t t_idle;         /* T_idle in frames: 120 */
  float alpha, beta, eta; /* EMA rates of c, p and (mu, Sigma): 0.05 */
  float sigma_eps;        /* added to the diagonal of Sigma_k before inversion (reading 4): 1e-4 */
  float cos_eps;          /* lower bound of |K||c| in the cosine (reading 6): 1e-12 */
  double pq_eps;          /* epsilon of Eq. 3 (value not given in the paper): 1e-6 */
  uint32_t flags;
  float gamma;            /* Alg. 2 idle decay rate (Table 5: 0.05); used with PROTOKV_MAINTENANCE */
  float eps_k, eps_v;     /* Alg. 2 merge thresholds on |c_i - c_j|, |p_i - p_j| (Table 5: 0.20, 0.25) */
  double rope_theta;      /* rotary base (rotate-half convention, angle of pair (i, i + d/2) at position p = p theta^(-2i/d));
                             the paper fixes none: 1e6 (Qwen2-family backbones).  Used with PROTOKV_ROPE */
  int32_t rope_anchor;    /* D.1: 0 = most recent absorbed position (default), 1 = first, 2 = average */
  int64_t pos0;           /* stream position of token 0 of frame 0; token j of frame f sits at pos0 + f T + j */
  int32_t t_warm;         /* PROTOKV_WARMUP: warm-up length T_warm in streaming steps = frames (the paper gives no value, L478) */
  int32_t warm_reservoir; /* residual pairs the reservoir of a bank holds (<= 65536) */
  int32_t km_iters, km_batch; /* mini-batch k-means: iterations, samples drawn per iteration (km_batch <= 1024) */
  uint64_t km_seed;       /* bank b draws from the counter-based generator (SplitMix64 output function) seeded km_seed + b */
  int32_t s_cap;          /* PROTOKV_VAR_ALLOC: upper bound of S_k, <= beam and <= 32 */
  const float *codebook_k, *codebook_v; /* device; copied at create.  NULL => no residual statistics */
  void *workspace;        /* device memory from the caller, >= protokv_workspace_bytes(cfg), 256-byte aligned */
  size_t workspace_bytes;
  void *cuda_stream;      /* cudaStream_t of the caller (NULL = legacy default stream) */
} protokv_config;

/* Bytes of device workspace a state with this configuration needs: the two-tier state of PAPER.md:L300-312 (§A.1) --
 * B_near (ring of W = near_frames * T exact K, V rows per bank, L300) and B_far (k_max prototypes
 * (c, p, n, R, mu, Sigma, tau) per bank, L302-310, R = two G x C histograms + n_res) -- plus the per-frame scratch, the
 * derived copies the kernels stream and the host-variant staging buffers; constant in the
 * stream length (L81, L102).  0 if the configuration is invalid (protokv_last_error() says why).  Pointer fields of
 * cfg are ignored.  Host-only, no CUDA call. */
size_t protokv_workspace_bytes(const protokv_config *cfg);

/* Builds the empty state of PAPER.md:L300-312 inside cfg->workspace: empty near window, every prototype slot inactive
 * (L83: slots are opened by the first evicted tokens), codebooks copied from cfg (L312: fixed after warm-up; their
 * training is the caller's, reading 11).  The workspace is zeroed asynchronously on the stream.
 * The state is bound to the CUDA device that is current at this call; later calls may be made with any device
 * current.  NULL on failure (protokv_last_error()). */
protokv_state *protokv_create(const protokv_config *cfg);

/* Releases host-side resources (the paper's state lives entirely in the caller's workspace).  NULL is a no-op. */
void protokv_destroy(protokv_state *st);

/*
 * Alg. 1 for one frame of every bank, frame-synchronous reading (reading 1):
 * the frame is appended to the ring; if the ring was full its oldest frame (T tokens, in stored order) is
 * evicted and absorbed:  (A) while free slots remain each evicted token opens the lowest free slot (l.3-4, L83);
 * (B) the others are assigned by Eq. 1 (L93) against the bank as it stands after (A), lowest index on ties;
 * (C) Alg. 1 l.8-13 is replayed token by token in eviction order (EMA centres, mass, recency, spatial mean and
 * covariance, PQ residual histograms of the just-updated centres).  Alg. 1 l.15 (maintenance, Alg. 2)
 * runs only with PROTOKV_MAINTENANCE, once per frame after (C) and after the frame has entered the ring: idle
 * prototypes decay n <- floor((1 - gamma) n), pairs with |c_i - c_j| < eps_k and |p_i - p_j| < eps_v merge into the lower
 * index (mass-weighted c, p, mu; n, H, n_res summed; Sigma, tau, pos of the survivor kept), and every slot emptied by
 * decay or merging is re-initialised from the newest near-window tokens (readings 20, 24-27).
 * K, V, grid_pos: device.
 */
int protokv_append_frame(protokv_state *st, const void *K, const void *V, const float *grid_pos);

/*
 * Alg. 4: for every active prototype decode the top-S residual modes of H^K and H^V by
 * Alg. 3 / Eq. 3 (zero residuals when n_res = 0), then O = softmax(Q K~^T / sqrt(d) + b) V~ over
 * [near window || pseudo-tokens], b = log n_k on pseudo-tokens (Eq. 2/4) and 0 on near tokens; no mask.
 * Pseudo-tokens are built on chip and never written to HBM.  Q, out: device.  Does not modify the memory.
 */
int protokv_query_attention(protokv_state *st, const void *Q, void *out);

/* The same two calls with HOST buffers (pinned memory recommended): inputs are copied to the device and, for
 * the query, the result copied back.  The host-to-device copies run on a copy stream the library owns, next to the work
 * that does not need them (Eq. 1 scoring and the prototype update only read the evicted frame already in the ring; the
 * synthesis does not read Q); the state's stream waits for them before the ring append / the attention, so synchronising
 * cfg.cuda_stream still covers the whole call.  append returns without synchronising; the query variant synchronises
 * the stream before returning so `out` is ready. */
int protokv_append_frame_host(protokv_state *st, const void *K, const void *V, const float *grid_pos);
int protokv_query_attention_host(protokv_state *st, const void *Q, void *out);

/* Thread-local description of the last error returned on this thread ("" if none). */
const char *protokv_last_error(void);

/* ------------------------------------------------------------------------------------------------------ */
/* Parity / debug surface (not on the timed path).                                                          */
/* ------------------------------------------------------------------------------------------------------ */

/* Attention for n_q query tokens (<= cfg.n_query_tokens) of layers [layer_begin, layer_begin + layer_count):
 * Q, out [n_streams][layer_count][n_q][n_q_heads][head_dim] device; lse (optional, device)
 * [n_streams][layer_count][n_q][n_q_heads] fp32 natural-log-sum-exp of the logits.  run_synthesis = 0 reuses
 * the codes of the previous synthesis (or of protokv_import_codes). */
int protokv_query_attention_ex(protokv_state *st, const void *Q, int32_t n_q, int32_t layer_begin,
                               int32_t layer_count, void *out, float *lse, int32_t run_synthesis);

/* The same with the stream position of the first query token given explicitly (PROTOKV_ROPE; query token i is rotated
 * at q_pos0 + i).  protokv_query_attention(_ex) use q_pos0 = pos0 + frames_seen * T, the next stream position. */
int protokv_query_attention_at(protokv_state *st, const void *Q, int32_t n_q, int32_t layer_begin, int32_t layer_count,
                               void *out, float *lse, int32_t run_synthesis, int64_t q_pos0);

/* protokv_query_attention_ex for callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same arguments and the same result (Alg. 4; Eq. 4), computed by the fp32 SIMT
 * attention kernel whatever the state's default route is, with the split-context partials in a file-scope device array of
 * the library (csrc/static_scratch.cu) instead of the workspace.  The call and everything under it performs no cudaMalloc,
 * cudaFree or other allocating call.  The array holds protokv_static_scratch_bytes() = 8 MiB; every GPU that loads the
 * library holds it until the process exits.  A query needs n_streams * layer_count * n_kv_heads * n_q * (n_q_heads /
 * n_kv_heads) * (head_dim + 2) * 4 bytes per context split: one that does not fit with a single split returns
 * PROTOKV_EUNSUPPORTED and leaves the state unchanged (config 3's one-token query needs 0.4 MB, its 32-token query 13 MB).
 * The array is shared by every state and call on the GPU and keeps the last call's contents; nothing in it has to start at
 * zero (each call rewrites every partial it reads).  Calls that overlap on one GPU (different streams) RACE on it; calls
 * on one stream are ordered.  Q, out, lse: device, as for protokv_query_attention_ex; the stream is cfg.cuda_stream. */
int protokv_query_attention_static(protokv_state *st, const void *Q, int32_t n_q, int32_t layer_begin,
                                   int32_t layer_count, void *out, float *lse, int32_t run_synthesis);
size_t protokv_static_scratch_bytes(void);

/* Alg. 3 for every bank without the attention (timing / parity of the synthesis kernel alone). */
int protokv_synthesize(protokv_state *st);

/* Host views of one bank; NULL members are skipped.  Both calls synchronise the stream. */
typedef struct {
  float *c, *p;                 /* [k_max][head_dim] key / value centres                                  */
  int32_t *n;                   /* [k_max] mass                                                           */
  float *mu, *sigma;            /* [k_max][2]; [k_max][3] = (xx, xy, yy)                                  */
  int32_t *tau;                 /* [k_max] frame index of the last absorption (idle test)                 */
  int64_t *pos;                 /* [k_max] stream position of the last absorbed token (RoPE anchor, L126) */
  uint32_t *hist_k, *hist_v;    /* [k_max][G][C]                                                          */
  uint32_t *nres;               /* [k_max]                                                                */
  uint8_t *active;              /* [k_max]                                                                */
  int64_t *pos_first, *pos_sum; /* [k_max] D.1 anchors: position of the initialising token; sum of all absorbed positions */
  int32_t *pos_cnt;             /* [k_max] number of absorbed positions (average anchor = pos_sum / pos_cnt)           */
} protokv_bank_view;
int protokv_export_state(protokv_state *st, int32_t bank, const protokv_bank_view *host_dst);
int protokv_import_state(protokv_state *st, int32_t bank, const protokv_bank_view *host_src);

/* Near window of one bank in chronological order, as fp32 on the host: K, V [n][T][head_dim], s [n][T][2],
 * frame_index [n]; *n_frames receives n (<= near_frames).  NULL members are skipped.  Synchronises. */
int protokv_export_ring(protokv_state *st, int32_t bank, float *K, float *V, float *s, int32_t *frame_index,
                        int32_t *n_frames);

/* Result of the last synthesis for one bank, on the host: codes [k_max][S][G] (one code per byte) and
 * kind [k_max] (0 = decoded modes, 1 = zero residuals, 2 = slot not in the context).  Synchronises. */
int protokv_export_codes(protokv_state *st, int32_t bank, uint8_t *codes_k, uint8_t *codes_v, uint8_t *kind);
/* Overwrites the tuples of one bank (parity aid: attention with the checker's codes).  They stay in force until the
 * next synthesis, which re-decodes the whole bank from its histograms. */
int protokv_import_codes(protokv_state *st, int32_t bank, const uint8_t *codes_k, const uint8_t *codes_v);

/* What the last append_frame decided, all banks, on the host: assign [banks][T] (slot index; -1 if no frame
 * was evicted; -2 for a token without any finite Eq. 1 score, see protokv_error_flags), best [banks][T] (Eq. 1 score
 * of the choice; 0 for slot fills), codes_k/v [banks][T][G] (255 = no residual update); *n_fill = tokens per bank that
 * opened a new slot; *evicted_frame = index of the evicted frame or -1.  NULL members are skipped.  Synchronises.
 * The runner-up score is deliberately not part of the trace: the parity rule needs "the ORACLE's score of the GPU's
 * choice minus the oracle's best" (north_star's 1e-5 gap), which only the checker can evaluate, and the kernels keep
 * one running minimum per token (a second one would cost the epilogue a compare per score for no consumer). */
int protokv_last_frame_trace(protokv_state *st, int32_t *assign, float *best, uint8_t *codes_k,
                             uint8_t *codes_v, int32_t *n_fill, int32_t *evicted_frame);

/* Counters: frames appended so far; kernels launched by this state since create (bench's gpu_launches). */
int64_t protokv_frames_seen(const protokv_state *st);
int64_t protokv_kernel_launches(const protokv_state *st);

/* Sticky device-side error bits raised by the kernels since create (or the last clear); synchronises the stream.
 *   bit 0 (PROTOKV_ERRBIT_UNASSIGNED): an evicted token had no finite Eq. 1 score against any prototype (NaN / Inf in
 *   its key row or in the bank).  Eq. 1's argmin is undefined for it; the token is dropped (not absorbed, trace
 *   assign = -2) and the rest of the frame proceeds.  *flags (host) receives the bits; clear != 0 resets them. */
/*   bit 1 (PROTOKV_ERRBIT_MAINT_OVERFLOW): Alg. 2 met more merge candidates in one frame of one bank than its list holds
 *   (2,048); the excess pairs were not merged in that frame. */
/*   bit 2 (PROTOKV_ERRBIT_WARMUP_SHORT): the warm-up ended with fewer residuals than codewords (C) in the reservoir; no
 *   codebooks were trained and the state keeps running without residual statistics. */
enum { PROTOKV_ERRBIT_UNASSIGNED = 1u, PROTOKV_ERRBIT_MAINT_OVERFLOW = 2u, PROTOKV_ERRBIT_WARMUP_SHORT = 4u };
int protokv_error_flags(protokv_state *st, uint32_t *flags, int32_t clear);

/* What Alg. 2 has done since create, summed over all banks: counts[0] = mass removed by aging, counts[1] = prototypes
 * merged away, counts[2] = slots recycled (host, 3 entries).  Synchronises.  The generalised mass invariant reads
 * sum_k n_k = tokens absorbed - counts[0] + counts[2]. */
int protokv_maintenance_counters(protokv_state *st, int64_t *counts);

/* PQ codebook warm-up ("initialized via mini-batch k-means on a warm-up reservoir of residuals collected
 * during the first T_warm streaming steps, run separately for each subspace and for key/value ... kept fixed
 * thereafter"; PROTOKV_WARMUP states only).
 * protokv_train_codebooks ends the warm-up of every bank now: k-means on what the reservoirs hold, codebooks written,
 * histogram updates start with the next absorbed token.  Called by the library itself at the end of the append of frame
 * t_warm - 1 unless PROTOKV_WARMUP_MANUAL is set.  PROTOKV_ESTATE if the state has no warm-up or is already trained.
 * export/import_reservoir: rows [fill][head_dim] fp32 of r^K and r^V of one bank (host); *fill = rows held, *seen =
 * residuals offered so far; import overwrites the first n rows and sets both counts to n (parity aid).
 * export_codebooks: the bank's [G][C][head_dim / G] fp32 codebooks (host); PROTOKV_ESTATE if it has none.
 * All four synchronise. */
int protokv_train_codebooks(protokv_state *st);
int protokv_export_reservoir(protokv_state *st, int32_t bank, float *res_k, float *res_v, int64_t *fill, int64_t *seen);
int protokv_import_reservoir(protokv_state *st, int32_t bank, const float *res_k, const float *res_v, int64_t n);
int protokv_export_codebooks(protokv_state *st, int32_t bank, float *codebook_k, float *codebook_v);

/* D.3 (PROTOKV_VAR_ALLOC states): the pseudo-token counts S_k [k_max] (int32, host) and fixed-point variances
 * v_k = floor(Var(H_k) 2^20 + 1/2) [k_max] (int64, host; may be NULL) of one bank as of the last synthesis; with the
 * flag off S_k = S for every prototype in the context.  PROTOKV_ESTATE without a valid synthesis.  Synchronises. */
int protokv_export_allocation(protokv_state *st, int32_t bank, int32_t *s_count, int64_t *variance_fx);

/* Stage timing (measurement aid, off by default).  When enabled the library brackets every kernel group it launches
 * with CUDA events on the state's stream; protokv_profile_read synchronises the stream and returns, per stage, the
 * summed device time in milliseconds and the number of bracketed launches since the last enable, then resets.
 * ms_sum and launches hold PROTOKV_N_STAGES entries (host). */
enum {
  PROTOKV_STAGE_FILL = 0,    /* U2 slot fill                       */
  PROTOKV_STAGE_SCORE = 1,   /* U3 Eq. 1 scores + argmin           */
  PROTOKV_STAGE_UPDATE = 2,  /* U4-U6 segmenting, update, PQ hist  */
  PROTOKV_STAGE_APPEND = 3,  /* U1 ring append                     */
  PROTOKV_STAGE_SYNTH = 4,   /* Q1 synthesis                       */
  PROTOKV_STAGE_ATTN = 5,    /* Q2 fused attention (+ split combine) */
  PROTOKV_N_STAGES = 6
};
int protokv_profile_enable(protokv_state *st, int32_t on);
int protokv_profile_read(protokv_state *st, double *ms_sum, int64_t *launches);

/* Names the kernel variant each stage uses for this state, for reports: "simt", "tcgen05", "mma.sync register-resident"
 * (+ " (blocks)": the rotating / ragged 8-row-block variants), "mma.sync split-KV".  stage: 0 = assignment, 1 = attention (multi-token queries), 2 = attention of
 * decode-style queries (<= 16 rows per bank).  Returns a static string, never NULL. */
const char *protokv_stage_impl(const protokv_state *st, int32_t stage);

#ifdef __cplusplus
}
#endif
#endif /* PROTOKV_H_ */
