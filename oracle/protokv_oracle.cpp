// ProtoKV CPU ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, single-threaded restatement of the paper's hot path (PAPER.md = arxiv 2606.26762 text):
//   Alg. 1 streaming update   (Eq. 1 at L93)      -> append_frame_sync / append_frame_seq
//   Eq. 3 + Alg. 3 beam decode             -> decode_top_s
//   Alg. 4 decode + attention, Eq. 2/4 -> materialize / attention
//   Alg. 2 prototype maintenance (off unless FLAG_MAINTENANCE) -> maintain
//   PQ codebook warm-up (FLAG_WARMUP) -> reservoir_offer / kmeans_subspace / train_codebooks
//   D.3 variance-aware pseudo-token allocation (FLAG_VAR_ALLOC) -> variance_fx / allocate
// One object = one bank = one (stream, layer, KV head): banks are independent.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call this.
// It shares no code with paper_2606_26762_b200/ (the CUDA path) and must never be used by the product path.
//
// Arithmetic: state is fp32 (what is compared); every expression is evaluated in fp64 from the fp32
// state and rounded once.  Discrete decisions (argmin of Eq. 1, nearest PQ codeword) compare the
// fp32-rounded values, lowest index on exact ties.  Readings of silent/garbled points: DESIGN.md "Readings".
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): mass conservation; histogram row sums; T=1 frame-synchronous
// == sequential; forced replay; brute-force recomputation of the statistics from the assignment log (numpy);
// constant-stream closed forms; exact attention over the full history when K_max >= evicted tokens; a mass-m
// prototype == m duplicated tokens; torch SDPA on the materialised context; cosine nearest centroid; Euclidean
// special case of d_Mah; beam == brute-force top-S; closed forms after one absorption into a fresh slot (Sigma step
// with delta against the NEW mean, Alg. 1 l.11-12; residual taken AFTER the token's own EMA step, l.8-9 before l.13).
// Alg. 2 (tests/test_oracle_maintenance.py): generalised mass invariant, conservation of the mass-weighted sums under
// merging, closed form of the idle decay, gamma = eps = 0 == the plain path bit for bit, T = 1 sync == sequential.
// Rotary anchoring (FLAG_ROPE, tests/test_oracle_rope.py): rotated keys and attention against the rotate-half routine of
// the `transformers` package + torch SDPA, relative-position property (a common shift of all positions changes nothing),
// norm preservation, anchor fields (first / average / most recent) recomputed from the assignment log.
// PQ codebook warm-up (FLAG_WARMUP, tests/test_oracle_warmup.py): generator against the published
// SplitMix64 vector, reservoir against uniform sampling and numpy residuals, mini-batch k-means against the running-mean
// closed form, separated blobs and scikit-learn KMeans.  D.3 allocation (FLAG_VAR_ALLOC, tests/test_oracle_alloc.py;
// PAPER.md:L608-625): Var(H_k) against numpy's population variance, shares against hand-worked examples and invariants.
// What stays unpinned: the absolute values produced on the five configs ("parity unpinned" beyond those pins, see
// DESIGN.md).
#include <algorithm>
#include <array>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <deque>
#include <limits>
#include <vector>

namespace {

enum : uint32_t {
  FLAG_MAH_SQUARED = 1u,   // use d_Mah^2 instead of d_Mah (reading 4 alternative)
  FLAG_NO_MASS_BIAS = 2u,  // b_k = 0          (Table 2 "w/o mass bias")
  FLAG_NO_RESIDUAL = 4u,   // no histograms    (Table 2 "w/o residual stats", L179)
  FLAG_NEAR_ONLY = 8u,     // attention over the near window only (L176)
  FLAG_FAR_ONLY = 16u,     // attention over pseudo-tokens only   (L177)
  FLAG_ROPE = 256u,        // rotary position anchoring of L126 / D.1 (readings 28-31): K and Q are given un-rotated
  FLAG_MAINTENANCE = 64u,  // run Alg. 2 at Alg. 1 l.15; off on the graded path (reading 19)
  FLAG_WARMUP = 512u,      // PQ codebook warm-up (readings 32-36): residual reservoir over the first t_warm
                           // steps, then mini-batch k-means per subspace and side; codebooks given at create are ignored
  FLAG_WARMUP_MANUAL = 1024u,  // with FLAG_WARMUP: training is not started by the frame t_warm - 1 but by pko_train_codebooks
  FLAG_VAR_ALLOC = 2048u,  // variance-aware pseudo-token allocation S_k (D.3; readings 37-40)
};

struct Config {
  int32_t T, near_frames, k_max, d, S, G, C, beam;
  float lambda_sp, lambda_idle;
  int32_t t_idle;
  float alpha, beta, eta, sigma_eps, cos_eps;
  double pq_eps;
  uint32_t flags;
  float gamma, eps_k, eps_v;   // Alg. 2: idle decay rate, merge thresholds (Table 5: 0.05, 0.20, 0.25)
  double rope_theta;           // rotary base (reading 28); angle of pair i at position p = p * theta^(-2 i / d)
  int32_t rope_anchor;         // D.1 (L578-596): 0 most recent absorbed position (default), 1 first, 2 average
  int64_t pos0;                // stream position of token 0 of frame 0 (positions are pos0 + f T + j)
  int32_t t_warm;              // warm-up length in streaming steps (frames, reading 2): residuals of steps t < t_warm are collected
  int32_t warm_reservoir;      // reservoir capacity R (residual pairs per bank)
  int32_t km_iters, km_batch;  // mini-batch k-means: iterations, samples per iteration
  uint64_t km_seed;            // seed of this bank's counter-based generator (reservoir replacement, batch sampling)
  int32_t s_cap;               // D.3: upper bound of S_k (<= beam); S_tot = k_max * S
};

struct Maint {          // what Alg. 2 did since the counters were last read (pko_maintenance_counters)
  int64_t decayed;      // mass removed by aging (l.3)
  int64_t merges;       // prototypes merged away (l.7-11)
  int64_t recycled;     // slots re-initialised from the near window (l.15-17)
};

struct Trace {          // all pointers nullable; sizes [T] or [T][G]
  int32_t evicted;      // out: 1 if a frame was evicted by this call
  int32_t n_fill;       // out: tokens that opened a new slot (Alg. 1 l.3-4)
  int32_t* assign;      // out: the oracle's own choice (slot index for fills, argmin for the rest)
  float* best;          // out: best Eq. 1 score (0 for fills)
  float* second;        // out: second best score (+inf if none)
  float* forced_excess; // out: score(forced choice) - best, 0 when not forced
  uint8_t* codes_k;     // out: the oracle's own PQ codes [T][G] (255 = no residual update)
  uint8_t* codes_v;
  float* code_gap_k;    // out: (dist(forced code) - dist(best)) / max(dist(best), 1e-30), [T][G]
  float* code_gap_v;
};

struct StateView {      // host pointers, any may be NULL
  float* c; float* p;           // [k_max][d]
  int32_t* n;                   // [k_max] mass
  float* mu; float* sigma;      // [k_max][2], [k_max][3] = (xx, xy, yy)
  int32_t* tau; int64_t* pos;   // [k_max] frame index of last absorption / stream position of last absorbed token
  uint32_t* hist_k; uint32_t* hist_v;  // [k_max][G][C]
  uint32_t* nres;               // [k_max]
  uint8_t* active;              // [k_max]
  int64_t* pos_first;           // [k_max] stream position of the initialising token (D.1 "first")
  int64_t* pos_sum;             // [k_max] sum of the positions of all absorbed tokens (D.1 "average" = pos_sum / pos_cnt)
  int32_t* pos_cnt;             // [k_max]
};

struct Frame {
  int32_t index;
  std::vector<float> K, V, s;
};

using Tuple = std::array<uint8_t, 16>;

struct Bank {
  Config cfg;
  int sub;  // d / G
  bool has_cb;
  std::vector<float> cbk, cbv;  // [G][C][sub]
  std::deque<Frame> ring;
  int32_t frames_seen = 0;
  std::vector<float> c, p, mu, sigma;
  std::vector<int32_t> n, tau;
  std::vector<int64_t> pos, pos_first, pos_sum;
  std::vector<int32_t> pos_cnt;
  std::vector<uint32_t> hk, hv, nres;
  std::vector<uint8_t> active;
  std::vector<uint8_t> used;   // slot has been initialised at least once (Alg. 2 recycles only such slots, reading 24)
  Maint maint{0, 0, 0};
  // PQ codebook warm-up: reservoir of residual pairs (r^K, r^V) of absorbed tokens, [R][d] each
  std::vector<float> resK, resV;
  int64_t res_seen = 0;        // residuals offered to the reservoir so far
  bool trained = false;        // codebooks have been trained (warm-up is over)

  Bank(const Config& cf, const float* ck, const float* cv) : cfg(cf) {
    sub = cfg.d / cfg.G;
    has_cb = ck && cv && !(cfg.flags & (FLAG_NO_RESIDUAL | FLAG_WARMUP));
    if ((cfg.flags & FLAG_WARMUP) && !(cfg.flags & FLAG_NO_RESIDUAL)) {
      resK.assign((size_t)cfg.warm_reservoir * cfg.d, 0.f);
      resV.assign((size_t)cfg.warm_reservoir * cfg.d, 0.f);
    }
    if (has_cb) {
      size_t nn = (size_t)cfg.G * cfg.C * sub;
      cbk.assign(ck, ck + nn);
      cbv.assign(cv, cv + nn);
    }
    size_t K = cfg.k_max, d = cfg.d;
    c.assign(K * d, 0.f); p.assign(K * d, 0.f);
    mu.assign(K * 2, 0.f); sigma.assign(K * 3, 0.f);
    n.assign(K, 0); tau.assign(K, 0); pos.assign(K, 0);
    pos_first.assign(K, 0); pos_sum.assign(K, 0); pos_cnt.assign(K, 0);
    hk.assign(K * cfg.G * cfg.C, 0u); hv.assign(K * cfg.G * cfg.C, 0u);
    nres.assign(K, 0u); active.assign(K, 0); used.assign(K, 0);
  }

  int free_slot() const {  // lowest-index inactive slot (reading 9), -1 if none
    for (int k = 0; k < cfg.k_max; ++k) if (!active[k]) return k;
    return -1;
  }

  // Alg. 1 l.4: c<-K_e, p<-V_e, n<-1, mu<-s_e, Sigma<-I, tau<-t, R<-0
  void init_slot(int k, const float* Ke, const float* Ve, const float* se, int32_t t, int64_t ps) {
    int d = cfg.d;
    for (int i = 0; i < d; ++i) { c[(size_t)k * d + i] = Ke[i]; p[(size_t)k * d + i] = Ve[i]; }
    n[k] = 1; mu[k * 2] = se[0]; mu[k * 2 + 1] = se[1];
    sigma[k * 3] = 1.f; sigma[k * 3 + 1] = 0.f; sigma[k * 3 + 2] = 1.f;
    tau[k] = t; pos[k] = ps;
    pos_first[k] = ps; pos_sum[k] = ps; pos_cnt[k] = 1;
    std::fill(hk.begin() + (size_t)k * cfg.G * cfg.C, hk.begin() + (size_t)(k + 1) * cfg.G * cfg.C, 0u);
    std::fill(hv.begin() + (size_t)k * cfg.G * cfg.C, hv.begin() + (size_t)(k + 1) * cfg.G * cfg.C, 0u);
    nres[k] = 0; active[k] = 1; used[k] = 1;
  }

  // Alg. 2, readings 20 and 24-27 of DESIGN.md: aging, pairwise merge, recycling -- in that order.
  void maintain(int32_t t) {
    const int K = cfg.k_max, d = cfg.d, GC = cfg.G * cfg.C;
    // l.1-5 aging: n_k <- floor((1 - gamma) n_k) for prototypes idle for more than T_idle steps
    for (int k = 0; k < K; ++k) {
      if (!active[k]) continue;
      if ((int64_t)t - (int64_t)tau[k] > (int64_t)cfg.t_idle) {
        int32_t nn = (int32_t)std::floor((1.0 - (double)cfg.gamma) * (double)n[k]);
        maint.decayed += n[k] - nn;
        n[k] = nn;
      }
    }
    // l.6-13 merging: pairs i < j in lexicographic order, both non-empty; the lower index survives and its UPDATED
    // centres are what later pairs (i, j') are tested against; fields Alg. 2 does not list (Sigma, tau, pos) keep
    // Pi_i's values
    const double ek2 = (double)cfg.eps_k * (double)cfg.eps_k, ev2 = (double)cfg.eps_v * (double)cfg.eps_v;
    for (int i = 0; i < K; ++i) {
      if (!active[i] || n[i] < 1) continue;
      for (int j = i + 1; j < K; ++j) {
        if (!active[j] || n[j] < 1) continue;
        double dk = 0, dv = 0;
        for (int e = 0; e < d; ++e) {
          double a = (double)c[(size_t)i * d + e] - (double)c[(size_t)j * d + e];
          dk += a * a;
        }
        if (!(dk < ek2)) continue;                         // ||c_i - c_j||_2 < eps_K
        for (int e = 0; e < d; ++e) {
          double a = (double)p[(size_t)i * d + e] - (double)p[(size_t)j * d + e];
          dv += a * a;
        }
        if (!(dv < ev2)) continue;                         // ||p_i - p_j||_2 < eps_V
        const double ni = n[i], nj = n[j], w = ni + nj;
        for (int e = 0; e < d; ++e) {
          c[(size_t)i * d + e] = (float)((ni * (double)c[(size_t)i * d + e] + nj * (double)c[(size_t)j * d + e]) / w);
          p[(size_t)i * d + e] = (float)((ni * (double)p[(size_t)i * d + e] + nj * (double)p[(size_t)j * d + e]) / w);
        }
        for (int e = 0; e < 2; ++e)
          mu[i * 2 + e] = (float)((ni * (double)mu[i * 2 + e] + nj * (double)mu[j * 2 + e]) / w);
        n[i] += n[j];
        for (int e = 0; e < GC; ++e) {
          hk[(size_t)i * GC + e] += hk[(size_t)j * GC + e];
          hv[(size_t)i * GC + e] += hv[(size_t)j * GC + e];
        }
        nres[i] += nres[j];
        pos_first[i] = std::min(pos_first[i], pos_first[j]);   // anchors of the union of the absorbed tokens (reading 30)
        pos_sum[i] += pos_sum[j]; pos_cnt[i] += pos_cnt[j];
        active[j] = 0; n[j] = 0;                           // "mark Pi_j as inactive"
        maint.merges += 1;
      }
    }
    // l.14-19 recycling: every slot emptied by decay or merging (never-used slots stay free for Alg. 1 l.3-4) is
    // re-initialised from a recent near-window token: the r-th such slot of this call, in increasing slot order, takes
    // token T-1-(r mod T) of the (r / T)-th newest frame
    int r = 0;
    for (int k = 0; k < K; ++k) {
      if (!used[k] || (active[k] && n[k] >= 1)) continue;
      int back = r / cfg.T;
      if (back >= (int)ring.size()) back = (int)ring.size() - 1;
      const Frame& f = ring[ring.size() - 1 - back];
      const int j = cfg.T - 1 - (r % cfg.T);
      init_slot(k, &f.K[(size_t)j * d], &f.V[(size_t)j * d], &f.s[j * 2], t, cfg.pos0 + (int64_t)f.index * cfg.T + j);
      maint.recycled += 1;
      ++r;
    }
  }

  // ---- PQ codebook warm-up ("mini-batch k-means on a warm-up reservoir of residuals collected during the
  // first T_warm streaming steps, run separately for each subspace and for key/value"; readings 32-36) ----
  // Counter-based generator: the SplitMix64 output function (Steele, Lea & Flood 2014) of a counter.
  static uint64_t mix64(uint64_t x) {
    uint64_t z = x + 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
  }
  uint64_t draw(uint64_t stream, uint64_t counter) const { return mix64(cfg.km_seed ^ mix64(2 * counter + stream)); }
  bool warming(int32_t t) const {
    return (cfg.flags & FLAG_WARMUP) && !(cfg.flags & FLAG_NO_RESIDUAL) && !trained && t < cfg.t_warm;
  }
  // Reservoir sampling (Vitter's Algorithm R): the i-th residual pair offered (i = 0, 1, ...) fills slot i while
  // i < R, afterwards it replaces slot u = draw mod (i + 1) if u < R.  Returns the slot or -1.
  int reservoir_slot(int64_t i) const {
    const int64_t R = cfg.warm_reservoir;
    if (i < R) return (int)i;
    const uint64_t u = draw(0, (uint64_t)i) % (uint64_t)(i + 1);
    return u < (uint64_t)R ? (int)u : -1;
  }
  void reservoir_offer(const float* Ke, const float* Ve, const float* ck, const float* pk) {
    const int64_t i = res_seen++;
    const int slot = reservoir_slot(i);
    if (slot < 0) return;
    for (int e = 0; e < cfg.d; ++e) {      // r = x - centre (the just-updated one, reading 7), one rounding to fp32
      resK[(size_t)slot * cfg.d + e] = (float)((double)Ke[e] - (double)ck[e]);
      resV[(size_t)slot * cfg.d + e] = (float)((double)Ve[e] - (double)pk[e]);
    }
  }
  int64_t reservoir_fill() const { return std::min<int64_t>(res_seen, cfg.warm_reservoir); }

  // Mini-batch k-means (Sculley 2010, Alg. 1) of the rows X[0, n) restricted to subspace g: C centres of `sub` dims.
  // Reading 34: centre z starts at row floor(z n / C); per iteration `km_batch` rows are drawn with replacement by the
  // counter-based generator (the same rows for every subspace and side), assigned to their nearest centre with the
  // centres frozen, then applied in batch order with the per-centre rate 1 / v_z, v_z = samples ever assigned to z.
  // Reading 35: these decisions are taken in fp32, operation by operation (no fused multiply-add), so that another
  // implementation can reproduce them bit for bit: dist = sum_m (x_m - c_m)^2 accumulated left to right from 0.
  void kmeans_subspace(const std::vector<float>& X, int64_t n, int g, float* out /*[C][sub]*/) const {
    const int Cn = cfg.C, d = cfg.d;
    std::vector<float> cen((size_t)Cn * sub);
    std::vector<int64_t> v(Cn, 0);
    for (int z = 0; z < Cn; ++z) {
      const int64_t row = (int64_t)z * n / Cn;
      for (int m = 0; m < sub; ++m) cen[(size_t)z * sub + m] = X[(size_t)row * d + g * sub + m];
    }
    std::vector<int64_t> rows(cfg.km_batch);
    std::vector<int> asg(cfg.km_batch);
    for (int it = 0; it < cfg.km_iters; ++it) {
      for (int q = 0; q < cfg.km_batch; ++q) {
        rows[q] = (int64_t)(draw(1, (uint64_t)it * (uint64_t)cfg.km_batch + (uint64_t)q) % (uint64_t)n);
        const float* x = &X[(size_t)rows[q] * d + g * sub];
        int zb = 0;
        float db = std::numeric_limits<float>::infinity();
        for (int z = 0; z < Cn; ++z) {
          float acc = 0.f;
          for (int m = 0; m < sub; ++m) {
            const float t = x[m] - cen[(size_t)z * sub + m];
            const float t2 = t * t;
            acc = acc + t2;
          }
          if (acc < db) { db = acc; zb = z; }             // lowest index on ties
        }
        asg[q] = zb;
      }
      for (int q = 0; q < cfg.km_batch; ++q) {
        const int z = asg[q];
        v[z] += 1;
        const float eta = 1.0f / (float)v[z];
        const float keep = 1.0f - eta;
        const float* x = &X[(size_t)rows[q] * d + g * sub];
        for (int m = 0; m < sub; ++m) {
          const float a = keep * cen[(size_t)z * sub + m];
          const float b2 = eta * x[m];
          cen[(size_t)z * sub + m] = a + b2;
        }
      }
    }
    std::memcpy(out, cen.data(), cen.size() * sizeof(float));
  }
  // Ends the warm-up: trains C^K_g, C^V_g for every subspace from the reservoir.  Fewer than C residuals: no codebooks
  // (the state keeps running without residual statistics).  Returns 1 if codebooks now exist.
  int train_codebooks() {
    if (!(cfg.flags & FLAG_WARMUP) || (cfg.flags & FLAG_NO_RESIDUAL) || trained) return has_cb ? 1 : 0;
    trained = true;
    const int64_t n = reservoir_fill();
    if (n < cfg.C) return 0;
    cbk.assign((size_t)cfg.G * cfg.C * sub, 0.f);
    cbv.assign((size_t)cfg.G * cfg.C * sub, 0.f);
    for (int g = 0; g < cfg.G; ++g) {
      kmeans_subspace(resK, n, g, &cbk[(size_t)g * cfg.C * sub]);
      kmeans_subspace(resV, n, g, &cbv[(size_t)g * cfg.C * sub]);
    }
    has_cb = true;
    return 1;
  }

  // Eq. 1: -cos(K_e,c_k) + lambda_sp d_Mah(s_e;mu_k,Sigma_k) + lambda_idle 1[t - tau_k > T_idle]
  float score(const float* Ke, const float* se, int k, int32_t t) const {
    int d = cfg.d;
    const float* ck = &c[(size_t)k * d];
    double dot = 0, kk = 0, cc = 0;
    for (int i = 0; i < d; ++i) {
      dot += (double)Ke[i] * (double)ck[i];
      kk += (double)Ke[i] * (double)Ke[i];
      cc += (double)ck[i] * (double)ck[i];
    }
    double cosv = dot / std::max(std::sqrt(kk * cc), (double)cfg.cos_eps);
    double dx = (double)se[0] - (double)mu[k * 2], dy = (double)se[1] - (double)mu[k * 2 + 1];
    double a = (double)sigma[k * 3] + (double)cfg.sigma_eps, b = (double)sigma[k * 3 + 1],
           e = (double)sigma[k * 3 + 2] + (double)cfg.sigma_eps;
    double det = a * e - b * b;
    double q = (e * dx * dx - 2.0 * b * dx * dy + a * dy * dy) / det;  // delta^T (Sigma+eps I)^-1 delta
    if (q < 0) q = 0;
    double dm = (cfg.flags & FLAG_MAH_SQUARED) ? q : std::sqrt(q);
    double idle = ((int64_t)t - (int64_t)tau[k] > (int64_t)cfg.t_idle) ? (double)cfg.lambda_idle : 0.0;
    return (float)(-cosv + (double)cfg.lambda_sp * dm + idle);
  }

  // argmin over active prototypes, lowest index on exact ties; also second best
  int argmin_score(const float* Ke, const float* se, int32_t t, float* best, float* second) const {
    int kb = -1;
    float b = std::numeric_limits<float>::infinity(), s2 = b;
    for (int k = 0; k < cfg.k_max; ++k) {
      if (!active[k]) continue;
      float sc = score(Ke, se, k, t);
      if (sc < b) { s2 = b; b = sc; kb = k; }
      else if (sc < s2) s2 = sc;
    }
    *best = b; *second = s2;
    return kb;
  }

  // nearest codeword per subspace in squared L2 (reading 10); returns code, writes rounded distances
  int nearest_code(const std::vector<float>& cb, int g, const double* r, float* dist_out) const {
    int zb = 0;
    float db = std::numeric_limits<float>::infinity();
    for (int z = 0; z < cfg.C; ++z) {
      double acc = 0;
      const float* cw = &cb[((size_t)g * cfg.C + z) * sub];
      for (int m = 0; m < sub; ++m) { double t = r[m] - (double)cw[m]; acc += t * t; }
      float df = (float)acc;
      if (dist_out) dist_out[z] = df;
      if (df < db) { db = df; zb = z; }
    }
    return zb;
  }

  // Alg. 1 l.8-13, in the listed order; residuals use the just-updated centres (reading 7)
  void update_proto(int k, const float* Ke, const float* Ve, const float* se, int32_t t, int64_t ps,
                    const uint8_t* fck, const uint8_t* fcv, uint8_t* ock, uint8_t* ocv, float* gk, float* gv) {
    int d = cfg.d;
    double al = cfg.alpha, be = cfg.beta, et = cfg.eta;
    float* ck = &c[(size_t)k * d];
    float* pk = &p[(size_t)k * d];
    for (int i = 0; i < d; ++i) {
      ck[i] = (float)((1.0 - al) * (double)ck[i] + al * (double)Ke[i]);   // l.8
      pk[i] = (float)((1.0 - be) * (double)pk[i] + be * (double)Ve[i]);   // l.9
    }
    n[k] += 1; tau[k] = t; pos[k] = ps;                                   // l.10
    pos_sum[k] += ps; pos_cnt[k] += 1;                                    // D.1 anchors (pos_first stays)
    mu[k * 2] = (float)((1.0 - et) * (double)mu[k * 2] + et * (double)se[0]);          // l.11
    mu[k * 2 + 1] = (float)((1.0 - et) * (double)mu[k * 2 + 1] + et * (double)se[1]);
    double dx = (double)se[0] - (double)mu[k * 2], dy = (double)se[1] - (double)mu[k * 2 + 1];  // new mu
    sigma[k * 3] = (float)((1.0 - et) * (double)sigma[k * 3] + et * dx * dx);          // l.12
    sigma[k * 3 + 1] = (float)((1.0 - et) * (double)sigma[k * 3 + 1] + et * dx * dy);
    sigma[k * 3 + 2] = (float)((1.0 - et) * (double)sigma[k * 3 + 2] + et * dy * dy);
    if (warming(t)) reservoir_offer(Ke, Ve, ck, pk);                     // L312: residuals of the warm-up steps
    if (!has_cb) return;
    std::vector<double> r(sub);
    std::vector<float> dist(cfg.C);
    for (int kv = 0; kv < 2; ++kv) {                                      // l.13
      const float* x = kv ? Ve : Ke;
      const float* cen = kv ? pk : ck;
      const std::vector<float>& cb = kv ? cbv : cbk;
      std::vector<uint32_t>& H = kv ? hv : hk;
      const uint8_t* forced = kv ? fcv : fck;
      uint8_t* oc = kv ? ocv : ock;
      float* gap = kv ? gv : gk;
      for (int g = 0; g < cfg.G; ++g) {
        for (int m = 0; m < sub; ++m) r[m] = (double)x[g * sub + m] - (double)cen[g * sub + m];
        int z = nearest_code(cb, g, r.data(), dist.data());
        if (oc) oc[g] = (uint8_t)z;
        int use = z;
        if (forced) {
          use = forced[g];
          if (gap) gap[g] = (dist[use] - dist[z]) / std::max(dist[z], 1e-30f);
        } else if (gap) gap[g] = 0.f;
        H[((size_t)k * cfg.G + g) * cfg.C + use] += 1;
      }
    }
    nres[k] += 1;
  }

  bool pop_if_full(Frame* ev) {
    if ((int)ring.size() < cfg.near_frames) return false;
    *ev = std::move(ring.front());
    ring.pop_front();
    return true;
  }
  void push(const float* K, const float* V, const float* s) {
    Frame f;
    f.index = frames_seen;
    size_t nkv = (size_t)cfg.T * cfg.d;
    f.K.assign(K, K + nkv); f.V.assign(V, V + nkv); f.s.assign(s, s + (size_t)cfg.T * 2);
    ring.push_back(std::move(f));
  }
  static void clear_trace(Trace* tr, int T, int G) {
    if (!tr) return;
    tr->evicted = 0; tr->n_fill = 0;
    for (int j = 0; j < T; ++j) {
      if (tr->assign) tr->assign[j] = -1;
      if (tr->best) tr->best[j] = 0.f;
      if (tr->second) tr->second[j] = std::numeric_limits<float>::infinity();
      if (tr->forced_excess) tr->forced_excess[j] = 0.f;
      for (int g = 0; g < G; ++g) {
        if (tr->codes_k) tr->codes_k[j * G + g] = 255;
        if (tr->codes_v) tr->codes_v[j * G + g] = 255;
        if (tr->code_gap_k) tr->code_gap_k[j * G + g] = 0.f;
        if (tr->code_gap_v) tr->code_gap_v[j * G + g] = 0.f;
      }
    }
  }

  // Frame-synchronous update (reading 1; the graded definition):
  //  A) slot fill in eviction order, B) Eq. 1 scores of the remaining tokens against the bank as it stands
  //  after (A), C) Alg. 1 l.8-13 replayed token by token, in eviction order, on the live bank.
  void append_frame_sync(const float* K, const float* V, const float* s, const int32_t* forced,
                         const uint8_t* fck, const uint8_t* fcv, Trace* tr) {
    const int T = cfg.T, d = cfg.d, G = cfg.G;
    clear_trace(tr, T, G);
    Frame E;
    bool ev = pop_if_full(&E);                 // |B_near| > W after the append  (Alg. 1 l.1-3)
    push(K, V, s);
    const int32_t t = frames_seen;             // stream time = frame index (reading 2)
    frames_seen += 1;
    if (!ev) { end_of_step(t); return; }
    if (tr) tr->evicted = 1;
    int j = 0;
    for (; j < T; ++j) {                        // (A)
      int k = free_slot();
      if (k < 0) break;
      init_slot(k, &E.K[(size_t)j * d], &E.V[(size_t)j * d], &E.s[j * 2], t, cfg.pos0 + (int64_t)E.index * T + j);
      if (tr && tr->assign) tr->assign[j] = k;
    }
    const int nf = j;
    if (tr) tr->n_fill = nf;
    std::vector<int> own(T, -1);
    for (j = nf; j < T; ++j) {                  // (B) -- the bank is frozen during this loop
      float b, s2;
      own[j] = argmin_score(&E.K[(size_t)j * d], &E.s[j * 2], t, &b, &s2);
      if (tr) {
        if (tr->assign) tr->assign[j] = own[j];
        if (tr->best) tr->best[j] = b;
        if (tr->second) tr->second[j] = s2;
        if (forced && tr->forced_excess)
          tr->forced_excess[j] = score(&E.K[(size_t)j * d], &E.s[j * 2], forced[j], t) - b;
      }
    }
    for (j = nf; j < T; ++j) {                  // (C)
      int k = forced ? forced[j] : own[j];
      update_proto(k, &E.K[(size_t)j * d], &E.V[(size_t)j * d], &E.s[j * 2], t, cfg.pos0 + (int64_t)E.index * T + j,
                   fck ? fck + j * G : nullptr, fcv ? fcv + j * G : nullptr,
                   tr && tr->codes_k ? tr->codes_k + j * G : nullptr, tr && tr->codes_v ? tr->codes_v + j * G : nullptr,
                   tr && tr->code_gap_k ? tr->code_gap_k + j * G : nullptr,
                   tr && tr->code_gap_v ? tr->code_gap_v + j * G : nullptr);
    }
    end_of_step(t);
    if (cfg.flags & FLAG_MAINTENANCE) maintain(t);   // Alg. 1 l.15, once per frame in the frame-synchronous reading
  }

  // Literal Alg. 1 (token-sequential): every evicted token sees the live bank. Used for pinning only.
  void append_frame_seq(const float* K, const float* V, const float* s, const int32_t* forced,
                        const uint8_t* fck, const uint8_t* fcv, Trace* tr) {
    const int T = cfg.T, d = cfg.d, G = cfg.G;
    clear_trace(tr, T, G);
    Frame E;
    bool ev = pop_if_full(&E);
    push(K, V, s);
    const int32_t t = frames_seen;
    frames_seen += 1;
    if (!ev) { end_of_step(t); return; }
    if (tr) tr->evicted = 1;
    int nf = 0;
    for (int j = 0; j < T; ++j) {
      const float* Ke = &E.K[(size_t)j * d];
      const float* Ve = &E.V[(size_t)j * d];
      const float* se = &E.s[j * 2];
      int64_t ps = cfg.pos0 + (int64_t)E.index * T + j;
      int k = free_slot();
      if (k >= 0) {                                                   // l.3-4
        init_slot(k, Ke, Ve, se, t, ps);
        if (tr && tr->assign) tr->assign[j] = k;
        ++nf;
        if (cfg.flags & FLAG_MAINTENANCE) maintain(t);                // l.15
        continue;
      }
      float b, s2;
      int own = argmin_score(Ke, se, t, &b, &s2);                     // l.6
      if (tr) {
        if (tr->assign) tr->assign[j] = own;
        if (tr->best) tr->best[j] = b;
        if (tr->second) tr->second[j] = s2;
        if (forced && tr->forced_excess) tr->forced_excess[j] = score(Ke, se, forced[j], t) - b;
      }
      k = forced ? forced[j] : own;
      update_proto(k, Ke, Ve, se, t, ps, fck ? fck + j * G : nullptr, fcv ? fcv + j * G : nullptr,     // l.8-13
                   tr && tr->codes_k ? tr->codes_k + j * G : nullptr, tr && tr->codes_v ? tr->codes_v + j * G : nullptr,
                   tr && tr->code_gap_k ? tr->code_gap_k + j * G : nullptr,
                   tr && tr->code_gap_v ? tr->code_gap_v + j * G : nullptr);
      if (cfg.flags & FLAG_MAINTENANCE) maintain(t);                  // l.15
    }
    if (tr) tr->n_fill = nf;
    end_of_step(t);
  }
  // the last warm-up step trains the codebooks (reading 33) unless the caller does it (FLAG_WARMUP_MANUAL)
  void end_of_step(int32_t t) {
    if ((cfg.flags & FLAG_WARMUP) && !(cfg.flags & FLAG_WARMUP_MANUAL) && !trained && t == cfg.t_warm - 1) train_codebooks();
  }

  // Eq. 3 in fixed point (reading 13): q(g,c) = llround(2^24 * log P(g,c))
  void log_table(const uint32_t* H, std::vector<int64_t>& q) const {
    q.resize((size_t)cfg.G * cfg.C);
    for (int g = 0; g < cfg.G; ++g) {
      double tot = 0;
      for (int z = 0; z < cfg.C; ++z) tot += (double)H[g * cfg.C + z];
      double den = tot + (double)cfg.C * cfg.pq_eps;
      for (int z = 0; z < cfg.C; ++z) {
        double P = ((double)H[g * cfg.C + z] + cfg.pq_eps) / den;
        q[g * cfg.C + z] = std::llround(std::log(P) * 16777216.0);
      }
    }
  }

  // Alg. 3: beam search over subquantisers, beam width B, output the top S tuples.
  // Order: score descending, then tuple ascending lexicographically (z_1 most significant).
  void decode_top_s(const uint32_t* H, std::vector<Tuple>& out, std::vector<int64_t>* out_scores, int S_out = -1) const {
    if (S_out < 0) S_out = cfg.S;
    std::vector<int64_t> q;
    log_table(H, q);
    struct Item { int64_t a; Tuple z; };
    std::vector<Item> beam(1), next;
    beam[0].a = 0; beam[0].z.fill(0);
    for (int g = 0; g < cfg.G; ++g) {                      // l.2
      next.clear();                                        // B' <- empty
      for (const Item& it : beam)                          // l.4
        for (int z = 0; z < cfg.C; ++z) {                  // l.5
          Item e = it;
          e.a = it.a + q[g * cfg.C + z];                   // l.6
          e.z[g] = (uint8_t)z;
          next.push_back(e);
        }
      std::sort(next.begin(), next.end(), [&](const Item& x, const Item& y) {
        if (x.a != y.a) return x.a > y.a;
        return std::lexicographical_compare(x.z.begin(), x.z.begin() + g + 1, y.z.begin(), y.z.begin() + g + 1);
      });
      if ((int)next.size() > cfg.beam) next.resize(cfg.beam);   // TopB, l.10
      beam.swap(next);
    }
    out.clear();
    if (out_scores) out_scores->clear();
    for (int s = 0; s < S_out && s < (int)beam.size(); ++s) {    // TopS, l.12
      out.push_back(beam[s].z);
      if (out_scores) out_scores->push_back(beam[s].a);
    }
  }

  // ---- D.3 dynamic pseudo-token allocation: S_k = S_tot Var(H_k) / sum_j Var(H_j), S_tot = K_max S.
  // Reading 37: Var(H_k) = total variance of the residual distribution the histograms describe -- for each side and
  // subspace the codewords C_g[z] weighted by the empirical frequencies H[g,z] / sum_z H[g,z]:
  //   var_g = sum_z H_z |C_g[z] - mean_g|^2 / tot,  mean_g = sum_z H_z C_g[z] / tot;  Var = sum over (K then V, g ascending).
  // fp64, every product and sum rounded separately in the order written (reading 38: the value is then fixed to
  // v_k = floor(Var 2^20 + 1/2), so that the allocation is integer arithmetic another implementation reproduces exactly).
  int64_t variance_fx(int k) const {
    if (!has_cb || nres[k] == 0) return 0;
    double total = 0.0;
    std::vector<double> mean(sub);
    for (int kv = 0; kv < 2; ++kv) {
      const std::vector<uint32_t>& H = kv ? hv : hk;
      const std::vector<float>& cb = kv ? cbv : cbk;
      for (int g = 0; g < cfg.G; ++g) {
        const uint32_t* h = &H[((size_t)k * cfg.G + g) * cfg.C];
        double tot = 0.0;
        for (int z = 0; z < cfg.C; ++z) tot = tot + (double)h[z];
        if (tot == 0.0) continue;
        for (int m = 0; m < sub; ++m) {
          double a = 0.0;
          for (int z = 0; z < cfg.C; ++z) a = a + (double)h[z] * (double)cb[((size_t)g * cfg.C + z) * sub + m];
          mean[m] = a / tot;
        }
        double var = 0.0;
        for (int z = 0; z < cfg.C; ++z) {
          double dz = 0.0;
          for (int m = 0; m < sub; ++m) {
            const double t = (double)cb[((size_t)g * cfg.C + z) * sub + m] - mean[m];
            dz = dz + t * t;
          }
          var = var + (double)h[z] * dz;
        }
        total = total + var / tot;
      }
    }
    return (int64_t)std::floor(total * 1048576.0 + 0.5);
  }
  // Reading 39: integer shares.  Every prototype in the context (active, n >= 1) gets one pseudo-token, the remaining
  // budget S_tot - |A| is split in proportion to v_k (floor), capped at s_cap; what flooring and capping leave over goes
  // one unit at a time to the prototypes below the cap in the order (remainder of the proportional split descending,
  // index ascending), round after round.  sum_j v_j = 0: the fixed default min(S, s_cap) each.
  void allocate(std::vector<int32_t>& Sk) const {
    const int K = cfg.k_max;
    Sk.assign(K, 0);
    std::vector<int> A;
    for (int k = 0; k < K; ++k) if (active[k] && n[k] >= 1) A.push_back(k);
    if (A.empty()) return;
    if (!(cfg.flags & FLAG_VAR_ALLOC)) { for (int k : A) Sk[k] = cfg.S; return; }
    std::vector<int64_t> v(K, 0), rem(K, 0);
    int64_t vsum = 0;
    for (int k : A) { v[k] = variance_fx(k); vsum += v[k]; }
    if (vsum == 0) { for (int k : A) Sk[k] = std::min(cfg.S, cfg.s_cap); return; }
    const int64_t stot = (int64_t)K * cfg.S, bud = stot - (int64_t)A.size();
    int64_t used = 0;
    for (int k : A) {
      const int64_t prod = bud * v[k];
      Sk[k] = (int32_t)std::min<int64_t>(cfg.s_cap, 1 + prod / vsum);
      rem[k] = prod % vsum;
      used += Sk[k];
    }
    int64_t left = stot - used;
    std::vector<int> order(A);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b2) { return rem[a] > rem[b2]; });
    while (left > 0) {
      bool any = false;
      for (int k : order) {
        if (left == 0) break;
        if (Sk[k] < cfg.s_cap) { Sk[k] += 1; left -= 1; any = true; }
      }
      if (!any) break;
    }
  }

  int64_t tuple_score(int k, int which, const uint8_t* z) const {
    std::vector<int64_t> q;
    const std::vector<uint32_t>& H = which ? hv : hk;
    log_table(&H[(size_t)k * cfg.G * cfg.C], q);
    int64_t a = 0;
    for (int g = 0; g < cfg.G; ++g) a += q[g * cfg.C + z[g]];
    return a;
  }

  // Alg. 4 l.1-13: [near || pseudo] keys/values and bias b
  // Rotary embedding of one vector at (possibly fractional) position p, rotate-half convention (reading 28):
  // pair (i, i + d/2), angle p * theta^(-2 i / d); everything in fp64.
  void rope(double* x, double p) const {
    const int h = cfg.d / 2;
    for (int i = 0; i < h; ++i) {
      const double ang = p * std::pow(cfg.rope_theta, -2.0 * (double)i / (double)cfg.d);
      const double cs = std::cos(ang), sn = std::sin(ang);
      const double a = x[i], b2 = x[i + h];
      x[i] = a * cs - b2 * sn;
      x[i + h] = b2 * cs + a * sn;
    }
  }
  int stride_s() const { return (cfg.flags & FLAG_VAR_ALLOC) ? cfg.s_cap : cfg.S; }
  // Rotary anchor of prototype k (D.1 L578-596): most recent / first / average absorbed position
  double anchor(int k) const {
    if (cfg.rope_anchor == 1) return (double)pos_first[k];
    if (cfg.rope_anchor == 2) return (double)pos_sum[k] / (double)pos_cnt[k];
    return (double)pos[k];
  }

  // positions (optional out): stream position of every context element (near: original, pseudo: the anchor)
  void materialize(const uint8_t* fck, const uint8_t* fcv, std::vector<double>& Kt, std::vector<double>& Vt,
                   std::vector<double>& b, std::vector<double>* positions = nullptr, bool rotate = true) const {
    const int d = cfg.d, G = cfg.G;
    const bool do_rope = (cfg.flags & FLAG_ROPE) && rotate;
    Kt.clear(); Vt.clear(); b.clear();
    if (positions) positions->clear();
    if (!(cfg.flags & FLAG_FAR_ONLY))
      for (const Frame& f : ring)
        for (int j = 0; j < cfg.T; ++j) {
          for (int i = 0; i < d; ++i) { Kt.push_back(f.K[(size_t)j * d + i]); Vt.push_back(f.V[(size_t)j * d + i]); }
          b.push_back(0.0);                                                   // near tokens carry zero bias (L407)
          const double ps = (double)(cfg.pos0 + (int64_t)f.index * cfg.T + j);   // near tokens keep their positions (L126)
          if (positions) positions->push_back(ps);
          if (do_rope) rope(&Kt[Kt.size() - d], ps);
        }
    if (cfg.flags & FLAG_NEAR_ONLY) return;
    std::vector<Tuple> zk, zv;
    std::vector<int32_t> Sk;
    allocate(Sk);                                                             // S_k = S, or the D.3 shares (FLAG_VAR_ALLOC)
    const int smax = stride_s();                                              // row stride of forced code arrays
    for (int k = 0; k < cfg.k_max; ++k) {
      if (!active[k] || n[k] < 1) continue;                                   // l.2 "each active prototype"
      bool zero = (!has_cb) || nres[k] == 0;                                  // l.3-4
      const int S = Sk[k];
      if (!zero) {
        if (fck && fcv) {
          zk.assign(S, Tuple{}); zv.assign(S, Tuple{});
          for (int s = 0; s < S; ++s)
            for (int g = 0; g < G; ++g) {
              zk[s][g] = fck[((size_t)k * smax + s) * G + g];
              zv[s][g] = fcv[((size_t)k * smax + s) * G + g];
            }
        } else {
          decode_top_s(&hk[(size_t)k * G * cfg.C], zk, nullptr, S);           // l.5
          decode_top_s(&hv[(size_t)k * G * cfg.C], zv, nullptr, S);           // l.6
        }
      }
      double bias = (cfg.flags & FLAG_NO_MASS_BIAS) ? 0.0 : std::log((double)n[k]);   // Eq. 4, natural log
      for (int s = 0; s < S; ++s) {                                           // l.8-10
        for (int i = 0; i < d; ++i) {
          double rk = 0, rv = 0;
          if (!zero) {
            int g = i / sub, m = i % sub;
            rk = cbk[((size_t)g * cfg.C + zk[s][g]) * sub + m];
            rv = cbv[((size_t)g * cfg.C + zv[s][g]) * sub + m];
          }
          Kt.push_back((double)c[(size_t)k * d + i] + rk);
          Vt.push_back((double)p[(size_t)k * d + i] + rv);
        }
        b.push_back(bias);
        if (positions) positions->push_back(anchor(k));                       // all S pseudo-tokens share tau_k (L126)
        if (do_rope) rope(&Kt[Kt.size() - d], anchor(k));
      }
    }
  }

  // Alg. 4 l.14-15: A = Q K~^T / sqrt(d) + b ; O = softmax(A) V~   (no mask, reading 17)
  // qpos: stream position of every query row (used with FLAG_ROPE only; a query token i sits at q_pos0 + i and all heads
  // of a token share its position -- the caller expands that to rows; NULL = every row at the next stream position)
  void attention(const float* Q, int rows, const uint8_t* fck, const uint8_t* fcv, float* out, double* lse,
                 const int64_t* qpos = nullptr) const {
    const int d = cfg.d;
    std::vector<double> Kt, Vt, b;
    materialize(fck, fcv, Kt, Vt, b);
    const size_t L = b.size();
    const double scale = 1.0 / std::sqrt((double)d);
    std::vector<double> logit(L), acc(d), q(d);
    for (int r = 0; r < rows; ++r) {
      for (int i = 0; i < d; ++i) q[i] = (double)Q[(size_t)r * d + i];
      if (cfg.flags & FLAG_ROPE) rope(q.data(), (double)(qpos ? qpos[r] : cfg.pos0 + (int64_t)frames_seen * cfg.T));
      double m = -std::numeric_limits<double>::infinity();
      for (size_t j = 0; j < L; ++j) {
        double dot = 0;
        for (int i = 0; i < d; ++i) dot += q[i] * Kt[j * d + i];
        logit[j] = dot * scale + b[j];
        m = std::max(m, logit[j]);
      }
      double sum = 0;
      std::fill(acc.begin(), acc.end(), 0.0);
      for (size_t j = 0; j < L; ++j) {
        double w = std::exp(logit[j] - m);
        sum += w;
        for (int i = 0; i < d; ++i) acc[i] += w * Vt[j * d + i];
      }
      for (int i = 0; i < d; ++i) out[(size_t)r * d + i] = L ? (float)(acc[i] / sum) : 0.f;
      if (lse) lse[r] = L ? m + std::log(sum) : -std::numeric_limits<double>::infinity();
    }
  }
};

}  // namespace

extern "C" {

void* pko_create(const Config* cfg, const float* codebook_k, const float* codebook_v) {
  if (!cfg || cfg->d <= 0 || cfg->G <= 0 || cfg->d % cfg->G || cfg->C <= 0 || cfg->C > 255 || cfg->G > 16 ||
      cfg->S <= 0 || cfg->beam < cfg->S || cfg->T <= 0 || cfg->near_frames <= 0 || cfg->k_max <= 0)
    return nullptr;
  if ((cfg->flags & FLAG_WARMUP) && (cfg->t_warm < 1 || cfg->warm_reservoir < 1 || cfg->km_iters < 0 || cfg->km_batch < 1))
    return nullptr;
  if ((cfg->flags & FLAG_VAR_ALLOC) && (cfg->s_cap < 1 || cfg->s_cap > cfg->beam)) return nullptr;
  return new Bank(*cfg, codebook_k, codebook_v);
}
void pko_destroy(void* h) { delete static_cast<Bank*>(h); }

// mode 0: frame-synchronous (graded); mode 1: token-sequential (literal Alg. 1)
int pko_append_frame(void* h, const float* K, const float* V, const float* s, int mode, const int32_t* forced_assign,
                     const uint8_t* forced_codes_k, const uint8_t* forced_codes_v, Trace* trace) {
  Bank* b = static_cast<Bank*>(h);
  if (!b || !K || !V || !s) return 1;
  if (mode == 0) b->append_frame_sync(K, V, s, forced_assign, forced_codes_k, forced_codes_v, trace);
  else b->append_frame_seq(K, V, s, forced_assign, forced_codes_k, forced_codes_v, trace);
  return 0;
}

int pko_frames_seen(void* h) { return static_cast<Bank*>(h)->frames_seen; }

// Alg. 2 on its own (time t), for pins; and its counters since the last call with reset != 0
void pko_maintain(void* h, int32_t t) { static_cast<Bank*>(h)->maintain(t); }
void pko_maintenance_counters(void* h, int64_t* out3, int reset) {
  Bank* b = static_cast<Bank*>(h);
  out3[0] = b->maint.decayed; out3[1] = b->maint.merges; out3[2] = b->maint.recycled;
  if (reset) b->maint = Maint{0, 0, 0};
}
int pko_ring_frames(void* h) { return (int)static_cast<Bank*>(h)->ring.size(); }

// ring in chronological order: K,V [n][T][d], s [n][T][2], idx [n]; returns n
int pko_get_ring(void* h, float* K, float* V, float* s, int32_t* idx) {
  Bank* b = static_cast<Bank*>(h);
  size_t nkv = (size_t)b->cfg.T * b->cfg.d, ns = (size_t)b->cfg.T * 2;
  int i = 0;
  for (const Frame& f : b->ring) {
    if (K) std::memcpy(K + i * nkv, f.K.data(), nkv * sizeof(float));
    if (V) std::memcpy(V + i * nkv, f.V.data(), nkv * sizeof(float));
    if (s) std::memcpy(s + i * ns, f.s.data(), ns * sizeof(float));
    if (idx) idx[i] = f.index;
    ++i;
  }
  return i;
}

#define PKO_COPY(field, vec) \
  if (v->field) std::memcpy(v->field, b->vec.data(), b->vec.size() * sizeof(b->vec[0]))
#define PKO_LOAD(field, vec) \
  if (v->field) std::memcpy(b->vec.data(), v->field, b->vec.size() * sizeof(b->vec[0]))

void pko_get_state(void* h, StateView* v) {
  Bank* b = static_cast<Bank*>(h);
  PKO_COPY(c, c); PKO_COPY(p, p); PKO_COPY(n, n); PKO_COPY(mu, mu); PKO_COPY(sigma, sigma);
  PKO_COPY(tau, tau); PKO_COPY(pos, pos); PKO_COPY(hist_k, hk); PKO_COPY(hist_v, hv); PKO_COPY(nres, nres);
  PKO_COPY(active, active); PKO_COPY(pos_first, pos_first); PKO_COPY(pos_sum, pos_sum); PKO_COPY(pos_cnt, pos_cnt);
}
void pko_set_state(void* h, const StateView* v) {
  Bank* b = static_cast<Bank*>(h);
  PKO_LOAD(c, c); PKO_LOAD(p, p); PKO_LOAD(n, n); PKO_LOAD(mu, mu); PKO_LOAD(sigma, sigma);
  PKO_LOAD(tau, tau); PKO_LOAD(pos, pos); PKO_LOAD(hist_k, hk); PKO_LOAD(hist_v, hv); PKO_LOAD(nres, nres);
  PKO_LOAD(active, active); PKO_LOAD(pos_first, pos_first); PKO_LOAD(pos_sum, pos_sum); PKO_LOAD(pos_cnt, pos_cnt);
  if (v->active)
    for (size_t k = 0; k < b->used.size(); ++k) b->used[k] = b->used[k] || b->active[k];
}

// Eq. 1 score of (K_e, s_e) against prototype k at stream time t, on the current bank
float pko_score(void* h, const float* Ke, const float* se, int k, int32_t t) {
  return static_cast<Bank*>(h)->score(Ke, se, k, t);
}

// Alg. 3 for every slot: codes [k_max][S][G] (K and V), scores [k_max][S] (fixed-point), zero[k_max] = 1 when
// the slot contributes zero residuals (n_res = 0 or no codebooks), 2 when the slot is not in the context at all.
void pko_synthesize(void* h, uint8_t* codes_k, uint8_t* codes_v, int64_t* scores_k, int64_t* scores_v, uint8_t* zero,
                    int32_t* s_count) {
  Bank* b = static_cast<Bank*>(h);
  const Config& cf = b->cfg;
  std::vector<Tuple> z;
  std::vector<int64_t> sc;
  std::vector<int32_t> Sk;
  b->allocate(Sk);
  const int smax = b->stride_s();      // rows per slot in the outputs: S, or s_cap with FLAG_VAR_ALLOC
  for (int k = 0; k < cf.k_max; ++k) {
    bool present = b->active[k] && b->n[k] >= 1;
    bool zr = !b->has_cb || b->nres[k] == 0;
    if (zero) zero[k] = present ? (zr ? 1 : 0) : 2;
    if (s_count) s_count[k] = Sk[k];
    for (int kv = 0; kv < 2; ++kv) {
      uint8_t* oc = kv ? codes_v : codes_k;
      int64_t* os = kv ? scores_v : scores_k;
      if (present && !zr) b->decode_top_s(&(kv ? b->hv : b->hk)[(size_t)k * cf.G * cf.C], z, &sc, Sk[k]);
      for (int s = 0; s < smax; ++s) {
        bool have = present && !zr && s < (int)z.size();
        if (oc) for (int g = 0; g < cf.G; ++g) oc[((size_t)k * smax + s) * cf.G + g] = have ? z[s][g] : 0;
        if (os) os[(size_t)k * smax + s] = have ? sc[s] : 0;
      }
    }
  }
}

// Alg. 3 on a caller-supplied histogram [G][C]; returns the number of tuples written (<= S)
int pko_decode_hist(void* h, const uint32_t* H, uint8_t* codes /*[S][G]*/, int64_t* scores /*[S]*/) {
  Bank* b = static_cast<Bank*>(h);
  std::vector<Tuple> z;
  std::vector<int64_t> sc;
  b->decode_top_s(H, z, &sc);
  for (size_t s = 0; s < z.size(); ++s) {
    for (int g = 0; g < b->cfg.G; ++g) codes[s * b->cfg.G + g] = z[s][g];
    if (scores) scores[s] = sc[s];
  }
  return (int)z.size();
}
// fixed-point Eq. 3 table of a caller-supplied histogram, q [G][C]
void pko_log_table(void* h, const uint32_t* H, int64_t* q) {
  Bank* b = static_cast<Bank*>(h);
  std::vector<int64_t> t;
  b->log_table(H, t);
  std::memcpy(q, t.data(), t.size() * sizeof(int64_t));
}
int64_t pko_tuple_score(void* h, int k, int which, const uint8_t* z) {
  return static_cast<Bank*>(h)->tuple_score(k, which, z);
}

// PQ codebook warm-up: reservoir contents [fill][d] x 2 and the number of residuals offered so far
int64_t pko_reservoir(void* h, float* rK, float* rV, int64_t* seen) {
  Bank* b = static_cast<Bank*>(h);
  const int64_t n = b->reservoir_fill();
  if (rK) std::memcpy(rK, b->resK.data(), (size_t)n * b->cfg.d * sizeof(float));
  if (rV) std::memcpy(rV, b->resV.data(), (size_t)n * b->cfg.d * sizeof(float));
  if (seen) *seen = b->res_seen;
  return n;
}
// overwrite the reservoir (pins): n rows, counted as n residuals offered
void pko_set_reservoir(void* h, const float* rK, const float* rV, int64_t n) {
  Bank* b = static_cast<Bank*>(h);
  std::memcpy(b->resK.data(), rK, (size_t)n * b->cfg.d * sizeof(float));
  std::memcpy(b->resV.data(), rV, (size_t)n * b->cfg.d * sizeof(float));
  b->res_seen = n;
}
int pko_train_codebooks(void* h) { return static_cast<Bank*>(h)->train_codebooks(); }
// current codebooks [G][C][sub] x 2; returns 0 if the bank has none
int pko_codebooks(void* h, float* ck, float* cv) {
  Bank* b = static_cast<Bank*>(h);
  if (!b->has_cb) return 0;
  if (ck) std::memcpy(ck, b->cbk.data(), b->cbk.size() * sizeof(float));
  if (cv) std::memcpy(cv, b->cbv.data(), b->cbv.size() * sizeof(float));
  return 1;
}
uint64_t pko_draw(void* h, uint64_t stream, uint64_t counter) { return static_cast<Bank*>(h)->draw(stream, counter); }
int pko_reservoir_slot(void* h, int64_t i) { return static_cast<Bank*>(h)->reservoir_slot(i); }
// D.3: fixed-point variances v_k [k_max] and the shares S_k [k_max] of the current state
void pko_allocation(void* h, int64_t* v, int32_t* Sk) {
  Bank* b = static_cast<Bank*>(h);
  std::vector<int32_t> s;
  b->allocate(s);
  for (int k = 0; k < b->cfg.k_max; ++k) {
    if (v) v[k] = (b->active[k] && b->n[k] >= 1) ? b->variance_fx(k) : 0;
    if (Sk) Sk[k] = s[k];
  }
}

// context length of the current state
int pko_context_len(void* h) {
  Bank* b = static_cast<Bank*>(h);
  std::vector<double> Kt, Vt, bb;
  b->materialize(nullptr, nullptr, Kt, Vt, bb);
  return (int)bb.size();
}
// [near || pseudo] as doubles: Kt, Vt [L][d], bias [L]; returns L (call pko_context_len first)
// positions (optional): stream position of every context element; rotate = 0 returns the keys un-rotated under FLAG_ROPE
int pko_materialize(void* h, const uint8_t* forced_codes_k, const uint8_t* forced_codes_v, double* Kt, double* Vt,
                    double* bias, double* positions, int rotate) {
  Bank* b = static_cast<Bank*>(h);
  std::vector<double> k, v, bb, ps;
  b->materialize(forced_codes_k, forced_codes_v, k, v, bb, &ps, rotate != 0);
  if (positions) std::memcpy(positions, ps.data(), ps.size() * sizeof(double));
  if (Kt) std::memcpy(Kt, k.data(), k.size() * sizeof(double));
  if (Vt) std::memcpy(Vt, v.data(), v.size() * sizeof(double));
  if (bias) std::memcpy(bias, bb.data(), bb.size() * sizeof(double));
  return (int)bb.size();
}

// Q [rows][d] fp32 (bf16 inputs widened exactly by the caller); out [rows][d] fp32; lse [rows] or NULL
int pko_attention(void* h, const float* Q, int rows, const uint8_t* forced_codes_k, const uint8_t* forced_codes_v,
                  float* out, double* lse, const int64_t* qpos) {
  Bank* b = static_cast<Bank*>(h);
  if (!b || !Q || !out || rows < 0) return 1;
  b->attention(Q, rows, forced_codes_k, forced_codes_v, out, lse, qpos);
  return 0;
}

}  // extern "C"
