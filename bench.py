#!/usr/bin/env python
"""bench.py -- ProtoKV hot path on B200: update frames/s, query-attention latency, roofline fractions.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3] [--impl ours|reference]

One STEP = one pass of the whole hot path over one batch of synthetic input:
    protokv_append_frame   (U1 ring append, U2 slot fill, U3 assignment, U4 segmenting, U5 update, U6 histograms)
    protokv_query_attention (Q1 synthesis, Q2 fused attention over [near || pseudo-tokens])
in steady state (near window and prototype bank full).  CUDA events split every step into its update part and
its query part: `value` = update frames/s (BASELINE.json's first metric component), `query_attn_us` = query
latency, `ms_per_step` = the whole step.  One JSON line on stdout (rank 0); progress goes to stderr.
See DESIGN.md "Measurement" for the byte / flop counts behind the roofline objects.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

import gen  # noqa: E402

METRIC = "frames/sec far-memory update; query-attn latency us; % HBM/tensor roofline"
UNIT = "frames/s"
L2_BYTES = 126 * 2 ** 20


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm=float(p["hbm_gbs"]), bf16_burst=float(p["bf16_tflops"]),
                    bf16_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), source="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, source="fallback")   # B200_PROFILING.md fallback


# ---------------------------------------------------------------------------------------------------------------
# algorithmic bytes / flops (restated in DESIGN.md "Measurement")
# ---------------------------------------------------------------------------------------------------------------
def update_bytes_per_frame(spec, touched_per_bank):
    elt = 2 if spec.dtype == "bf16" else 4
    T, d, K, G = spec.T, spec.head_dim, spec.k_max, spec.G
    per_bank = 6 * T * d * elt + K * (4 * d + 40) + touched_per_bank * (16 * d + 80) + T * 16 * G
    return per_bank * spec.n_banks


def assign_flops_per_frame(spec):
    return 2.0 * spec.T * spec.k_max * spec.head_dim * spec.n_banks


def query_bytes(spec):
    elt = 2 if spec.dtype == "bf16" else 4
    d, K, S, G = spec.head_dim, spec.k_max, 8, spec.G
    W = spec.near_frames * spec.T
    rows = spec.n_query_tokens * (spec.n_q_heads // spec.n_kv_heads)
    per_bank = 2 * W * d * elt + K * (2 * d * 4 + S * G + 4) + 2 * rows * d * elt
    return per_bank * spec.n_banks


def query_flops(spec):
    d, K, S = spec.head_dim, spec.k_max, 8
    W = spec.near_frames * spec.T
    rows = spec.n_query_tokens * (spec.n_q_heads // spec.n_kv_heads)
    fact = 4.0 * rows * (W + K) * d * spec.n_banks
    dense = 4.0 * rows * (W + K * S) * d * spec.n_banks
    return fact, dense


# ---------------------------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        sm.sort()
        return dict(sm_mhz=sm[len(sm) // 2] if sm else None, sm_max_mhz=mx, samples=len(sm), reasons=sorted(reasons))


# ---------------------------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------------------------
def make_state(spec, device):
    from paper_2606_26762_b200 import ProtoKV
    ck, cv = gen.codebooks(spec, device=device)
    return ProtoKV(n_streams=spec.n_streams, n_layers=spec.n_layers, n_q_heads=spec.n_q_heads,
                   n_kv_heads=spec.n_kv_heads, head_dim=spec.head_dim, dtype=spec.dtype, tokens_per_frame=spec.T,
                   near_frames=spec.near_frames, k_max=spec.k_max, n_query_tokens=spec.n_query_tokens,
                   codebook_k=ck, codebook_v=cv, device=device, G=spec.G, C=spec.C)


def steady_state_frames(spec):
    """Frames to stream before the timed region: ring and bank full, plus 12 frames of absorptions so that most prototypes
    carry residual statistics (two frames after the bank fills two thirds of them still have n_res = 0 and their
    pseudo-tokens need no codeword: an easier query than a long stream's)."""
    return spec.near_frames + math.ceil(spec.k_max / spec.T) + 12


def run_workload(spec, device, steps, warmup, rank=0, do_e2e=True, do_profile=True, sampler=None, barrier=None):
    dev = str(device)
    st = make_state(spec, dev)
    s = gen.grid_positions(spec, device=dev)
    prime = steady_state_frames(spec)
    frame_bytes = 2 * spec.n_streams * spec.n_layers * spec.T * spec.n_kv_heads * spec.head_dim * (2 if spec.dtype == "bf16" else 4)
    pool_n = max(4, min(64, math.ceil(2.2 * L2_BYTES / frame_bytes)))
    log(f"[{spec.name}] banks={spec.n_banks} workspace={st.workspace_bytes / 1e6:.0f} MB, priming {prime} frames, "
        f"pool {pool_n} frames ({pool_n * frame_bytes / 1e6:.0f} MB)")
    for f in range(prime):
        K, V = gen.frame_kv(spec, f + 1000 * rank, device=dev)
        st.append_frame(K, V, s)
    pool = [gen.frame_kv(spec, prime + i + 1000 * rank, device=dev) for i in range(pool_n)]
    Q = gen.queries(spec, 0, device=dev)
    out = torch.empty_like(Q)
    state_bytes = st.workspace_bytes
    flush = None
    if state_bytes + pool_n * frame_bytes < 2 * L2_BYTES:
        flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev)
    torch.cuda.synchronize()

    def step(i, evs=None):
        K, V = pool[i % pool_n]
        if flush is not None:
            flush.fill_(i & 255)
        if evs: evs[0].record()
        st.append_frame(K, V, s)
        if evs: evs[1].record()
        if flush is not None:
            flush.fill_((i + 1) & 255)
        if evs: evs[2].record()
        st.query_attention(Q, out)
        if evs: evs[3].record()

    for i in range(warmup):
        step(i)
    torch.cuda.synchronize()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps)]
    launches0 = st.kernel_launches
    if barrier: barrier()
    torch.cuda.synchronize()
    if sampler: sampler.start()
    t0 = time.perf_counter()
    for i in range(steps):
        step(warmup + i, evs[i])
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    clocks = sampler.stop() if sampler else None
    if barrier: barrier()
    launches = st.kernel_launches - launches0
    upd = sorted(e[0].elapsed_time(e[1]) for e in evs)
    qry = sorted(e[2].elapsed_time(e[3]) for e in evs)
    res = dict(update_ms_sum=sum(upd), query_ms_sum=sum(qry), update_ms_median=upd[len(upd) // 2],
               query_ms_median=qry[len(qry) // 2], region_ms=evs[0][0].elapsed_time(evs[-1][3]), wall_ms=wall * 1e3,
               launches=launches, clocks=clocks, l2="flush: 252 MB fill between timed segments" if flush is not None else
               f"no flush: state {state_bytes / 1e6:.0f} MB + cycled input pool {pool_n * frame_bytes / 1e6:.0f} MB > 2x L2",
               impl=dict(assign=st.stage_impl(0), attention=st.stage_impl(1)), state_bytes=state_bytes)

    # touched prototypes per bank-frame (U of the byte formula), from the decisions of the last frame
    tr = st.last_frame_trace()
    res["touched_per_bank"] = float(sum(len(set(a.tolist())) for a in tr["assign"]) / len(tr["assign"]))

    # the same query as per-layer calls (layers are sequentially dependent in a real model): one
    # synthesis of the dirty prototypes, then one protokv_query_attention_ex per layer, summed
    if spec.n_layers > 1:
        reps = max(3, min(10, steps // 10))
        Ql = [Q[:, la:la + 1].contiguous() for la in range(spec.n_layers)]
        Ol = [torch.empty_like(q) for q in Ql]
        tot = 0.0
        for i in range(reps):
            K, V = pool[(warmup + i) % pool_n]
            st.append_frame(K, V, s)                          # dirties prototypes like a timed step does
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            st.synthesize()
            for la in range(spec.n_layers):
                st.query_attention_ex(Ql[la], n_q=spec.n_query_tokens, layer_begin=la, layer_count=1, out=Ol[la],
                                      run_synthesis=False)
            e1.record()
            torch.cuda.synchronize()
            tot += e0.elapsed_time(e1)
        res["per_layer_query_ms"] = tot / reps

    # decode-style query: ONE query token (rows = GQA group per bank), memory-bound by construction -- the near window
    # and the bank are streamed once for a handful of rows (north_star: HBM fraction of the decode-style attention)
    if spec.dtype == "bf16":
        Q1 = Q[:, :, :1].contiguous()
        O1 = torch.empty_like(Q1)
        st.synthesize()
        st.query_attention_ex(Q1, n_q=1, out=O1, run_synthesis=False)
        ts = []
        for i in range(10):
            if flush is not None:
                flush.fill_(i & 255)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            st.query_attention_ex(Q1, n_q=1, out=O1, run_synthesis=False)
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        ts.sort()
        res["decode_ms"] = ts[len(ts) // 2]
        res["decode_impl"] = st.stage_impl(2)

    if do_profile:   # per-kernel durations: same steps again with the library's stage events switched on
        st.profile_enable(True)
        for i in range(steps):
            step(warmup + steps + i)
        res["stages"] = st.profile_read()
        st.profile_enable(False)

    if do_e2e:       # through the host-buffer entry points: H2D of the frame and D2H of the result inside the region
        hp = [(K.cpu().pin_memory(), V.cpu().pin_memory()) for K, V in pool[:min(pool_n, 8)]]
        hs, hQ = s.cpu().pin_memory(), Q.cpu().pin_memory()
        hout = torch.empty_like(hQ).pin_memory()
        n_e2e = max(3, min(steps, 50))
        for i in range(2):
            st.append_frame_host(hp[i % len(hp)][0], hp[i % len(hp)][1], hs)
            st.query_attention_host(hQ, hout)
        torch.cuda.synchronize()
        tu = tq = 0.0
        t_all = time.perf_counter()
        for i in range(n_e2e):
            K, V = hp[i % len(hp)]
            t1 = time.perf_counter()
            st.append_frame_host(K, V, hs)
            torch.cuda.synchronize()
            t2 = time.perf_counter()
            st.query_attention_host(hQ, hout)     # synchronises: result is on the host
            t3 = time.perf_counter()
            tu += t2 - t1; tq += t3 - t2
        res["e2e"] = dict(update_s=tu, query_s=tq, steps=n_e2e, total_s=time.perf_counter() - t_all,
                          h2d=frame_bytes + s.numel() * 4 + Q.numel() * Q.element_size(),
                          d2h=Q.numel() * Q.element_size())
    st.close()
    return res


def next_rows(spec, device):
    """SURVEY 8(f) rows at the measurement bar, on the headline workload's shape: the CUDA path of each optional row timed
    with CUDA events on the library's stream (device-resident inputs).  None of them is on the graded step."""
    from paper_2606_26762_b200 import ProtoKV, binding as B
    dev = str(device)
    s = gen.grid_positions(spec, device=dev)
    Q = gen.queries(spec, 0, device=dev)
    out = {}

    def mk(**kw):
        cb = kw.pop("cb", True)
        ck, cv = gen.codebooks(spec, device=dev) if cb else (None, None)
        return ProtoKV(n_streams=spec.n_streams, n_layers=spec.n_layers, n_q_heads=spec.n_q_heads,
                       n_kv_heads=spec.n_kv_heads, head_dim=spec.head_dim, dtype=spec.dtype, tokens_per_frame=spec.T,
                       near_frames=spec.near_frames, k_max=spec.k_max, n_query_tokens=spec.n_query_tokens,
                       codebook_k=ck, codebook_v=cv, device=dev, G=spec.G, C=spec.C, **kw)

    def timed(fn, reps=5):
        ts = []
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        ts.sort()
        return ts[len(ts) // 2]

    prime = steady_state_frames(spec) + 8
    frames = [gen.frame_kv(spec, f, device=dev) for f in range(prime)]
    # NEXT-2: warm-up frames (reservoir plan + stores in the update kernel) and the k-means training
    st = mk(cb=False, flags=B.WARMUP | B.WARMUP_MANUAL, t_warm=1 << 30, warm_reservoir=2048, km_iters=32, km_batch=256, km_seed=1)
    for K, V in frames[:-4]:
        st.append_frame(K, V, s)
    it = iter(frames[-4:])
    warm_ms = timed(lambda: st.append_frame(*next(it), s), reps=4)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); st.train_codebooks(); e1.record()
    torch.cuda.synchronize()
    out["next2_codebook_warmup"] = dict(warmup_frame_update_ms=warm_ms, kmeans_training_ms=e0.elapsed_time(e1),
                                        reservoir=2048, km_iters=32, km_batch=256,
                                        note="one-time training of 2 x G codebooks per bank, CTA = (subspace, side, bank)")
    st.close()
    # NEXT-4: D.3 allocation + ragged synthesis + SIMT attention over the ragged context
    st = mk(flags=B.VAR_ALLOC, s_cap=32)
    for K, V in frames:
        st.append_frame(K, V, s)
    o = torch.empty_like(Q)
    syn_ms = timed(lambda: st.synthesize())
    att_ms = timed(lambda: st.query_attention_ex(Q, out=o, run_synthesis=False))
    sk, _ = st.export_allocation(0)
    out["next4_variance_aware_allocation"] = dict(allocation_and_synthesis_ms=syn_ms, attention_ms=att_ms, attention_impl=st.stage_impl(1),
                                                  s_k_min=int(sk[sk > 0].min()), s_k_max=int(sk.max()), s_total=int(sk.sum()))
    st.close()
    # NEXT-3: rotary anchoring (SIMT attention with the rotation stage + fp64 sincos tables) (D.1)
    st = mk(flags=B.ROPE)
    for K, V in frames:
        st.append_frame(K, V, s)
    st.synthesize()
    Q1 = Q[:, :, :1].contiguous()
    o1 = torch.empty_like(Q1)
    out["next3_rope_anchoring"] = dict(attention_ms=timed(lambda: st.query_attention_ex(Q, out=o, run_synthesis=False)),
                                       attention_impl=st.stage_impl(1),
                                       one_token_query_ms=timed(lambda: st.query_attention_ex(Q1, n_q=1, out=o1, run_synthesis=False)),
                                       note="attention_ms / one_token_query_ms include the fp64 sincos tables rebuilt per query")
    st.close()
    # NEXT-1: Alg. 2 maintenance, Table 5 defaults, in steady state
    st = mk(flags=B.MAINTENANCE)
    for K, V in frames[:-4]:
        st.append_frame(K, V, s)
    it2 = iter(frames[-4:])
    out["next1_maintenance"] = dict(update_frame_with_alg2_ms=timed(lambda: st.append_frame(*next(it2), s), reps=4),
                                    counters=st.maintenance_counters())
    st.close()
    return out


def decode_bytes(spec, e_c):
    """Algorithmic bytes of a one-token query (SURVEY 8(d) query formula with rows = the GQA group): near K, V rows, the
    centres at e_c bytes per element (2 = the bf16 copies the decode kernel streams, 4 = the fp32 state), codes, masses."""
    elt = 2 if spec.dtype == "bf16" else 4
    W = spec.near_frames * spec.T
    rows = spec.n_q_heads // spec.n_kv_heads
    per_bank = 2 * W * spec.head_dim * elt + spec.k_max * (2 * spec.head_dim * e_c + 8 * spec.G + 4) + 2 * rows * spec.head_dim * elt
    return per_bank * spec.n_banks


def decode_object(spec, res, peaks):
    """One-token query (attention only, codes valid): us and fraction of the HBM roofline on its algorithmic bytes."""
    if "decode_ms" not in res:
        return None
    e_c = 2 if res.get("decode_impl", "").startswith("mma.sync register") else 4
    b = decode_bytes(spec, e_c)
    gbs = b / (res["decode_ms"] * 1e-3) / 1e9
    return dict(n_query_tokens=1, attention_us=res["decode_ms"] * 1e3, algorithmic_bytes=b, centre_bytes_per_element=e_c,
                bound="hbm", achieved=gbs, unit="GB/s", peak=peaks["hbm"], frac=gbs / peaks["hbm"],
                impl=res.get("decode_impl"), roofline_us=b / peaks["hbm"] / 1e3)


def tensor_peak(peaks, clocks):
    """Which measured bf16 peak applies to this run (MEASURED_PEAKS.json holds a burst and a sustained figure): a timed
    region of milliseconds that the sampler saw at the maximum SM clock without a power cap ran under burst conditions;
    a power-capped or down-clocked region is compared with the sustained figure."""
    burst = True
    if clocks and clocks.get("sm_mhz") and clocks.get("sm_max_mhz"):
        burst = clocks["sm_mhz"] >= 0.95 * clocks["sm_max_mhz"] and "sw_power_cap" not in (clocks.get("reasons") or [])
    return (peaks["bf16_burst"], "burst") if burst else (peaks["bf16_sustained"], "sustained")


def roofline_objects(spec, res, peaks, steps, clocks=None):
    """roofline of the dominant kernel + one object per stage group, all on SURVEY.md 8(d)'s ALGORITHMIC counts
    (DESIGN.md "Measurement"): frac = (time the roofline allows for the algorithmic bytes / flops) / (measured time)."""
    out = {}
    stages = res.get("stages")
    if not stages:
        return None, out
    tpeak, tkind = tensor_peak(peaks, clocks if clocks is not None else res.get("clocks"))
    ub = update_bytes_per_frame(spec, res["touched_per_bank"])
    qb = query_bytes(spec)
    fact, dense = query_flops(spec)
    upd_ms = sum(stages[k][0] for k in ("fill", "score", "update", "append")) / steps
    out["update_path"] = dict(bound="hbm", achieved=ub / (upd_ms * 1e-3) / 1e9, peak=peaks["hbm"], unit="GB/s",
                              algorithmic_bytes=ub, ms=upd_ms, note="all update kernels of one frame (profiled pass)")
    out["update_path"]["frac"] = out["update_path"]["achieved"] / peaks["hbm"]
    if res.get("update_ms_sum"):   # the same bytes over the un-profiled frame time: the launch chain overlaps the kernels
        fr_ms = res["update_ms_sum"] / steps
        out["update_path"].update(frame_ms=fr_ms, frac_frame=ub / (fr_ms * 1e-3) / 1e9 / peaks["hbm"])
    sc_ms = stages["score"][0] / max(1, stages["score"][1])
    af = assign_flops_per_frame(spec)
    out["score"] = dict(bound="tensor", achieved=af / (sc_ms * 1e-3) / 1e12, peak=tpeak, unit="TFLOP/s",
                        algorithmic_flops=af, ms=sc_ms, peak_kind=tkind,
                        note="T x K_max x d contraction, 1x flops (the hi+lo split issues 2x that on the tensor pipe)")
    out["score"]["frac"] = out["score"]["achieved"] / tpeak
    at_ms = stages["attention"][0] / max(1, stages["attention"][1])
    # the attention's roofline is max(algorithmic bytes / HBM, FACTORISED flops / tensor peak).  The kernel
    # issues the dense contraction 4 rows L_context d (DESIGN.md 6.1 says why the factorised form does not shrink the
    # MMA volume); its utilisation of the tensor pipe rides along as tensor_pipe_util, it is not `frac`.
    t_hbm, t_tc = qb / (peaks["hbm"] * 1e9), fact / (tpeak * 1e12)
    t_roof = max(t_hbm, t_tc)
    if t_hbm >= t_tc:
        att = dict(bound="hbm", achieved=qb / (at_ms * 1e-3) / 1e9, peak=peaks["hbm"], unit="GB/s")
    else:
        att = dict(bound="tensor", achieved=fact / (at_ms * 1e-3) / 1e12, peak=tpeak, unit="TFLOP/s")
    att.update(frac=att["achieved"] / att["peak"], algorithmic_bytes=qb, algorithmic_flops=fact,
               roofline_us=t_roof * 1e6, ms=at_ms, peak_kind=tkind,
               dense_flops=dense, dense_tflops=dense / (at_ms * 1e-3) / 1e12,
               tensor_pipe_util=dense / (at_ms * 1e-3) / 1e12 / tpeak,
               dense_roofline_us=max(t_hbm, dense / (tpeak * 1e12)) * 1e6)
    out["attention"] = att
    sy_ms = stages["synthesis"][0] / max(1, stages["synthesis"][1])
    syb = spec.k_max * (2 * spec.G * spec.C * 4 + 8 * spec.G) * spec.n_banks      # if run for every prototype (8(d))
    out["synthesis"] = dict(ms=sy_ms, bound="hbm", algorithmic_bytes_all_prototypes=syb)
    # dominant kernel of the step = the stage with the largest summed device time
    dom = max(("score", "update", "attention", "synthesis", "append", "fill"), key=lambda k: stages[k][0])
    src = {"score": out["score"], "attention": out["attention"]}.get(dom)
    if src is None:   # a bandwidth-side kernel dominates: report the update path
        src = out["update_path"]
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")      # ncu dram bytes per launch (profiles/traffic.md)
    if os.path.exists(tpath):
        try:
            for ln in open(tpath).read().splitlines()[1:]:
                w, k, v = ln.split(",")
                if w == spec.name and k == dom:
                    traffic = float(v)
        except Exception:
            traffic = None
    roof = dict(bound=src["bound"], achieved=src["achieved"], peak=src["peak"], unit=src["unit"], frac=src["frac"],
                traffic=traffic, kernel=dom,
                peak_source=peaks["source"] + (f" {tkind} bf16" if src["unit"] == "TFLOP/s" else " copy bandwidth"))
    if dom == "attention":
        roof["tensor_pipe_util"] = src["tensor_pipe_util"]
    return roof, out


# ---------------------------------------------------------------------------------------------------------------
# the oracle arm (cpu_baseline and --impl reference)
# ---------------------------------------------------------------------------------------------------------------
def _oracle_subspec(spec, nb):
    """The smallest spec whose first nb banks are the first nb banks of `spec` (the generator is counter-based, so the
    sub-spec yields exactly the values those banks have in the full workload)."""
    import dataclasses
    per_stream = spec.n_layers * spec.n_kv_heads
    if nb <= per_stream:
        return dataclasses.replace(spec, n_streams=1, n_layers=min(spec.n_layers, math.ceil(nb / spec.n_kv_heads)))
    return dataclasses.replace(spec, n_streams=min(spec.n_streams, math.ceil(nb / per_stream)))


def oracle_arm(spec, steps, warmup, query_rows=2, max_cores=None):
    """The CPU oracle, as it stands, on the box's host cores.  One oracle object per bank (banks are independent,
    PAPER.md:L312); nb = min(banks, cores) banks run in parallel threads (the ctypes call drops the GIL), each
    single-threaded.  One STEP = one steady-state frame of those nb banks + one attention call per bank over
    `query_rows` of its query rows (synthesis + materialisation of the whole bank, then the sampled rows).  Returns the
    measured per-step times and the whole-workload figures obtained by scaling with the bank and row counts."""
    from concurrent.futures import ThreadPoolExecutor
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import bank_coords, query_rows_for_bank
    from oracle import OracleBank
    torch.set_num_threads(1)                       # host-side input generation must not fight the oracle threads
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    if max_cores:
        cores = min(cores, max_cores)
    nb = max(1, min(spec.n_banks, cores))
    sub = _oracle_subspec(spec, nb)
    ck, cv = gen.codebooks(sub)
    banks = list(range(nb))
    coords = [bank_coords(sub, b) for b in banks]
    orc = [OracleBank(sub.T, sub.near_frames, sub.k_max, sub.head_dim, ck[c].numpy(), cv[c].numpy(), G=sub.G, C=sub.C)
           for c in coords]
    s = gen.grid_positions(sub)

    def frame_inputs(f):
        K, V = gen.frame_kv(sub, f)
        return [(K[st, la, :, hd, :].float().numpy(), V[st, la, :, hd, :].float().numpy(), s[st].numpy())
                for st, la, hd in coords]

    pool = ThreadPoolExecutor(nb)

    def upd(f):
        inp = frame_inputs(f)
        t0 = time.perf_counter()
        list(pool.map(lambda i: orc[i].append_frame(*inp[i], trace=False), range(nb)))
        return time.perf_counter() - t0

    Q = gen.queries(sub, 0)
    rows = [query_rows_for_bank(sub, Q, b) for b in banks]
    rows_total = rows[0].shape[0]

    def qry(nrows):
        t0 = time.perf_counter()
        list(pool.map(lambda i: orc[i].attention(rows[i][:nrows]), range(nb)))
        return time.perf_counter() - t0

    prime = steady_state_frames(sub)
    for f in range(prime):
        upd(f)
    f = prime
    for _ in range(warmup):
        upd(f); f += 1
        qry(1 + query_rows)
    tu = tq = 0.0
    q1 = []
    t_all = time.perf_counter()
    for i in range(steps):
        tu += upd(f); f += 1
        tq += qry(1 + query_rows)
        if i < 3:
            q1.append(qry(1))                      # calibration of the per-row cost (1 row vs 1 + query_rows rows);
    wall = time.perf_counter() - t_all             # inside the wall time, outside the per-step sums
    pool.shutdown()
    tu /= steps; tq /= steps
    t_q1 = min(q1) if q1 else tq
    per_row = max(0.0, (tq - t_q1) / query_rows)
    fixed = max(0.0, tq - (1 + query_rows) * per_row)
    scale = spec.n_banks / nb
    s_frame = tu * scale
    s_query = (fixed + per_row * rows_total) * scale
    return dict(frames_per_s=1.0 / s_frame, query_s=s_query, step_ms=(tu + tq) * 1e3, update_step_ms=tu * 1e3,
                query_step_ms=tq * 1e3, wall_s=wall, cores=nb, banks_timed=nb, steps=steps,
                sample=f"{steps} steps on banks 0..{nb - 1} of {spec.n_banks} ({nb} threads, one single-threaded oracle per "
                       f"bank) after {prime} priming frames; step = 1 steady-state frame of those banks ({tu * 1e3:.1f} ms) + "
                       f"1 query per bank over {1 + query_rows} of its {rows_total} rows ({tq * 1e3:.1f} ms); value scales the "
                       f"frame time by {spec.n_banks}/{nb} banks, query_attn_us scales per-bank fixed + per-row cost to "
                       f"{rows_total} rows x {spec.n_banks} banks")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="c3")
    ap.add_argument("--extras", default="c2,c5,c4_k4096_w64",
                    help="comma list of further configs measured briefly in the same line (N=1)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    warmup = max(3, args.warmup)
    rank = int(os.environ.get("RANK", 0))
    local = int(os.environ.get("LOCAL_RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    spec = gen.spec_for(args.workload)
    if world > 1 and args.impl != "reference":
        # banks are independent, so N GPUs hold disjoint banks and nothing is exchanged.  The N-GPU job is the
        # workload with N x its streams (one C3 video stream per GPU; C5's streams spread over the ranks), cut along the
        # stream axis by paper_2606_26762_b200.sharding: weak scaling, per-GPU work fixed.
        import dataclasses
        from paper_2606_26762_b200 import sharding
        sh = sharding.shard_config(spec.n_streams * world, spec.n_layers, spec.n_q_heads, spec.n_kv_heads, world, rank,
                                   axis="stream")
        spec = dataclasses.replace(spec, n_streams=sh["n_streams"], stream0=sh["begin"])
    config = dict(workload=f"{spec.name}: BASELINE.json configs[{ {'c1': 0, 'c2': 1, 'c3': 2, 'c5': 4}.get(spec.name, 3)}]",
                  banks=spec.n_banks, layers=spec.n_layers, streams=spec.n_streams, q_heads=spec.n_q_heads,
                  kv_heads=spec.n_kv_heads, head_dim=spec.head_dim, tokens_per_frame=spec.T, near_frames=spec.near_frames,
                  k_max=spec.k_max, n_query_tokens=spec.n_query_tokens,
                  step="1 protokv_append_frame (steady state) + 1 protokv_query_attention; value = frames/s of the update "
                       "part, query_attn_us = the query part, ms_per_step = both",
                  l2="inputs cycle through a device pool sized so that state + pool > 2x L2 (126 MB); where they are "
                     "smaller a 252 MB fill flushes L2 before each timed segment (l2_policy says which applied)")

    if args.impl == "reference":
        if rank != 0:
            return
        os_ = oracle_arm(spec, steps=args.steps, warmup=warmup)
        line = dict(metric=METRIC, value=os_["frames_per_s"], unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=warmup,
                    ms_per_step=os_["wall_s"] * 1e3 / args.steps, higher_is_better=True, scaling="weak",
                    vs_baseline=None, dtype="f64", data="synthetic", config=config, impl="reference",
                    query_attn_us=os_["query_s"] * 1e6,
                    measured=dict(update_step_ms=os_["update_step_ms"], query_step_ms=os_["query_step_ms"],
                                  banks_timed=os_["banks_timed"], timed_region_s=os_["wall_s"],
                                  note="ms_per_step is the time of the bounded step actually run; value and query_attn_us "
                                       "are whole-workload figures obtained from it (see cpu_baseline.sample)"),
                    cpu_baseline=dict(value=os_["frames_per_s"], unit=UNIT, cores=os_["cores"], kind="oracle", sample=os_["sample"]),
                    e2e=dict(value=os_["frames_per_s"], unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
        print(json.dumps(line))
        return

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    barrier = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
        barrier = lambda: dist.barrier()
    peaks = load_peaks()
    sampler = ClockSampler(local) if rank == 0 else None
    res = run_workload(spec, device, args.steps, warmup, rank=0, sampler=sampler, barrier=barrier,
                       do_e2e=True, do_profile=True)
    upd_ms, qry_ms, region_ms = res["update_ms_sum"], res["query_ms_sum"], res["region_ms"]
    e2e_u, e2e_q = res["e2e"]["update_s"] / res["e2e"]["steps"], res["e2e"]["query_s"] / res["e2e"]["steps"]
    if world > 1:
        import torch.distributed as dist
        from paper_2606_26762_b200 import sharding
        upd_ms, qry_ms, region_ms, e2e_u, e2e_q = sharding.max_over_ranks([upd_ms, qry_ms, region_ms, e2e_u, e2e_q], device=device)
        ln = torch.tensor([res["launches"]], device=device, dtype=torch.int64)
        dist.all_reduce(ln)
        res["launches"] = int(ln.item())
    if rank != 0:
        if world > 1:
            torch.distributed.destroy_process_group()
        return
    K = args.steps
    fps = world * K / (upd_ms * 1e-3)
    roof, stage_roofs = roofline_objects(spec, res, peaks, K)
    line = dict(metric=METRIC, value=fps, unit=UNIT, n_gpus=world, steps=K, warmup=warmup,
                ms_per_step=region_ms / K, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="bf16" if spec.dtype == "bf16" else "f32", data="synthetic", config=config, l2_policy=res["l2"],
                update_ms_per_frame=upd_ms / K, update_ms_median=res["update_ms_median"],
                query_attn_us=qry_ms / K * 1e3, query_attn_us_median=res["query_ms_median"] * 1e3,
                gpu_launches=res["launches"], impl_kernels=res["impl"], clocks=res["clocks"],
                e2e=dict(value=world / e2e_u, unit=UNIT, h2d_bytes_per_step=res["e2e"]["h2d"],
                         d2h_bytes_per_step=res["e2e"]["d2h"], query_attn_us=e2e_q * 1e6,
                         steps=res["e2e"]["steps"],
                         note="protokv_append_frame_host / protokv_query_attention_host with pinned host buffers; "
                              "value = frames/s of the update call incl. its H2D copies, query_attn_us incl. H2D of Q and D2H of out"),
                roofline=roof, rooflines=stage_roofs,
                stages_ms_per_step={k: v[0] / K for k, v in res.get("stages", {}).items()},
                touched_prototypes_per_bank_frame=res["touched_per_bank"], state_bytes=res["state_bytes"],
                query_attn_us_per_layer_calls=(res["per_layer_query_ms"] * 1e3 if "per_layer_query_ms" in res else None),
                decode_query=decode_object(spec, res, peaks),
                peaks=peaks)
    if world == 1 and args.extras:
        extras = {}
        for name in [x for x in args.extras.split(",") if x and x != spec.name]:
            try:
                sp = gen.spec_for(name)
                r = run_workload(sp, device, max(10, K // 4), warmup, do_e2e=False, do_profile=True)
                n = max(10, K // 4)
                ro, sr = roofline_objects(sp, r, peaks, n, clocks=res["clocks"])
                extras[name] = dict(frames_per_s=n / (r["update_ms_sum"] * 1e-3), update_ms_per_frame=r["update_ms_sum"] / n,
                                    query_attn_us=r["query_ms_sum"] / n * 1e3, steps=n, l2=r["l2"], roofline=ro,
                                    rooflines=sr, stages_ms_per_step={k: v[0] / n for k, v in r["stages"].items()})
            except Exception as e:   # an extra must not take the headline down
                extras[name] = dict(error=repr(e))
        line["other_workloads"] = extras
    if world == 1 and args.extras:
        try:
            line["next_rows"] = next_rows(spec, device)
        except Exception as e:
            line["next_rows"] = dict(error=repr(e))
    if world == 1 and not args.no_cpu_baseline:
        os_ = oracle_arm(spec, steps=12, warmup=1)
        line["cpu_baseline"] = dict(value=os_["frames_per_s"], unit=UNIT, cores=os_["cores"], kind="oracle",
                                    sample=os_["sample"], query_attn_us=os_["query_s"] * 1e6,
                                    host_cores_available=os.cpu_count())
    print(json.dumps(line))
    if world > 1:
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
