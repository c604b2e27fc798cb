"""Helpers of the -m gpu parity tests: drive the CUDA path (through the C ABI binding) and the CPU oracle on the
same seeded inputs, teacher-forced.  No ProtoKV arithmetic here."""
import numpy as np
import torch

import gen
from helpers import bank_coords, codebooks_for_bank, query_rows_for_bank
from oracle import OracleBank
from paper_2606_26762_b200 import ProtoKV

ASSIGN_GAP = 1e-5      # north_star: assignments bit-exact except where the fp32 score gap is below 1e-5
CODE_GAP = 1e-5        # same rule for the nearest-codeword decision, on the relative squared distance
STAT_RTOL, STAT_ATOL = 1e-4, 1e-6   # north_star: statistics within 1e-4 relative (abs floor: DESIGN.md reading 23)


def make_gpu(spec, with_codebooks=True, n_query_tokens=None, **hyper):
    cb = gen.codebooks(spec) if with_codebooks else (None, None)
    hyper.setdefault("G", spec.G)
    hyper.setdefault("C", spec.C)
    return ProtoKV(n_streams=spec.n_streams, n_layers=spec.n_layers, n_q_heads=spec.n_q_heads,
                   n_kv_heads=spec.n_kv_heads, head_dim=spec.head_dim, dtype=spec.dtype,
                   tokens_per_frame=spec.T, near_frames=spec.near_frames, k_max=spec.k_max,
                   n_query_tokens=n_query_tokens or spec.n_query_tokens,
                   codebook_k=cb[0], codebook_v=cb[1], **hyper)


def make_oracles(spec, banks, with_codebooks=True, **hyper):
    out = {}
    cb = gen.codebooks(spec) if with_codebooks else None
    hyper.setdefault("G", spec.G)
    hyper.setdefault("C", spec.C)
    for b in banks:
        ck = cv = None
        if with_codebooks:
            ck, cv = codebooks_for_bank(spec, b, cb)
        out[b] = OracleBank(spec.T, spec.near_frames, spec.k_max, spec.head_dim, ck, cv, **hyper)
    return out


def bank_frame(spec, K, V, s, bank):
    st, la, hd = bank_coords(spec, bank)
    return (K[st, la, :, hd, :].float().numpy(), V[st, la, :, hd, :].float().numpy(), s[st].numpy())


def compare_state(gs, os_, where=""):
    """GPU state dict vs oracle state dict of one bank."""
    for f in ("n", "tau", "pos", "nres", "active", "hist_k", "hist_v", "pos_first", "pos_sum", "pos_cnt"):
        assert np.array_equal(gs[f], os_[f]), f"{where}: {f} differs"
    act = os_["active"].astype(bool)
    for f in ("c", "p", "mu", "sigma"):
        a, b = gs[f][act], os_[f][act]
        err = np.abs(a - b)
        tol = STAT_RTOL * np.maximum(np.abs(a), np.abs(b)) + STAT_ATOL
        assert (err <= tol).all(), f"{where}: {f} max err {err.max():.3e}"


def _follow_bank(spec, f, b, o, Kb, Vb, sb, tr, with_codebooks):
    """Oracle side of one bank-frame: checks the GPU's decisions against the oracle's own and advances the oracle in
    follow mode.  Returns the counters of this bank-frame.  Runs on a worker thread (ctypes drops the GIL)."""
    st = new_stats()
    _check_bank_frame(spec, f, b, o, Kb, Vb, sb, tr, st, with_codebooks)
    return st


def step_teacher_forced(spec, gpu, oracles, f, K, V, s, stats, with_codebooks=True, pool=None):
    """Append frame f on the GPU, check its decisions against the oracle's own, then advance every oracle bank with
    the GPU's decisions (follow mode).  K, V, s may live on the device (only the followed banks are pulled to the
    host); with a thread pool the oracle banks advance in parallel."""
    dev = gpu.device
    gpu.append_frame(K.to(dev), V.to(dev), s.to(dev))
    tr = gpu.last_frame_trace()
    if K.is_cuda:
        s_host = s.cpu()
        frames = {}
        for b in oracles:
            st_, la, hd = bank_coords(spec, b)
            frames[b] = (K[st_, la, :, hd, :].float().cpu().numpy(), V[st_, la, :, hd, :].float().cpu().numpy(),
                         s_host[st_].numpy())
    else:
        frames = {b: bank_frame(spec, K, V, s, b) for b in oracles}
    if pool is not None:
        futs = [pool.submit(_follow_bank, spec, f, b, o, *frames[b], tr, with_codebooks) for b, o in oracles.items()]
        for fu in futs:
            for k, v in fu.result().items():
                stats[k] = max(stats[k], v) if k == "max_score_err" else stats[k] + v
        return
    for b, o in oracles.items():
        _check_bank_frame(spec, f, b, o, *frames[b], tr, stats, with_codebooks)


def _check_bank_frame(spec, f, b, o, Kb, Vb, sb, tr, stats, with_codebooks):
    ga = tr["assign"][b]
    evicted = tr["evicted_frame"] >= 0
    forced = ga.copy()
    fk = tr["codes_k"][b] if with_codebooks else None
    fv = tr["codes_v"][b] if with_codebooks else None
    if evicted and with_codebooks:
        # fills carry 255 in the GPU trace; the oracle ignores forced codes for fills
        fk = np.where(fk == 255, 0, fk).astype(np.uint8)
        fv = np.where(fv == 255, 0, fv).astype(np.uint8)
    ot = o.append_frame(Kb, Vb, sb, mode=0, forced_assign=forced if evicted else None,
                        forced_codes_k=fk if evicted else None, forced_codes_v=fv if evicted else None)
    assert bool(ot["evicted"]) == evicted, f"frame {f} bank {b}: eviction mismatch"
    if not evicted:
        assert (ga == -1).all()
        return
    assert ot["n_fill"] == tr["n_fill"]
    nf = ot["n_fill"]
    assert np.array_equal(ga[:nf], ot["assign"][:nf]), f"frame {f} bank {b}: slot fill differs"
    diff = ga[nf:] != ot["assign"][nf:]
    excess = ot["forced_excess"][nf:]
    bad = diff & ~(excess <= ASSIGN_GAP)
    assert not bad.any(), (f"frame {f} bank {b}: {bad.sum()} assignments differ beyond the 1e-5 gap rule; "
                           f"worst excess {excess[bad].max():.3e}")
    stats["scored"] += int(diff.size)
    stats["assign_flips"] += int(diff.sum())
    # the GPU's score of its choice vs the oracle's score of that choice
    sc_err = np.abs(tr["best"][b][nf:] - (ot["best"][nf:] + excess))
    stats["max_score_err"] = max(stats["max_score_err"], float(sc_err.max()) if sc_err.size else 0.0)
    assert (sc_err <= ASSIGN_GAP).all(), f"frame {f} bank {b}: score error {sc_err.max():.3e}"
    if with_codebooks:
        for name, gc, oc, gap in (("K", tr["codes_k"][b], ot["codes_k"], ot["code_gap_k"]),
                                  ("V", tr["codes_v"][b], ot["codes_v"], ot["code_gap_v"])):
            assert (gc[:nf] == 255).all()
            d = gc[nf:] != oc[nf:]
            badc = d & ~(gap[nf:] <= CODE_GAP)
            assert not badc.any(), f"frame {f} bank {b}: {badc.sum()} PQ codes ({name}) differ beyond the gap rule"
            stats["codes"] += int(d.size)
            stats["code_flips"] += int(d.sum())


def new_stats():
    return dict(scored=0, assign_flips=0, max_score_err=0.0, codes=0, code_flips=0)


def run_stream(spec, gpu, oracles, n_frames, check_state_every=8, with_codebooks=True, stats=None, first_frame=0,
               on_device=False, pool=None, after_frame=None):
    """Teacher-forced stream of frames [first_frame, first_frame + n_frames).  on_device: frames are generated on the
    GPU (bit-identical generator) and only the followed banks are pulled to the host -- what makes the full-length
    streams of BASELINE.json's configs affordable.  after_frame(f) is called after frame f has been checked."""
    stats = stats if stats is not None else new_stats()
    dev = str(gpu.device) if on_device else "cpu"
    s = gen.grid_positions(spec, device=dev)
    for f in range(first_frame, first_frame + n_frames):
        K, V = gen.frame_kv(spec, f, device=dev)
        step_teacher_forced(spec, gpu, oracles, f, K, V, s, stats, with_codebooks, pool=pool)
        if check_state_every and ((f + 1) % check_state_every == 0 or f == first_frame + n_frames - 1):
            for b, o in oracles.items():
                compare_state(gpu.export_state(b), o.state(), f"frame {f} bank {b}")
        if after_frame is not None:
            after_frame(f)
    return stats


def compare_ring(gpu, oracles):
    for b, o in oracles.items():
        gK, gV, gs, gi = gpu.export_ring(b)
        oK, oV, os_, oi = o.ring()
        assert np.array_equal(gi, oi) and np.array_equal(gK, oK) and np.array_equal(gV, oV) and np.array_equal(gs, os_), \
            f"bank {b}: near window differs"


def compare_codes(gpu, oracles, G):
    """Synthesis parity (DESIGN.md "Parity protocol" iii): GPU codes equal the oracle's, or differ only in tuples
    whose oracle score is within G fixed-point units of the oracle's S-th score."""
    gpu.synthesize()
    flips = 0
    for b, o in oracles.items():
        gk, gv, kind = gpu.export_codes(b)
        syn = o.synthesize()
        assert np.array_equal(kind, syn["zero"]), f"bank {b}: kind differs"
        dec = np.nonzero(kind == 0)[0]
        for which, g_codes, o_codes, o_scores in ((0, gk, syn["codes_k"], syn["scores_k"]),
                                                  (1, gv, syn["codes_v"], syn["scores_v"])):
            neq = np.nonzero((g_codes[dec] != o_codes[dec]).any(axis=(1, 2)))[0]
            for k in dec[neq]:
                flips += 1
                sth = o_scores[k][-1]
                for s in range(g_codes.shape[1]):
                    if not np.array_equal(g_codes[k, s], o_codes[k, s]):
                        sc = o.tuple_score(int(k), which, g_codes[k, s])
                        assert abs(sc - o_scores[k][s]) <= G and sc >= sth - G, \
                            f"bank {b} prototype {k}: decoded tuple {s} differs beyond a last-bit tie"
    return flips


def attention_tolerance(spec):
    # north_star: 1e-2 absolute and 2e-2 relative for bf16 with fp32 accumulation; fp32 inputs: DESIGN.md derives 2e-4
    return (1e-2, 2e-2) if spec.dtype == "bf16" else (2e-4, 2e-4)


def compare_attention(spec, gpu, oracles, Q, n_q=None, layer_begin=0, layer_count=None, run_synthesis=True,
                      use_gpu_codes=False, rows_sample=None, q_pos0=None):
    """GPU attention of all banks vs the oracle on the given banks.  Q: CPU tensor in the ABI layout
    [n_streams][layer_count][n_q][Hq][d]."""
    n_q = Q.shape[2]
    layer_count = Q.shape[1]
    out, lse = gpu.query_attention_ex(Q.to(gpu.device), n_q=n_q, layer_begin=layer_begin, layer_count=layer_count,
                                      return_lse=True, run_synthesis=run_synthesis, q_pos0=q_pos0)
    out = out.float().cpu()
    lse = lse.cpu().numpy()
    atol, rtol = attention_tolerance(spec)
    group = spec.n_q_heads // spec.n_kv_heads
    worst = 0.0
    for b, o in oracles.items():
        st, la, hd = bank_coords(spec, b)
        if not (layer_begin <= la < layer_begin + layer_count):
            continue
        ll = la - layer_begin
        q = Q[st, ll, :, hd * group:(hd + 1) * group, :].float().numpy().reshape(-1, spec.head_dim)
        g = out[st, ll, :, hd * group:(hd + 1) * group, :].numpy().reshape(-1, spec.head_dim)
        gl = lse[st, ll, :, hd * group:(hd + 1) * group].reshape(-1)
        rows = np.arange(q.shape[0]) if rows_sample is None else np.asarray(rows_sample)
        fk = fv = None
        if use_gpu_codes:
            fk, fv, _ = gpu.export_codes(b)
        # query token i sits at q_pos0 + i (default: the next stream position); row = token * group + head.  Ignored by
        # the oracle unless FLAG_ROPE is set.
        qp0 = q_pos0 if q_pos0 is not None else int(gpu.cfg.pos0) + gpu.frames_seen * spec.T
        qpos = (qp0 + rows // group).astype(np.int64)
        ref, rl = o.attention(q[rows], forced_codes_k=fk, forced_codes_v=fv, return_lse=True, qpos=qpos)
        ref_r = torch.from_numpy(ref).to(spec.torch_dtype).float().numpy()   # output rounded to the I/O dtype
        err = np.abs(g[rows] - ref_r)
        tol = atol + rtol * np.abs(ref_r)
        assert (err <= tol).all(), f"bank {b}: attention max err {err.max():.3e}"
        worst = max(worst, float(err.max()))
        fin = np.isfinite(rl)
        assert np.array_equal(np.isfinite(gl[rows]), fin)
        if fin.any():
            assert np.abs(gl[rows][fin] - rl[fin]).max() <= 5e-3, f"bank {b}: lse differs"
    return worst
