"""Pins of the CPU oracle (oracle/) against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  The paper prints no worked numeric example, so the pins are
invariants, closed forms, brute force on tiny inputs and special cases that reduce to library routines.
"""
import itertools
import math

import numpy as np
import pytest
import torch

import gen
from helpers import make_oracle, frame_for_bank, query_rows_for_bank, codebooks_for_bank
from oracle import (OracleBank, DEFAULTS, FLAG_NEAR_ONLY, FLAG_FAR_ONLY, FLAG_NO_MASS_BIAS, FLAG_NO_RESIDUAL,
                    FLAG_MAH_SQUARED)

SMALL = gen.spec_for("c1")                       # BASELINE.json configs[0]


def run_stream(spec, o, n_frames, mode=0, bank=0, log=None, **kw):
    for f in range(n_frames):
        K, V, s = frame_for_bank(spec, f, bank)
        tr = o.append_frame(K, V, s, mode=mode, **kw)
        if log is not None:
            log.append((f, K, V, s, tr))
    return o


# ---------------------------------------------------------------------------------------------------------
# Table 5 defaults: golden text fixture
# ---------------------------------------------------------------------------------------------------------
def test_defaults_match_table5_golden():
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "table5_defaults.txt")
    gold = {}
    for line in open(path):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            gold[k.strip()] = float(v)
    for k, v in gold.items():
        assert float(DEFAULTS[k]) == pytest.approx(v, rel=1e-6), k


# ---------------------------------------------------------------------------------------------------------
# pin 1 + 2: mass conservation, histogram row sums (north_star invariant 1)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", [0, 1])
def test_mass_conservation_and_histogram_rows(mode):
    spec = SMALL
    o = make_oracle(spec)
    for f in range(spec.n_frames):
        K, V, s = frame_for_bank(spec, f, 0)
        o.append_frame(K, V, s, mode=mode)
        st = o.state()
        evicted = max(0, f + 1 - spec.near_frames) * spec.T
        assert int(st["n"].sum()) == evicted
        act = st["active"].astype(bool)
        assert act.sum() == min(evicted, spec.k_max)
        assert np.all(act[:act.sum()]) and not np.any(act[act.sum():])       # lowest free slot first (prefix)
        for H in (st["hist_k"], st["hist_v"]):
            rows = H.sum(axis=2)                                              # [k][G]
            assert np.all(rows == st["nres"][:, None])
        assert np.all(st["n"][act] - st["nres"][act].astype(np.int64) == 1)  # reading 8
        assert np.all(st["n"][~act] == 0)


# ---------------------------------------------------------------------------------------------------------
# pin 3: frame-synchronous with T=1 == sequential, bit for bit
# ---------------------------------------------------------------------------------------------------------
def test_sync_with_one_token_frames_equals_sequential():
    spec = gen.spec_for("c1", grid_h=1, grid_w=1, near_frames=5, k_max=6, n_frames=80)
    a, b = make_oracle(spec), make_oracle(spec)
    for f in range(spec.n_frames):
        K, V, s = frame_for_bank(spec, f, 0)
        s = np.array([[(f % 7 + 0.5) / 7, (f % 3 + 0.5) / 3]], np.float32)
        ta, tb = a.append_frame(K, V, s, mode=0), b.append_frame(K, V, s, mode=1)
        assert np.array_equal(ta["assign"], tb["assign"])
    sa, sb = a.state(), b.state()
    for k in sa:
        assert np.array_equal(sa[k], sb[k]), k


# ---------------------------------------------------------------------------------------------------------
# pin 4: sequential mode forced with a frame-synchronous run's assignments reproduces its state bit for bit
# ---------------------------------------------------------------------------------------------------------
def test_forced_replay_reproduces_state():
    spec = SMALL
    a, b = make_oracle(spec), make_oracle(spec)
    n_diff = 0
    for f in range(spec.n_frames):
        K, V, s = frame_for_bank(spec, f, 0)
        ta = a.append_frame(K, V, s, mode=0)
        tb = b.append_frame(K, V, s, mode=1, forced_assign=ta["assign"], forced_codes_k=ta["codes_k"],
                            forced_codes_v=ta["codes_v"])
        n_diff += int((ta["assign"] != tb["assign"]).sum())
        assert np.all(tb["forced_excess"] >= 0)
    sa, sb = a.state(), b.state()
    for k in sa:
        assert np.array_equal(sa[k], sb[k]), k
    # and a free-running sequential run agrees on most, not necessarily all, assignments (reading 1)
    c = make_oracle(spec)
    run_stream(spec, c, spec.n_frames, mode=1)
    assert int(c.state()["n"].sum()) == int(sa["n"].sum())


# ---------------------------------------------------------------------------------------------------------
# pin 5: brute-force recomputation of every statistic from the assignment log (numpy, fp64, own code)
# ---------------------------------------------------------------------------------------------------------
def _recompute_from_log(spec, log, ck, cv, alpha, beta, eta):
    """Independent re-derivation: EMA closed forms for c, p, mu; re-simulation for Sigma and H."""
    d, G, Cn = spec.head_dim, spec.G, spec.C
    sub = d // G
    members = {}                       # slot -> list of (K, V, s, frame t of absorption, stream position)
    for (f, K, V, s, tr) in log:
        if not tr["evicted"]:
            continue
        fe = f - spec.near_frames      # index of the evicted frame
        Ke, Ve, se = log[fe][1], log[fe][2], log[fe][3]
        for j in range(spec.T):
            members.setdefault(int(tr["assign"][j]), []).append((Ke[j], Ve[j], se[j], f, fe * spec.T + j))
    out = {}
    for k, lst in members.items():
        m = len(lst) - 1               # absorbed after the initialising token
        Ks = np.array([x[0] for x in lst], np.float64)
        Vs = np.array([x[1] for x in lst], np.float64)
        ss = np.array([x[2] for x in lst], np.float64)

        def ema(x, a):                 # (1-a)^m x_0 + a sum_j (1-a)^(m-j) x_j
            w = np.array([(1 - a) ** m] + [a * (1 - a) ** (m - j) for j in range(1, m + 1)])
            return (w[:, None] * x).sum(0)
        c, p, mu = ema(Ks, alpha), ema(Vs, beta), ema(ss, eta)
        # Sigma and H need the running centres: re-simulate in fp64
        cc, pp, mm = Ks[0].copy(), Vs[0].copy(), ss[0].copy()
        Sg = np.eye(2)
        HK = np.zeros((G, Cn), np.int64)
        HV = np.zeros((G, Cn), np.int64)
        for j in range(1, m + 1):
            cc = (1 - alpha) * cc + alpha * Ks[j]
            pp = (1 - beta) * pp + beta * Vs[j]
            mm = (1 - eta) * mm + eta * ss[j]
            dl = ss[j] - mm
            Sg = (1 - eta) * Sg + eta * np.outer(dl, dl)
            for (x, cen, cb, H) in ((Ks[j], cc, ck, HK), (Vs[j], pp, cv, HV)):
                r = (x - cen).reshape(G, 1, sub)
                dist = ((r - cb.astype(np.float64)) ** 2).sum(-1)          # [G][C]
                H[np.arange(G), dist.argmin(1)] += 1
        out[k] = dict(n=len(lst), c=c, p=p, mu=mu, sigma=np.array([Sg[0, 0], Sg[0, 1], Sg[1, 1]]), hk=HK, hv=HV,
                      tau=lst[-1][3], pos=lst[-1][4], nres=m)
    return out


def test_bruteforce_recomputation_matches_online_statistics():
    spec = SMALL
    o = make_oracle(spec)
    log = []
    run_stream(spec, o, spec.n_frames, log=log)
    ck, cv = codebooks_for_bank(spec, 0)
    a = float(np.float32(0.05))
    ref = _recompute_from_log(spec, log, ck, cv, a, a, a)
    st = o.state()
    assert sorted(ref) == list(range(int(st["active"].sum())))
    flips = 0
    for k, r in ref.items():
        assert st["n"][k] == r["n"] and st["nres"][k] == r["nres"]
        assert st["tau"][k] == r["tau"] and st["pos"][k] == r["pos"]
        np.testing.assert_allclose(st["c"][k], r["c"], rtol=1e-5, atol=2e-6)
        np.testing.assert_allclose(st["p"][k], r["p"], rtol=1e-5, atol=2e-6)
        np.testing.assert_allclose(st["mu"][k], r["mu"], rtol=1e-5, atol=1e-6)
        np.testing.assert_allclose(st["sigma"][k], r["sigma"], rtol=1e-4, atol=1e-7)
        # histogram bins may differ only where fp32-vs-fp64 state rounding flips a near-tie; count them
        flips += int(np.abs(st["hist_k"][k].astype(np.int64) - r["hk"]).sum() // 2)
        flips += int(np.abs(st["hist_v"][k].astype(np.int64) - r["hv"]).sum() // 2)
    total = int(st["nres"].sum()) * spec.G * 2
    assert flips <= max(2, total // 5000), (flips, total)


# ---------------------------------------------------------------------------------------------------------
# pin 6: constant stream closed forms
# ---------------------------------------------------------------------------------------------------------
def test_constant_stream_closed_forms():
    d, G, Cn, T = 16, 4, 5, 3
    rng = np.random.default_rng(1)
    ck = rng.normal(size=(G, Cn, d // G)).astype(np.float32)
    cv = rng.normal(size=(G, Cn, d // G)).astype(np.float32)
    o = OracleBank(T, 2, 1, d, ck, cv, G=G, C=Cn, S=2, beam=4)
    k0 = rng.normal(size=d).astype(np.float32)
    v0 = rng.normal(size=d).astype(np.float32)
    K, V = np.tile(k0, (T, 1)), np.tile(v0, (T, 1))
    s = np.tile(np.array([[0.25, 0.75]], np.float32), (T, 1))
    n_frames = 12
    for _ in range(n_frames):
        o.append_frame(K, V, s)
    st = o.state()
    m = (n_frames - 2) * T - 1
    assert st["n"][0] == m + 1 and st["nres"][0] == m
    assert np.array_equal(st["c"][0], k0) and np.array_equal(st["p"][0], v0)        # EMA of a constant is exact
    assert np.array_equal(st["mu"][0], s[0])
    eta = float(np.float32(0.05))
    np.testing.assert_allclose(st["sigma"][0], [(1 - eta) ** m, 0.0, (1 - eta) ** m], rtol=1e-5)
    zk = (ck.astype(np.float64) ** 2).sum(-1).argmin(1)                              # codeword nearest to 0
    zv = (cv.astype(np.float64) ** 2).sum(-1).argmin(1)
    for g in range(G):
        assert st["hist_k"][0, g, zk[g]] == m and st["hist_v"][0, g, zv[g]] == m


# ---------------------------------------------------------------------------------------------------------
# attention helpers: exact softmax attention written out in numpy fp64
# ---------------------------------------------------------------------------------------------------------
def exact_attention(Q, K, V, bias=None):
    Q, K, V = (np.asarray(x, np.float64) for x in (Q, K, V))
    A = Q @ K.T / math.sqrt(Q.shape[1])
    if bias is not None:
        A = A + np.asarray(bias, np.float64)[None, :]
    A = A - A.max(1, keepdims=True)
    W = np.exp(A)
    W /= W.sum(1, keepdims=True)
    return W @ V


# ---------------------------------------------------------------------------------------------------------
# pin 7: capacity >= evicted tokens, zero residuals: attention over the state == exact attention over the
# full history (S=1), or with +log S on every evicted token (S>1; reading 15)   (north_star invariant 2)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("S", [1, 3])
def test_full_capacity_equals_exact_attention_over_history(S):
    spec = gen.spec_for("c1", k_max=16 * 8, n_frames=12)          # 8 evicted frames * 16 tokens = 128 slots
    o = make_oracle(spec, with_codebooks=False, S=S, beam=4)
    log = []
    run_stream(spec, o, spec.n_frames, log=log)
    Kall = np.concatenate([x[1] for x in log])
    Vall = np.concatenate([x[2] for x in log])
    n_ev = (spec.n_frames - spec.near_frames) * spec.T
    Q = query_rows_for_bank(spec, gen.queries(spec), 0)
    bias = np.zeros(len(Kall))
    bias[:n_ev] = math.log(S)
    ref = exact_attention(Q, Kall, Vall, bias)
    out = o.attention(Q)
    np.testing.assert_allclose(out, ref, rtol=1e-5, atol=1e-6)
    assert o.materialize()[2].shape[0] == spec.near_frames * spec.T + n_ev * S


# ---------------------------------------------------------------------------------------------------------
# pin 8: a zero-residual prototype of mass m == m duplicated tokens (S=1); S*m duplicates in general
# (north_star invariant 3)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("S", [1, 2])
def test_mass_m_prototype_equals_m_duplicates(S):
    d, T = 8, 2
    rng = np.random.default_rng(3)
    o = OracleBank(T, 2, 4, d, None, None, S=S, beam=4)
    for _ in range(2):                                             # fill the near window only
        o.append_frame(rng.normal(size=(T, d)), rng.normal(size=(T, d)), rng.random(size=(T, 2)))
    c = rng.normal(size=(4, d)).astype(np.float32)
    p = rng.normal(size=(4, d)).astype(np.float32)
    masses = np.array([5, 1, 17, 0], np.int32)
    o.set_state(c=c, p=p, n=masses, active=np.array([1, 1, 1, 0], np.uint8))
    Kn, Vn, _, _ = o.ring()
    Kd = [Kn.reshape(-1, d)] + [np.tile(c[k], (S * masses[k], 1)) for k in range(3)]
    Vd = [Vn.reshape(-1, d)] + [np.tile(p[k], (S * masses[k], 1)) for k in range(3)]
    Q = rng.normal(size=(5, d)).astype(np.float32)
    ref = exact_attention(Q, np.concatenate(Kd), np.concatenate(Vd))
    np.testing.assert_allclose(o.attention(Q), ref, rtol=1e-5, atol=1e-6)


# ---------------------------------------------------------------------------------------------------------
# pin 9: against a library routine (torch SDPA on CPU): NEAR_ONLY == sliding-window attention; any state ==
# plain attention over the materialised [K~;V~] with additive mask b; NO_MASS_BIAS == b = 0; FAR_ONLY
# ---------------------------------------------------------------------------------------------------------
def _sdpa(Q, K, V, b=None):
    q = torch.from_numpy(np.asarray(Q, np.float64))[None]
    k = torch.from_numpy(np.asarray(K, np.float64))[None]
    v = torch.from_numpy(np.asarray(V, np.float64))[None]
    m = None if b is None else torch.from_numpy(np.asarray(b, np.float64))[None, None, :].expand(1, q.shape[1], -1)
    return torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=m)[0].numpy()


def test_attention_against_torch_sdpa():
    spec = SMALL
    Q = query_rows_for_bank(spec, gen.queries(spec), 0)
    for flags in (0, FLAG_NEAR_ONLY, FLAG_FAR_ONLY, FLAG_NO_MASS_BIAS):
        o = make_oracle(spec, flags=flags)
        run_stream(spec, o, 40)
        Kt, Vt, b = o.materialize()
        st = o.state()
        n_act = int(st["active"].sum())
        W = spec.near_frames * spec.T
        exp_len = {0: W + n_act * 8, FLAG_NEAR_ONLY: W, FLAG_FAR_ONLY: n_act * 8, FLAG_NO_MASS_BIAS: W + n_act * 8}
        assert len(b) == exp_len[flags]
        if flags == FLAG_NEAR_ONLY:
            Kn, Vn, _, _ = o.ring()
            assert np.array_equal(Kt, Kn.reshape(-1, spec.head_dim)) and np.all(b == 0)
        if flags == FLAG_NO_MASS_BIAS:
            assert np.all(b == 0)
        if flags == 0:                                            # Eq. 4: b = log n_k on pseudo tokens, 0 on near
            assert np.all(b[:W] == 0)
            np.testing.assert_allclose(b[W:], np.repeat(np.log(st["n"][:n_act].astype(np.float64)), 8))
            # pseudo keys = centre + concatenated codewords of the decoded tuple (Alg. 4 l.9)
            syn = o.synthesize()
            ck, cv = codebooks_for_bank(spec, 0)
            k = n_act - 1
            for s_ in (0, 7):
                z = syn["codes_k"][k, s_]
                r = np.concatenate([ck[g, z[g]] for g in range(spec.G)]) if not syn["zero"][k] else 0.0
                np.testing.assert_allclose(Kt[W + k * 8 + s_], st["c"][k].astype(np.float64) + r, rtol=0, atol=1e-12)
        out, lse = o.attention(Q, return_lse=True)
        ref = _sdpa(Q, Kt, Vt, b)
        np.testing.assert_allclose(out, ref, rtol=1e-5, atol=1e-6)
        A = np.asarray(Q, np.float64) @ Kt.T / math.sqrt(spec.head_dim) + b
        np.testing.assert_allclose(lse, torch.logsumexp(torch.from_numpy(A), 1).numpy(), rtol=1e-10)


# ---------------------------------------------------------------------------------------------------------
# pin 12: invariances and bounded footprint
# ---------------------------------------------------------------------------------------------------------
def test_attention_invariances_and_bounded_context():
    spec = SMALL
    o = make_oracle(spec)
    lens = []
    for f in range(spec.n_frames):
        K, V, s = frame_for_bank(spec, f, 0)
        o.append_frame(K, V, s)
        lens.append(o.materialize()[2].shape[0])
    L_context = spec.near_frames * spec.T + spec.k_max * 8
    assert max(lens) == L_context and all(x == L_context for x in lens[10:])
    st = o.state()
    det = st["sigma"][:, 0].astype(np.float64) * st["sigma"][:, 2] - st["sigma"][:, 1].astype(np.float64) ** 2
    assert np.all(st["sigma"][:, 0] >= 0) and np.all(st["sigma"][:, 2] >= 0) and np.all(det >= -1e-12)   # PSD
    Kt, Vt, b = o.materialize()
    Q = query_rows_for_bank(spec, gen.queries(spec), 0)
    ref = o.attention(Q)
    perm = np.random.default_rng(0).permutation(len(b))
    np.testing.assert_allclose(exact_attention(Q, Kt[perm], Vt[perm], b[perm]), ref, rtol=1e-5, atol=1e-6)
    np.testing.assert_allclose(exact_attention(Q, Kt, Vt, b + 3.7), ref, rtol=1e-5, atol=1e-6)


# ---------------------------------------------------------------------------------------------------------
# pin 10: assignment special cases (Eq. 1)
# ---------------------------------------------------------------------------------------------------------
def test_assignment_reduces_to_cosine_nearest_centroid():
    spec = SMALL
    o = make_oracle(spec, lambda_sp=0.0, lambda_idle=0.0)
    log = []
    run_stream(spec, o, 20, log=log)
    st = o.state()
    K, V, s = frame_for_bank(spec, 20, 0)
    tr = o.append_frame(K, V, s)
    Ke = log[20 - spec.near_frames][1].astype(np.float64)
    c = st["c"].astype(np.float64)
    cos = (Ke / np.linalg.norm(Ke, axis=1, keepdims=True)) @ (c / np.linalg.norm(c, axis=1, keepdims=True)).T
    assert tr["n_fill"] == 0
    assert np.array_equal(tr["assign"], cos.argmax(1))
    np.testing.assert_allclose(tr["best"], -cos.max(1), rtol=1e-6)
    srt = np.sort(cos, axis=1)
    np.testing.assert_allclose(tr["second"], -srt[:, -2], rtol=1e-6)


def test_mahalanobis_special_cases_and_idle_term():
    d = 8
    rng = np.random.default_rng(5)
    o = OracleBank(1, 1, 2, d, None, None, lambda_sp=1.0, lambda_idle=0.5, t_idle=10, sigma_eps=0.0)
    c = rng.normal(size=(2, d)).astype(np.float32)
    mu = np.array([[0.2, 0.3], [0.6, 0.1]], np.float32)
    o.set_state(c=c, p=c, n=[1, 1], active=[1, 1], mu=mu, sigma=[[1, 0, 1], [0.04, 0.01, 0.09]], tau=[0, 95])
    Ke = rng.normal(size=d).astype(np.float32)
    se = np.array([0.7, 0.9], np.float32)
    cos = [float(Ke.astype(np.float64) @ c[k] / np.linalg.norm(Ke.astype(np.float64)) / np.linalg.norm(c[k].astype(np.float64)))
           for k in range(2)]
    # Sigma = I, eps = 0  =>  d_Mah = Euclidean distance
    eu = float(np.linalg.norm(se.astype(np.float64) - mu[0]))
    assert o.score(Ke, se, 0, 5) == pytest.approx(-cos[0] + eu, rel=1e-6)
    # idle indicator is strict: t - tau > T_idle
    assert o.score(Ke, se, 0, 10) == pytest.approx(-cos[0] + eu, rel=1e-6)
    assert o.score(Ke, se, 0, 11) == pytest.approx(-cos[0] + eu + 0.5, rel=1e-6)
    # general 2x2 covariance against numpy's inverse
    Sg = np.array([[0.04, 0.01], [0.01, 0.09]], np.float32).astype(np.float64)
    dl = se.astype(np.float64) - mu[1]
    dm = math.sqrt(dl @ np.linalg.inv(Sg) @ dl)
    assert o.score(Ke, se, 1, 100) == pytest.approx(-cos[1] + dm, rel=1e-6)
    o2 = OracleBank(1, 1, 2, d, None, None, lambda_sp=1.0, lambda_idle=0.5, t_idle=10, sigma_eps=0.0,
                    flags=FLAG_MAH_SQUARED)
    o2.set_state(c=c, p=c, n=[1, 1], active=[1, 1], mu=mu, sigma=[[1, 0, 1], [0.04, 0.01, 0.09]], tau=[0, 95])
    assert o2.score(Ke, se, 1, 100) == pytest.approx(-cos[1] + dm * dm, rel=1e-6)
    # the regulariser is added to the diagonal before inversion (reading 4)
    o3 = OracleBank(1, 1, 2, d, None, None, lambda_sp=1.0, lambda_idle=0.0, sigma_eps=0.5)
    o3.set_state(c=c, p=c, n=[1, 1], active=[1, 1], mu=mu, sigma=[[1, 0, 1], [0.04, 0.01, 0.09]], tau=[0, 0])
    dm3 = math.sqrt(dl @ np.linalg.inv(Sg + np.float64(np.float32(0.5)) * np.eye(2)) @ dl)
    assert o3.score(Ke, se, 1, 0) == pytest.approx(-cos[1] + dm3, rel=1e-6)


# ---------------------------------------------------------------------------------------------------------
# pin 11: Alg. 3 beam search == brute-force top-S over all C^G tuples (small G, C), == enumeration of rank
# vectors with prod r_g <= S at full size; top-1 = per-subspace mode; one-hot histograms decode themselves
# ---------------------------------------------------------------------------------------------------------
def _bruteforce_top_s(q, S):
    """q [G][C] integer scores -> the S best tuples under (score desc, tuple lexicographic asc)."""
    G, Cn = q.shape
    items = []
    for z in itertools.product(range(Cn), repeat=G):
        items.append((-int(sum(q[g, z[g]] for g in range(G))), z))
    items.sort()
    return [z for _, z in items[:S]], [-a for a, _ in items[:S]]


@pytest.mark.parametrize("G,Cn,S,beam", [(3, 4, 5, 8), (4, 5, 8, 32), (2, 6, 8, 8), (5, 3, 6, 6)])
def test_beam_equals_bruteforce_small(G, Cn, S, beam):
    rng = np.random.default_rng(G * 100 + Cn)
    o = OracleBank(1, 1, 1, G * 2, None, None, G=G, C=Cn, S=S, beam=beam)
    for trial in range(60):
        kind = trial % 4
        if kind == 0:
            H = rng.integers(0, 3, size=(G, Cn))               # tie-heavy
        elif kind == 1:
            H = rng.integers(0, 50, size=(G, Cn))
        elif kind == 2:
            H = np.zeros((G, Cn), np.int64)
            H[np.arange(G), rng.integers(0, Cn, size=G)] = 1   # one-hot rows
        else:
            H = rng.permuted(np.tile(rng.integers(0, 9, size=Cn), (G, 1)), axis=1)   # permuted multisets
        H = H.astype(np.uint32)
        q = o.log_table(H)
        codes, scores = o.decode_hist(H)
        ref_z, ref_a = _bruteforce_top_s(q, S)
        assert [tuple(int(v) for v in z) for z in codes] == ref_z
        assert [int(a) for a in scores] == ref_a


def test_log_table_is_eq3_in_fixed_point():
    o = OracleBank(1, 1, 1, 16, None, None, pq_eps=1e-6)
    rng = np.random.default_rng(2)
    H = rng.integers(0, 1000, size=(8, 16)).astype(np.uint32)
    H[3] = 0
    q = o.log_table(H)
    P = (H.astype(np.float64) + 1e-6) / (H.sum(1, keepdims=True).astype(np.float64) + 16 * 1e-6)   # Eq. 3
    np.testing.assert_allclose(P.sum(1), 1.0, rtol=1e-12)
    assert np.array_equal(q, np.rint(np.log(P) * 2.0 ** 24).astype(np.int64))


def _rank_vector_top_s(q, S):
    """Full-size cross-check: only tuples whose per-subspace ranks multiply to <= S can be in the top S."""
    G, Cn = q.shape
    order = [sorted(range(Cn), key=lambda c: (-int(q[g, c]), c)) for g in range(G)]

    def rec(g, budget):
        if g == G:
            yield ()
            return
        for r in range(1, budget + 1):
            for rest in rec(g + 1, budget // r):
                yield (r,) + rest
    items = []
    for rv in rec(0, S):
        z = tuple(order[g][rv[g] - 1] for g in range(G))
        items.append((-int(sum(q[g, z[g]] for g in range(G))), z))
    items.sort()
    return [z for _, z in items[:S]], len(items)


def test_beam_full_size_against_rank_vector_enumeration():
    rng = np.random.default_rng(11)
    o = OracleBank(1, 1, 1, 16, None, None)                    # G=8, C=16, S=8, beam=32
    n_vec = None
    for trial in range(40):
        if trial % 3 == 0:
            H = rng.integers(0, 2, size=(8, 16))
        elif trial % 3 == 1:
            H = rng.multinomial(int(rng.integers(1, 400)), rng.dirichlet(np.ones(16) * 0.3), size=8)
        else:
            H = np.zeros((8, 16), np.int64)
            H[np.arange(8), rng.integers(0, 16, size=8)] = 7
        H = H.astype(np.uint32)
        q = o.log_table(H)
        codes, scores = o.decode_hist(H)
        ref, n_vec = _rank_vector_top_s(q, 8)
        assert [tuple(int(v) for v in z) for z in codes] == ref
        mode = tuple(int(np.lexsort((np.arange(16), -q[g]))[0]) for g in range(8))
        assert tuple(int(v) for v in codes[0]) == mode         # top-1 = per-subspace mode (lowest index on ties)
        assert int(scores[0]) == int(sum(q[g, mode[g]] for g in range(8)))
        assert all(scores[i] >= scores[i + 1] for i in range(7))
    assert n_vec == 253


def test_zero_nres_gives_zero_residuals_and_no_codebooks_flag():
    spec = SMALL
    o = make_oracle(spec)
    run_stream(spec, o, spec.near_frames + 1)                  # one evicted frame: 16 fills, nothing absorbed
    st = o.state()
    assert int(st["nres"].sum()) == 0
    Kt, Vt, b = o.materialize()
    W = spec.near_frames * spec.T
    for k in range(16):                                        # Alg. 4 l.3-4: all S pseudo-tokens == centre
        for s_ in range(8):
            assert np.array_equal(Kt[W + k * 8 + s_], st["c"][k].astype(np.float64))
            assert np.array_equal(Vt[W + k * 8 + s_], st["p"][k].astype(np.float64))
    assert np.all(o.synthesize()["zero"][:16] == 1) and np.all(o.synthesize()["zero"][16:] == 2)
    o2 = make_oracle(spec, flags=FLAG_NO_RESIDUAL)
    run_stream(spec, o2, 30)
    assert int(o2.state()["nres"].sum()) == 0 and int(o2.state()["hist_k"].sum()) == 0


# ---------------------------------------------------------------------------------------------------------
# pins 13 + 14 (closed forms of Alg. 1 l.11-13 after ONE absorption into a fresh slot): they pin
# the two statements the re-simulation of pin 5 only restates -- "Sigma uses delta = s_e - mu_NEW" (l.12 after l.11)
# and "the residual is taken after the token's own EMA step" (l.13 after l.8-9, reading 7).
#   slot opened by token 0: c = K0, p = V0, mu = s0, Sigma = I.  Token 1 absorbed:
#     mu' = (1-eta) s0 + eta s1,  delta = s1 - mu' = (1-eta)(s1 - s0)
#     Sigma' = (1-eta) I + eta (1-eta)^2 (s1-s0)(s1-s0)^T          [with the OLD mu it would be eta (s1-s0)(s1-s0)^T]
#     r^K = K1 - c' = (1-alpha)(K1 - K0),  r^V = (1-beta)(V1 - V0)  [before the EMA step it would be K1 - K0]
# ---------------------------------------------------------------------------------------------------------
def _one_absorption(alpha, beta, eta, ck=None, cv=None, G=2, Cn=2, d=8, seed=7):
    rng = np.random.default_rng(seed)
    K = rng.normal(size=(3, 1, d)).astype(np.float32)
    V = rng.normal(size=(3, 1, d)).astype(np.float32)
    s = np.array([[[0.125, 0.75]], [[0.875, 0.25]], [[0.5, 0.5]]], np.float32)
    o = OracleBank(1, 1, 1, d, ck, cv, G=G, C=Cn, S=1, beam=1, alpha=alpha, beta=beta, eta=eta)
    traces = [o.append_frame(K[f], V[f], s[f]) for f in range(3)]   # f=1 evicts token 0 (fill), f=2 evicts token 1
    assert traces[1]["n_fill"] == 1 and traces[2]["n_fill"] == 0 and traces[2]["assign"][0] == 0
    return o.state(), K[:, 0], V[:, 0], s[:, 0], traces


def test_sigma_after_one_absorption_closed_form():
    eta = 0.25
    st, K, V, s, _ = _one_absorption(0.5, 0.5, eta)
    ds = s[1].astype(np.float64) - s[0].astype(np.float64)
    want = (1 - eta) * np.eye(2) + eta * (1 - eta) ** 2 * np.outer(ds, ds)
    got = st["sigma"][0].astype(np.float64)
    assert np.allclose([got[0], got[1], got[2]], [want[0, 0], want[0, 1], want[1, 1]], rtol=0, atol=2e-7)
    wrong = (1 - eta) * np.eye(2) + eta * np.outer(ds, ds)                    # delta against the old mean
    assert abs(wrong[0, 0] - want[0, 0]) > 1e-2                               # the pin separates the two readings
    assert np.allclose(st["mu"][0], (1 - eta) * s[0] + eta * s[1], rtol=0, atol=1e-7)


def test_residual_is_taken_after_the_ema_step():
    alpha, beta, d, G = 0.5, 0.25, 8, 2
    sub = d // G
    _, K, V, s, _ = _one_absorption(alpha, beta, 0.05, d=d)                   # same seeded tokens, no codebooks yet
    # codeword 0 sits on the BEFORE-update residual K1-K0 (V1-V0), codeword 1 on the AFTER-update residual
    # (1-alpha)(K1-K0): the literal order of Alg. 1 must hit codeword 1 in every subspace, the other order codeword 0
    rk_before, rv_before = K[1] - K[0], V[1] - V[0]
    ck = np.stack([rk_before.reshape(G, sub), ((1 - alpha) * rk_before).reshape(G, sub)], axis=1).astype(np.float32)
    cv = np.stack([rv_before.reshape(G, sub), ((1 - beta) * rv_before).reshape(G, sub)], axis=1).astype(np.float32)
    for g in range(G):                                                        # the two candidates are well separated
        assert np.linalg.norm(ck[g, 0] - ck[g, 1]) > 0.05 and np.linalg.norm(cv[g, 0] - cv[g, 1]) > 0.05
    st, K2, V2, _, tr = _one_absorption(alpha, beta, 0.05, ck=ck, cv=cv, d=d)
    assert np.array_equal(K2, K) and np.array_equal(V2, V)
    assert np.array_equal(st["hist_k"][0], np.tile([0, 1], (G, 1)))
    assert np.array_equal(st["hist_v"][0], np.tile([0, 1], (G, 1)))
    assert st["nres"][0] == 1 and st["n"][0] == 2
    assert (tr[2]["codes_k"][0] == 1).all() and (tr[2]["codes_v"][0] == 1).all()
    assert np.allclose(st["c"][0], (1 - alpha) * K[0] + alpha * K[1], atol=1e-7)
