"""Pins of the oracle's Alg. 2 (PrototypeMaintenance) against what the paper
and the mathematics fix: conservation laws of merging, the closed form of the idle decay, the degenerate settings that
must reproduce the maintenance-free path bit for bit, and the recycling rule.  CPU only; nothing here touches the CUDA
path.  The readings of what Alg. 2 leaves open are DESIGN.md readings 20, 24-27."""
import math

import numpy as np
import pytest

import gen
from helpers import make_oracle, frame_for_bank
from oracle import OracleBank, FLAG_MAINTENANCE

SMALL = gen.spec_for("c1")


def _stream(o, spec, n_frames, mode=0):
    for f in range(n_frames):
        K, V, s = frame_for_bank(spec, f, 0)
        o.append_frame(K, V, s, mode=mode, trace=False)


# gamma = 0 and eps = 0: no decay (floor(n) = n), no pair is closer than 0, nothing to recycle => Alg. 1 alone
@pytest.mark.parametrize("mode", [0, 1])
def test_neutral_maintenance_is_the_plain_path_bit_for_bit(mode):
    spec = SMALL
    a = make_oracle(spec, t_idle=3)
    b = make_oracle(spec, t_idle=3, flags=FLAG_MAINTENANCE, gamma=0.0, eps_k=0.0, eps_v=0.0)
    _stream(a, spec, 40, mode)
    _stream(b, spec, 40, mode)
    sa, sb = a.state(), b.state()
    for f in sa:
        assert np.array_equal(sa[f], sb[f]), f
    assert b.maintenance_counters() == dict(decayed=0, merges=0, recycled=0)


# generalised mass invariant: sum n = absorbed - decayed + recycled; every used slot is active with n >= 1
# after a call; never-used slots stay free for Alg. 1 l.3-4
@pytest.mark.parametrize("mode", [0, 1])
def test_generalised_mass_invariant(mode):
    spec = gen.spec_for("c1", k_max=40)
    o = make_oracle(spec, flags=FLAG_MAINTENANCE, t_idle=2, gamma=0.3, eps_k=1.5, eps_v=1.5)
    seen = dict(decayed=0, merges=0, recycled=0)
    for f in range(spec.n_frames):
        K, V, s = frame_for_bank(spec, f, 0)
        o.append_frame(K, V, s, mode=mode, trace=False)
        st = o.state()
        c = o.maintenance_counters()
        absorbed = max(0, f + 1 - spec.near_frames) * spec.T
        assert int(st["n"].sum()) == absorbed - c["decayed"] + c["recycled"]
        act = st["active"].astype(bool)
        assert (st["n"][act] >= 1).all() and (st["n"][~act] == 0).all()
        na = int(act.sum())
        assert act[:na].all()                                     # the active set stays a prefix
        for H in (st["hist_k"], st["hist_v"]):
            assert np.all(H.sum(axis=2) == st["nres"][:, None])   # rows still sum to n_res (L310) after merges
        seen = c
    assert seen["decayed"] > 0 and seen["merges"] > 0 and seen["recycled"] >= seen["merges"]


def _two_cluster_state(o, spec, rng, n_proto=6):
    """A hand-made bank: prototypes 0, 2, 4 are copies of one point (+ tiny offsets), 1, 3, 5 of another."""
    st = o.state()
    d = spec.head_dim
    base = rng.normal(size=(2, 2, d)).astype(np.float32)          # [cluster][c|p][d]
    for k in range(n_proto):
        off = (0.001 * k * rng.normal(size=(2, d))).astype(np.float32)
        st["c"][k] = base[k % 2, 0] + off[0]
        st["p"][k] = base[k % 2, 1] + off[1]
        st["n"][k] = 3 + 2 * k
        st["nres"][k] = st["n"][k] - 1
        st["mu"][k] = rng.uniform(size=2)
        st["sigma"][k] = (0.5 + k, 0.01 * k, 0.25 + k)
        st["tau"][k] = 10 + k
        st["pos"][k] = 1000 + k
        st["active"][k] = 1
        for H in (st["hist_k"], st["hist_v"]):
            H[k] = 0
            for g in range(H.shape[1]):
                H[k, g, (g + k) % H.shape[2]] = st["nres"][k]
    return st


# merging: conservation of mass, of the mass-weighted centres / spatial means, of histograms and residual counts;
# the lower index survives; fields Alg. 2 does not list (Sigma, tau, pos) keep the survivor's values
def test_merge_conserves_weighted_sums_and_keeps_the_lower_index():
    spec = SMALL
    rng = np.random.default_rng(3)
    o = make_oracle(spec, flags=FLAG_MAINTENANCE, gamma=0.0, eps_k=0.2, eps_v=0.25, t_idle=10 ** 6)
    _stream(o, spec, spec.near_frames)                            # a full near window, nothing evicted yet
    st = _two_cluster_state(o, spec, rng)
    o.set_state(**st)
    o.maintain(50)
    af = o.state()
    m = o.maintenance_counters()
    assert m["merges"] == 4 and m["decayed"] == 0 and m["recycled"] == 4
    n0 = st["n"].astype(np.float64)
    for cl in (0, 1):                                             # survivors: slots 0 and 1
        grp = [cl, cl + 2, cl + 4]
        assert af["n"][cl] == st["n"][grp].sum()
        assert af["nres"][cl] == st["nres"][grp].sum()
        assert np.array_equal(af["hist_k"][cl], st["hist_k"][grp].sum(axis=0))
        assert np.array_equal(af["hist_v"][cl], st["hist_v"][grp].sum(axis=0))
        for f in ("c", "p", "mu"):
            want = (n0[grp, None] * st[f][grp].astype(np.float64)).sum(axis=0) / n0[grp].sum()
            assert np.allclose(af[f][cl], want, rtol=0, atol=2e-6), f
        assert np.array_equal(af["sigma"][cl], st["sigma"][cl]) and af["tau"][cl] == st["tau"][cl]
        assert af["pos"][cl] == st["pos"][cl]
    # the merged-away slots 2..5 were recycled in the same call from the newest frame's last tokens, in slot order
    K, V, s = frame_for_bank(spec, spec.near_frames - 1, 0)
    for r, k in enumerate((2, 3, 4, 5)):
        j = spec.T - 1 - r
        assert np.array_equal(af["c"][k], K[j]) and np.array_equal(af["p"][k], V[j])
        assert af["n"][k] == 1 and af["nres"][k] == 0 and af["tau"][k] == 50
        assert np.array_equal(af["mu"][k], s[j]) and np.array_equal(af["sigma"][k], [1, 0, 1])
        assert af["pos"][k] == (spec.near_frames - 1) * spec.T + j
        assert not af["hist_k"][k].any() and not af["hist_v"][k].any()
    assert not af["active"][6:].any()                            # never-used slots are not recycled (reading 24)


# two IDENTICAL prototypes merge into one of summed mass / histograms with unchanged centres
def test_merge_of_identical_prototypes():
    spec = SMALL
    o = make_oracle(spec, flags=FLAG_MAINTENANCE, gamma=0.0, eps_k=0.2, eps_v=0.25, t_idle=10 ** 6)
    _stream(o, spec, spec.near_frames)
    st = o.state()
    rng = np.random.default_rng(5)
    c, p = rng.normal(size=spec.head_dim).astype(np.float32), rng.normal(size=spec.head_dim).astype(np.float32)
    for k, n in ((0, 7), (1, 12)):
        st["c"][k], st["p"][k], st["n"][k], st["nres"][k], st["active"][k] = c, p, n, n - 1, 1
        st["mu"][k] = (0.25, 0.75)
        st["sigma"][k] = (1, 0, 1)
        st["hist_k"][k, :, k] = n - 1
        st["hist_v"][k, :, 3] = n - 1
    o.set_state(**st)
    o.maintain(9)
    af = o.state()
    assert np.array_equal(af["c"][0], c) and np.array_equal(af["p"][0], p) and af["n"][0] == 19 and af["nres"][0] == 17
    assert (af["hist_k"][0, :, 0] == 6).all() and (af["hist_k"][0, :, 1] == 11).all() and (af["hist_v"][0, :, 3] == 17).all()
    assert np.array_equal(af["mu"][0], np.float32([0.25, 0.75]))


# a pair is merged only if BOTH distances are below their thresholds (strict), and the test is on the L2 norm
def test_merge_needs_both_thresholds():
    spec = SMALL
    d = spec.head_dim
    for dk, dv, expect in ((0.19, 0.24, 1), (0.21, 0.24, 0), (0.19, 0.26, 0), (0.2000001, 0.1, 0)):
        o = make_oracle(spec, flags=FLAG_MAINTENANCE, gamma=0.0, eps_k=0.2, eps_v=0.25, t_idle=10 ** 6)
        _stream(o, spec, spec.near_frames)
        st = o.state()
        for k in (0, 1):
            st["c"][k] = 1.0
            st["p"][k] = -2.0
            st["n"][k], st["active"][k] = 5, 1
        st["c"][1, :4] += dk / 2.0                                  # ||c_0 - c_1|| = dk (4 coordinates x dk/2)
        st["p"][1, :4] += dv / 2.0
        o.set_state(**st)
        o.maintain(1)
        assert o.maintenance_counters()["merges"] == expect, (dk, dv)


# aging: n <- floor((1 - gamma) n) on every call while t - tau > T_idle (strict), down to 0, then the slot is recycled
def test_idle_decay_closed_form_then_recycling():
    spec = SMALL
    gamma = 0.25
    o = make_oracle(spec, flags=FLAG_MAINTENANCE, gamma=gamma, eps_k=0.0, eps_v=0.0, t_idle=5)
    _stream(o, spec, spec.near_frames)
    st = o.state()
    st["c"][0], st["p"][0], st["n"][0], st["tau"][0], st["active"][0] = 1.0, 2.0, 37, 10, 1
    st["c"][1], st["p"][1], st["n"][1], st["tau"][1], st["active"][1] = -1.0, 3.0, 50, 14, 1
    o.set_state(**st)
    g32 = float(np.float32(gamma))
    n0, n1 = 37, 50
    for t in range(11, 40):
        o.maintain(t)
        if n0 > 0 and t - 10 > 5:
            n0 = math.floor((1.0 - g32) * n0)
        if n1 > 0 and t - 14 > 5:
            n1 = math.floor((1.0 - g32) * n1)
        af = o.state()
        if n0 == 0:
            break
        assert af["n"][0] == n0 and af["n"][1] == n1, t
    assert n0 == 0 and t - 10 > 5
    # the call that took slot 0 to zero recycled it at once: mass 1, tau = t, centres of the newest frame's last token
    K, V, s = frame_for_bank(spec, spec.near_frames - 1, 0)
    assert af["n"][0] == 1 and af["tau"][0] == t and np.array_equal(af["c"][0], K[spec.T - 1])
    assert o.maintenance_counters()["recycled"] == 1
    # not idle (t - tau == T_idle is not "> T_idle"): untouched
    o2 = make_oracle(spec, flags=FLAG_MAINTENANCE, gamma=gamma, eps_k=0.0, eps_v=0.0, t_idle=5)
    _stream(o2, spec, spec.near_frames)
    st["n"][0], st["tau"][0] = 37, 10
    o2.set_state(**st)
    o2.maintain(15)
    assert o2.state()["n"][0] == 37
    o2.maintain(16)
    assert o2.state()["n"][0] == math.floor((1.0 - g32) * 37)


# frame-synchronous with one-token frames == literal per-token Alg. 1 + Alg. 2, bit for bit
def test_sync_one_token_frames_equals_sequential_with_maintenance():
    spec = gen.spec_for("c1", grid_h=1, grid_w=1, near_frames=5, k_max=6, n_frames=120)
    kw = dict(flags=FLAG_MAINTENANCE, t_idle=4, gamma=0.4, eps_k=2.0, eps_v=2.0)
    a, b = make_oracle(spec, **kw), make_oracle(spec, **kw)
    for f in range(spec.n_frames):
        K, V, s = frame_for_bank(spec, f, 0)
        s = np.array([[(f % 7 + 0.5) / 7, (f % 3 + 0.5) / 3]], np.float32)
        a.append_frame(K, V, s, mode=0, trace=False)
        b.append_frame(K, V, s, mode=1, trace=False)
    sa, sb = a.state(), b.state()
    for f in sa:
        assert np.array_equal(sa[f], sb[f]), f
    assert a.maintenance_counters() == b.maintenance_counters() and a.maintenance_counters()["recycled"] > 0
