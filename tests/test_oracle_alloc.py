"""Pins of the oracle's variance-aware pseudo-token allocation (D.3; DESIGN.md
readings 37-40): Var(H_k) against numpy's population variance of the multiset of codewords the histogram describes,
the integer shares against worked examples computed by hand from the stated rule, and the invariants the paper states
(total count S_tot = K_max S, so L_context is unchanged).  CPU only; nothing here touches the CUDA path."""
import numpy as np
import pytest

from oracle import OracleBank, FLAG_VAR_ALLOC


def _bank(k_max, S, G, C, sub, ck, cv, s_cap=32, flags=FLAG_VAR_ALLOC, beam=32):
    return OracleBank(1, 1, k_max, G * sub, ck, cv, S=S, G=G, C=C, beam=beam, s_cap=s_cap, flags=flags)


def _load(o, hk, hv, n=None):
    k_max = hk.shape[0]
    nres = hk.sum(axis=2)[:, 0].astype(np.uint32)
    o.set_state(hist_k=hk, hist_v=hv, nres=nres, n=(nres + 1).astype(np.int32) if n is None else n,
                active=np.ones(k_max, np.uint8), c=np.zeros((k_max, o.d), np.float32), p=np.zeros((k_max, o.d), np.float32),
                mu=np.zeros((k_max, 2), np.float32), sigma=np.tile(np.array([1, 0, 1], np.float32), (k_max, 1)))


# Var(H_k): expand each histogram row into the list of codewords it counts; the variance of the residual distribution is
# the population variance of that list summed over dimensions, subspaces and the two sides (numpy, fp64)
def test_variance_is_the_population_variance_of_the_counted_codewords():
    rng = np.random.default_rng(0)
    G, C, sub, k_max = 2, 4, 3, 6
    ck = rng.standard_normal((G, C, sub)).astype(np.float32)
    cv = rng.standard_normal((G, C, sub)).astype(np.float32)
    o = _bank(k_max, 2, G, C, sub, ck, cv)
    hk = np.zeros((k_max, G, C), np.uint32)
    hv = np.zeros((k_max, G, C), np.uint32)
    for k in range(k_max):
        tot = 3 + 2 * k
        for g in range(G):
            hk[k, g] = rng.multinomial(tot, np.ones(C) / C)
            hv[k, g] = rng.multinomial(tot, np.ones(C) / C)
    hk[0] = 0; hk[0, :, 1] = 3; hv[0] = 0; hv[0, :, 2] = 3         # all counts on one codeword: variance 0
    _load(o, hk, hv)
    v, _ = o.allocation()
    for k in range(k_max):
        want = 0.0
        for cb, H in ((ck, hk), (cv, hv)):
            for g in range(G):
                rows = np.repeat(cb[g].astype(np.float64), H[k, g], axis=0)
                want += np.var(rows, axis=0).sum()
        assert abs(v[k] / 2.0 ** 20 - want) < 1e-6 + 1e-9 * want, (k, v[k] / 2.0 ** 20, want)
    assert v[0] == 0


def _two_point(a=2.0):
    """G = 1, C = 2, sub = 1, key codewords {0, a}, value codewords {0, 0}: Var = a^2 p (1 - p), p = h1 / (h0 + h1)."""
    ck = np.array([[[0.0], [a]]], np.float32)
    cv = np.zeros((1, 2, 1), np.float32)
    return ck, cv


def _hists(pairs):
    hk = np.array([[list(p)] for p in pairs], np.uint32)             # [k][1][2]
    return hk, hk.copy()


# worked examples (reading 39), by hand.  k_max = 4, S = 2: S_tot = 8, one each => budget 4.
#   variances (a = 2): (1,1) -> 1, (1,3) -> 3/4, (0,4) -> 0;  v = [1, 1, 3/4, 0] 2^20, sum = 11/4 2^20
#   shares 4 v / sum = 16/11, 16/11, 12/11, 0 -> floor 1, 1, 1, 0 with remainders 5, 5, 1, 0 (in units of 2^18)
#   S = [2, 2, 2, 1], one unit left -> largest remainder, lowest index on the tie: S = [3, 2, 2, 1]
def test_worked_example_largest_remainder():
    ck, cv = _two_point()
    o = _bank(4, 2, 1, 2, 1, ck, cv)
    hk, hv = _hists([(1, 1), (1, 1), (1, 3), (0, 4)])
    _load(o, hk, hv)
    v, sk = o.allocation()
    assert list(v) == [2 ** 20, 2 ** 20, 3 * 2 ** 18, 0]
    assert list(sk) == [3, 2, 2, 1] and sk.sum() == 8
    # with the cap s_cap = 2 the same split is [2, 2, 2, 1]; the unit left goes to the only prototype below the cap
    o2 = _bank(4, 2, 1, 2, 1, ck, cv, s_cap=2)
    _load(o2, hk, hv)
    assert list(o2.allocation()[1]) == [2, 2, 2, 2]
    # one prototype holds all the variance: budget 4 -> S = [5, 1, 1, 1]; capped at 3 the surplus goes round in
    # (remainder, index) order: [3, 2, 2, 1] after the first round (2 units left for three prototypes)
    hk, hv = _hists([(2, 2), (0, 4), (0, 4), (0, 4)])
    o3 = _bank(4, 2, 1, 2, 1, ck, cv)
    _load(o3, hk, hv)
    assert list(o3.allocation()[1]) == [5, 1, 1, 1]
    o4 = _bank(4, 2, 1, 2, 1, ck, cv, s_cap=3)
    _load(o4, hk, hv)
    assert list(o4.allocation()[1]) == [3, 2, 2, 1]


# all variances zero (no residual statistics yet): the fixed default; flag off: S for everybody whatever the histograms
def test_degenerate_cases_fall_back_to_the_fixed_default():
    ck, cv = _two_point()
    hk, hv = _hists([(0, 4), (4, 0), (0, 1), (0, 2)])
    o = _bank(4, 2, 1, 2, 1, ck, cv)
    _load(o, hk, hv)
    assert list(o.allocation()[1]) == [2, 2, 2, 2]
    hk, hv = _hists([(1, 1), (1, 1), (1, 3), (0, 4)])
    o = _bank(4, 2, 1, 2, 1, ck, cv, flags=0)
    _load(o, hk, hv)
    assert list(o.allocation()[1]) == [2, 2, 2, 2]
    # inactive slots and slots of mass 0 get nothing and do not count against the one-each floor
    o = _bank(4, 2, 1, 2, 1, ck, cv)
    _load(o, hk, hv)
    o.set_state(active=np.array([1, 1, 0, 1], np.uint8))
    _, sk = o.allocation()
    assert sk[2] == 0 and sk.sum() == 8 and list(sk) == [4, 3, 0, 1]   # budget 5: 5/2 each -> 2 r 1, tie -> index 0


# invariants on random states: total = S_tot while the cap does not bind, 1 <= S_k <= s_cap, monotone in the variance,
# within one unit of the proportional share; the context the attention sees has exactly W + S_tot elements (L_context
# unchanged) and prototype k contributes S_k of them
def test_invariants_and_context_length():
    rng = np.random.default_rng(3)
    G, C, sub, k_max, S = 2, 4, 2, 24, 4
    ck = (0.3 * rng.standard_normal((G, C, sub))).astype(np.float32)
    cv = (0.3 * rng.standard_normal((G, C, sub))).astype(np.float32)
    for trial in range(20):
        o = _bank(k_max, S, G, C, sub, ck, cv, s_cap=32)
        hk = np.zeros((k_max, G, C), np.uint32)
        hv = np.zeros((k_max, G, C), np.uint32)
        for k in range(k_max):
            tot = int(rng.integers(0, 40))
            conc = rng.dirichlet(np.ones(C) * rng.choice([0.05, 1.0, 10.0]))
            for g in range(G):
                hk[k, g] = rng.multinomial(tot, conc)
                hv[k, g] = rng.multinomial(tot, conc)
        _load(o, hk, hv)
        v, sk = o.allocation()
        if v.sum() == 0:
            continue
        assert sk.min() >= 1 and sk.max() <= 32
        bud = k_max * S - k_max
        share = 1 + bud * v / v.sum()
        if share.max() <= 32:
            assert sk.sum() == k_max * S
            assert np.all(np.abs(sk - share) < 1.0 + 1e-9)
        order = np.argsort(v, kind="stable")
        assert np.all(np.diff(sk[order]) >= -0)                      # larger variance never gets fewer
        Kt, Vt, b = o.materialize()
        assert Kt.shape[0] == sk.sum()                                # near window is empty here
        syn = o.synthesize()
        assert np.array_equal(syn["s_count"], sk)
        # the S_k modes of a prototype are the top S_k of Alg. 3: a prefix of the top s_cap
        full = _bank(k_max, 32, G, C, sub, ck, cv, flags=0, beam=32)
        _load(full, hk, hv)
        ref = full.synthesize()
        for k in range(k_max):
            if syn["zero"][k] == 0:
                m = min(int(sk[k]), C ** G)
                assert np.array_equal(syn["codes_k"][k, :m], ref["codes_k"][k, :m])
                assert np.array_equal(syn["codes_v"][k, :m], ref["codes_v"][k, :m])
