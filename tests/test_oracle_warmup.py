"""Pins of the oracle's PQ codebook warm-up (readings 32-36):
the counter-based generator against the published SplitMix64 test vector, the reservoir against the definition of
uniform sampling and against residuals recomputed in numpy, mini-batch k-means against closed forms (running mean),
against well-separated blobs and against scikit-learn's KMeans.  CPU only; nothing here touches the CUDA path."""
import numpy as np
import pytest

import gen
from helpers import frame_for_bank
from oracle import OracleBank, FLAG_WARMUP, FLAG_WARMUP_MANUAL

GOLD = __import__("os").path.join(__import__("os").path.dirname(__file__), "golden", "splitmix64_seed0.txt")


def _bank(T=1, near=1, k_max=1, d=4, G=1, C=2, R=64, iters=8, batch=32, seed=0, t_warm=10 ** 6, manual=True, **kw):
    flags = FLAG_WARMUP | (FLAG_WARMUP_MANUAL if manual else 0)
    return OracleBank(T, near, k_max, d, None, None, G=G, C=C, S=min(2, C ** G), beam=min(2, C ** G), flags=flags,
                      t_warm=t_warm, warm_reservoir=R, km_iters=iters, km_batch=batch, km_seed=seed, **kw)


# the generator is SplitMix64's output function: draw(stream, i) = mix(seed ^ mix(2 i + stream)); mix(0) is the first
# output of the reference generator seeded with 0 (value from the reference implementation's published test vector)
def test_generator_is_splitmix64():
    want = [int(x, 16) for x in open(GOLD).read().split("#")[0].split()]
    o = _bank(seed=0)
    mask = (1 << 64) - 1

    def mix(x):   # the published sequence: state += golden gamma each call; output function of the new state
        z = (x + 0x9E3779B97F4A7C15) & mask
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & mask
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & mask
        return z ^ (z >> 31)
    assert mix(0) == want[0]                                  # pins the python restatement to the published vector
    assert mix(0x9E3779B97F4A7C15) == want[1]
    for stream in (0, 1):
        for i in (0, 1, 7, 12345678901):
            assert o.draw(stream, i) == mix(0 ^ mix(2 * i + stream))
    o2 = _bank(seed=0xDEADBEEF)
    assert o2.draw(1, 5) == mix(0xDEADBEEF ^ mix(11))


# Algorithm R: the first R offers fill the slots in order; offer i >= R lands with probability R / (i + 1); every offer
# survives to the end with probability R / N (the definition of a uniform sample of the stream)
def test_reservoir_is_a_uniform_sample():
    R, N, trials = 8, 96, 600
    kept = np.zeros(N)
    for seed in range(trials):
        o = _bank(R=R, seed=seed)
        owner = {}
        for i in range(N):
            s = o.reservoir_slot(i)
            if i < R:
                assert s == i
            assert -1 <= s < R
            if s >= 0:
                owner[s] = i
        for i in owner.values():
            kept[i] += 1
    p = R / N
    sd = np.sqrt(trials * p * (1 - p))
    assert np.all(np.abs(kept - trials * p) < 5 * sd), (kept.min(), kept.max(), trials * p)
    assert abs(kept.sum() - trials * R) < 1e-9


# one prototype, one token per frame: residual i is K_i - c_i with c_i the EMA after absorbing K_i (reading 7); with
# R >= all residuals the reservoir holds them in order; recomputed in numpy fp64 from the inputs alone
def test_reservoir_rows_are_the_residuals_of_the_updated_centres():
    rng = np.random.default_rng(5)
    d, n = 4, 30
    K = rng.standard_normal((n, d)).astype(np.float32)
    V = rng.standard_normal((n, d)).astype(np.float32)
    o = _bank(d=d, R=64, alpha=0.25, beta=0.5)
    s = np.array([[0.5, 0.5]], np.float32)
    for i in range(n):
        o.append_frame(K[i:i + 1], V[i:i + 1], s, trace=False)
    rk, rv, seen = o.reservoir()
    # frame 0 is evicted at step 1 and fills the slot; frames 1..n-2 are absorbed at steps 2..n-1
    assert seen == n - 2 and rk.shape == (n - 2, d)
    c, p = K[0].astype(np.float64), V[0].astype(np.float64)
    for i in range(1, n - 1):
        c = np.float32(0.75 * c + 0.25 * K[i]).astype(np.float64)
        p = np.float32(0.5 * p + 0.5 * V[i]).astype(np.float64)
        assert np.allclose(rk[i - 1], K[i] - c, rtol=0, atol=1e-6)
        assert np.allclose(rv[i - 1], V[i] - p, rtol=0, atol=1e-6)
    # residuals of steps t >= t_warm are not collected
    o2 = _bank(d=d, R=64, t_warm=10)
    for i in range(n):
        o2.append_frame(K[i:i + 1], V[i:i + 1], s, trace=False)
    assert o2.reservoir()[2] == 8          # absorptions at steps 2..9


# C = 1: every sample goes to the only centre and the rate 1 / v makes it the running mean of the samples drawn
# (Sculley 2010); the draws are with replacement from the reservoir, so the centre estimates the data mean with
# standard error sigma / sqrt(iters * batch) whatever the seed
def test_single_centre_is_the_running_mean():
    rng = np.random.default_rng(1)
    n, d = 64, 4
    X = (rng.standard_normal((n, d)) + np.array([3.0, -1.0, 0.5, 10.0])).astype(np.float32)
    for seed in (0, 1, 2):
        o = _bank(d=d, G=1, C=1, R=64, iters=40, batch=100, seed=seed)
        o.set_reservoir(X, 2 * X)
        assert o.train_codebooks() == 1
        ck, cv = o.codebooks()
        se = X.std(axis=0) / np.sqrt(4000)
        assert np.all(np.abs(ck[0, 0] - X.mean(axis=0)) < 6 * se)
        assert np.allclose(cv, 2 * ck, rtol=1e-5)          # same rows drawn for both sides, linear update
    # identical rows: the centre is that row (up to the rounding of (1 - eta) x + eta x)
    o = _bank(d=d, G=1, C=1, R=64, iters=3, batch=10)
    row = np.array([[1.25, -2.5, 3.0, 0.1]], np.float32).repeat(8, 0)
    o.set_reservoir(row, row)
    o.train_codebooks()
    assert np.allclose(o.codebooks()[0][0, 0], row[0], rtol=1e-6)


def _blobs(rng, C, per, sub, G, spread=0.01):
    """C well-separated blobs per subspace, rows grouped by blob so that the strided initialisation hits every blob."""
    centres = rng.standard_normal((G, C, sub)) * 10.0
    X = np.zeros((C * per, G * sub), np.float32)
    for g in range(G):
        for z in range(C):
            X[z * per:(z + 1) * per, g * sub:(g + 1) * sub] = centres[g, z] + spread * rng.standard_normal((per, sub))
    return X, centres


# well-separated blobs: every centre converges to the mean of its blob (each subspace separately, both sides), and
# scikit-learn's KMeans started from the same rows finds the same centres
def test_blobs_and_scikit_learn():
    from sklearn.cluster import KMeans
    rng = np.random.default_rng(2)
    G, C, sub, per = 2, 4, 3, 40
    X, centres = _blobs(rng, C, per, sub, G)
    Xv, centres_v = _blobs(rng, C, per, sub, G)
    o = _bank(d=G * sub, G=G, C=C, R=C * per, iters=30, batch=64, seed=3)
    o.set_reservoir(X, Xv)
    assert o.train_codebooks() == 1
    ck, cv = o.codebooks()
    for side, (cb, data, cen) in enumerate(((ck, X, centres), (cv, Xv, centres_v))):
        for g in range(G):
            sl = data[:, g * sub:(g + 1) * sub]
            for z in range(C):
                blob_mean = sl[z * per:(z + 1) * per].mean(axis=0)
                assert np.allclose(cb[g, z], blob_mean, atol=0.01), (side, g, z)      # 0.01 spread / sqrt(samples)
            init = np.stack([sl[(z * C * per) // C] for z in range(C)])
            km = KMeans(n_clusters=C, init=init, n_init=1, algorithm="lloyd").fit(sl.astype(np.float64))
            assert np.allclose(km.cluster_centers_, cb[g], atol=0.01)


# the quantisation error of the trained codebook is not worse than that of its initialisation (rows of the data)
def test_training_lowers_the_quantisation_error():
    rng = np.random.default_rng(4)
    n, G, sub, C = 512, 2, 8, 16
    X = rng.standard_normal((n, G * sub)).astype(np.float32) * 0.1
    o = _bank(d=G * sub, G=G, C=C, R=n, iters=32, batch=256, seed=9)
    o.set_reservoir(X, X[::-1].copy())
    o.train_codebooks()
    ck, cv = o.codebooks()

    def err(cb, data, g):
        sl = data[:, g * sub:(g + 1) * sub].astype(np.float64)
        return ((sl[:, None, :] - cb[None]) ** 2).sum(-1).min(1).mean()
    for g in range(G):
        init = np.stack([X[(z * n) // C, g * sub:(g + 1) * sub] for z in range(C)]).astype(np.float64)
        assert err(ck[g].astype(np.float64), X, g) < err(init, X, g)


# fewer residuals than codewords: no codebooks, the stream keeps running without residual statistics
def test_short_warmup_leaves_the_state_without_codebooks():
    o = _bank(d=4, G=1, C=2, R=8)
    o.set_reservoir(np.ones((1, 4), np.float32), np.ones((1, 4), np.float32))
    assert o.train_codebooks() == 0 and o.codebooks() is None


# end to end on C1: warm-up over the first t_warm steps, automatic training at step t_warm - 1, histograms only count
# absorptions of later steps; the codebooks equal those of a manual training on the same reservoir
def test_stream_with_automatic_training():
    spec = gen.spec_for("c1")
    t_warm = 20
    kw = dict(G=spec.G, C=spec.C, t_warm=t_warm, warm_reservoir=128, km_iters=8, km_batch=64, km_seed=11)
    auto = OracleBank(spec.T, spec.near_frames, spec.k_max, spec.head_dim, None, None, flags=FLAG_WARMUP, **kw)
    man = OracleBank(spec.T, spec.near_frames, spec.k_max, spec.head_dim, None, None,
                     flags=FLAG_WARMUP | FLAG_WARMUP_MANUAL, **kw)
    for f in range(40):
        K, V, s = frame_for_bank(spec, f, 0)
        auto.append_frame(K, V, s, trace=False)
        man.append_frame(K, V, s, trace=False)
        if f == t_warm - 2:
            assert auto.codebooks() is None
            ra, rb = auto.reservoir(), man.reservoir()
            assert np.array_equal(ra[0], rb[0]) and ra[2] == rb[2]
        if f == t_warm - 1:
            assert man.codebooks() is None and man.train_codebooks() == 1
            assert np.array_equal(auto.codebooks()[0], man.codebooks()[0])
            assert np.array_equal(auto.codebooks()[1], man.codebooks()[1])
            seen = auto.reservoir()[2]
            # tokens absorbed (not slot fills) during steps near_frames .. t_warm - 1
            assert seen == (t_warm - spec.near_frames) * spec.T - spec.k_max and seen > 128
    sa, sm = auto.state(), man.state()
    for f in sa:
        assert np.array_equal(sa[f], sm[f]), f
    absorbed_after = (40 - t_warm) * spec.T
    assert int(sa["nres"].sum()) == absorbed_after                      # histograms start after the warm-up
    assert np.all(sa["hist_k"].sum(axis=2) == sa["nres"][:, None])
    assert auto.reservoir()[2] == seen                                   # nothing is collected after the warm-up
