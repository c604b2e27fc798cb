"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Protocol: teacher-forced streams -- after every frame the GPU's decisions (assignment,
PQ codes) are checked against the oracle's own, under north_star's gap rule, and the oracle then follows the GPU's
decisions so that one accepted near-tie cannot cascade; statistics are compared field by field; synthesis codes
and attention outputs are compared at the query.
"""
import dataclasses

import numpy as np
import pytest
import torch

import gen
from gpu_helpers import (make_gpu, make_oracles, run_stream, compare_ring, compare_codes, compare_attention,
                         compare_state, new_stats, step_teacher_forced)
from oracle import FLAG_NEAR_ONLY, FLAG_FAR_ONLY, FLAG_NO_MASS_BIAS, FLAG_MAH_SQUARED
from paper_2606_26762_b200 import (ProtoKV, ProtoKVError, NEAR_ONLY, FAR_ONLY, NO_MASS_BIAS, MAH_SQUARED, FORCE_SIMT,
                                   DECODE_SPLITKV, NO_DECODE_KERNEL, SERIAL_LAUNCH)

pytestmark = pytest.mark.gpu


def _query_and_check(spec, gpu, oracles, query_index=0, **kw):
    flips = compare_codes(gpu, oracles, spec.G)
    Q = gen.queries(spec, query_index)
    worst = compare_attention(spec, gpu, oracles, Q, run_synthesis=False, **kw)
    return flips, worst


# ---------------------------------------------------------------------------------------------------------
# config 1 (BASELINE.json configs[0]): the whole 64-frame stream, every frame, every field, then the query
# ---------------------------------------------------------------------------------------------------------
def test_c1_full_stream():
    spec = gen.spec_for("c1")
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, [0])
    stats = run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=1)
    assert stats["scored"] == (spec.n_frames - spec.near_frames) * spec.T - spec.k_max
    compare_ring(gpu, oracles)
    st = gpu.export_state(0)
    assert int(st["n"].sum()) == (spec.n_frames - spec.near_frames) * spec.T      # mass conservation
    _query_and_check(spec, gpu, oracles)
    # end to end without forced codes
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=True)
    assert gpu.frames_seen == spec.n_frames and gpu.kernel_launches > 0


# ---------------------------------------------------------------------------------------------------------
# config 2 shape (bf16, GQA 28/4, d=128, T=196 -> ragged tiles), all 4 banks, first frames incl. the fill phase
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("force_simt", [False, True])
def test_c2_shape_short_stream(force_simt):
    spec = gen.spec_for("c2", n_frames=30)
    gpu = make_gpu(spec, flags=FORCE_SIMT if force_simt else 0)
    oracles = make_oracles(spec, range(spec.n_banks))
    stats = run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=7)
    assert stats["scored"] > 0
    compare_ring(gpu, oracles)
    _query_and_check(spec, gpu, oracles)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 1), run_synthesis=True)


# ---------------------------------------------------------------------------------------------------------
# config 3 shape: several layers in one state; attention of a layer subset and of fewer query tokens
# ---------------------------------------------------------------------------------------------------------
def test_c3_shape_layers_subset():
    spec = gen.spec_for("c3", n_layers=3, n_frames=26, k_max=512)
    gpu = make_gpu(spec)
    banks = [0, 5, 11]     # (layer 0, head 0), (layer 1, head 1), (layer 2, head 3)
    oracles = make_oracles(spec, banks)
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=13)
    compare_codes(gpu, oracles, spec.G)
    Q = gen.queries(spec, 0)
    compare_attention(spec, gpu, oracles, Q, run_synthesis=False)
    # layers [1, 3), 5 query tokens
    Qs = Q[:, 1:3, :5].contiguous()
    compare_attention(spec, gpu, oracles, Qs, layer_begin=1, run_synthesis=False)


# ---------------------------------------------------------------------------------------------------------
# config 5 shape: 2 streams x 8 KV heads, T = 576, K_max = 2048, N_q = 64 (256 rows per bank)
# ---------------------------------------------------------------------------------------------------------
def test_c5_shape_multi_stream():
    spec = gen.spec_for("c5", n_streams=2, n_frames=14)
    gpu = make_gpu(spec)
    banks = [0, 7, 9]
    oracles = make_oracles(spec, banks)
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=7)
    compare_ring(gpu, oracles)
    compare_codes(gpu, oracles, spec.G)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=False, rows_sample=range(0, 256, 5))


# ---------------------------------------------------------------------------------------------------------
# full sizes in the launch configuration bench.py times (C3: 112 banks, C5: 64 banks): the same grids, tile plans and
# stream-K splits as the timed runs; the oracle follows a sample of banks (first, middle, last) frame by frame and
# checks a sample of query rows -- every output it checks is computed one by one from the definition
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,banks,frames", [("c3", [0, 57, 111], 25), ("c5", [0, 31, 63], 13)])
def test_full_size_bench_configuration_sampled(name, banks, frames):
    spec = gen.spec_for(name, n_frames=frames)
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, banks)
    stats = run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=frames - 1)
    assert stats["scored"] > 0
    compare_codes(gpu, oracles, spec.G)
    rows = spec.n_query_tokens * (spec.n_q_heads // spec.n_kv_heads)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=True, rows_sample=range(0, rows, 11))
    for b in banks:                                          # mass conservation on the sampled banks
        assert int(gpu.export_state(b)["n"].sum()) == (spec.n_frames - spec.near_frames) * spec.T


# ---------------------------------------------------------------------------------------------------------
# config 4 cells (small ends of the sweep): K_max 256 with W_f 4, and a bank larger than the stream ever fills
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k_max,near", [(256, 4), (4096, 4)])
def test_c4_cells(k_max, near):
    spec = gen.spec_for(f"c4_k{k_max}_w{near}", n_frames=14)
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, [0, 3])
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=7)
    compare_codes(gpu, oracles, spec.G)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=False, rows_sample=range(0, 224, 3))


# ---------------------------------------------------------------------------------------------------------
# Eq. 1's idle term and non-default hyper-parameters: with T_idle = 2 frames most prototypes are idle at any step
# (the default 120 frames never triggers in a short stream), larger lambda_sp / lambda_idle move decisions, and the
# EMA rates differ per statistic
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("force_simt", [False, True])
def test_idle_penalty_and_hyperparameters(force_simt):
    spec = gen.spec_for("c2", n_frames=32)
    hyper = dict(t_idle=2, lambda_idle=0.05, lambda_sp=0.3, alpha=0.1, beta=0.2, eta=0.02)
    gpu = make_gpu(spec, flags=FORCE_SIMT if force_simt else 0, **hyper)
    oracles = make_oracles(spec, [0, 3], **hyper)
    stats = run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=8)
    assert stats["scored"] > 0
    st = oracles[0].state()
    t_last = spec.n_frames - 1
    idle = int(((t_last - st["tau"][st["active"].astype(bool)]) > hyper["t_idle"]).sum())
    assert idle > 50, f"only {idle} idle prototypes: the idle term is not exercised"
    _query_and_check(spec, gpu, oracles)


# ---------------------------------------------------------------------------------------------------------
# long stream: the bank has been full for > 100 frames, segments hold several tokens per prototype, histograms are
# deep, and with the default T_idle = 120 frames the idle term of Eq. 1 starts to fire near the end
# ---------------------------------------------------------------------------------------------------------
def test_c2_long_stream_steady_state():
    spec = gen.spec_for("c2", n_frames=150)
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, [1])
    stats = run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=30)
    assert stats["scored"] > 100 * spec.T
    st = oracles[1].state()
    assert int(st["n"].max()) >= 8                           # prototypes that absorbed many tokens
    assert int(((spec.n_frames - 1 - st["tau"]) > 120).sum()) > 0, "no prototype went idle"
    compare_ring(gpu, oracles)
    _query_and_check(spec, gpu, oracles)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 2), run_synthesis=True, rows_sample=range(0, 224, 3))


# ---------------------------------------------------------------------------------------------------------
# the lazily moved reference maximum of the fused attention: keys of the later ring slots are 8x larger, so the
# logits of later tiles exceed the first tile's row maximum by far more than the 2^8 head-room and O, l have to be
# rescaled in flight (tcgen05 kernel) -- same inputs to the oracle, which has no such mechanism
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("force_simt", [False, True])
def test_attention_reference_maximum_moves(force_simt):
    spec = gen.spec_for("c2", n_frames=24)
    gpu = make_gpu(spec, flags=FORCE_SIMT if force_simt else 0)
    oracles = make_oracles(spec, [0, 2])
    stats = new_stats()
    s = gen.grid_positions(spec)
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        if f % spec.near_frames >= 6:                        # ring slot = f mod W_f; exact in bf16
            K = K * 8
        step_teacher_forced(spec, gpu, oracles, f, K, V, s, stats)
    Q = gen.queries(spec, 0)
    compare_codes(gpu, oracles, spec.G)
    worst = compare_attention(spec, gpu, oracles, Q, run_synthesis=False)
    # the construction does what it claims: the kernel walks the ring in slot order, slot 0 holds frame 16 (unscaled);
    # for most rows the largest near-window logit lies far above the maximum over that first tile
    from gpu_helpers import bank_frame
    q = Q[0, 0, :, 0:7, :].float().numpy().reshape(-1, spec.head_dim)
    first = None
    top = np.full(q.shape[0], -np.inf)
    for f in range(spec.n_frames - spec.near_frames, spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        if f % spec.near_frames >= 6:
            K = K * 8
        Kb = bank_frame(spec, K, V, s, 0)[0]
        lg = q @ Kb.T / np.sqrt(spec.head_dim)
        top = np.maximum(top, lg.max(axis=1))
        if f % spec.near_frames == 0:
            first = lg[:, :128].max(axis=1)
    assert ((top - first) > 8 * np.log(2.0)).mean() > 0.5, "the reference maximum never has to move"
    assert worst < 1e-1


# ---------------------------------------------------------------------------------------------------------
# degenerate cases of the method
# ---------------------------------------------------------------------------------------------------------
def test_empty_and_near_only_states():
    spec = gen.spec_for("c1")
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, [0])
    Q = gen.queries(spec, 0)
    # no frame yet: empty context -> zeros, lse = -inf
    out, lse = gpu.query_attention_ex(Q.to(gpu.device), return_lse=True)
    assert (out == 0).all() and torch.isinf(lse).all()
    # fewer frames than the window holds: nothing evicted, attention = plain attention over the partial window
    run_stream(spec, gpu, oracles, 3, check_state_every=1)
    assert gpu.last_frame_trace()["evicted_frame"] == -1
    compare_attention(spec, gpu, oracles, Q, run_synthesis=True)
    # exactly the first eviction
    run_stream(spec, gpu, oracles, 2, check_state_every=1, first_frame=3)
    compare_attention(spec, gpu, oracles, Q, run_synthesis=True)


@pytest.mark.parametrize("gflag,oflag", [(NEAR_ONLY, FLAG_NEAR_ONLY), (FAR_ONLY, FLAG_FAR_ONLY),
                                         (NO_MASS_BIAS, FLAG_NO_MASS_BIAS), (MAH_SQUARED, FLAG_MAH_SQUARED)])
def test_ablation_flags(gflag, oflag):
    spec = gen.spec_for("c1", n_frames=24)
    gpu = make_gpu(spec, flags=gflag)
    oracles = make_oracles(spec, [0], flags=oflag)
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=4)
    if gflag != NEAR_ONLY:
        compare_codes(gpu, oracles, spec.G)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=True)


def test_no_codebooks_zero_residuals():
    spec = gen.spec_for("c1", n_frames=20)
    gpu = make_gpu(spec, with_codebooks=False)
    oracles = make_oracles(spec, [0], with_codebooks=False)
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=4, with_codebooks=False)
    compare_codes(gpu, oracles, spec.G)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=True)


def test_small_pq_and_single_mode():
    # G = 2, C = 4, S = 3: C^G = 16 >= S; exercises ragged code tables and S < 8
    spec = gen.spec_for("c1", n_frames=30, G=2, C=4)
    gpu = make_gpu(spec, S=3, beam=3)
    oracles = make_oracles(spec, [0], S=3, beam=3)
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=5)
    compare_codes(gpu, oracles, spec.G)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=False)


def test_ragged_frame_size_and_bf16_d64():
    spec = dataclasses.replace(gen.spec_for("c1"), name="ragged", dtype="bf16", grid_h=5, grid_w=7, k_max=50,
                               n_q_heads=6, n_kv_heads=2, n_frames=20, n_query_tokens=3)
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, [0, 1])
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=5)
    compare_codes(gpu, oracles, spec.G)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=False)


# ---------------------------------------------------------------------------------------------------------
# boundary behaviour: host variants, state import/export, errors
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,frames", [("c1", 12), ("c2", 30)])
def test_host_variants_match_device_calls(name, frames):
    """The host-buffer entry points (copies on the library's copy stream, overlapped with the scoring / update kernels and
    the synthesis) produce exactly what the device-pointer calls produce."""
    spec = gen.spec_for(name, n_frames=frames)
    a, b = make_gpu(spec), make_gpu(spec)
    s = gen.grid_positions(spec)
    hs = s.pin_memory()
    keep = []
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        a.append_frame(K.cuda(), V.cuda(), s.cuda())
        keep.append((K.pin_memory(), V.pin_memory()))        # arguments stay valid until the stream has passed the call
        b.append_frame_host(keep[-1][0], keep[-1][1], hs)
        if f % 7 == 3:
            torch.cuda.synchronize()
            keep.clear()
    torch.cuda.synchronize()
    Q = gen.queries(spec, 0)
    oa = a.query_attention(Q.cuda()).cpu()
    ob = torch.empty_like(Q).pin_memory()
    b.query_attention_host(Q.pin_memory(), ob)
    assert torch.equal(oa, ob)
    for f in ("c", "p", "n", "hist_k", "hist_v", "mu", "sigma"):
        assert np.array_equal(a.export_state(0)[f], b.export_state(0)[f])


def test_import_state_round_trip():
    spec = gen.spec_for("c1", n_frames=16)
    a, b = make_gpu(spec), make_gpu(spec)
    s = gen.grid_positions(spec).cuda()
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        a.append_frame(K.cuda(), V.cuda(), s)
        b.append_frame(K.cuda(), V.cuda(), s)
    st = a.export_state(0)
    st2 = {k: v.copy() for k, v in st.items()}
    st2["c"][:] *= 0.5
    b.import_state(0, **st2)
    got = b.export_state(0)
    assert np.array_equal(got["c"], st2["c"]) and np.array_equal(got["hist_k"], st["hist_k"])
    b.import_state(0, **st)
    K, V = gen.frame_kv(spec, spec.n_frames)
    a.append_frame(K.cuda(), V.cuda(), s)
    b.append_frame(K.cuda(), V.cuda(), s)
    ta, tb = a.last_frame_trace(), b.last_frame_trace()
    # bit for bit: the slot fill, the update kernels and refresh_derived_kernel all reduce |c|^2 in the same per-lane
    # order, so the derived 1/|c| (and with it every score) is reproduced exactly after an import
    assert np.array_equal(ta["assign"], tb["assign"]) and np.array_equal(ta["best"], tb["best"])
    for f in ("c", "p", "n", "hist_k", "mu", "sigma"):
        assert np.array_equal(a.export_state(0)[f], b.export_state(0)[f])


def test_stage_profile_counts_launches():
    spec = gen.spec_for("c1", n_frames=10)
    gpu = make_gpu(spec)
    s = gen.grid_positions(spec).cuda()
    gpu.profile_enable(True)
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        gpu.append_frame(K.cuda(), V.cuda(), s)
    gpu.query_attention(gen.queries(spec, 0).cuda())
    prof = gpu.profile_read()
    assert prof["append"][1] == 10 and prof["fill"][1] == 2 and prof["score"][1] == 4 and prof["update"][1] == 4
    assert prof["synthesis"][1] == 1 and prof["attention"][1] == 1
    assert all(ms >= 0 for ms, _ in prof.values()) and prof["attention"][0] > 0
    gpu.profile_enable(False)


def test_errors_leave_state_unchanged():
    spec = gen.spec_for("c1")
    gpu = make_gpu(spec)
    K, V = gen.frame_kv(spec, 0)
    s = gen.grid_positions(spec)
    with pytest.raises(ProtoKVError):
        gpu.append_frame(K.cuda()[..., :32].contiguous(), V.cuda(), s.cuda())      # wrong size
    with pytest.raises(ProtoKVError):
        gpu.append_frame(K, V, s)                                                  # host tensors
    assert gpu.frames_seen == 0
    Q = gen.queries(spec, 0).cuda()
    with pytest.raises(ProtoKVError) as ei:
        gpu.query_attention_ex(Q[:, :, :4].contiguous(), n_q=4, layer_begin=1)     # layer range
    assert ei.value.code == 1
    with pytest.raises(ProtoKVError) as ei:
        gpu.export_state(7)
    assert ei.value.code == 1
    with pytest.raises(ProtoKVError) as ei:
        make_gpu(dataclasses.replace(spec, head_dim=96))
    with pytest.raises(ProtoKVError):
        gpu.export_codes(0)                                                        # nothing synthesised yet


# ---------------------------------------------------------------------------------------------------------
# non-finite inputs are contained: a NaN / Inf key row has no finite Eq. 1 score -- the token is dropped
# and flagged instead of indexing a prototype with garbage; a NaN query row yields NaN for that row only and the
# persistent attention kernel terminates
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,force_simt", [("c2", False), ("c2", True), ("c1", False)])
def test_nonfinite_key_row_is_dropped_and_flagged(name, force_simt):
    spec = gen.spec_for(name, n_frames=spec_frames(name))
    gpu = make_gpu(spec, flags=FORCE_SIMT if force_simt else 0)
    s = gen.grid_positions(spec).cuda()
    bad_frame, bad_tok = spec.n_frames - spec.near_frames - 2, 5
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        if f == bad_frame:
            K[0, 0, bad_tok, 0, 3] = float("nan")
            K[0, 0, bad_tok + 1, 0, 7] = float("inf")
        gpu.append_frame(K.cuda(), V.cuda(), s)
        tr = gpu.last_frame_trace()
        if tr["evicted_frame"] == bad_frame:
            a = tr["assign"][0]
            assert a[bad_tok] == -2 and a[bad_tok + 1] == -2
            assert (np.delete(a, [bad_tok, bad_tok + 1]) >= 0).all()
            assert (tr["assign"][1:] >= 0).all()                 # the other banks are untouched by it
    assert gpu.error_flags() & 1
    st = gpu.export_state(0)
    evicted = (spec.n_frames - spec.near_frames) * spec.T
    assert int(st["n"].sum()) == evicted - 2                     # exactly the two tokens are missing from the mass
    assert np.isfinite(st["c"]).all() and np.isfinite(st["p"]).all()
    assert gpu.error_flags(clear=True) & 1 and gpu.error_flags() == 0


def spec_frames(name):
    return 14 if name == "c1" else 26


@pytest.mark.parametrize("force_simt", [False, True])
def test_nan_query_row_stays_in_its_row(force_simt):
    spec = gen.spec_for("c2", n_frames=24)
    gpu = make_gpu(spec, flags=FORCE_SIMT if force_simt else 0)
    s = gen.grid_positions(spec).cuda()
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        gpu.append_frame(K.cuda(), V.cuda(), s)
    Q = gen.queries(spec, 0)
    ref = gpu.query_attention(Q.cuda()).float().cpu()
    Qn = Q.clone()
    Qn[0, 0, 3, 9, 17] = float("nan")            # query token 3, query head 9 (KV head 1)
    Qn[0, 0, 5, 20, 1] = float("inf")
    out = gpu.query_attention(Qn.cuda()).float().cpu()   # must return (a hang would trip the suite's timeout)
    assert torch.isnan(out[0, 0, 3, 9]).all() and not torch.isfinite(out[0, 0, 5, 20]).any()
    mask = torch.ones(out.shape[:4], dtype=torch.bool)
    mask[0, 0, 3, 9] = False
    mask[0, 0, 5, 20] = False
    # (a NaN row makes its warp re-reference its rows' maxima once: other rows may differ in rounding, not in value)
    assert torch.allclose(out[mask], ref[mask], atol=1e-2, rtol=2e-2)


def test_imported_codes_last_until_the_next_synthesis():
    spec = gen.spec_for("c1", n_frames=20)
    gpu = make_gpu(spec)
    s = gen.grid_positions(spec).cuda()
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        gpu.append_frame(K.cuda(), V.cuda(), s)
    gpu.synthesize()
    ck, cv, kind = gpu.export_codes(0)
    forced_k, forced_v = (ck + 1) % spec.C, (cv + 3) % spec.C
    gpu.import_codes(0, forced_k, forced_v)
    assert np.array_equal(gpu.export_codes(0)[0], forced_k)      # in force for queries with run_synthesis = 0
    K, V = gen.frame_kv(spec, spec.n_frames)
    gpu.append_frame(K.cuda(), V.cuda(), s)                       # touches only a few prototypes
    gpu.synthesize()
    ck2, cv2, kind2 = gpu.export_codes(0)
    fresh = make_gpu(spec)
    for f in range(spec.n_frames + 1):
        K, V = gen.frame_kv(spec, f)
        fresh.append_frame(K.cuda(), V.cuda(), s)
    fresh.synthesize()
    ek, ev, ekind = fresh.export_codes(0)
    assert np.array_equal(ck2, ek) and np.array_equal(cv2, ev) and np.array_equal(kind2, ekind)


# ---------------------------------------------------------------------------------------------------------
# synthesis with deep histograms: counts beyond the 4,096-entry numerator table of Eq. 3 take the kernel's own
# log() branch; masses in the thousands enter the log n_k bias
# ---------------------------------------------------------------------------------------------------------
def test_synthesis_and_bias_with_counts_beyond_the_log_table():
    spec = gen.spec_for("c1", n_frames=16)
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, [0])
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=0)
    st = oracles[0].state()
    rng = np.random.default_rng(11)
    act = st["active"].astype(bool)
    big = rng.integers(0, 3, size=st["hist_k"].shape) * rng.integers(3000, 200000, size=st["hist_k"].shape)
    hk = (st["hist_k"].astype(np.int64) + big).astype(np.uint32)
    hv = np.roll(hk, 1, axis=2)
    # rows of a prototype must all sum to n_res: top the first bin of every row up to a common total
    tot = max(int(hk.sum(axis=2).max()), int(hv.sum(axis=2).max())) + 5
    for H in (hk, hv):
        H[:, :, 0] += (tot - H.sum(axis=2)).astype(np.uint32)
    hk[~act] = 0
    hv[~act] = 0
    st["hist_k"], st["hist_v"] = hk, hv
    st["nres"] = np.where(act, tot, 0).astype(np.uint32)
    st["n"] = np.where(act, tot + 1, 0).astype(np.int32)
    assert hk.max() > 4095
    oracles[0].set_state(**st)
    gpu.import_state(0, **st)
    compare_codes(gpu, oracles, spec.G)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=False)


# ---------------------------------------------------------------------------------------------------------
# decode-style queries (<= 16 rows per bank) through the opt-in split-KV mma.sync kernel (csrc/decode_attention.cu): one- and
# two-token queries against the oracle at every stage of a stream -- partial window (ragged near tail), bank still
# filling (ragged prototype tail, zero-residual prototypes), steady state -- and under the ablation flags
# ---------------------------------------------------------------------------------------------------------
_ROUTES = {0: "mma.sync register-resident", DECODE_SPLITKV: "mma.sync split-KV", NO_DECODE_KERNEL: "tcgen05"}


@pytest.mark.parametrize("flags,oflags,route", [(0, 0, 0), (NEAR_ONLY, FLAG_NEAR_ONLY, 0), (FAR_ONLY, FLAG_FAR_ONLY, 0),
                                                (NO_MASS_BIAS, FLAG_NO_MASS_BIAS, 0), (0, 0, DECODE_SPLITKV),
                                                (FAR_ONLY, FLAG_FAR_ONLY, DECODE_SPLITKV), (0, 0, NO_DECODE_KERNEL)])
def test_decode_query_kernel(flags, oflags, route):
    """Default route = the register-resident decode kernel (csrc/decode_attention2.cu); the opt-in split-KV kernel and the
    128-row tcgen05 kernel serve the same queries as cross-checks."""
    spec = gen.spec_for("c2", n_frames=40)
    gpu = make_gpu(spec, flags=flags | route)
    assert gpu.stage_impl(2) == _ROUTES[route]
    oracles = make_oracles(spec, [0, 3], flags=oflags)
    Q = gen.queries(spec, 5)
    checkpoints = {2: 1, 9: 2, 17: 1, 19: 2, 23: 1, 39: 2}      # frame -> query tokens (7 or 14 rows per bank)
    stats = new_stats()
    s = gen.grid_positions(spec)
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        step_teacher_forced(spec, gpu, oracles, f, K, V, s, stats)
        if f in checkpoints:
            nq = checkpoints[f]
            if not (flags & NEAR_ONLY):
                compare_codes(gpu, oracles, spec.G)
            Qs = Q[:, :, 3:3 + nq].contiguous()
            compare_attention(spec, gpu, oracles, Qs, run_synthesis=True)
            # and against the 128-row tcgen05 kernel on the same state (a 3-token query has 21 rows)
            Q3 = Q[:, :, 3:6].contiguous()
            o3 = gpu.query_attention_ex(Q3.cuda(), n_q=3, run_synthesis=False).float().cpu()
            o1 = gpu.query_attention_ex(Qs.cuda(), n_q=nq, run_synthesis=False).float().cpu()
            assert torch.allclose(o1, o3[:, :, :nq], atol=1e-2, rtol=2e-2)


def test_decode_query_full_size_c3_sampled():
    spec = gen.spec_for("c3", n_frames=24)
    for flags in (0, DECODE_SPLITKV, NO_DECODE_KERNEL):   # default (register-resident decode kernel) and the two others
        gpu = make_gpu(spec, flags=flags)
        assert gpu.stage_impl(2) == _ROUTES[flags]
        banks = [0, 57, 111]
        oracles = make_oracles(spec, banks)
        run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=0, on_device=True)
        Q = gen.queries(spec, 1)[:, :, :1].contiguous()
        compare_attention(spec, gpu, oracles, Q, run_synthesis=True)
        gpu.close()


def test_decode_query_c5_shape():
    """GQA group 4, T = 576, K_max = 2048 (config 5's bank shape, one stream): 1-, 3- and 4-token queries (4, 12, 16 rows)
    through the register-resident decode kernel while the bank fills and in steady state."""
    spec = gen.spec_for("c5", n_frames=16, n_streams=1)
    gpu = make_gpu(spec)
    assert gpu.stage_impl(2) == _ROUTES[0]
    oracles = make_oracles(spec, [0, 5])
    Q = gen.queries(spec, 2)
    stats = new_stats()
    s = gen.grid_positions(spec)
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        step_teacher_forced(spec, gpu, oracles, f, K, V, s, stats)
        if f in (3, 9, 11, 15):
            nq = {3: 1, 9: 4, 11: 3, 15: 4}[f]
            compare_attention(spec, gpu, oracles, Q[:, :, :nq].contiguous(), run_synthesis=True)
    gpu.close()


def test_decode_query_without_codebooks():
    """No residual statistics (Table 2 "w/o residual stats"): every prototype contributes S copies of (c_k, p_k); the decode
    kernels must not touch a codebook."""
    spec = gen.spec_for("c2", n_frames=30)
    gpu = make_gpu(spec, with_codebooks=False)
    oracles = make_oracles(spec, [0, 2], with_codebooks=False)
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=0, with_codebooks=False)
    Q = gen.queries(spec, 4)
    compare_attention(spec, gpu, oracles, Q[:, :, :1].contiguous(), run_synthesis=True)
    compare_attention(spec, gpu, oracles, Q[:, :, :2].contiguous(), run_synthesis=False)
    gpu.close()


@pytest.mark.parametrize("name,frames", [("c2", 40), ("c1", 24)])
def test_dependent_launch_chain_equals_serial_launches(name, frames):
    """The default launch mode overlaps each kernel's set-up with its predecessor's tail (programmatic dependent launch,
    csrc/common.cuh pdl_wait); PROTOKV_SERIAL_LAUNCH serialises every launch.  Same inputs, ONE pair of K / V buffers that a
    copy kernel of the caller refills right before every append and overwrites right after it (the ring append reads them
    ahead of its wait): ring, bank state, pseudo-token codes and attention outputs must agree bit for bit."""
    spec = gen.spec_for(name, n_frames=frames)
    s = gen.grid_positions(spec, device="cuda")
    src = [gen.frame_kv(spec, f, device="cuda") for f in range(frames)]
    Q = gen.queries(spec, 0).cuda()
    Q1 = Q[:, :, :1].contiguous()
    got = []
    for flags in (0, SERIAL_LAUNCH):
        gpu = make_gpu(spec, flags=flags)
        K, V = torch.empty_like(src[0][0]), torch.empty_like(src[0][1])
        outs = []
        for f in range(frames):
            K.copy_(src[f][0]); V.copy_(src[f][1])
            gpu.append_frame(K, V, s)
            K.fill_(7.0); V.fill_(-3.0)                                  # the caller reuses its buffers at once
            if f % 9 == 8:
                outs.append(gpu.query_attention(Q).float().cpu())
                outs.append(gpu.query_attention_ex(Q1, n_q=1, run_synthesis=False).float().cpu())
        gpu.synthesize()
        for la in range(spec.n_layers):                                  # back-to-back per-layer calls
            outs.append(gpu.query_attention_ex(Q[:, la:la + 1].contiguous(), layer_begin=la, layer_count=1,
                                               run_synthesis=False).float().cpu())
        banks = [0, spec.n_banks - 1]
        got.append((outs, [gpu.export_state(b) for b in banks], [gpu.export_ring(b) for b in banks],
                    [gpu.export_codes(b) for b in banks]))
        gpu.close()
    (oa, sa, ra, ca), (ob, sb, rb, cb) = got
    assert len(oa) == len(ob) and all(torch.equal(x, y) for x, y in zip(oa, ob))
    for x, y in zip(sa, sb):
        assert all(np.array_equal(x[k], y[k], equal_nan=True) for k in x), [k for k in x if not np.array_equal(x[k], y[k])]
    for x, y in zip(ra + ca, rb + cb):
        assert all(np.array_equal(u, v) for u, v in zip(x, y))
