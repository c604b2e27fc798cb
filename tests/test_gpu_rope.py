"""-m gpu parity of the rotary position anchoring (D.1 L578-596) against the
oracle: un-rotated K / Q in, near tokens rotated at their stream positions, the S pseudo-tokens of a prototype at its
anchor (most recent / first / average absorbed position), query tokens at q_pos0 + i.  The anchor fields are part of
the state comparison of every teacher-forced stream (gpu_helpers.compare_state)."""
import dataclasses

import numpy as np
import pytest

import gen
from gpu_helpers import make_gpu, make_oracles, run_stream, compare_codes, compare_attention
from oracle import FLAG_ROPE, FLAG_MAINTENANCE
from paper_2606_26762_b200 import ROPE, MAINTENANCE, FORCE_SIMT

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("anchor", [0, 1, 2])
def test_rope_c1_all_anchor_variants(anchor):
    spec = gen.spec_for("c1", n_frames=40)
    hyper = dict(rope_theta=10000.0, rope_anchor=anchor, pos0=1000)
    gpu = make_gpu(spec, flags=ROPE, **hyper)
    assert gpu.stage_impl(1) == "simt"
    oracles = make_oracles(spec, [0], flags=FLAG_ROPE, **hyper)
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=4)
    compare_codes(gpu, oracles, spec.G)
    Q = gen.queries(spec, 0)
    compare_attention(spec, gpu, oracles, Q, run_synthesis=False)                       # default: next stream position
    compare_attention(spec, gpu, oracles, Q, run_synthesis=False, q_pos0=1000 + spec.n_frames * spec.T)   # the same, explicit
    compare_attention(spec, gpu, oracles, Q, run_synthesis=False, q_pos0=5000)
    # the rotation is not a no-op
    a = gpu.query_attention_ex(Q.cuda(), q_pos0=5000, run_synthesis=False).float().cpu()
    b = gpu.query_attention_ex(Q.cuda(), q_pos0=5037, run_synthesis=False).float().cpu()
    assert (a - b).abs().max() > 1e-3


@pytest.mark.parametrize("route,impl", [(0, "mma.sync register-resident (blocks)"), (FORCE_SIMT, "simt")])
def test_rope_bf16_gqa_shape_long_positions(route, impl):
    # config-2 shape (bf16, d = 128, GQA 28/4), default base 1e6, positions beyond 10^6 (pos0): fp32 angles would be off.
    # Default route: the rotating variant of the register-resident kernel (8-row blocks); cross-check: the fp32 SIMT kernel
    spec = gen.spec_for("c2", n_frames=26)
    hyper = dict(pos0=1_500_000)
    gpu = make_gpu(spec, flags=ROPE | route, **hyper)
    assert gpu.stage_impl(1) == impl
    oracles = make_oracles(spec, [0, 3], flags=FLAG_ROPE, **hyper)
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=13)
    compare_codes(gpu, oracles, spec.G)
    rows = spec.n_query_tokens * (spec.n_q_heads // spec.n_kv_heads)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=False, rows_sample=np.arange(0, rows, 5))
    compare_attention(spec, gpu, oracles, gen.queries(spec, 1)[:, :, :3].contiguous(), run_synthesis=False, q_pos0=1_500_000)


def test_rope_with_maintenance_merges_anchors():
    spec = gen.spec_for("c1", n_frames=48)
    hyper = dict(t_idle=3, gamma=0.3, eps_k=1.2, eps_v=1.2, rope_anchor=2, rope_theta=10000.0)
    gpu = make_gpu(spec, flags=ROPE | MAINTENANCE, **hyper)
    oracles = make_oracles(spec, [0], flags=FLAG_ROPE | FLAG_MAINTENANCE, **hyper)
    run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=2)
    assert gpu.maintenance_counters()["merges"] > 0
    compare_codes(gpu, oracles, spec.G)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=False)


@pytest.mark.parametrize("anchor", [0, 1, 2])
def test_rope_decode_query_anchor_variants(anchor):
    """One- and three-token queries (7 / 21 rows per bank) of a bf16 state through the rotating decode kernel at every stage
    of a stream (partial window, bank filling, steady state), all three D.1 anchors."""
    spec = gen.spec_for("c2", n_frames=30)
    hyper = dict(rope_anchor=anchor, pos0=250_000)
    gpu = make_gpu(spec, flags=ROPE, **hyper)
    assert gpu.stage_impl(2) == "mma.sync register-resident (blocks)"
    oracles = make_oracles(spec, [1, 2], flags=FLAG_ROPE, **hyper)
    Q = gen.queries(spec, 3)
    from gpu_helpers import step_teacher_forced, new_stats
    stats = new_stats()
    s = gen.grid_positions(spec)
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        step_teacher_forced(spec, gpu, oracles, f, K, V, s, stats)
        if f in (3, 18, 22, 29):
            nq = 1 if f % 2 else 3
            compare_attention(spec, gpu, oracles, Q[:, :, 2:2 + nq].contiguous(), run_synthesis=True)
    compare_attention(spec, gpu, oracles, Q[:, :, :1].contiguous(), run_synthesis=False, q_pos0=7)
    gpu.close()
