"""Pins of the oracle's rotary position anchoring (§3.3; §D.1; SURVEY.md 8(f) NEXT-3;
DESIGN.md readings 28-31).  CPU only.  The rotary embedding is pinned to the rotate-half routine of the installed
`transformers` package and to the relative-position property of RoPE; the three anchor variants (most recent / first /
average absorbed position) are pinned by recomputing them from the assignment log."""
import numpy as np
import pytest
import torch

import gen
from helpers import make_oracle, frame_for_bank, query_rows_for_bank
from oracle import FLAG_ROPE

SPEC = gen.spec_for("c1", n_frames=24)


def _stream(o, spec, n_frames, log=None):
    for f in range(n_frames):
        K, V, s = frame_for_bank(spec, f, 0)
        tr = o.append_frame(K, V, s)
        if log is not None:
            log.append(tr)


def _library_rope(x, pos, theta):
    """x [n][d] fp64, pos [n]: the rotate-half formulation of transformers (x cos + rotate_half(x) sin)."""
    from transformers.models.llama.modeling_llama import rotate_half
    d = x.shape[1]
    inv_freq = 1.0 / (theta ** (torch.arange(0, d, 2, dtype=torch.float64) / d))
    freqs = torch.as_tensor(pos, dtype=torch.float64)[:, None] * inv_freq[None, :]
    emb = torch.cat((freqs, freqs), dim=-1)
    xt = torch.as_tensor(x, dtype=torch.float64)
    return xt * emb.cos() + rotate_half(xt) * emb.sin()


@pytest.mark.parametrize("anchor", [0, 1, 2])
def test_rope_attention_against_transformers_rotate_half(anchor):
    theta = 10000.0
    o = make_oracle(SPEC, flags=FLAG_ROPE, rope_theta=theta, rope_anchor=anchor)
    _stream(o, SPEC, SPEC.n_frames)
    Q = query_rows_for_bank(SPEC, gen.queries(SPEC, 0), 0)
    qpos = np.arange(Q.shape[0], dtype=np.int64) + SPEC.n_frames * SPEC.T + 3
    Ku, V, b, ps = o.materialize(positions=True, rotate=False)
    Kr = o.materialize()[0]
    k_rot = _library_rope(Ku, ps, theta)
    assert np.allclose(Kr, k_rot.numpy(), rtol=0, atol=1e-9)                 # the oracle's rotated keys
    q_rot = _library_rope(Q.astype(np.float64), qpos, theta)
    ref = torch.nn.functional.scaled_dot_product_attention(q_rot[None], k_rot[None], torch.as_tensor(V)[None],
                                                           attn_mask=torch.as_tensor(b)[None, None, :])[0]
    got = o.attention(Q, qpos=qpos)
    assert np.allclose(got, ref.numpy(), rtol=0, atol=2e-6)
    # and rotation matters: the un-rotated attention differs
    plain = make_oracle(SPEC)
    _stream(plain, SPEC, SPEC.n_frames)
    assert np.abs(plain.attention(Q) - got).max() > 1e-3


def test_rope_depends_on_relative_positions_only():
    a = make_oracle(SPEC, flags=FLAG_ROPE, pos0=0)
    b = make_oracle(SPEC, flags=FLAG_ROPE, pos0=987654)
    _stream(a, SPEC, SPEC.n_frames)
    _stream(b, SPEC, SPEC.n_frames)
    Q = query_rows_for_bank(SPEC, gen.queries(SPEC, 1), 0)
    qpos = np.arange(Q.shape[0], dtype=np.int64) * 5 + 400
    oa, ob = a.attention(Q, qpos=qpos), b.attention(Q, qpos=qpos + 987654)
    assert np.allclose(oa, ob, rtol=0, atol=5e-6)
    # default query position = the next stream position, pos0 + frames_seen * T
    assert np.array_equal(a.attention(Q), a.attention(Q, qpos=np.full(Q.shape[0], SPEC.n_frames * SPEC.T, np.int64)))


def test_rope_preserves_norms_and_unrotated_values():
    o = make_oracle(SPEC, flags=FLAG_ROPE)
    _stream(o, SPEC, SPEC.n_frames)
    Ku, Vu, _, _ = o.materialize(positions=True, rotate=False)
    Kr, Vr, _ = o.materialize()
    assert np.allclose(np.linalg.norm(Kr, axis=1), np.linalg.norm(Ku, axis=1), rtol=1e-12)   # rotations are orthogonal
    assert np.array_equal(Vr, Vu)                                                            # values are not rotated


def test_anchor_fields_from_the_assignment_log():
    spec = SPEC
    log = []
    o = make_oracle(spec)
    _stream(o, spec, spec.n_frames, log)
    st = o.state()
    first, last, total, cnt = {}, {}, {}, {}
    for f, tr in enumerate(log):
        if not tr["evicted"]:
            continue
        fe = f - spec.near_frames                                  # index of the evicted frame
        for j, k in enumerate(tr["assign"]):
            ps = fe * spec.T + j
            first.setdefault(int(k), ps)
            last[int(k)] = ps
            total[int(k)] = total.get(int(k), 0) + ps
            cnt[int(k)] = cnt.get(int(k), 0) + 1
    for k in first:
        assert st["pos_first"][k] == first[k] and st["pos"][k] == last[k]
        assert st["pos_sum"][k] == total[k] and st["pos_cnt"][k] == cnt[k] == st["n"][k]
    # the anchors the attention uses: positions of the pseudo-tokens under each variant
    n_near = spec.near_frames * spec.T
    act = np.nonzero(st["active"])[0]
    for anchor, want in ((0, st["pos"][act].astype(np.float64)), (1, st["pos_first"][act].astype(np.float64)),
                         (2, st["pos_sum"][act] / st["pos_cnt"][act])):
        oa = make_oracle(spec, flags=FLAG_ROPE, rope_anchor=anchor)
        _stream(oa, spec, spec.n_frames)
        ps = oa.materialize(positions=True)[3]
        assert np.array_equal(ps[:n_near], np.arange((spec.n_frames - spec.near_frames) * spec.T, spec.n_frames * spec.T))
        assert np.allclose(ps[n_near:].reshape(len(act), 8), want[:, None], rtol=1e-15)
