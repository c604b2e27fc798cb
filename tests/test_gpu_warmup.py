"""-m gpu parity of the PQ codebook warm-up (readings 32-36) through the
C ABI: reservoir contents against the oracle's (teacher-forced stream), k-means codebooks bit for bit from the same
reservoir, the stream after the warm-up with the trained codebooks, the automatic trigger and the short-warm-up case."""
import numpy as np
import pytest
import torch

import gen
from gpu_helpers import (make_gpu, run_stream, compare_state, compare_codes, compare_attention, new_stats)
from helpers import codebooks_for_bank
from oracle import OracleBank, FLAG_WARMUP, FLAG_WARMUP_MANUAL
from paper_2606_26762_b200 import binding as B

pytestmark = pytest.mark.gpu


def _oracles(spec, banks, flags, **kw):
    out = {}
    seed = kw.pop("km_seed")
    for b in banks:
        out[b] = OracleBank(spec.T, spec.near_frames, spec.k_max, spec.head_dim, None, None, G=spec.G, C=spec.C,
                            flags=flags, km_seed=seed + b, **kw)
    return out


@pytest.mark.parametrize("name,t_warm,R,after", [("c2", 40, 2048, 12), ("c1", 24, 96, 16)])
def test_reservoir_kmeans_and_the_stream_after_the_warmup(name, t_warm, R, after):
    """Manual training: (1) the reservoirs agree after the warm-up (slots bit-exact by construction of the stream,
    rows within the tolerance of the centres); (2) with the oracle's reservoir imported, the GPU's k-means reproduces
    the oracle's codebooks bit for bit; (3) the stream continues teacher-forced with residual histograms."""
    spec = gen.spec_for(name, n_frames=t_warm + after)
    kw = dict(t_warm=t_warm, warm_reservoir=R, km_iters=12, km_batch=128, km_seed=77)
    gpu = make_gpu(spec, with_codebooks=False, flags=B.WARMUP | B.WARMUP_MANUAL, **kw)
    banks = list(range(spec.n_banks))
    orc = _oracles(spec, banks, FLAG_WARMUP | FLAG_WARMUP_MANUAL, **kw)
    stats = run_stream(spec, gpu, orc, t_warm, check_state_every=8, with_codebooks=False)
    assert stats["scored"] > 0
    absorbed = (t_warm - spec.near_frames) * spec.T - spec.k_max
    for b, o in orc.items():
        gk, gv, gseen = gpu.export_reservoir(b)
        ok, ov, oseen = o.reservoir()
        assert gseen == oseen == absorbed and gk.shape == ok.shape and gk.shape[0] == min(R, absorbed)
        assert absorbed > R                                              # replacement was exercised
        assert np.abs(gk - ok).max() <= 2e-5 and np.abs(gv - ov).max() <= 2e-5, (np.abs(gk - ok).max(), np.abs(gv - ov).max())
    for b, o in orc.items():                                             # (the import resets the state-wide residual count)
        ok, ov, _ = o.reservoir()
        gpu.import_reservoir(b, ok, ov)
    with pytest.raises(B.ProtoKVError):
        gpu.export_codebooks(0)                                          # no codebooks before the training
    gpu.train_codebooks()
    for b, o in orc.items():
        assert o.train_codebooks() == 1
        gck, gcv = gpu.export_codebooks(b)
        ock, ocv = o.codebooks()
        assert np.array_equal(gck, ock) and np.array_equal(gcv, ocv), f"bank {b}: codebooks differ"
    with pytest.raises(B.ProtoKVError):
        gpu.train_codebooks()                                            # once
    st2 = run_stream(spec, gpu, orc, after, check_state_every=4, with_codebooks=True, first_frame=t_warm)
    assert st2["codes"] > 0
    for b, o in orc.items():
        s = o.state()
        assert int(s["nres"].sum()) == after * spec.T                    # histograms count only post-warm-up tokens
    compare_codes(gpu, orc, spec.G)
    compare_attention(spec, gpu, orc, gen.queries(spec, 0), run_synthesis=False, use_gpu_codes=True,
                      rows_sample=range(0, spec.n_query_tokens * (spec.n_q_heads // spec.n_kv_heads), 5))
    # a decode-style query reads the bf16 copies of the TRAINED codebooks (Dev::cb_bf, rewritten by the training)
    compare_attention(spec, gpu, orc, gen.queries(spec, 2)[:, :, :1].contiguous(), run_synthesis=False, use_gpu_codes=True)
    assert gpu.error_flags() == 0
    gpu.close()


def test_automatic_training_at_the_end_of_the_warmup():
    """Default mode: the append of frame t_warm - 1 trains the codebooks.  The k-means step is checked by handing the
    oracle the reservoir the GPU trained on (follow mode: one rounding difference in a residual may move a k-means
    decision, so the two reservoirs are compared by tolerance and the training bit for bit from equal inputs)."""
    spec = gen.spec_for("c2", n_frames=40)
    kw = dict(t_warm=36, warm_reservoir=1024, km_iters=8, km_batch=256, km_seed=5)
    gpu = make_gpu(spec, with_codebooks=False, flags=B.WARMUP, **kw)
    orc = _oracles(spec, [0, 3], FLAG_WARMUP | FLAG_WARMUP_MANUAL, **kw)
    run_stream(spec, gpu, orc, 35, check_state_every=0, with_codebooks=False)
    with pytest.raises(B.ProtoKVError):
        gpu.export_codebooks(0)
    run_stream(spec, gpu, orc, 1, check_state_every=0, with_codebooks=False, first_frame=35)
    for b, o in orc.items():
        gk, gv, gseen = gpu.export_reservoir(b)
        ok, ov, oseen = o.reservoir()
        assert gseen == oseen and np.abs(gk - ok).max() <= 2e-5 and np.abs(gv - ov).max() <= 2e-5
        o.set_reservoir(gk, gv)
        assert o.train_codebooks() == 1
        gck, gcv = gpu.export_codebooks(b)
        assert np.array_equal(gck, o.codebooks()[0]) and np.array_equal(gcv, o.codebooks()[1])
    # later frames update histograms and leave the reservoir alone
    s = gen.grid_positions(spec, device="cuda")
    for f in range(36, 40):
        K, V = gen.frame_kv(spec, f, device="cuda")
        gpu.append_frame(K, V, s)
    st = gpu.export_state(0)
    assert int(st["nres"].sum()) == 4 * spec.T
    assert gpu.export_reservoir(0)[2] == gseen
    gpu.close()


def test_short_warmup_raises_the_flag_and_keeps_running():
    spec = gen.spec_for("c1", n_frames=12)
    gpu = make_gpu(spec, with_codebooks=False, flags=B.WARMUP, t_warm=spec.near_frames, warm_reservoir=64, km_iters=4,
                   km_batch=32, km_seed=1)
    s = gen.grid_positions(spec, device="cuda")
    for f in range(12):
        K, V = gen.frame_kv(spec, f, device="cuda")
        gpu.append_frame(K, V, s)
    assert gpu.error_flags() & 4
    st = gpu.export_state(0)
    assert int(st["nres"].sum()) == 0 and int(st["n"].sum()) == (12 - spec.near_frames) * spec.T
    out = gpu.query_attention(gen.queries(spec, 0).to("cuda"))
    assert torch.isfinite(out.float()).all()
    gpu.close()
