"""-m gpu parity of the variance-aware pseudo-token allocation (D.3; DESIGN.md
readings 37-40) through the C ABI: fixed-point variances and integer shares bit-exact against the oracle, ragged
synthesis under the tie rule of the parity protocol, attention over the ragged context."""
import numpy as np
import pytest

import gen
from gpu_helpers import make_gpu, make_oracles, run_stream, compare_attention
from oracle import FLAG_VAR_ALLOC
from paper_2606_26762_b200 import binding as B

pytestmark = pytest.mark.gpu


def _compare_ragged_codes(gpu, orc, G):
    """GPU tuples equal the oracle's, or differ only where the oracle's fixed-point score of the GPU's tuple is within G
    units of the oracle's score at that rank and of its S_k-th score (last-bit log differences)."""
    flips = 0
    for b, o in orc.items():
        gk, gv, kind = gpu.export_codes(b)
        sk, v = gpu.export_allocation(b)
        ov, osk = o.allocation()
        assert np.array_equal(v, ov), f"bank {b}: variances differ ({np.abs(v - ov).max()})"
        assert np.array_equal(sk, osk), f"bank {b}: shares differ"
        syn = o.synthesize()
        assert np.array_equal(kind, syn["zero"]) and np.array_equal(syn["s_count"], sk)
        for which, gc, oc, osc in ((0, gk, syn["codes_k"], syn["scores_k"]), (1, gv, syn["codes_v"], syn["scores_v"])):
            for k in np.nonzero(kind == 0)[0]:
                m = int(sk[k])
                if np.array_equal(gc[k, :m], oc[k, :m]):
                    continue
                flips += 1
                for s in range(m):
                    if not np.array_equal(gc[k, s], oc[k, s]):
                        sc = o.tuple_score(int(k), which, gc[k, s])
                        assert abs(sc - osc[k][s]) <= G and sc >= osc[k][m - 1] - G, f"bank {b} prototype {k} tuple {s}"
    return flips


@pytest.mark.parametrize("name,frames,s_cap,kmax", [("c2", 40, 32, 256), ("c2", 30, 10, 128), ("c1", 40, 16, 32)])
def test_allocation_synthesis_and_attention(name, frames, s_cap, kmax):
    spec = gen.spec_for(name, n_frames=frames, k_max=kmax)
    gpu = make_gpu(spec, flags=B.VAR_ALLOC, s_cap=s_cap, beam=32)
    banks = list(range(spec.n_banks))
    orc = make_oracles(spec, banks, flags=FLAG_VAR_ALLOC, s_cap=s_cap, beam=32)
    # production shape: the ragged variant of the register-resident kernel (8-row blocks); fp32 / d = 64: the SIMT kernel
    assert gpu.stage_impl(1) == ("mma.sync register-resident (blocks)" if name == "c2" else "simt")
    run_stream(spec, gpu, orc, frames, check_state_every=10)
    gpu.synthesize()
    _compare_ragged_codes(gpu, orc, spec.G)
    for b, o in orc.items():
        sk, v = gpu.export_allocation(b)
        assert sk.max() <= s_cap and sk[sk > 0].min() >= 1
        assert v.max() > 0 and len(set(sk.tolist())) > 2                 # the shares really are unequal
        if sk.max() < s_cap:
            assert sk.sum() == spec.k_max * 8                            # S_tot = K_max S: L_context unchanged (L616)
    compare_attention(spec, gpu, orc, gen.queries(spec, 0), run_synthesis=False, use_gpu_codes=True,
                      rows_sample=range(0, spec.n_query_tokens * (spec.n_q_heads // spec.n_kv_heads), 5))
    compare_attention(spec, gpu, orc, gen.queries(spec, 1)[:, :, :1].contiguous(), run_synthesis=False, use_gpu_codes=True)
    gpu.close()


def test_ragged_attention_routes_agree():
    """The same VAR_ALLOC state through the ragged register-resident kernel and through the SIMT kernel (FORCE_SIMT)."""
    spec = gen.spec_for("c2", n_frames=36, k_max=256)
    outs = []
    for route in (0, B.FORCE_SIMT):
        gpu = make_gpu(spec, flags=B.VAR_ALLOC | route, s_cap=24)
        s = gen.grid_positions(spec, device="cuda")
        for f in range(spec.n_frames):
            K, V = gen.frame_kv(spec, f, device="cuda")
            gpu.append_frame(K, V, s)
        outs.append(gpu.query_attention(gen.queries(spec, 0).cuda()).float().cpu())
        gpu.close()
    import torch
    assert torch.allclose(outs[0], outs[1], atol=1e-2, rtol=2e-2)


def test_ragged_allocation_with_rotary_anchoring():
    """PROTOKV_VAR_ALLOC | PROTOKV_ROPE: ragged pseudo-token counts, every prototype's rows rotated at its anchor."""
    from oracle import FLAG_ROPE
    spec = gen.spec_for("c2", n_frames=32, k_max=128)
    hyper = dict(s_cap=20, pos0=40_000, rope_anchor=2)
    gpu = make_gpu(spec, flags=B.VAR_ALLOC | B.ROPE, **hyper)
    orc = make_oracles(spec, [0, 3], flags=FLAG_VAR_ALLOC | FLAG_ROPE, **hyper)
    run_stream(spec, gpu, orc, spec.n_frames, check_state_every=16)
    gpu.synthesize()
    _compare_ragged_codes(gpu, orc, spec.G)
    compare_attention(spec, gpu, orc, gen.queries(spec, 0)[:, :, :5].contiguous(), run_synthesis=False, use_gpu_codes=True)
    compare_attention(spec, gpu, orc, gen.queries(spec, 0)[:, :, :1].contiguous(), run_synthesis=False, use_gpu_codes=True)
    gpu.close()


def test_no_residual_statistics_fall_back_to_fixed_s():
    """Without codebooks every variance is 0: S_k = S for every prototype, the attention equals the fixed-S one."""
    spec = gen.spec_for("c1", n_frames=20)
    gpu = make_gpu(spec, with_codebooks=False, flags=B.VAR_ALLOC, s_cap=16)
    orc = make_oracles(spec, [0], with_codebooks=False, flags=FLAG_VAR_ALLOC, s_cap=16)
    run_stream(spec, gpu, orc, 20, check_state_every=0, with_codebooks=False)
    gpu.synthesize()
    sk, v = gpu.export_allocation(0)
    act = gpu.export_state(0)["active"].astype(bool)
    assert (v == 0).all() and (sk[act] == 8).all() and (sk[~act] == 0).all()
    assert np.array_equal(sk, orc[0].allocation()[1])
    compare_attention(spec, gpu, orc, gen.queries(spec, 0), run_synthesis=False)
    gpu.close()
