"""CPU-side checks of the boundary (-m "not gpu"): the C-ABI library builds, loads and exports every symbol that
include/protokv.h declares; host-only entry points work without a device; there is no CPU fallback."""
import ctypes
import os
import re

import pytest
import torch

import paper_2606_26762_b200 as pkv
from paper_2606_26762_b200.binding import make_config, ProtoKVConfig

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "protokv.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(protokv_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = pkv.load_library()
    names = _declared_functions()
    assert len(names) >= 19
    for n in names:
        assert hasattr(lib, n), f"{n} declared in protokv.h but not exported"
    assert sorted(pkv.EXPORTED_SYMBOLS) == names


def _cfg(**kw):
    base = dict(n_streams=1, n_layers=1, n_q_heads=28, n_kv_heads=4, head_dim=128, dtype=pkv.BF16,
                tokens_per_frame=196, near_frames=16, k_max=1024, n_query_tokens=32)
    base.update(kw)
    return make_config(**base)


def test_workspace_bytes_is_host_only_and_scales():
    a = pkv.protokv_workspace_bytes(_cfg())
    b = pkv.protokv_workspace_bytes(_cfg(n_layers=2))
    assert a > 0 and 1.4 * a < b < 2.1 * a     # a constant split-KV scratch term does not scale
    # config 2: ring 2 * 4 * 16 * 196 * 128 * 2 B = 6.4 MB, bank fp32 centres 2 * 4 * 1024 * 128 * 4 = 4.2 MB, ...
    assert 15e6 < a < 45e6     # (+ 2 MB of bf16 centre copies for the decode-style kernel since round 2)
    assert a % 256 == 0


@pytest.mark.parametrize("kw,code_substr", [
    (dict(head_dim=96), "head_dim"), (dict(n_q_heads=30), "n_q_heads"), (dict(S=9), "S <= 8"),
    (dict(C=17), "C <= 16"), (dict(G=3), "G in"), (dict(beam=4), "beam"), (dict(tokens_per_frame=0), "shape"),
    (dict(tokens_per_frame=5000), "4096"), (dict(alpha=1.5), "alpha"), (dict(pq_eps=0.0), "pq_eps"),
    (dict(flags=pkv.NEAR_ONLY | pkv.FAR_ONLY), "exclusive"), (dict(G=1, C=2, S=8, beam=8), "C^G"),
    (dict(flags=pkv.WARMUP, t_warm=0), "warm-up"), (dict(flags=pkv.WARMUP, t_warm=8, km_batch=4096), "warm-up"),
    (dict(flags=pkv.WARMUP_MANUAL), "WARMUP_MANUAL"), (dict(flags=pkv.VAR_ALLOC, s_cap=33), "s_cap"),
    (dict(flags=pkv.VAR_ALLOC, s_cap=0), "s_cap"), (dict(flags=pkv.ROPE, rope_anchor=3), "rope"),
])
def test_invalid_configs_are_rejected_with_a_message(kw, code_substr):
    assert pkv.protokv_workspace_bytes(_cfg(**kw)) == 0
    assert code_substr in pkv.protokv_last_error()


def test_optional_rows_change_the_workspace_only_by_their_own_arrays():
    base = pkv.protokv_workspace_bytes(_cfg())
    warm = pkv.protokv_workspace_bytes(_cfg(flags=pkv.WARMUP, t_warm=40, warm_reservoir=2048))
    # two reservoirs of 2,048 x 128 fp32 rows per bank + claim words + the per-frame slot plan
    assert warm - base >= 4 * (2 * 2048 * 128 * 4 + 2048 * 8 + 196 * 4)
    assert warm - base < 4 * (2 * 2048 * 128 * 4 + 2048 * 8 + 196 * 4) + 4096
    var = pkv.protokv_workspace_bytes(_cfg(flags=pkv.VAR_ALLOC))
    assert 0 < var - base < 4 * 1024 * 32 + 4096


def test_struct_size_is_checked():
    cfg = _cfg()
    cfg.struct_size = 8
    assert pkv.protokv_workspace_bytes(cfg) == 0
    assert "struct_size" in pkv.protokv_last_error()
    assert ctypes.sizeof(ProtoKVConfig) % 8 == 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback():
    with pytest.raises(pkv.ProtoKVError):
        pkv.ProtoKV(n_streams=1, n_layers=1, n_q_heads=1, n_kv_heads=1, head_dim=64, dtype="f32",
                    tokens_per_frame=16, near_frames=4, k_max=32, n_query_tokens=8)
    # straight through the C ABI as well: create must fail with "unsupported", never compute on the host
    lib = pkv.load_library()
    cfg = _cfg()
    buf = ctypes.create_string_buffer(1024)
    cfg.workspace = (ctypes.addressof(buf) + 255) // 256 * 256
    cfg.workspace_bytes = 1 << 40
    assert lib.protokv_create(ctypes.byref(cfg)) is None
    assert "no CUDA device" in pkv.protokv_last_error() or "sm_" in pkv.protokv_last_error()


def test_null_arguments_are_errors():
    lib = pkv.load_library()
    assert lib.protokv_append_frame(None, None, None, None) == 1
    assert lib.protokv_query_attention(None, None, None) == 1
    assert lib.protokv_frames_seen(None) == -1
    lib.protokv_destroy(None)      # no-op
