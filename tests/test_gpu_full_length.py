"""-m gpu parity at the stream lengths BASELINE.json's configs state (bank subsets listed
there): C2 all 600 frames on all 4 banks; C3 all 3,600 frames (event cluster at frames 300-304, query after the last
frame) with the full 112-bank state on the GPU and the oracle following layers 0 and 27 x KV heads 0 and 3; every cell of
the C4 sweep (3 x 3, 1,200 frames, oracle on one bank per cell); C5 all 2,000 frames with the full 8-stream state on the
GPU, the oracle following two banks, and a 64-token query every 200 frames.

Same teacher-forced protocol as test_gpu_parity.py.  Frames are generated on the device (the generator is counter-based
and bit-identical on CPU and GPU) and only the followed banks are pulled to the host; the followed oracle banks advance
on a thread pool (the oracle call drops the GIL)."""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import gen
from gpu_helpers import (make_gpu, make_oracles, run_stream, compare_ring, compare_codes, compare_attention, new_stats)

pytestmark = pytest.mark.gpu


def _rows(spec):
    return spec.n_query_tokens * (spec.n_q_heads // spec.n_kv_heads)


def _final_checks(spec, gpu, oracles, rows_sample, query_index=0):
    compare_ring(gpu, oracles)
    compare_codes(gpu, oracles, spec.G)
    Q = gen.queries(spec, query_index)
    compare_attention(spec, gpu, oracles, Q, run_synthesis=False, rows_sample=rows_sample)   # the GPU's own tuples
    compare_attention(spec, gpu, oracles, Q, run_synthesis=True, rows_sample=rows_sample)
    evicted = (gpu.frames_seen - spec.near_frames) * spec.T
    for b in oracles:
        assert int(gpu.export_state(b)["n"].sum()) == evicted                               # mass conservation
    assert gpu.error_flags() == 0


def test_c2_all_600_frames_all_banks():
    spec = gen.spec_for("c2")
    assert spec.n_frames == 600
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, range(spec.n_banks))
    with ThreadPoolExecutor(4) as pool:
        stats = run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=50, on_device=True, pool=pool)
    assert stats["scored"] > 500 * spec.T * spec.n_banks
    _final_checks(spec, gpu, oracles, range(0, _rows(spec), 5))


def test_c3_all_3600_frames_with_event():
    spec = gen.spec_for("c3")
    assert spec.n_frames == 3600 and spec.event[:2] == (300, 305)
    banks = [0, 3, 108, 111]                      # layers 0 and 27 x KV heads 0 and 3
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, banks)
    seen_event = []

    def after(f):
        if 300 + spec.near_frames <= f < 305 + spec.near_frames:     # the step that evicts event frame f - W_f
            seen_event.append(gpu.last_frame_trace()["evicted_frame"])

    with ThreadPoolExecutor(4) as pool:
        stats = run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=300, on_device=True, pool=pool,
                           after_frame=after)
    assert seen_event == [300, 301, 302, 303, 304]
    assert stats["scored"] > 3500 * spec.T * len(banks)
    st = oracles[0].state()
    t_last = spec.n_frames - 1
    assert int(((t_last - st["tau"]) > 120).sum()) > 100, "T_idle = 120 does not fire on > 100 prototypes"
    assert int(st["n"].max()) > 4096, "no prototype with a mass in the thousands (log n_k bias of Eq. 4)"
    _final_checks(spec, gpu, oracles, range(0, _rows(spec), 9))
    print("c3 full length:", stats, "max mass", int(st["n"].max()), "max bin",
          int(max(st["hist_k"].max(), st["hist_v"].max())))


def _c4_cell(k_max, near):
    spec = gen.spec_for(f"c4_k{k_max}_w{near}")
    assert spec.n_frames == 1200
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, [{256: 0, 1024: 1, 4096: 3}[k_max]])   # one bank per cell
    stats = run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=400, on_device=True)
    _final_checks(spec, gpu, oracles, range(0, _rows(spec), 13))
    gpu.close()
    return stats


def test_c4_every_cell_1200_frames():
    cells = [(k, w) for k in (256, 1024, 4096) for w in (4, 16, 64)]
    with ThreadPoolExecutor(len(cells)) as pool:
        futs = {c: pool.submit(_c4_cell, *c) for c in cells}
        for c, fu in futs.items():
            st = fu.result()
            assert st["scored"] > 0, c


def test_c5_all_2000_frames_query_every_200():
    spec = gen.spec_for("c5")
    assert spec.n_frames == 2000 and spec.query_every == 200
    banks = [2, 45]                               # stream 0 head 2; stream 5 head 5
    gpu = make_gpu(spec)
    oracles = make_oracles(spec, banks)
    queries = []

    def after(f):
        if (f + 1) % spec.query_every == 0:
            qi = (f + 1) // spec.query_every
            compare_codes(gpu, oracles, spec.G)
            w = compare_attention(spec, gpu, oracles, gen.queries(spec, qi), run_synthesis=False,
                                  rows_sample=range(qi % 7, _rows(spec), 37))
            queries.append((f, w))

    with ThreadPoolExecutor(2) as pool:
        stats = run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=250, on_device=True, pool=pool,
                           after_frame=after)
    assert len(queries) == 10
    assert stats["scored"] > 1900 * spec.T * len(banks)
    _final_checks(spec, gpu, oracles, range(0, _rows(spec), 31), query_index=11)
    print("c5 full length:", stats, queries)
