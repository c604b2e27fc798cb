"""-m gpu parity of Alg. 2 prototype maintenance (csrc/maintenance.cu) against
the oracle's Bank::maintain, teacher-forced like every other stream test: after each frame the GPU's assignment / PQ
decisions are checked and followed, and the whole state -- masses after decay, merged centres and histograms, recycled
slots -- is compared field by field (integers bit-exact, c / p / mu / Sigma within 1e-4 relative)."""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import gen
from gpu_helpers import make_gpu, make_oracles, run_stream, compare_codes, compare_attention, compare_state
from oracle import FLAG_MAINTENANCE
from paper_2606_26762_b200 import MAINTENANCE, FORCE_SIMT

pytestmark = pytest.mark.gpu


def _oracle_counters(oracles):
    tot = dict(decayed=0, merges=0, recycled=0)
    for o in oracles.values():
        for k, v in o.maintenance_counters().items():
            tot[k] += v
    return tot


# aggressive settings so that all three passes of Alg. 2 fire within a short stream: prototypes idle for more than 6
# frames lose 30 % of their mass per frame, same-cluster prototypes closer than 1.0 / 1.2 merge, emptied slots recycle
@pytest.mark.parametrize("name,force_simt", [("c2", False), ("c2", True), ("c1", False)])
def test_maintenance_all_three_passes(name, force_simt):
    spec = gen.spec_for(name, n_frames=70 if name == "c2" else 64)
    hyper = dict(t_idle=6, gamma=0.3, eps_k=1.0, eps_v=1.2) if name == "c2" else dict(t_idle=3, gamma=0.3, eps_k=1.2, eps_v=1.2)
    gpu = make_gpu(spec, flags=MAINTENANCE | (FORCE_SIMT if force_simt else 0), **hyper)
    banks = list(range(spec.n_banks))
    oracles = make_oracles(spec, banks, flags=FLAG_MAINTENANCE, **hyper)
    with ThreadPoolExecutor(len(banks)) as pool:
        run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=2, pool=pool)
    got, want = gpu.maintenance_counters(), _oracle_counters(oracles)
    assert got == want, (got, want)
    assert want["decayed"] > 0 and want["merges"] > 0 and want["recycled"] >= want["merges"]
    assert gpu.error_flags() == 0
    # generalised mass invariant on the GPU state: sum n = absorbed - decayed + recycled
    absorbed = (spec.n_frames - spec.near_frames) * spec.T * spec.n_banks
    assert sum(int(gpu.export_state(b)["n"].sum()) for b in banks) == absorbed - got["decayed"] + got["recycled"]
    compare_codes(gpu, oracles, spec.G)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=True)
    # decode-style queries over a bank with merged-away (absent) slots in the middle of the active prefix
    compare_attention(spec, gpu, oracles, gen.queries(spec, 1)[:, :, :1].contiguous(), run_synthesis=False)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 1)[:, :, 1:3].contiguous(), run_synthesis=False)


# neutral settings: Alg. 2 runs every frame and must leave the plain path untouched, bit for bit in the integers
def test_neutral_maintenance_changes_nothing():
    spec = gen.spec_for("c2", n_frames=40)
    a = make_gpu(spec)
    b = make_gpu(spec, flags=MAINTENANCE, gamma=0.0, eps_k=0.0, eps_v=0.0)
    s = gen.grid_positions(spec).cuda()
    for f in range(spec.n_frames):
        K, V = gen.frame_kv(spec, f)
        a.append_frame(K.cuda(), V.cuda(), s)
        b.append_frame(K.cuda(), V.cuda(), s)
    for bank in range(spec.n_banks):
        sa, sb = a.export_state(bank), b.export_state(bank)
        for f in sa:
            assert np.array_equal(sa[f], sb[f]), f
    assert b.maintenance_counters() == dict(decayed=0, merges=0, recycled=0)


# config 3 (full 112-bank state on the GPU) through the rare-event cluster of frames 300-304 with the Table 5 defaults
# (T_idle 120, gamma 0.05, eps 0.20 / 0.25): by then the bank has been full for ~280 frames and idle prototypes have
# started to decay, so slots are being recycled while the event passes through the near window
def test_c3_through_the_event_with_default_maintenance():
    spec = gen.spec_for("c3", n_frames=345)
    gpu = make_gpu(spec, flags=MAINTENANCE)
    banks = [1, 110]
    oracles = make_oracles(spec, banks, flags=FLAG_MAINTENANCE)
    recycled_by_frame = {}

    def after(f):
        if f in (299, 304, 320, 344):
            recycled_by_frame[f] = _oracle_counters(oracles)["recycled"]

    with ThreadPoolExecutor(len(banks)) as pool:
        run_stream(spec, gpu, oracles, spec.n_frames, check_state_every=15, on_device=True, pool=pool, after_frame=after)
    want = _oracle_counters(oracles)
    assert want["decayed"] > 0 and want["recycled"] > 0, want
    # slots were (re)opened while the event frames sat in the near window / were being absorbed
    assert recycled_by_frame[344] > recycled_by_frame[299], recycled_by_frame
    for b in banks:
        compare_state(gpu.export_state(b), oracles[b].state(), f"end bank {b}")
    assert gpu.error_flags() == 0
    compare_codes(gpu, oracles, spec.G)
    rows = spec.n_query_tokens * (spec.n_q_heads // spec.n_kv_heads)
    compare_attention(spec, gpu, oracles, gen.queries(spec, 0), run_synthesis=True, rows_sample=range(0, rows, 9))
    print("c3 maintenance:", want, recycled_by_frame)
