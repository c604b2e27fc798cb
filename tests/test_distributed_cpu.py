"""N>1 path on CPU (-m "not gpu"): world_size-2 gloo processes.  Banks are independent, so the
multi-GPU design is "one state per rank over a disjoint slice of streams / layers / KV heads, no data-path
collective".  Checked here: the slices partition the banks; a rank that runs only its slice gets, bank for bank, the
bits the single-process run gets (with the oracle standing in for the state, since there is no GPU here); timings
reduce by MAX over ranks; the oracle arm of bench.py prints on rank 0 only."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import gen
from helpers import make_oracle, frame_for_bank, bank_coords
from paper_2606_26762_b200 import sharding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("axis", sharding.AXES)
@pytest.mark.parametrize("world", [1, 2, 3])
def test_slices_partition_the_banks(axis, world):
    NS, L, HQ, HKV = 3, 5, 28, 4
    seen = []
    for r in range(world):
        sh = sharding.shard_config(NS, L, HQ, HKV, world, r, axis)
        assert sh["n_q_heads"] // sh["n_kv_heads"] == HQ // HKV
        banks = sharding.owned_banks(NS, L, HKV, sh)
        assert len(banks) == sh["n_streams"] * sh["n_layers"] * sh["n_kv_heads"]
        seen += list(banks)
    assert sorted(seen) == list(range(NS * L * HKV))
    with pytest.raises(ValueError):
        sharding.shard_config(1, 1, 4, 4, 5, 0, axis)


def test_slicing_follows_the_abi_layout():
    NS, L, T, HKV, HQ, d, NQ = 2, 3, 4, 4, 8, 8, 2
    K = torch.arange(NS * L * T * HKV * d, dtype=torch.float32).reshape(NS, L, T, HKV, d)
    Q = torch.arange(NS * L * NQ * HQ * d, dtype=torch.float32).reshape(NS, L, NQ, HQ, d)
    sh = sharding.shard_config(NS, L, HQ, HKV, 2, 1, "kv_head")
    assert torch.equal(sharding.slice_kv(K, sh), K[:, :, :, 2:4])
    assert torch.equal(sharding.slice_q(Q, sh, HQ // HKV), Q[:, :, :, 4:8])
    sh = sharding.shard_config(NS, L, HQ, HKV, 2, 0, "layer")
    assert torch.equal(sharding.slice_kv(K, sh), K[:, 0:2]) and sharding.slice_kv(K, sh).is_contiguous()
    s = torch.zeros(NS, T, 2)
    assert sharding.slice_grid_pos(s, sh).shape[0] == NS
    sh = sharding.shard_config(NS, L, HQ, HKV, 2, 1, "stream")
    assert sharding.slice_grid_pos(s, sh).shape[0] == 1


def _worker(rank, world, port, axis, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        spec = gen.spec_for("c1", n_frames=12)
        import dataclasses
        spec = dataclasses.replace(spec, n_streams=2, n_layers=2, n_q_heads=4, n_kv_heads=2)
        sh = sharding.shard_config(spec.n_streams, spec.n_layers, spec.n_q_heads, spec.n_kv_heads, world, rank, axis)
        banks = sharding.owned_banks(spec.n_streams, spec.n_layers, spec.n_kv_heads, sh)
        local = dataclasses.replace(spec, n_streams=sh["n_streams"], n_layers=sh["n_layers"], n_q_heads=sh["n_q_heads"],
                                    n_kv_heads=sh["n_kv_heads"])
        oracles = {b: make_oracle(spec, b) for b in banks}
        s_all = gen.grid_positions(spec)
        for f in range(spec.n_frames):
            K, V = gen.frame_kv(spec, f)                       # the full job's frame ...
            Kl, Vl = sharding.slice_kv(K, sh), sharding.slice_kv(V, sh)   # ... and what this rank's state would be fed
            sl = sharding.slice_grid_pos(s_all, sh)
            if axis == "stream":   # what bench.py --gpus N feeds a rank: the shard generated directly (stream0 = begin)
                shard = dataclasses.replace(local, stream0=sh["begin"])
                Kd, Vd = gen.frame_kv(shard, f)
                assert torch.equal(Kd, Kl) and torch.equal(Vd, Vl)
                if f == 0:
                    group = spec.n_q_heads // spec.n_kv_heads
                    assert torch.equal(gen.queries(shard, 3), sharding.slice_q(gen.queries(spec, 3), sh, group))
                    assert torch.equal(gen.codebooks(shard)[0], gen.codebooks(spec)[0][sh["begin"]:sh["end"]])
            for i, b in enumerate(banks):                      # rank-local bank i  <->  global bank b
                st, la, hd = bank_coords(local, i)
                k_loc, v_loc = Kl[st, la, :, hd].float().numpy(), Vl[st, la, :, hd].float().numpy()
                k_glob, v_glob, s_glob = frame_for_bank(spec, f, b, kv=(K, V))
                assert np.array_equal(k_loc, k_glob) and np.array_equal(v_loc, v_glob)
                assert np.array_equal(sl[st].numpy(), s_glob)
                oracles[b].append_frame(k_loc, v_loc, sl[st].numpy(), trace=False)
        masses = {b: int(np.asarray(oracles[b].state()["n"]).sum()) for b in banks}
        # timing rule: max over ranks; whole-job rate = world * units / slowest
        t = sharding.max_over_ranks([1.0 + rank, 5.0 - rank])
        gathered = [None] * world
        dist.all_gather_object(gathered, masses)
        if rank == 0:
            q.put((t, gathered))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("axis", ["stream", "kv_head"])
def test_two_ranks_over_disjoint_banks_match_the_single_process_run(axis):
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = 29500 + (os.getpid() % 400) + (7 if axis == "stream" else 11)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, axis, q)) for r in range(2)]
    for p in procs: p.start()
    for p in procs: p.join(180)
    assert all(p.exitcode == 0 for p in procs)
    t, gathered = q.get()
    assert t == [2.0, 5.0]
    merged = {}
    for g in gathered:
        assert not (set(g) & set(merged))
        merged.update(g)
    # single-process run over all banks: every absorbed token carries mass 1 (mass conservation per bank)
    import dataclasses
    spec = dataclasses.replace(gen.spec_for("c1", n_frames=12), n_streams=2, n_layers=2, n_q_heads=4, n_kv_heads=2)
    assert sorted(merged) == list(range(spec.n_banks))
    evicted = (spec.n_frames - spec.near_frames) * spec.T
    assert all(m == evicted for m in merged.values())
    assert sharding.whole_job_rate(100, 2.0, 2) == 100.0


def test_reference_arm_prints_on_rank_zero_only():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "c1",
                        "--steps", "1", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"; env["LOCAL_RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "c1",
                        "--steps", "1", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
