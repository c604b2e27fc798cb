"""Shared test helpers: feed generator output (gen/) to oracle banks. No ProtoKV arithmetic here."""
import numpy as np
import torch

import gen
from oracle import OracleBank


def bank_index(spec, stream, layer, head):
    return (stream * spec.n_layers + layer) * spec.n_kv_heads + head


def bank_coords(spec, bank):
    head = bank % spec.n_kv_heads
    layer = (bank // spec.n_kv_heads) % spec.n_layers
    stream = bank // (spec.n_kv_heads * spec.n_layers)
    return stream, layer, head


def frame_for_bank(spec, frame, bank, kv=None):
    """(K [T][d], V [T][d], s [T][2]) fp32 numpy for one bank, from gen.frame_kv (values exactly as the dtype holds)."""
    K, V = kv if kv is not None else gen.frame_kv(spec, frame)
    st, la, hd = bank_coords(spec, bank)
    s = gen.grid_positions(spec)[st].numpy()
    return (K[st, la, :, hd, :].float().numpy(), V[st, la, :, hd, :].float().numpy(), s)


def codebooks_for_bank(spec, bank, cb=None):
    ck, cv = cb if cb is not None else gen.codebooks(spec)
    st, la, hd = bank_coords(spec, bank)
    return ck[st, la, hd].numpy(), cv[st, la, hd].numpy()


def make_oracle(spec, bank=0, with_codebooks=True, **kw):
    ck = cv = None
    if with_codebooks:
        ck, cv = codebooks_for_bank(spec, bank)
    kw.setdefault("G", spec.G)
    kw.setdefault("C", spec.C)
    return OracleBank(spec.T, spec.near_frames, spec.k_max, spec.head_dim, ck, cv, **kw)


def query_rows_for_bank(spec, Q, bank):
    """Q [S][L][Nq][Hq][d] -> rows [Nq * group][d] fp32 numpy for one bank, row = i * group + h_in_group."""
    st, la, hd = bank_coords(spec, bank)
    group = spec.n_q_heads // spec.n_kv_heads
    q = Q[st, la, :, hd * group:(hd + 1) * group, :].float().numpy()
    return np.ascontiguousarray(q.reshape(-1, spec.head_dim))
