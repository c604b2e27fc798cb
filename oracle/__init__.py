"""ctypes front-end of the ProtoKV CPU oracle (oracle/protokv_oracle.cpp) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It shares no code with paper_2606_26762_b200/ (the CUDA path) and neither imports the other.

`build()` compiles the C++ file with g++ -O2 into oracle/libprotokv_oracle.so (git-ignored).
`OracleBank` wraps one bank = one (stream, layer, KV head).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "protokv_oracle.cpp")
_LIB = os.path.join(_HERE, "libprotokv_oracle.so")

FLAG_MAH_SQUARED, FLAG_NO_MASS_BIAS, FLAG_NO_RESIDUAL, FLAG_NEAR_ONLY, FLAG_FAR_ONLY = 1, 2, 4, 8, 16
FLAG_MAINTENANCE = 64
FLAG_ROPE = 256
FLAG_WARMUP, FLAG_WARMUP_MANUAL, FLAG_VAR_ALLOC = 512, 1024, 2048


def build(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off",
                               "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class _Config(C.Structure):
    _fields_ = [("T", C.c_int32), ("near_frames", C.c_int32), ("k_max", C.c_int32), ("d", C.c_int32),
                ("S", C.c_int32), ("G", C.c_int32), ("C", C.c_int32), ("beam", C.c_int32),
                ("lambda_sp", C.c_float), ("lambda_idle", C.c_float), ("t_idle", C.c_int32),
                ("alpha", C.c_float), ("beta", C.c_float), ("eta", C.c_float),
                ("sigma_eps", C.c_float), ("cos_eps", C.c_float), ("pq_eps", C.c_double),
                ("flags", C.c_uint32), ("gamma", C.c_float), ("eps_k", C.c_float), ("eps_v", C.c_float),
                ("rope_theta", C.c_double), ("rope_anchor", C.c_int32), ("pos0", C.c_int64),
                ("t_warm", C.c_int32), ("warm_reservoir", C.c_int32), ("km_iters", C.c_int32),
                ("km_batch", C.c_int32), ("km_seed", C.c_uint64), ("s_cap", C.c_int32)]


class _Trace(C.Structure):
    _fields_ = [("evicted", C.c_int32), ("n_fill", C.c_int32), ("assign", C.c_void_p), ("best", C.c_void_p),
                ("second", C.c_void_p), ("forced_excess", C.c_void_p), ("codes_k", C.c_void_p),
                ("codes_v", C.c_void_p), ("code_gap_k", C.c_void_p), ("code_gap_v", C.c_void_p)]


class _StateView(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("c", "p", "n", "mu", "sigma", "tau", "pos", "hist_k", "hist_v",
                                          "nres", "active", "pos_first", "pos_sum", "pos_cnt")]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.pko_create.restype = C.c_void_p
        lib.pko_create.argtypes = [C.POINTER(_Config), C.c_void_p, C.c_void_p]
        lib.pko_destroy.argtypes = [C.c_void_p]
        lib.pko_append_frame.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                         C.c_void_p, C.c_void_p, C.POINTER(_Trace)]
        lib.pko_frames_seen.argtypes = [C.c_void_p]
        lib.pko_ring_frames.argtypes = [C.c_void_p]
        lib.pko_maintain.argtypes = [C.c_void_p, C.c_int32]
        lib.pko_maintenance_counters.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        lib.pko_get_ring.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        lib.pko_get_state.argtypes = [C.c_void_p, C.POINTER(_StateView)]
        lib.pko_set_state.argtypes = [C.c_void_p, C.POINTER(_StateView)]
        lib.pko_score.restype = C.c_float
        lib.pko_score.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int32]
        lib.pko_synthesize.argtypes = [C.c_void_p] + [C.c_void_p] * 6
        lib.pko_reservoir.restype = C.c_int64
        lib.pko_reservoir.argtypes = [C.c_void_p] * 4
        lib.pko_set_reservoir.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64]
        lib.pko_train_codebooks.argtypes = [C.c_void_p]
        lib.pko_codebooks.argtypes = [C.c_void_p] * 3
        lib.pko_draw.restype = C.c_uint64
        lib.pko_draw.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64]
        lib.pko_reservoir_slot.argtypes = [C.c_void_p, C.c_int64]
        lib.pko_allocation.argtypes = [C.c_void_p] * 3
        lib.pko_decode_hist.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.pko_log_table.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        lib.pko_tuple_score.restype = C.c_int64
        lib.pko_tuple_score.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        lib.pko_context_len.argtypes = [C.c_void_p]
        lib.pko_materialize.argtypes = [C.c_void_p] + [C.c_void_p] * 6 + [C.c_int]
        lib.pko_attention.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                      C.c_void_p, C.c_void_p]
        _lib = lib
    return _lib


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


DEFAULTS = dict(S=8, G=8, C=16, beam=32, lambda_sp=0.1, lambda_idle=0.01, t_idle=120, alpha=0.05, beta=0.05,
                eta=0.05, sigma_eps=1e-4, cos_eps=1e-12, pq_eps=1e-6, flags=0,
                gamma=0.05, eps_k=0.20, eps_v=0.25,   # Table 5
                rope_theta=1.0e6, rope_anchor=0, pos0=0,   # readings 28-30 (the paper fixes no rotary base)
                t_warm=0, warm_reservoir=2048, km_iters=32, km_batch=256, km_seed=0,   # readings 32-36 (L312, L478)
                s_cap=32)                                  # reading 39 (D.3)


class OracleBank:
    """One bank of the oracle. All tensors are numpy, fp32 unless noted (bf16 inputs widened by the caller)."""

    def __init__(self, T, near_frames, k_max, d, codebook_k=None, codebook_v=None, **kw):
        p = dict(DEFAULTS)
        p.update(kw)
        self.cfg = _Config(T=T, near_frames=near_frames, k_max=k_max, d=d, **p)
        self.T, self.near_frames, self.k_max, self.d = T, near_frames, k_max, d
        self.S, self.G, self.C = p["S"], p["G"], p["C"]
        self.smax = p["s_cap"] if p["flags"] & FLAG_VAR_ALLOC else self.S   # rows per slot of code arrays
        self._lib = _load()
        ck = _f32(codebook_k) if codebook_k is not None else None
        cv = _f32(codebook_v) if codebook_v is not None else None
        if ck is not None:
            assert ck.size == self.G * self.C * (d // self.G) and cv.size == ck.size
        self._h = self._lib.pko_create(C.byref(self.cfg), _ptr(ck), _ptr(cv))
        if not self._h:
            raise ValueError("oracle rejected the configuration")

    def __del__(self):
        if getattr(self, "_h", None):
            self._lib.pko_destroy(self._h)
            self._h = None

    # ---- update -------------------------------------------------------------------------------------------
    def append_frame(self, K, V, s, mode=0, forced_assign=None, forced_codes_k=None, forced_codes_v=None,
                     trace=True):
        """Alg. 1 on one frame. mode 0 = frame-synchronous (graded), 1 = token-sequential (literal).
        Returns a dict trace (or None)."""
        K, V, s = _f32(K), _f32(V), _f32(s)
        assert K.shape == (self.T, self.d) and V.shape == K.shape and s.shape == (self.T, 2)
        fa = None if forced_assign is None else np.ascontiguousarray(forced_assign, dtype=np.int32)
        fk = None if forced_codes_k is None else np.ascontiguousarray(forced_codes_k, dtype=np.uint8)
        fv = None if forced_codes_v is None else np.ascontiguousarray(forced_codes_v, dtype=np.uint8)
        tr, out = None, None
        if trace:
            T, G = self.T, self.G
            out = dict(assign=np.empty(T, np.int32), best=np.empty(T, np.float32), second=np.empty(T, np.float32),
                       forced_excess=np.empty(T, np.float32), codes_k=np.empty((T, G), np.uint8),
                       codes_v=np.empty((T, G), np.uint8), code_gap_k=np.empty((T, G), np.float32),
                       code_gap_v=np.empty((T, G), np.float32))
            tr = _Trace(0, 0, *[_ptr(out[k]) for k in ("assign", "best", "second", "forced_excess", "codes_k",
                                                         "codes_v", "code_gap_k", "code_gap_v")])
        rc = self._lib.pko_append_frame(self._h, _ptr(K), _ptr(V), _ptr(s), mode, _ptr(fa), _ptr(fk), _ptr(fv),
                                        C.byref(tr) if tr is not None else None)
        assert rc == 0
        if out is not None:
            out["evicted"], out["n_fill"] = int(tr.evicted), int(tr.n_fill)
        return out

    @property
    def frames_seen(self):
        return self._lib.pko_frames_seen(self._h)

    def maintain(self, t):
        """Alg. 2 at stream time t on the current state (pins)."""
        self._lib.pko_maintain(self._h, int(t))

    def maintenance_counters(self, reset=False):
        out = np.zeros(3, np.int64)
        self._lib.pko_maintenance_counters(self._h, _ptr(out), int(reset))
        return dict(decayed=int(out[0]), merges=int(out[1]), recycled=int(out[2]))

    def ring(self):
        n = self._lib.pko_ring_frames(self._h)
        K = np.empty((n, self.T, self.d), np.float32)
        V = np.empty_like(K)
        s = np.empty((n, self.T, 2), np.float32)
        idx = np.empty(n, np.int32)
        self._lib.pko_get_ring(self._h, _ptr(K), _ptr(V), _ptr(s), _ptr(idx))
        return K, V, s, idx

    def _state_arrays(self):
        k, d, G, Cc = self.k_max, self.d, self.G, self.C
        return dict(c=np.zeros((k, d), np.float32), p=np.zeros((k, d), np.float32), n=np.zeros(k, np.int32),
                    mu=np.zeros((k, 2), np.float32), sigma=np.zeros((k, 3), np.float32), tau=np.zeros(k, np.int32),
                    pos=np.zeros(k, np.int64), hist_k=np.zeros((k, G, Cc), np.uint32),
                    hist_v=np.zeros((k, G, Cc), np.uint32), nres=np.zeros(k, np.uint32),
                    active=np.zeros(k, np.uint8), pos_first=np.zeros(k, np.int64), pos_sum=np.zeros(k, np.int64),
                    pos_cnt=np.zeros(k, np.int32))

    def state(self):
        st = self._state_arrays()
        v = _StateView(*[_ptr(st[f]) for f, _ in _StateView._fields_])
        self._lib.pko_get_state(self._h, C.byref(v))
        return st

    def set_state(self, **fields):
        ref = self._state_arrays()
        keep = {}
        for f, a in fields.items():
            keep[f] = np.ascontiguousarray(a, dtype=ref[f].dtype).reshape(ref[f].shape)
        v = _StateView(*[_ptr(keep.get(f)) for f, _ in _StateView._fields_])
        self._lib.pko_set_state(self._h, C.byref(v))

    def score(self, Ke, se, k, t):
        Ke, se = _f32(Ke), _f32(se)
        return float(self._lib.pko_score(self._h, _ptr(Ke), _ptr(se), int(k), int(t)))

    # ---- synthesis ----------------------------------------------------------------------------------------
    def synthesize(self):
        k, S, G = self.k_max, self.smax, self.G
        out = dict(codes_k=np.zeros((k, S, G), np.uint8), codes_v=np.zeros((k, S, G), np.uint8),
                   scores_k=np.zeros((k, S), np.int64), scores_v=np.zeros((k, S), np.int64),
                   zero=np.zeros(k, np.uint8), s_count=np.zeros(k, np.int32))
        self._lib.pko_synthesize(self._h, *[_ptr(out[f]) for f in ("codes_k", "codes_v", "scores_k", "scores_v",
                                                                    "zero", "s_count")])
        return out

    # ---- PQ codebook warm-up and D.3 allocation ---------------------------------------------
    def reservoir(self):
        """(r^K [n][d], r^V [n][d], residuals offered so far)."""
        R = self.cfg.warm_reservoir
        rk = np.zeros((R, self.d), np.float32)
        rv = np.zeros((R, self.d), np.float32)
        seen = np.zeros(1, np.int64)
        n = self._lib.pko_reservoir(self._h, _ptr(rk), _ptr(rv), _ptr(seen))
        return rk[:n], rv[:n], int(seen[0])

    def set_reservoir(self, rk, rv):
        rk, rv = _f32(rk), _f32(rv)
        assert rk.shape == rv.shape and rk.shape[1] == self.d and rk.shape[0] <= self.cfg.warm_reservoir
        self._lib.pko_set_reservoir(self._h, _ptr(rk), _ptr(rv), rk.shape[0])

    def train_codebooks(self):
        return int(self._lib.pko_train_codebooks(self._h))

    def codebooks(self):
        sub = self.d // self.G
        ck = np.zeros((self.G, self.C, sub), np.float32)
        cv = np.zeros_like(ck)
        return (ck, cv) if self._lib.pko_codebooks(self._h, _ptr(ck), _ptr(cv)) else None

    def draw(self, stream, counter):
        return int(self._lib.pko_draw(self._h, int(stream), int(counter)))

    def reservoir_slot(self, i):
        return int(self._lib.pko_reservoir_slot(self._h, int(i)))

    def allocation(self):
        v = np.zeros(self.k_max, np.int64)
        sk = np.zeros(self.k_max, np.int32)
        self._lib.pko_allocation(self._h, _ptr(v), _ptr(sk))
        return v, sk

    def decode_hist(self, H):
        H = np.ascontiguousarray(H, dtype=np.uint32)
        assert H.shape == (self.G, self.C)
        codes = np.zeros((self.S, self.G), np.uint8)
        scores = np.zeros(self.S, np.int64)
        n = self._lib.pko_decode_hist(self._h, _ptr(H), _ptr(codes), _ptr(scores))
        return codes[:n], scores[:n]

    def log_table(self, H):
        H = np.ascontiguousarray(H, dtype=np.uint32)
        q = np.zeros((self.G, self.C), np.int64)
        self._lib.pko_log_table(self._h, _ptr(H), _ptr(q))
        return q

    def tuple_score(self, k, which, z):
        z = np.ascontiguousarray(z, dtype=np.uint8)
        return int(self._lib.pko_tuple_score(self._h, int(k), int(which), _ptr(z)))

    # ---- attention ----------------------------------------------------------------------------------------
    def materialize(self, forced_codes_k=None, forced_codes_v=None, positions=False, rotate=True):
        """[near || pseudo] keys, values, bias (fp64).  positions=True also returns the stream position of every
        element; rotate=False returns the keys before the rotary embedding (FLAG_ROPE only)."""
        fk = None if forced_codes_k is None else np.ascontiguousarray(forced_codes_k, dtype=np.uint8)
        fv = None if forced_codes_v is None else np.ascontiguousarray(forced_codes_v, dtype=np.uint8)
        L = self._lib.pko_context_len(self._h)
        Kt = np.empty((L, self.d), np.float64)
        Vt = np.empty((L, self.d), np.float64)
        b = np.empty(L, np.float64)
        ps = np.empty(L, np.float64)
        self._lib.pko_materialize(self._h, _ptr(fk), _ptr(fv), _ptr(Kt), _ptr(Vt), _ptr(b), _ptr(ps), int(rotate))
        return (Kt, Vt, b, ps) if positions else (Kt, Vt, b)

    def attention(self, Q, forced_codes_k=None, forced_codes_v=None, return_lse=False, qpos=None):
        """Q [rows][d] -> O [rows][d] fp32 (Alg. 4).  qpos [rows] int64: stream positions of the query rows (FLAG_ROPE)."""
        Q = _f32(Q)
        rows = Q.shape[0]
        assert Q.shape == (rows, self.d)
        fk = None if forced_codes_k is None else np.ascontiguousarray(forced_codes_k, dtype=np.uint8)
        fv = None if forced_codes_v is None else np.ascontiguousarray(forced_codes_v, dtype=np.uint8)
        out = np.empty((rows, self.d), np.float32)
        lse = np.empty(rows, np.float64)
        qp = None if qpos is None else np.ascontiguousarray(qpos, dtype=np.int64)
        assert qp is None or qp.shape == (rows,)
        rc = self._lib.pko_attention(self._h, _ptr(Q), rows, _ptr(fk), _ptr(fv), _ptr(out), _ptr(lse), _ptr(qp))
        assert rc == 0
        return (out, lse) if return_lse else out
