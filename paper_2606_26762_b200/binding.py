"""ctypes binding of include/protokv.h.  Same names as the C entry points; torch supplies device memory and
the stream.  Nothing here computes: tensors go in as raw pointers, results come back in caller tensors."""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from .build import build

F32, BF16 = 0, 1
MAH_SQUARED, NO_MASS_BIAS, NO_RESIDUAL, NEAR_ONLY, FAR_ONLY, FORCE_SIMT, MAINTENANCE, DECODE_SPLITKV, ROPE = 1, 2, 4, 8, 16, 32, 64, 128, 256
WARMUP, WARMUP_MANUAL, VAR_ALLOC, NO_DECODE_KERNEL, SERIAL_LAUNCH = 512, 1024, 2048, 4096, 8192

# Table 5 of the paper + the constants the paper leaves open (readings 4, 6, 12)
DEFAULTS = dict(S=8, G=8, C=16, beam=32, lambda_sp=0.1, lambda_idle=0.01, t_idle=120, alpha=0.05, beta=0.05,
                eta=0.05, sigma_eps=1e-4, cos_eps=1e-12, pq_eps=1e-6, flags=0, gamma=0.05, eps_k=0.20, eps_v=0.25,
                rope_theta=1.0e6, rope_anchor=0, pos0=0,
                t_warm=0, warm_reservoir=2048, km_iters=32, km_batch=256, km_seed=0, s_cap=32)

EXPORTED_SYMBOLS = [
    "protokv_workspace_bytes", "protokv_create", "protokv_destroy", "protokv_append_frame",
    "protokv_query_attention", "protokv_append_frame_host", "protokv_query_attention_host", "protokv_last_error",
    "protokv_query_attention_ex", "protokv_synthesize", "protokv_export_state", "protokv_import_state",
    "protokv_export_ring", "protokv_export_codes", "protokv_import_codes", "protokv_last_frame_trace",
    "protokv_frames_seen", "protokv_kernel_launches", "protokv_stage_impl", "protokv_profile_enable",
    "protokv_profile_read", "protokv_error_flags", "protokv_maintenance_counters", "protokv_query_attention_at",
    "protokv_query_attention_static", "protokv_static_scratch_bytes",
    "protokv_train_codebooks", "protokv_export_reservoir", "protokv_import_reservoir", "protokv_export_codebooks",
    "protokv_export_allocation",
]
STAGES = ["fill", "score", "update", "append", "synthesis", "attention"]


class ProtoKVError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"protokv error {code}: {msg}")
        self.code = code


class ProtoKVConfig(C.Structure):
    _fields_ = [("struct_size", C.c_uint32),
                ("n_streams", C.c_int32), ("n_layers", C.c_int32), ("n_q_heads", C.c_int32),
                ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("dtype", C.c_int32), ("tokens_per_frame", C.c_int32), ("near_frames", C.c_int32),
                ("k_max", C.c_int32), ("n_query_tokens", C.c_int32),
                ("S", C.c_int32), ("G", C.c_int32), ("C", C.c_int32), ("beam", C.c_int32),
                ("lambda_sp", C.c_float), ("lambda_idle", C.c_float), ("t_idle", C.c_int32),
                ("alpha", C.c_float), ("beta", C.c_float), ("eta", C.c_float),
                ("sigma_eps", C.c_float), ("cos_eps", C.c_float), ("pq_eps", C.c_double),
                ("flags", C.c_uint32), ("gamma", C.c_float), ("eps_k", C.c_float), ("eps_v", C.c_float),
                ("rope_theta", C.c_double), ("rope_anchor", C.c_int32), ("pos0", C.c_int64),
                ("t_warm", C.c_int32), ("warm_reservoir", C.c_int32), ("km_iters", C.c_int32), ("km_batch", C.c_int32),
                ("km_seed", C.c_uint64), ("s_cap", C.c_int32),
                ("codebook_k", C.c_void_p), ("codebook_v", C.c_void_p),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("cuda_stream", C.c_void_p)]


class _BankView(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("c", "p", "n", "mu", "sigma", "tau", "pos", "hist_k", "hist_v", "nres",
                                          "active", "pos_first", "pos_sum", "pos_cnt")]


_lib = None


def load_library():
    """dlopen lib/libprotokv.so (building it if needed) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    vp, i32 = C.c_void_p, C.c_int32
    lib.protokv_workspace_bytes.restype = C.c_size_t
    lib.protokv_workspace_bytes.argtypes = [C.POINTER(ProtoKVConfig)]
    lib.protokv_create.restype = vp
    lib.protokv_create.argtypes = [C.POINTER(ProtoKVConfig)]
    lib.protokv_destroy.restype = None
    lib.protokv_destroy.argtypes = [vp]
    lib.protokv_append_frame.argtypes = [vp, vp, vp, vp]
    lib.protokv_query_attention.argtypes = [vp, vp, vp]
    lib.protokv_append_frame_host.argtypes = [vp, vp, vp, vp]
    lib.protokv_query_attention_host.argtypes = [vp, vp, vp]
    lib.protokv_last_error.restype = C.c_char_p
    lib.protokv_query_attention_ex.argtypes = [vp, vp, i32, i32, i32, vp, vp, i32]
    lib.protokv_query_attention_at.argtypes = [vp, vp, i32, i32, i32, vp, vp, i32, C.c_int64]
    lib.protokv_query_attention_static.argtypes = [vp, vp, i32, i32, i32, vp, vp, i32]
    lib.protokv_static_scratch_bytes.argtypes = []
    lib.protokv_static_scratch_bytes.restype = C.c_size_t
    lib.protokv_synthesize.argtypes = [vp]
    lib.protokv_export_state.argtypes = [vp, i32, C.POINTER(_BankView)]
    lib.protokv_import_state.argtypes = [vp, i32, C.POINTER(_BankView)]
    lib.protokv_export_ring.argtypes = [vp, i32, vp, vp, vp, vp, C.POINTER(i32)]
    lib.protokv_export_codes.argtypes = [vp, i32, vp, vp, vp]
    lib.protokv_import_codes.argtypes = [vp, i32, vp, vp]
    lib.protokv_last_frame_trace.argtypes = [vp, vp, vp, vp, vp, C.POINTER(i32), C.POINTER(i32)]
    lib.protokv_frames_seen.restype = C.c_int64
    lib.protokv_frames_seen.argtypes = [vp]
    lib.protokv_kernel_launches.restype = C.c_int64
    lib.protokv_kernel_launches.argtypes = [vp]
    lib.protokv_profile_enable.argtypes = [vp, i32]
    lib.protokv_profile_read.argtypes = [vp, vp, vp]
    lib.protokv_error_flags.argtypes = [vp, C.POINTER(C.c_uint32), i32]
    lib.protokv_maintenance_counters.argtypes = [vp, vp]
    lib.protokv_train_codebooks.argtypes = [vp]
    lib.protokv_export_reservoir.argtypes = [vp, i32, vp, vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    lib.protokv_import_reservoir.argtypes = [vp, i32, vp, vp, C.c_int64]
    lib.protokv_export_codebooks.argtypes = [vp, i32, vp, vp]
    lib.protokv_export_allocation.argtypes = [vp, i32, vp, vp]
    lib.protokv_stage_impl.restype = C.c_char_p
    lib.protokv_stage_impl.argtypes = [vp, i32]
    _lib = lib
    return lib


def protokv_last_error() -> str:
    return load_library().protokv_last_error().decode()


def make_config(**kw) -> ProtoKVConfig:
    p = dict(DEFAULTS)
    p.update(kw)
    cfg = ProtoKVConfig()
    cfg.struct_size = C.sizeof(ProtoKVConfig)
    for k, v in p.items():
        setattr(cfg, k, v)
    return cfg


def protokv_workspace_bytes(cfg: ProtoKVConfig) -> int:
    return int(load_library().protokv_workspace_bytes(C.byref(cfg)))


def _np_ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class ProtoKV:
    """One state = n_streams * n_layers * n_kv_heads banks.  Tensors are torch CUDA tensors in the ABI layouts:
    K, V [n_streams][n_layers][T][n_kv_heads][d]; grid_pos [n_streams][T][2] fp32; Q, out
    [n_streams][n_layers][N_q][n_q_heads][d]; codebooks [n_streams][n_layers][n_kv_heads][G][C][d/G] fp32."""

    def __init__(self, *, n_streams, n_layers, n_q_heads, n_kv_heads, head_dim, dtype, tokens_per_frame,
                 near_frames, k_max, n_query_tokens, codebook_k=None, codebook_v=None, device="cuda:0",
                 stream=None, **hyper):
        import torch
        self._torch = torch
        self._lib = load_library()
        self._h = None
        self.device = torch.device(device)
        self.torch_dtype = torch.bfloat16 if dtype in (BF16, "bf16", torch.bfloat16) else torch.float32
        dt = BF16 if self.torch_dtype == torch.bfloat16 else F32
        cfg = make_config(n_streams=n_streams, n_layers=n_layers, n_q_heads=n_q_heads, n_kv_heads=n_kv_heads,
                          head_dim=head_dim, dtype=dt, tokens_per_frame=tokens_per_frame, near_frames=near_frames,
                          k_max=k_max, n_query_tokens=n_query_tokens, **hyper)
        self.cfg = cfg
        self.n_banks = n_streams * n_layers * n_kv_heads
        need = protokv_workspace_bytes(cfg)
        if need == 0:
            raise ProtoKVError(1, protokv_last_error())
        if not torch.cuda.is_available():
            raise ProtoKVError(2, "no CUDA device: the ProtoKV hot path has no CPU fallback")
        torch.cuda.set_device(self.device)
        self._ws = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
        base = (self._ws.data_ptr() + 255) // 256 * 256
        cfg.workspace = base
        cfg.workspace_bytes = need
        self._stream = stream
        cfg.cuda_stream = stream.cuda_stream if stream is not None else torch.cuda.current_stream(self.device).cuda_stream
        self._cb = None
        if codebook_k is not None:
            ck = codebook_k.to(self.device, torch.float32).contiguous()
            cv = codebook_v.to(self.device, torch.float32).contiguous()
            expect = self.n_banks * cfg.G * cfg.C * (head_dim // cfg.G)
            if ck.numel() != expect or cv.numel() != expect:
                raise ProtoKVError(1, "codebook shape mismatch")
            self._cb = (ck, cv)
            cfg.codebook_k, cfg.codebook_v = ck.data_ptr(), cv.data_ptr()
        self._h = self._lib.protokv_create(C.byref(cfg))
        if not self._h:
            raise ProtoKVError(-1, protokv_last_error())
        self.workspace_bytes = need

    # ---- lifetime -------------------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            self._lib.protokv_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    def _check(self, rc):
        if rc != 0:
            raise ProtoKVError(rc, protokv_last_error())

    def _dev(self, t, dtype, numel):
        if not t.is_cuda or t.dtype != dtype or not t.is_contiguous() or t.numel() != numel:
            raise ProtoKVError(1, f"expected a contiguous CUDA tensor of {numel} x {dtype}, got "
                                  f"{tuple(t.shape)} {t.dtype} on {t.device}")
        return t.data_ptr()

    # ---- shapes ---------------------------------------------------------------------------------------------
    @property
    def _frame_numel(self):
        c = self.cfg
        return c.n_streams * c.n_layers * c.tokens_per_frame * c.n_kv_heads * c.head_dim

    def _q_numel(self, n_q, layers):
        c = self.cfg
        return c.n_streams * layers * n_q * c.n_q_heads * c.head_dim

    # ---- the four calls of the hot path ---------------------------------------------------------------------
    def append_frame(self, K, V, grid_pos):
        """protokv_append_frame: Alg. 1 for one frame of every bank (device tensors)."""
        c = self.cfg
        self._check(self._lib.protokv_append_frame(
            self._h, self._dev(K, self.torch_dtype, self._frame_numel), self._dev(V, self.torch_dtype, self._frame_numel),
            self._dev(grid_pos, self._torch.float32, c.n_streams * c.tokens_per_frame * 2)))

    def query_attention(self, Q, out=None):
        """protokv_query_attention: synthesis + fused attention for N_q query tokens of every layer."""
        c = self.cfg
        n = self._q_numel(c.n_query_tokens, c.n_layers)
        if out is None:
            out = self._torch.empty_like(Q)
        self._check(self._lib.protokv_query_attention(self._h, self._dev(Q, self.torch_dtype, n),
                                                      self._dev(out, self.torch_dtype, n)))
        return out

    def append_frame_host(self, K, V, grid_pos):
        """protokv_append_frame_host: the same with host (pinned) tensors; copies run on the state's stream."""
        for t in (K, V, grid_pos):
            if t.is_cuda or not t.is_contiguous():
                raise ProtoKVError(1, "host variant needs contiguous CPU tensors")
        self._check(self._lib.protokv_append_frame_host(self._h, K.data_ptr(), V.data_ptr(), grid_pos.data_ptr()))

    def query_attention_host(self, Q, out):
        for t in (Q, out):
            if t.is_cuda or not t.is_contiguous():
                raise ProtoKVError(1, "host variant needs contiguous CPU tensors")
        self._check(self._lib.protokv_query_attention_host(self._h, Q.data_ptr(), out.data_ptr()))
        return out

    # ---- parity / debug surface -----------------------------------------------------------------------------
    def query_attention_ex(self, Q, n_q=None, layer_begin=0, layer_count=None, out=None, return_lse=False,
                           run_synthesis=True, q_pos0=None):
        c = self.cfg
        n_q = c.n_query_tokens if n_q is None else n_q
        layer_count = c.n_layers if layer_count is None else layer_count
        n = self._q_numel(n_q, layer_count)
        if out is None:
            out = self._torch.empty_like(Q)
        lse = None
        if return_lse:
            lse = self._torch.empty((c.n_streams, layer_count, n_q, c.n_q_heads), dtype=self._torch.float32,
                                    device=self.device)
        args = (self._h, self._dev(Q, self.torch_dtype, n), n_q, layer_begin, layer_count,
                self._dev(out, self.torch_dtype, n), lse.data_ptr() if lse is not None else None, int(run_synthesis))
        if q_pos0 is None:
            self._check(self._lib.protokv_query_attention_ex(*args))
        else:
            self._check(self._lib.protokv_query_attention_at(*args, int(q_pos0)))
        return (out, lse) if return_lse else out

    def query_attention_static(self, Q, out, n_q=None, layer_begin=0, layer_count=None, lse=None, run_synthesis=True):
        """protokv_query_attention_static: the partials live in the library's static device array; nothing is allocated
        (out, and lse if wanted, are the caller's)."""
        c = self.cfg
        n_q = c.n_query_tokens if n_q is None else n_q
        layer_count = c.n_layers if layer_count is None else layer_count
        n = self._q_numel(n_q, layer_count)
        self._check(self._lib.protokv_query_attention_static(
            self._h, self._dev(Q, self.torch_dtype, n), n_q, layer_begin, layer_count, self._dev(out, self.torch_dtype, n),
            lse.data_ptr() if lse is not None else None, int(run_synthesis)))
        return out

    @property
    def static_scratch_bytes(self):
        return int(self._lib.protokv_static_scratch_bytes())

    def synthesize(self):
        self._check(self._lib.protokv_synthesize(self._h))

    def _state_arrays(self):
        c = self.cfg
        k, d, G, Cc = c.k_max, c.head_dim, c.G, c.C
        return dict(c=np.zeros((k, d), np.float32), p=np.zeros((k, d), np.float32), n=np.zeros(k, np.int32),
                    mu=np.zeros((k, 2), np.float32), sigma=np.zeros((k, 3), np.float32), tau=np.zeros(k, np.int32),
                    pos=np.zeros(k, np.int64), hist_k=np.zeros((k, G, Cc), np.uint32),
                    hist_v=np.zeros((k, G, Cc), np.uint32), nres=np.zeros(k, np.uint32),
                    active=np.zeros(k, np.uint8), pos_first=np.zeros(k, np.int64), pos_sum=np.zeros(k, np.int64),
                    pos_cnt=np.zeros(k, np.int32))

    def export_state(self, bank):
        st = self._state_arrays()
        v = _BankView(*[_np_ptr(st[f]) for f, _ in _BankView._fields_])
        self._check(self._lib.protokv_export_state(self._h, bank, C.byref(v)))
        return st

    def import_state(self, bank, **fields):
        ref = self._state_arrays()
        keep = {f: np.ascontiguousarray(a, dtype=ref[f].dtype).reshape(ref[f].shape) for f, a in fields.items()}
        v = _BankView(*[_np_ptr(keep.get(f)) for f, _ in _BankView._fields_])
        self._check(self._lib.protokv_import_state(self._h, bank, C.byref(v)))

    def export_ring(self, bank):
        c = self.cfg
        K = np.zeros((c.near_frames, c.tokens_per_frame, c.head_dim), np.float32)
        V = np.zeros_like(K)
        s = np.zeros((c.near_frames, c.tokens_per_frame, 2), np.float32)
        idx = np.zeros(c.near_frames, np.int32)
        n = C.c_int32(0)
        self._check(self._lib.protokv_export_ring(self._h, bank, _np_ptr(K), _np_ptr(V), _np_ptr(s), _np_ptr(idx),
                                                  C.byref(n)))
        return K[:n.value], V[:n.value], s[:n.value], idx[:n.value]

    def train_codebooks(self):
        """protokv_train_codebooks: ends the warm-up now (PROTOKV_WARMUP_MANUAL states)."""
        self._check(self._lib.protokv_train_codebooks(self._h))

    def export_reservoir(self, bank):
        """(r^K [fill][d], r^V [fill][d], residuals offered so far) of one bank."""
        c = self.cfg
        rk = np.zeros((c.warm_reservoir, c.head_dim), np.float32)
        rv = np.zeros_like(rk)
        fill, seen = C.c_int64(0), C.c_int64(0)
        self._check(self._lib.protokv_export_reservoir(self._h, bank, _np_ptr(rk), _np_ptr(rv), C.byref(fill),
                                                       C.byref(seen)))
        return rk[:fill.value], rv[:fill.value], int(seen.value)

    def import_reservoir(self, bank, res_k, res_v):
        rk = np.ascontiguousarray(res_k, dtype=np.float32)
        rv = np.ascontiguousarray(res_v, dtype=np.float32)
        if rk.shape != rv.shape or rk.ndim != 2 or rk.shape[1] != self.cfg.head_dim:
            raise ProtoKVError(1, "reservoir rows must be [n][head_dim] for both sides")
        self._check(self._lib.protokv_import_reservoir(self._h, bank, _np_ptr(rk), _np_ptr(rv), rk.shape[0]))

    def export_codebooks(self, bank):
        c = self.cfg
        ck = np.zeros((c.G, c.C, c.head_dim // c.G), np.float32)
        cv = np.zeros_like(ck)
        self._check(self._lib.protokv_export_codebooks(self._h, bank, _np_ptr(ck), _np_ptr(cv)))
        return ck, cv

    def export_allocation(self, bank):
        """(S_k [k_max] int32, v_k [k_max] int64) of one bank as of the last synthesis (D.3)."""
        sk = np.zeros(self.cfg.k_max, np.int32)
        v = np.zeros(self.cfg.k_max, np.int64)
        self._check(self._lib.protokv_export_allocation(self._h, bank, _np_ptr(sk), _np_ptr(v)))
        return sk, v

    def export_codes(self, bank):
        c = self.cfg
        smax = c.s_cap if c.flags & VAR_ALLOC else c.S
        ck = np.zeros((c.k_max, smax, c.G), np.uint8)
        cv = np.zeros_like(ck)
        kind = np.zeros(c.k_max, np.uint8)
        self._check(self._lib.protokv_export_codes(self._h, bank, _np_ptr(ck), _np_ptr(cv), _np_ptr(kind)))
        return ck, cv, kind

    def import_codes(self, bank, codes_k, codes_v):
        ck = np.ascontiguousarray(codes_k, dtype=np.uint8)
        cv = np.ascontiguousarray(codes_v, dtype=np.uint8)
        self._check(self._lib.protokv_import_codes(self._h, bank, _np_ptr(ck), _np_ptr(cv)))

    def last_frame_trace(self):
        c = self.cfg
        B, T, G = self.n_banks, c.tokens_per_frame, c.G
        out = dict(assign=np.zeros((B, T), np.int32), best=np.zeros((B, T), np.float32),
                   codes_k=np.zeros((B, T, G), np.uint8), codes_v=np.zeros((B, T, G), np.uint8))
        nf, ev = C.c_int32(0), C.c_int32(0)
        self._check(self._lib.protokv_last_frame_trace(self._h, _np_ptr(out["assign"]), _np_ptr(out["best"]),
                                                       _np_ptr(out["codes_k"]), _np_ptr(out["codes_v"]),
                                                       C.byref(nf), C.byref(ev)))
        out["n_fill"], out["evicted_frame"] = nf.value, ev.value
        return out

    def profile_enable(self, on=True):
        self._check(self._lib.protokv_profile_enable(self._h, int(on)))

    def profile_read(self):
        """{stage: (summed device ms, bracketed launches)} since the last enable/read."""
        ms = np.zeros(len(STAGES), np.float64)
        n = np.zeros(len(STAGES), np.int64)
        self._check(self._lib.protokv_profile_read(self._h, _np_ptr(ms), _np_ptr(n)))
        return {s: (float(ms[i]), int(n[i])) for i, s in enumerate(STAGES)}

    @property
    def frames_seen(self):
        return int(self._lib.protokv_frames_seen(self._h))

    @property
    def kernel_launches(self):
        return int(self._lib.protokv_kernel_launches(self._h))

    def maintenance_counters(self):
        c = np.zeros(3, np.int64)
        self._check(self._lib.protokv_maintenance_counters(self._h, _np_ptr(c)))
        return dict(decayed=int(c[0]), merges=int(c[1]), recycled=int(c[2]))

    def error_flags(self, clear=False):
        f = C.c_uint32(0)
        self._check(self._lib.protokv_error_flags(self._h, C.byref(f), int(clear)))
        return int(f.value)

    def stage_impl(self, stage):
        return self._lib.protokv_stage_impl(self._h, stage).decode()
