"""Counter-based, stateless, seeded workload generator (inputs only).

Every value is a pure function of (seed, tag, indices): integer hashing (splitmix64)
plus an Irwin-Hall normal built from twelve 16-bit fields, then IEEE fp64 mul/add and
one rounding.  No transcendental functions, so the CPU and a CUDA device produce the
same bits (the `device` argument only chooses where the tensors live).

The streams stand in for a VLM's per-layer visual-token K/V (BASELINE.json configs):
a Gaussian cluster mixture whose cluster choice is correlated with the grid position,
optional slow drift of the centres, an optional rare "event" cluster.  The recipe is
restated in DESIGN.md.  Nothing here knows about prototypes, assignment or attention.
"""
from __future__ import annotations

import dataclasses
import functools
from typing import Optional, Tuple

import torch

_MASK = (1 << 64) - 1


def _i64(x: int) -> int:
    """Python int -> the signed value with the same low 64 bits."""
    x &= _MASK
    return x - (1 << 64) if x >= (1 << 63) else x


_GOLDEN = _i64(0x9E3779B97F4A7C15)
_MUL1 = _i64(0xBF58476D1CE4E5B9)
_MUL2 = _i64(0x94D049BB133111EB)

# tags (arbitrary distinct constants)
TAG_CENTRE_K, TAG_CENTRE_V, TAG_NOISE_K, TAG_NOISE_V = 0x11, 0x12, 0x13, 0x14
TAG_HOME, TAG_PICK, TAG_OTHER, TAG_Q, TAG_CB_K, TAG_CB_V = 0x21, 0x22, 0x23, 0x31, 0x41, 0x42

SIGMA_W = 0.1          # within-cluster std (BASELINE.json config 1)
HOME_PROB = 0.75       # probability that a token takes its block's home cluster
HOME_EPOCH = 32        # frames between re-draws of a block's home cluster
DRIFT_PERIOD = 100     # frames between independent key-frame centres


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    """Logical shift right on int64 tensors."""
    return (x >> k) & ((1 << (64 - k)) - 1)


def splitmix64(x: torch.Tensor) -> torch.Tensor:
    """The splitmix64 output function on int64 tensors (bit pattern = uint64 result)."""
    z = x + _GOLDEN
    z = (z ^ _lsr(z, 30)) * _MUL1
    z = (z ^ _lsr(z, 27)) * _MUL2
    return z ^ _lsr(z, 31)


def _key(seed: int, tag: int, *idx, device="cpu") -> torch.Tensor:
    """Fold indices (ints or broadcastable int64 tensors) into a 64-bit key."""
    h = splitmix64(torch.tensor(_i64(seed * 0x100 + tag), dtype=torch.int64, device=device))
    for i in idx:
        if not torch.is_tensor(i):
            i = torch.tensor(int(i), dtype=torch.int64, device=device)
        h = splitmix64(h ^ i)
    return h


def _fold(h: torch.Tensor, i) -> torch.Tensor:
    if not torch.is_tensor(i):
        i = torch.tensor(int(i), dtype=torch.int64, device=h.device)
    return splitmix64(h ^ i)


def standard_normal(h: torch.Tensor) -> torch.Tensor:
    """Irwin-Hall(12) normal from key h: fp32, exact (integer sum times 2^-17)."""
    total = torch.zeros_like(h)
    for m in (1, 2, 3):
        w = splitmix64(h ^ m)
        total = total + (w & 0xFFFF) + (_lsr(w, 16) & 0xFFFF) + (_lsr(w, 32) & 0xFFFF) + _lsr(w, 48)
    return (2 * total - 786420).to(torch.float32) / 131072.0


def _arange(n: int, device) -> torch.Tensor:
    return torch.arange(n, dtype=torch.int64, device=device)


@dataclasses.dataclass(frozen=True)
class WorkloadSpec:
    name: str
    n_streams: int
    n_layers: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    dtype: str                 # "f32" | "bf16"
    grid_h: int
    grid_w: int
    near_frames: int
    k_max: int
    n_frames: int
    n_clusters: int
    n_query_tokens: int
    seed: int
    drift: bool = False
    event: Optional[Tuple[int, int, int, int, int, int]] = None   # f0,f1(excl),r0,r1(excl),c0,c1(excl)
    query_every: int = 0       # 0: one query after the last frame
    G: int = 8
    C: int = 16
    stream0: int = 0           # global index of this spec's first stream (a rank's shard of a multi-stream workload)

    @property
    def T(self) -> int:
        return self.grid_h * self.grid_w

    @property
    def n_banks(self) -> int:
        return self.n_streams * self.n_layers * self.n_kv_heads

    @property
    def torch_dtype(self):
        return torch.float32 if self.dtype == "f32" else torch.bfloat16


def _c4(k_max: int, near: int) -> WorkloadSpec:
    return WorkloadSpec(f"c4_k{k_max}_w{near}", 1, 1, 28, 4, 128, "bf16", 14, 14, near, k_max, 1200, 64, 32,
                        seed=4, drift=True)


CONFIGS = {
    # BASELINE.json configs[0..4]; seeds: 0 is given for config 1, 2..5 are this repo's choice.
    "c1": WorkloadSpec("c1", 1, 1, 1, 1, 64, "f32", 4, 4, 4, 32, 64, 8, 8, seed=0),
    "c2": WorkloadSpec("c2", 1, 1, 28, 4, 128, "bf16", 14, 14, 16, 1024, 600, 64, 32, seed=2, drift=True),
    "c3": WorkloadSpec("c3", 1, 28, 28, 4, 128, "bf16", 14, 14, 16, 1024, 3600, 64, 32, seed=3, drift=True,
                       event=(300, 305, 5, 9, 5, 9)),
    "c5": WorkloadSpec("c5", 8, 1, 32, 8, 128, "bf16", 24, 24, 8, 2048, 2000, 128, 64, seed=5, query_every=200),
}
for _k in (256, 1024, 4096):
    for _w in (4, 16, 64):
        CONFIGS[f"c4_k{_k}_w{_w}"] = _c4(_k, _w)


def spec_for(name: str, **overrides) -> WorkloadSpec:
    return dataclasses.replace(CONFIGS[name], **overrides)


def grid_positions(spec: WorkloadSpec, device="cpu") -> torch.Tensor:
    """[n_streams][T][2] fp32 normalised (x, y) cell centres; identical for every frame."""
    j = _arange(spec.T, device)
    col = (j % spec.grid_w).to(torch.float64)
    row = (j // spec.grid_w).to(torch.float64)
    xy = torch.stack([(col + 0.5) / spec.grid_w, (row + 0.5) / spec.grid_h], dim=-1).to(torch.float32)
    return xy.unsqueeze(0).expand(spec.n_streams, -1, -1).contiguous()


def cluster_ids(spec: WorkloadSpec, frame: int, device="cpu") -> torch.Tensor:
    """[n_streams][T] int64 mixture component of each token (shared by all layers/heads)."""
    st = _arange(spec.n_streams, device)[:, None] + spec.stream0
    j = _arange(spec.T, device)[None, :]
    row, col = j // spec.grid_w, j % spec.grid_w
    block = (row // 2) * ((spec.grid_w + 1) // 2) + (col // 2)
    home = _lsr(_key(spec.seed, TAG_HOME, st, block, frame // HOME_EPOCH, device=device), 33) % spec.n_clusters
    u = _lsr(_key(spec.seed, TAG_PICK, st, frame, j, device=device), 11)          # 53 bits
    other = _lsr(_key(spec.seed, TAG_OTHER, st, frame, j, device=device), 33) % spec.n_clusters
    cl = torch.where(u < int(HOME_PROB * (1 << 53)), home, other)
    if spec.event is not None:
        f0, f1, r0, r1, c0, c1 = spec.event
        if f0 <= frame < f1:
            inside = (row >= r0) & (row < r1) & (col >= c0) & (col < c1)
            cl = torch.where(inside.expand_as(cl), torch.full_like(cl, spec.n_clusters), cl)
    return cl


@functools.lru_cache(maxsize=16)
def _centre_table(spec: WorkloadSpec, tag: int, epoch: int, device: str) -> torch.Tensor:
    """[n_layers][n_kv_heads][n_clusters+1][d] fp32 N(0,1) key-frame centres of one drift epoch."""
    la = _arange(spec.n_layers, device)[:, None, None, None]
    hd = _arange(spec.n_kv_heads, device)[None, :, None, None]
    cl = _arange(spec.n_clusters + 1, device)[None, None, :, None]
    dm = _arange(spec.head_dim, device)[None, None, None, :]
    return standard_normal(_key(spec.seed, tag, epoch, la, hd, cl, dm, device=device))


def _centres(spec: WorkloadSpec, tag: int, frame: int, device: str) -> torch.Tensor:
    if not spec.drift:
        return _centre_table(spec, tag, 0, device)
    e, r = divmod(frame, DRIFT_PERIOD)
    a0 = _centre_table(spec, tag, e, device).to(torch.float64)
    a1 = _centre_table(spec, tag, e + 1, device).to(torch.float64)
    return (a0 + (r / DRIFT_PERIOD) * (a1 - a0)).to(torch.float32)


def frame_kv(spec: WorkloadSpec, frame: int, device="cpu"):
    """K, V of one frame in the C-ABI layout [n_streams][n_layers][T][n_kv_heads][d], spec dtype."""
    dev = str(device)
    cl = cluster_ids(spec, frame, dev)                                   # [S][T]
    out = []
    st = _arange(spec.n_streams, dev)[:, None, None, None, None] + spec.stream0
    la = _arange(spec.n_layers, dev)[None, :, None, None, None]
    j = _arange(spec.T, dev)[None, None, :, None, None]
    hd = _arange(spec.n_kv_heads, dev)[None, None, None, :, None]
    dm = _arange(spec.head_dim, dev)[None, None, None, None, :]
    for tag_c, tag_n in ((TAG_CENTRE_K, TAG_NOISE_K), (TAG_CENTRE_V, TAG_NOISE_V)):
        table = _centres(spec, tag_c, frame, dev)                        # [L][H][n_cl+1][d]
        # gather -> [S][L][T][H][d]
        cen = table[:, :, cl, :].permute(2, 0, 3, 1, 4)
        z = standard_normal(_key(spec.seed, tag_n, frame, st, la, j, hd, dm, device=dev))
        x = (cen.to(torch.float64) + float(torch.tensor(SIGMA_W, dtype=torch.float32)) * z.to(torch.float64))
        out.append(x.to(torch.float32).to(spec.torch_dtype).contiguous())
    return out[0], out[1]


def codebooks(spec: WorkloadSpec, device="cpu"):
    """PQ codebooks (an input of the method, reading 11):
    two fp32 tensors [n_streams][n_layers][n_kv_heads][G][C][d/G], entries sigma_w * N(0,1)."""
    dev = str(device)
    sub = spec.head_dim // spec.G
    shape_idx = [_arange(n, dev) for n in (spec.n_streams, spec.n_layers, spec.n_kv_heads, spec.G, spec.C, sub)]
    idx = [a.reshape([-1 if i == k else 1 for i in range(6)]) for k, a in enumerate(shape_idx)]
    idx[0] = idx[0] + spec.stream0
    res = []
    for tag in (TAG_CB_K, TAG_CB_V):
        z = standard_normal(_key(spec.seed, tag, *idx, device=dev))
        res.append((float(torch.tensor(SIGMA_W, dtype=torch.float32)) * z.to(torch.float64)).to(torch.float32).contiguous())
    return res[0], res[1]


def queries(spec: WorkloadSpec, query_index: int = 0, n_q: Optional[int] = None, device="cpu") -> torch.Tensor:
    """Q ~ N(0,1): [n_streams][n_layers][N_q][n_q_heads][d], spec dtype."""
    dev = str(device)
    n_q = spec.n_query_tokens if n_q is None else n_q
    dims = (spec.n_streams, spec.n_layers, n_q, spec.n_q_heads, spec.head_dim)
    idx = [_arange(n, dev).reshape([-1 if i == k else 1 for i in range(5)]) for k, n in enumerate(dims)]
    idx[0] = idx[0] + spec.stream0
    z = standard_normal(_key(spec.seed, TAG_Q, query_index, *idx, device=dev))
    return z.to(spec.torch_dtype).contiguous()
