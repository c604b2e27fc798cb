"""B200-native (sm_100a) ProtoKV two-tier KV memory hot path -- Python binding of the C ABI (include/protokv.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of csrc/.  There is no CPU fallback;
creating a state without an sm_100 device raises ProtoKVError.
"""
from .binding import (  # noqa: F401
    ProtoKV, ProtoKVConfig, ProtoKVError, load_library, DEFAULTS,
    F32, BF16, MAH_SQUARED, NO_MASS_BIAS, NO_RESIDUAL, NEAR_ONLY, FAR_ONLY, FORCE_SIMT, MAINTENANCE, DECODE_SPLITKV, ROPE,
    WARMUP, WARMUP_MANUAL, VAR_ALLOC, NO_DECODE_KERNEL, SERIAL_LAUNCH,
    protokv_workspace_bytes, protokv_last_error, EXPORTED_SYMBOLS,
)
from .build import build  # noqa: F401
