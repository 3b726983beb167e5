"""ctypes front end of the CPU oracle (oracle/skv_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module.

All arrays are numpy, one request at a time, contiguous, in the oracle's canonical layouts:
  K, V : float16 [L][n][Hkv][d]      Q : float16 [L][Hq][w][d]
  I    : float32 [L][n]              tier : uint8 [L][n]  (16 / 8 / 4 / 0)
"""
import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_half_to_float.restype = C.c_float
        _lib.orc_half_to_float.argtypes = [C.c_uint16]
        _lib.orc_float_to_half.restype = C.c_uint16
        _lib.orc_float_to_half.argtypes = [C.c_float]
        _lib.orc_float_to_bf16.restype = C.c_uint16
        _lib.orc_float_to_bf16.argtypes = [C.c_float]
        _lib.orc_blob_bytes.restype = C.c_uint64
        _lib.orc_blob_bytes_low.restype = C.c_uint64
        _lib.orc_blob_bytes_mode.restype = C.c_uint64
        _lib.orc_max_threads.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _c(a, dtype):
    a = np.ascontiguousarray(a)
    assert a.dtype == dtype, (a.dtype, dtype)
    return a


@dataclass(frozen=True)
class Counts:
    n16: int
    n8: int
    n4: int
    n0: int
    budget_q4: int            # quarter-units; EIGHTH-units when low_bits == 2
    spent_q4: int
    low_bits: int = 4         # 4 = symmetric INT4 low tier (tier code 4); 2 = asymmetric 2-bit (tier code 2, NEXT-4)
    mode: int = 0             # NEXT-4 bit flags: 1 = INT8 hot tier (P21), 2 = 2-bit tier in groups of 32 elements (P22)

    def arr(self):
        return (C.c_int64 * 6)(self.n16, self.n8, self.n4, self.n0, self.budget_q4, self.spent_q4)


def half_to_float(bits: int) -> float:
    return float(lib().orc_half_to_float(int(bits)))


def float_to_half(x: float) -> int:
    return int(lib().orc_float_to_half(C.c_float(x)))


def max_threads() -> int:
    return int(lib().orc_max_threads())


def set_threads(t: int) -> None:
    lib().orc_set_threads(C.c_int(int(t)))


def _mode(allow_int4):
    """allow_int4: False/0 = 2-tier, True/1 = symmetric INT4 low tier, 2 = asymmetric 2-bit low tier (NEXT-4)."""
    return 2 if (allow_int4 == 2 and allow_int4 is not True) else (1 if allow_int4 else 0)


MODE_HOT_INT8 = 1      # P21: the hot tier ships INT8 (nothing at FP16; protected positions pinned to INT8)
MODE_GROUP2 = 2        # P22: the 2-bit low tier is quantised in groups of 32 elements


def tier_counts(n, b, n_sink=0, ranges=(), allow_int4=True, mode=0):
    """O2.  Returns (Counts, protected bitmap uint8[n]).  Raises ValueError on infeasible/invalid."""
    rng = np.asarray(ranges, dtype=np.int32).reshape(-1, 2)
    out = (C.c_int64 * 6)()
    prot = np.zeros(int(n), dtype=np.uint8)
    rc = lib().orc_tier_counts_mode(C.c_int64(int(n)), C.c_double(float(b)), C.c_int32(int(n_sink)),
                                    C.c_int32(len(rng)), _p(np.ascontiguousarray(rng)),
                                    C.c_int32(_mode(allow_int4)), C.c_int32(int(mode)), out, _p(prot))
    if rc != 0:
        raise ValueError(f"orc_tier_counts rc={rc}")
    return Counts(*[int(v) for v in out], low_bits=2 if _mode(allow_int4) == 2 else 4, mode=int(mode)), prot


def _elems(x, bf16):
    """fp16 caches travel as numpy float16; bfloat16 caches (numpy has no such type) as uint16 bit patterns."""
    return _c(x, np.uint16 if bf16 else np.float16)


def importance(K, Q, causal=True, lam=0.0, bf16=False):
    """O1.  K [L][n][Hkv][d] f16, Q [L][Hq][w][d] f16 -> I [L][n] f32."""
    K = _elems(K, bf16)
    Q = _elems(Q, bf16)
    L, n, Hkv, d = K.shape
    L2, Hq, w, d2 = Q.shape
    assert L == L2 and d == d2 and Hq % Hkv == 0 and 1 <= w <= n
    I = np.empty((L, n), dtype=np.float32)
    lib().orc_importance_dt(C.c_int32(L), C.c_int32(Hq), C.c_int32(Hkv), C.c_int32(d), C.c_int64(n),
                            C.c_int32(w), C.c_int32(1 if causal else 0), C.c_double(float(lam)),
                            _p(K), _p(Q), _p(I), C.c_int32(1 if bf16 else 0))
    return I


def importance_kvnorm(K, lam=0.0, bf16=False):
    K = _elems(K, bf16)
    L, n, Hkv, d = K.shape
    I = np.empty((L, n), dtype=np.float32)
    lib().orc_importance_kvnorm_dt(C.c_int32(L), C.c_int32(Hkv), C.c_int32(d), C.c_int64(n),
                                   C.c_double(float(lam)), _p(K), _p(I), C.c_int32(1 if bf16 else 0))
    return I


def assign(I, prot, counts: Counts):
    """O3.  I [L][n] f32, prot uint8[n] -> tier uint8 [L][n]."""
    I = _c(I, np.float32)
    prot = _c(prot, np.uint8)
    L, n = I.shape
    tier = np.empty((L, n), dtype=np.uint8)
    c4 = (C.c_int64 * 4)(counts.n16, counts.n8, counts.n4, counts.n0)
    lib().orc_assign_mode(C.c_int32(L), C.c_int64(n), _p(I), _p(prot), c4, C.c_int32(counts.low_bits),
                          C.c_int32(counts.mode), _p(tier))
    return tier


def blob_bytes(L, Hkv, d, n, counts: Counts) -> int:
    c4 = (C.c_int64 * 4)(counts.n16, counts.n8, counts.n4, counts.n0)
    return int(lib().orc_blob_bytes_mode(C.c_int32(L), C.c_int32(Hkv), C.c_int32(d), C.c_int64(n), c4,
                                         C.c_int32(counts.low_bits), C.c_int32(counts.mode)))


def pack(K, V, tier, counts: Counts, allow_int4=True, bf16=False):
    """O4+O5.  Returns the SKV1 blob as uint8[total_bytes]."""
    K = _elems(K, bf16)
    V = _elems(V, bf16)
    tier = _c(tier, np.uint8)
    L, n, Hkv, d = K.shape
    assert V.shape == K.shape and tier.shape == (L, n)
    blob = np.empty(blob_bytes(L, Hkv, d, n, counts), dtype=np.uint8)
    rc = lib().orc_pack_mode(C.c_int32(L), C.c_int32(Hkv), C.c_int32(d), C.c_int64(n), _p(K), _p(V),
                             _p(tier), counts.arr(), C.c_int32(2 if counts.low_bits == 2 else _mode(allow_int4)),
                             C.c_int32(counts.mode), _p(blob), C.c_int32(1 if bf16 else 0))
    if rc != 0:
        raise ValueError(f"orc_pack rc={rc} (tier map does not match counts)")
    return blob


def unpack(blob, L, Hkv, d, n, bf16=False):
    """O6.  Returns (K, V, tier) dense (K, V as uint16 bit patterns when the blob holds bfloat16 elements)."""
    blob = _c(blob, np.uint8)
    assert bool(blob[40] & 4) == bool(bf16), "element type of the blob (header flags bit2) differs from the request"
    et = np.uint16 if bf16 else np.float16
    K = np.empty((L, n, Hkv, d), dtype=et)
    V = np.empty((L, n, Hkv, d), dtype=et)
    tier = np.empty((L, n), dtype=np.uint8)
    rc = lib().orc_unpack(_p(blob), C.c_uint64(blob.size), C.c_int32(L), C.c_int32(Hkv), C.c_int32(d),
                          C.c_int64(n), _p(K), _p(V), _p(tier))
    if rc != 0:
        raise ValueError(f"orc_unpack rc={rc} (bad blob)")
    return K, V, tier


def unpack_patch(blob, K, V, tier):
    """NEXT-3 cold-tier upgrade: applies an upgrade blob to COPIES of the dense cache K, V [L][n][Hkv][d] and of the
    tier map [L][n]; returns (K, V, tier)."""
    blob = _c(blob, np.uint8)
    et = np.uint16 if (blob[40] & 4) else np.float16
    K = np.array(K, dtype=et, order="C", copy=True)
    V = np.array(V, dtype=et, order="C", copy=True)
    tier = np.array(tier, dtype=np.uint8, order="C", copy=True)
    L, n, Hkv, d = K.shape
    rc = lib().orc_unpack_patch(_p(blob), C.c_uint64(blob.size), C.c_int32(L), C.c_int32(Hkv), C.c_int32(d),
                                C.c_int64(n), _p(K), _p(V), _p(tier))
    if rc != 0:
        raise ValueError(f"orc_unpack_patch rc={rc} (bad blob)")
    return K, V, tier


def quantize2_vector(x, bf16=False):
    """NEXT-4 asymmetric 2-bit quantizer on one vector.  x float16[d] -> (lo_bits, hi_bits, uint8[d] codes 0..3)."""
    x = _elems(x, bf16)
    q = np.empty(x.size, dtype=np.uint8)
    lo, hi = C.c_uint16(0), C.c_uint16(0)
    lib().orc_quantize2_vector_dt(_p(x), C.c_int32(x.size), C.byref(lo), C.byref(hi), _p(q), C.c_int32(1 if bf16 else 0))
    return int(lo.value), int(hi.value), q


def dequantize2_vector(q, lo_bits, hi_bits, bf16=False):
    q = _c(q, np.uint8)
    y = np.empty(q.size, dtype=np.uint16 if bf16 else np.float16)
    lib().orc_dequantize2_vector_dt(_p(q), C.c_int32(q.size), C.c_uint16(int(lo_bits)), C.c_uint16(int(hi_bits)), _p(y),
                                    C.c_int32(1 if bf16 else 0))
    return y


def bf16_to_float(bits):
    """uint16 bit patterns -> float32 (exact)."""
    return (np.asarray(bits, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)


def float_to_bf16(x):
    """float32 array -> bfloat16 bit patterns, round to nearest even (through the oracle's scalar routine)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    f = lib().orc_float_to_bf16
    return np.array([f(C.c_float(float(v))) for v in x.ravel()], dtype=np.uint16).reshape(x.shape)


def quantize_vector(x, qmax, bf16=False):
    """O4 on one vector.  x float16[d] (or bfloat16 bits uint16[d]) -> (amax_bits, int8[d])."""
    x = _elems(x, bf16)
    q = np.empty(x.size, dtype=np.int8)
    ab = C.c_uint16(0)
    lib().orc_quantize_vector_dt(_p(x), C.c_int32(x.size), C.c_int32(int(qmax)), C.byref(ab), _p(q),
                                 C.c_int32(1 if bf16 else 0))
    return int(ab.value), q


def dequantize_vector(q, qmax, amax_bits, bf16=False):
    q = _c(q, np.int8)
    y = np.empty(q.size, dtype=np.uint16 if bf16 else np.float16)
    lib().orc_dequantize_vector_dt(_p(q), C.c_int32(q.size), C.c_int32(int(qmax)), C.c_uint16(int(amax_bits)), _p(y),
                                   C.c_int32(1 if bf16 else 0))
    return y
