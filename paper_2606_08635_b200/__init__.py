"""paper_2606_08635_b200 -- thin Python binding of libskv (include/skv.h), the B200-native SpectrumKV
per-token mixed-precision KV transfer path.

Argument marshalling only: every step of the path runs in the hand-written CUDA kernels behind the C
ABI.  PyTorch is used for device memory and streams.  There is no CPU fallback: if libskv.so is missing
the import of any entry point raises.

Entry points mirror the C ABI one to one (see include/skv.h for semantics and citations):
    skv_tier_counts, skv_blob_bytes, skv_workspace_bytes, skv_blob_check,
    skv_importance, skv_importance_kvnorm, skv_importance_kvnorm_noalloc, skv_assign_tiers, skv_pack, skv_unpack, skv_unpack_patch,
    skv_counts_from_populations, skv_strerror
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libskv.so")

SKV_OK = 0
SKV_ERR_INVALID_ARG = -1
SKV_ERR_UNSUPPORTED = -2
SKV_ERR_BUDGET_INFEASIBLE = -3
SKV_ERR_BUFFER_TOO_SMALL = -4
SKV_ERR_BAD_BLOB = -5
SKV_ERR_CUDA = -6
SKV_ERR_NOALLOC_LIMIT = -7
SKV_NOALLOC_SCRATCH_BYTES = 4352 * 1024


class SkvError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        super().__init__(f"{where}: {skv_strerror(status)} ({status})")


class skv_shape(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("n_tokens", C.c_int32), ("n_requests", C.c_int32),
                ("stride_request", C.c_int64), ("stride_layer", C.c_int64),
                ("stride_token", C.c_int64), ("stride_head", C.c_int64),
                ("dtype", C.c_int32), ("reserved", C.c_int32)]


class skv_policy(C.Structure):
    _fields_ = [("budget", C.c_double), ("n_sink", C.c_int32), ("n_ranges", C.c_int32),
                ("ranges", C.POINTER(C.c_int32)), ("allow_int4", C.c_int32), ("tier_mode", C.c_int32)]


class skv_counts(C.Structure):
    _fields_ = [("n16", C.c_int32), ("n8", C.c_int32), ("n4", C.c_int32), ("n0", C.c_int32),
                ("allow_int4", C.c_int32), ("tier_mode", C.c_int32),
                ("budget_q4", C.c_int64), ("spent_q4", C.c_int64)]

    def as_tuple(self):
        return (self.n16, self.n8, self.n4, self.n0)

    def __repr__(self):
        return (f"skv_counts(n16={self.n16}, n8={self.n8}, n4={self.n4}, n0={self.n0}, "
                f"allow_int4={self.allow_int4}, tier_mode={self.tier_mode}, budget_q4={self.budget_q4}, "
                f"spent_q4={self.spent_q4})")


EXPORTS = ("skv_tier_counts", "skv_blob_bytes", "skv_workspace_bytes", "skv_blob_check", "skv_importance",
           "skv_importance_kvnorm", "skv_assign_tiers", "skv_pack", "skv_unpack", "skv_unpack_patch",
           "skv_counts_from_populations", "skv_assign_tiers_counts", "skv_strerror", "skv_version",
           "skv_importance_kvnorm_noalloc")

_lib = None


def lib():
    """Loads libskv.so (built in-tree by paper_2606_08635_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2606_08635_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        P, V = C.POINTER, C.c_void_p
        L.skv_tier_counts.argtypes = [P(skv_shape), P(skv_policy), P(skv_counts)]
        L.skv_blob_bytes.argtypes = [P(skv_shape), P(skv_counts)]
        L.skv_blob_bytes.restype = C.c_size_t
        L.skv_workspace_bytes.argtypes = [P(skv_shape), C.c_int32]
        L.skv_workspace_bytes.restype = C.c_size_t
        L.skv_blob_check.argtypes = [V, C.c_size_t, P(skv_shape), P(skv_counts)]
        L.skv_importance.argtypes = [P(skv_shape), V, V, C.c_int32, C.c_int32, C.c_float, V, V, C.c_size_t, V]
        L.skv_importance_kvnorm.argtypes = [P(skv_shape), V, C.c_float, V, V, C.c_size_t, V]
        L.skv_importance_kvnorm_noalloc.argtypes = [P(skv_shape), V, C.c_float, V, V]
        L.skv_assign_tiers.argtypes = [P(skv_shape), P(skv_policy), V, V, P(skv_counts), V, C.c_size_t, V]
        L.skv_assign_tiers_counts.argtypes = [P(skv_shape), P(skv_counts), C.c_int32, C.c_int32, P(C.c_int32), V, V, V, C.c_size_t, V]
        L.skv_pack.argtypes = [P(skv_shape), V, V, V, P(skv_counts), V, C.c_size_t, V, C.c_size_t, V]
        L.skv_unpack.argtypes = [P(skv_shape), V, C.c_size_t, P(skv_counts), V, V, V, V, C.c_size_t, V]
        L.skv_unpack_patch.argtypes = L.skv_unpack.argtypes
        L.skv_counts_from_populations.argtypes = [P(skv_shape), C.c_int32, C.c_int32, C.c_int32, C.c_int32, P(skv_counts)]
        L.skv_strerror.argtypes = [C.c_int]
        L.skv_strerror.restype = C.c_char_p
        L.skv_version.restype = C.c_char_p
        _lib = L
    return _lib


# ------------------------------------------------------------------------------------------------
# marshalling helpers
# ------------------------------------------------------------------------------------------------
SKV_F16, SKV_BF16 = 0, 1


def make_shape(n_layers, n_q_heads, n_kv_heads, head_dim, n_tokens, n_requests=1, layout="token_major",
               strides=None, dtype="f16"):
    """skv_shape for a contiguous cache.  layout: "token_major" [R][L][n][Hkv][d] or "hf" [R][L][Hkv][n][d];
    or pass strides=(request, layer, token, head) in elements."""
    s = skv_shape(n_layers, n_q_heads, n_kv_heads, head_dim, n_tokens, n_requests)
    s.dtype = SKV_BF16 if dtype in ("bf16", SKV_BF16) and dtype is not False else SKV_F16
    if strides is not None:
        s.stride_request, s.stride_layer, s.stride_token, s.stride_head = [int(x) for x in strides]
    elif layout == "token_major":
        s.stride_head = head_dim
        s.stride_token = n_kv_heads * head_dim
        s.stride_layer = n_tokens * n_kv_heads * head_dim
        s.stride_request = n_layers * s.stride_layer
    elif layout == "hf":
        s.stride_token = head_dim
        s.stride_head = n_tokens * head_dim
        s.stride_layer = n_kv_heads * n_tokens * head_dim
        s.stride_request = n_layers * s.stride_layer
    else:
        raise ValueError(layout)
    return s


def _low_mode(allow_int4):
    """False/0 = 2-tier, True/1 = symmetric INT4 low tier, 2 = asymmetric 2-bit low tier (NEXT-4)."""
    return 2 if (allow_int4 == 2 and allow_int4 is not True) else (1 if allow_int4 else 0)


SKV_MODE_HOT_INT8, SKV_MODE_GROUP2 = 1, 2      # skv_policy.tier_mode / skv_counts.tier_mode bit flags (NEXT-4)


def make_policy(budget, n_sink=0, ranges=(), allow_int4=True, tier_mode=0):
    flat = [int(v) for r in ranges for v in r]
    arr = (C.c_int32 * max(1, len(flat)))(*flat)
    p = skv_policy(float(budget), int(n_sink), len(flat) // 2, C.cast(arr, C.POINTER(C.c_int32)), _low_mode(allow_int4),
                   int(tier_mode))
    p._keepalive = arr
    return p


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, int):
        return C.c_void_p(t) if t else None
    return C.c_void_p(t.data_ptr())


def _nbytes(t):
    if t is None or isinstance(t, int):
        return 0
    return t.numel() * t.element_size()


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return C.c_void_p(stream)
    return C.c_void_p(stream.cuda_stream)


def _check(rc, where):
    if rc != SKV_OK:
        raise SkvError(rc, where)


# ------------------------------------------------------------------------------------------------
# entry points (same names as the C ABI)
# ------------------------------------------------------------------------------------------------
def skv_strerror(status):
    return lib().skv_strerror(int(status)).decode()


def skv_version():
    return lib().skv_version().decode()


def skv_tier_counts(shape, policy):
    c = skv_counts()
    _check(lib().skv_tier_counts(C.byref(shape), C.byref(policy), C.byref(c)), "skv_tier_counts")
    return c


def skv_blob_bytes(shape, counts):
    return int(lib().skv_blob_bytes(C.byref(shape), C.byref(counts)))


def skv_workspace_bytes(shape, window=0):
    return int(lib().skv_workspace_bytes(C.byref(shape), int(window)))


def skv_blob_check(header_host, blob_bytes):
    """header_host: a HOST uint8 tensor / bytes-like holding at least the first 256 bytes of a blob."""
    if hasattr(header_host, "data_ptr"):
        assert not header_host.is_cuda and header_host.numel() * header_host.element_size() >= 256
        ptr = C.c_void_p(header_host.data_ptr())
    else:
        buf = (C.c_uint8 * 256).from_buffer_copy(bytes(header_host)[:256].ljust(256, b"\0"))
        ptr = C.cast(buf, C.c_void_p)
    s, c = skv_shape(), skv_counts()
    _check(lib().skv_blob_check(ptr, int(blob_bytes), C.byref(s), C.byref(c)), "skv_blob_check")
    return s, c


def skv_importance(shape, K, Q, window, importance, workspace, causal=True, lam=0.0, stream=None):
    _check(lib().skv_importance(C.byref(shape), _ptr(K), _ptr(Q), int(window), 1 if causal else 0, float(lam),
                                _ptr(importance), _ptr(workspace), _nbytes(workspace), _stream(stream)),
           "skv_importance")


def skv_importance_kvnorm(shape, K, importance, workspace, lam=0.0, stream=None):
    _check(lib().skv_importance_kvnorm(C.byref(shape), _ptr(K), float(lam), _ptr(importance), _ptr(workspace),
                                       _nbytes(workspace), _stream(stream)), "skv_importance_kvnorm")


def skv_importance_kvnorm_noalloc(shape, K, importance, lam=0.0, stream=None):
    """skv_importance_kvnorm without a workspace: for callers that cannot allocate device memory (code inside an engine
    whose pool owns the GPU's memory and that receives only the call's tensors).  The scratch is a fixed 4.25 MiB array
    inside libskv.so, shared by every call on the GPU: raises SkvError(SKV_ERR_NOALLOC_LIMIT) beyond
    R * L * n ~ 1 Mi scores, and calls that overlap on the GPU (different streams, no event between them) corrupt each
    other.  The first call on each GPU looks the array up; make it at start-up.  See include/skv.h."""
    _check(lib().skv_importance_kvnorm_noalloc(C.byref(shape), _ptr(K), float(lam), _ptr(importance), _stream(stream)),
           "skv_importance_kvnorm_noalloc")


def skv_assign_tiers(shape, policy, importance, tier_map, workspace, stream=None):
    c = skv_counts()
    _check(lib().skv_assign_tiers(C.byref(shape), C.byref(policy), _ptr(importance), _ptr(tier_map), C.byref(c),
                                  _ptr(workspace), _nbytes(workspace), _stream(stream)), "skv_assign_tiers")
    return c


def skv_pack(shape, K, V, tier_map, counts, blob, workspace, stream=None):
    _check(lib().skv_pack(C.byref(shape), _ptr(K), _ptr(V), _ptr(tier_map), C.byref(counts), _ptr(blob), _nbytes(blob),
                          _ptr(workspace), _nbytes(workspace), _stream(stream)), "skv_pack")


def skv_unpack(shape, blob, blob_bytes, counts, K_out, V_out, tier_map_out, workspace, stream=None):
    _check(lib().skv_unpack(C.byref(shape), _ptr(blob), int(blob_bytes), C.byref(counts), _ptr(K_out), _ptr(V_out),
                            _ptr(tier_map_out), _ptr(workspace), _nbytes(workspace), _stream(stream)), "skv_unpack")


def skv_unpack_patch(shape, blob, blob_bytes, counts, K_inout, V_inout, tier_map_inout, workspace, stream=None):
    _check(lib().skv_unpack_patch(C.byref(shape), _ptr(blob), int(blob_bytes), C.byref(counts), _ptr(K_inout),
                                  _ptr(V_inout), _ptr(tier_map_inout), _ptr(workspace), _nbytes(workspace),
                                  _stream(stream)), "skv_unpack_patch")


def skv_counts_from_populations(shape, n16, n8=0, n4=0, allow_int4=True):
    c = skv_counts()
    _check(lib().skv_counts_from_populations(C.byref(shape), int(n16), int(n8), int(n4), _low_mode(allow_int4),
                                             C.byref(c)), "skv_counts_from_populations")
    return c


def skv_assign_tiers_counts(shape, counts, importance, tier_map, workspace, n_sink=0, ranges=(), stream=None):
    flat = [int(v) for r in ranges for v in r]
    arr = (C.c_int32 * max(1, len(flat)))(*flat)
    _check(lib().skv_assign_tiers_counts(C.byref(shape), C.byref(counts), int(n_sink), len(flat) // 2,
                                         C.cast(arr, C.POINTER(C.c_int32)), _ptr(importance), _ptr(tier_map),
                                         _ptr(workspace), _nbytes(workspace), _stream(stream)), "skv_assign_tiers_counts")
