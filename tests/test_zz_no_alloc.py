"""skv_importance_kvnorm_noalloc: the KV-norm score for callers that cannot allocate device memory.

Some users of libskv run inside a serving engine that has handed all of the GPU's memory to its own pool and passes a
plug-in nothing but the tensors of the call: their cudaMalloc fails, and they have no workspace to give.  For them the
library carries one entry point whose scratch is a fixed 4.25 MiB array inside libskv.so (include/skv.h,
SKV_NOALLOC_SCRATCH_BYTES).  These tests check that it returns what skv_importance_kvnorm returns with a caller-owned
workspace -- twice in a row, the second call on a different shape, because every call reuses the same array and finds
the previous call's leftovers in it -- that device memory in use does not move across a call, and that a problem beyond
the built-in limit is refused with its own status instead of being run.

This file is named so that pytest collects it last: with `-x` a failure here cannot hide another test.
"""
import ctypes as C

import numpy as np
import pytest

import paper_2606_08635_b200 as skv


def test_noalloc_refuses_problems_beyond_the_built_in_scratch():
    # no GPU needed: the size check comes before the first CUDA call
    L = skv.lib()
    fits = skv.make_shape(32, 8, 8, 128, 32768, 1)               # one 32-layer, 32768-token request: exactly the limit
    assert 4 * 32 * 32768 + 8 * 32 * (32768 // 64) == skv.SKV_NOALLOC_SCRATCH_BYTES - 128 * 1024
    big = skv.make_shape(32, 8, 8, 128, 32768, 2)                # two of them: too much
    huge = skv.make_shape(65535, 8, 8, 128, 1 << 20, 65535)      # would overflow a careless 32-bit size computation
    for shape in (big, huge):
        rc = L.skv_importance_kvnorm_noalloc(C.byref(shape), C.c_void_p(256), 0.0, C.c_void_p(256), None)
        assert rc == skv.SKV_ERR_NOALLOC_LIMIT
    assert "scratch" in skv.skv_strerror(skv.SKV_ERR_NOALLOC_LIMIT)
    # a shape that fits gets past the size check and is then judged like skv_importance_kvnorm judges it
    rc = L.skv_importance_kvnorm_noalloc(C.byref(fits), None, 0.0, C.c_void_p(256), None)
    assert rc in (skv.SKV_ERR_INVALID_ARG, skv.SKV_ERR_CUDA)    # null K (SKV_ERR_CUDA: no device to look the array up on)
    bad = skv.make_shape(0, 8, 8, 128, 100, 1)
    assert L.skv_importance_kvnorm_noalloc(C.byref(bad), C.c_void_p(256), 0.0, C.c_void_p(256), None) == skv.SKV_ERR_INVALID_ARG
    assert L.skv_importance_kvnorm_noalloc(None, C.c_void_p(256), 0.0, C.c_void_p(256), None) == skv.SKV_ERR_INVALID_ARG


@pytest.mark.gpu
def test_noalloc_matches_the_workspace_path_on_two_calls_in_a_row():
    import torch

    import oracle
    from parity_util import to_layout

    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)           # the entry point looks its scratch up on the CURRENT device

    # (L, Hkv, d, n, R, layout, bf16, lambda): first a large problem that fills most of the array, then a small one
    # of another geometry and element type that lands on its leftovers
    calls = [(8, 2, 128, 16000, 4, "token_major", False, 0.005),
             (3, 2, 256, 777, 2, "hf", True, 0.0)]
    prepared = []
    for (L, Hkv, d, n, R, layout, bf16, lam) in calls:
        g = torch.Generator().manual_seed(97 * n + d)
        K = torch.randn((R, L, n, Hkv, d), generator=g) * (1.0 + 3.0 * torch.rand((R, L, n, 1, 1), generator=g))
        K[0, 0, 5] = 0.0
        K = K.to(torch.bfloat16 if bf16 else torch.float16)
        shape = skv.make_shape(L, Hkv, Hkv, d, n, R, layout=layout, dtype="bf16" if bf16 else "f16")
        Kd = to_layout(K, layout).to(dev)
        # the existing path, with a workspace the caller owns (this also gets the kernels loaded before memory is watched)
        ws = torch.full((skv.skv_workspace_bytes(shape, 0),), 0xCD, dtype=torch.uint8, device=dev)
        want = torch.full((R, L, n), float("nan"), dtype=torch.float32, device=dev)
        skv.skv_importance_kvnorm(shape, Kd, want, ws, lam=lam)
        got = torch.full((R, L, n), float("nan"), dtype=torch.float32, device=dev)
        prepared.append((shape, K, Kd, want, got, lam, bf16))
    torch.cuda.synchronize()

    # call 1 (looks the array up on this GPU), then call 2 straight behind it on the same stream
    shape, _, Kd, _, got, lam, _ = prepared[0]
    skv.skv_importance_kvnorm_noalloc(shape, Kd, got, lam=lam)
    free_before = torch.cuda.mem_get_info(dev)[0]
    shape, _, Kd, _, got, lam, _ = prepared[1]
    skv.skv_importance_kvnorm_noalloc(shape, Kd, got, lam=lam)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(dev)[0] == free_before        # the call took no device memory and gave none back

    for (shape, K, Kd, want, got, lam, bf16) in prepared:
        w, h = want.cpu().numpy().astype(np.float64), got.cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(h))
        assert np.all(np.abs(h - w) <= 1e-3 * w + 1e-30)          # the tolerance of the importance parity tests
        assert torch.equal(want, got)                             # and in fact the same bits: the same kernels ran

    # the small problem against the CPU oracle as well, like tests/test_gpu_parity.py does for the workspace path
    shape, K, _, _, got, lam, bf16 = prepared[1]
    for r in range(K.shape[0]):
        Kr = K[r].view(torch.int16).numpy().view(np.uint16) if bf16 else K[r].numpy()
        ref = oracle.importance_kvnorm(Kr, lam=lam, bf16=bf16).astype(np.float64)
        assert np.all(np.abs(got[r].cpu().numpy().astype(np.float64) - ref) <= 1e-3 * ref + 1e-30)

    # beyond the limit: its own status, and the output is not touched
    big = skv.make_shape(32, 8, 8, 128, 32768, 2)
    sentinel = torch.full((16,), -1.0, dtype=torch.float32, device=dev)
    with pytest.raises(skv.SkvError) as ei:
        skv.skv_importance_kvnorm_noalloc(big, prepared[0][2], sentinel)
    assert ei.value.status == skv.SKV_ERR_NOALLOC_LIMIT
    torch.cuda.synchronize()
    assert torch.all(sentinel == -1.0)
