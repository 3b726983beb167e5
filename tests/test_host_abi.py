"""CPU-only tests of the C-ABI library: it loads without a GPU, exports every symbol include/skv.h declares,
and its host-side logic (tier counts, blob sizes, header validation, argument errors) agrees with the oracle."""
import os
import re

import numpy as np
import pytest

import oracle
import paper_2606_08635_b200 as skv

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_08635_b200 import build
    build.build()


def test_library_exports_every_declared_symbol():
    text = open(os.path.join(ROOT, "include", "skv.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(skv_[a-z0-9_]+)\s*\(", text))
    assert declared == set(skv.EXPORTS)
    L = skv.lib()
    for name in declared:
        assert getattr(L, name) is not None
    assert "sm_100a" in skv.skv_version()


def test_tier_counts_match_oracle_sweep():
    rng = np.random.default_rng(0)
    for _ in range(2000):
        n = int(rng.integers(1, 6000))
        b = float(rng.choice([rng.uniform(0.01, 1.3), rng.integers(1, 41) / 40.0]))
        s = int(rng.integers(0, min(n, 9) + 1))
        rngs = []
        for _r in range(int(rng.integers(0, 4))):
            a = int(rng.integers(0, n + 1)); e = int(rng.integers(a, n + 1)); rngs.append((a, e))
        a4 = int(rng.integers(0, 3))                      # 0 = 2-tier, 1 = INT4 low tier, 2 = 2-bit low tier (NEXT-4)
        shape = skv.make_shape(2, 4, 2, 128, n)
        pol = skv.make_policy(b, s, rngs, a4)
        try:
            want, _ = oracle.tier_counts(n, b, s, rngs, a4)
        except ValueError:
            with pytest.raises(skv.SkvError) as ei:
                skv.skv_tier_counts(shape, pol)
            assert ei.value.status == skv.SKV_ERR_BUDGET_INFEASIBLE
            continue
        got = skv.skv_tier_counts(shape, pol)
        assert got.as_tuple() == (want.n16, want.n8, want.n4, want.n0)
        assert (got.budget_q4, got.spent_q4, got.allow_int4) == (want.budget_q4, want.spent_q4, int(a4))
        assert skv.skv_blob_bytes(shape, got) == oracle.blob_bytes(2, 2, 128, n, want)


def test_tier_counts_next4_modes_match_oracle_sweep_and_header_flags():
    """NEXT-4 tier modes (INT8 hot tier P21, group-wise 2-bit P22): closed-form counts and blob sizes against the oracle."""
    rng = np.random.default_rng(5)
    for _ in range(1500):
        n = int(rng.integers(1, 6000))
        b = float(rng.choice([rng.uniform(0.01, 1.3), rng.integers(1, 41) / 40.0]))
        s = int(rng.integers(0, min(n, 9) + 1))
        a4 = int(rng.integers(0, 3))
        mode = int(rng.integers(1, 4)) if a4 == 2 else 1
        rngs = [(int(a), int(a + rng.integers(0, n - a + 1))) for a in rng.integers(0, n + 1, size=int(rng.integers(0, 3)))]
        shape = skv.make_shape(2, 4, 2, 128, n)
        pol = skv.make_policy(b, s, rngs, a4, tier_mode=mode)
        try:
            want, _ = oracle.tier_counts(n, b, s, rngs, a4, mode=mode)
        except ValueError:
            with pytest.raises(skv.SkvError) as ei:
                skv.skv_tier_counts(shape, pol)
            assert ei.value.status == skv.SKV_ERR_BUDGET_INFEASIBLE
            continue
        got = skv.skv_tier_counts(shape, pol)
        assert got.as_tuple() == (want.n16, want.n8, want.n4, want.n0) and got.tier_mode == mode
        assert (got.budget_q4, got.spent_q4, got.allow_int4) == (want.budget_q4, want.spent_q4, a4)
        assert skv.skv_blob_bytes(shape, got) == oracle.blob_bytes(2, 2, 128, n, want)
    # group-wise records need the 2-bit tier; unknown mode bits are refused
    shape = skv.make_shape(2, 4, 2, 128, 100)
    for pol in (skv.make_policy(0.3, 0, (), 1, tier_mode=2), skv.make_policy(0.3, 0, (), 0, tier_mode=2),
                skv.make_policy(0.3, 0, (), 2, tier_mode=4)):
        with pytest.raises(skv.SkvError) as ei:
            skv.skv_tier_counts(shape, pol)
        assert ei.value.status == skv.SKV_ERR_INVALID_ARG
    # skv_blob_check: an oracle-written blob with both flags is accepted and reports the mode; FP16 tokens under the
    # INT8-hot-tier flag and groups without the 2-bit tier are refused
    L, n, Hkv, d = 1, 24, 2, 64
    c, prot = oracle.tier_counts(n, 0.2, 2, [], 2, mode=3)
    K = np.random.default_rng(6).standard_normal((L, n, Hkv, d)).astype(np.float16)
    tier = oracle.assign(np.random.default_rng(7).random((L, n)).astype(np.float32), prot, c)
    blob = oracle.pack(K, K, tier, c, 2)
    assert int.from_bytes(bytes(blob[40:44]), "little") == 1 | 2 | 8 | 16
    hs, hc = skv.skv_blob_check(bytes(blob[:256]), blob.size)
    assert hc.tier_mode == 3 and hc.allow_int4 == 2 and hc.as_tuple() == (0, c.n8, c.n4, c.n0)
    for off, val in ((24, 1), (40, 1 | 8 | 16)):
        bad = blob[:256].copy(); bad[off] = val
        with pytest.raises(skv.SkvError) as ei:
            skv.skv_blob_check(bytes(bad), blob.size)
        assert ei.value.status == skv.SKV_ERR_BAD_BLOB


def test_argument_errors():
    shape = skv.make_shape(2, 4, 2, 128, 100)
    for bad_b in (0.0, -1.0, float("nan")):
        with pytest.raises(skv.SkvError) as ei:
            skv.skv_tier_counts(shape, skv.make_policy(bad_b))
        assert ei.value.status == skv.SKV_ERR_INVALID_ARG
    for rngs in ([(5, 101)], [(-1, 3)], [(9, 4)]):
        with pytest.raises(skv.SkvError) as ei:
            skv.skv_tier_counts(shape, skv.make_policy(0.5, 0, rngs))
        assert ei.value.status == skv.SKV_ERR_INVALID_ARG
    c = skv.skv_tier_counts(shape, skv.make_policy(0.5, 4))
    # device entry points validate before launching anything: null pointers / bad dims / misalignment
    ws = 0
    for fn, args in (
        (skv.skv_pack, (shape, 0, 0, 0, c, 0, 0)),
        (skv.skv_unpack, (shape, 0, 0, c, 0, 0, None, 0)),
    ):
        with pytest.raises(skv.SkvError) as ei:
            fn(*args, stream=0)
        assert ei.value.status == skv.SKV_ERR_INVALID_ARG
    shape_bad = skv.make_shape(2, 4, 2, 96, 100)
    L = skv.lib()
    import ctypes as C
    rc = L.skv_pack(C.byref(shape_bad), 256, 256, 256, C.byref(c), 256, 1 << 30, 256, 1 << 30, None)
    assert rc == skv.SKV_ERR_UNSUPPORTED
    rc = L.skv_pack(C.byref(shape), 256 + 8, 256, 256, C.byref(c), 256, 1 << 30, 256, 1 << 30, None)
    assert rc == skv.SKV_ERR_UNSUPPORTED            # K not 16-byte aligned
    rc = L.skv_pack(C.byref(shape), 256, 256, 256, C.byref(c), 256, 16, 256, 1 << 30, None)
    assert rc == skv.SKV_ERR_BUFFER_TOO_SMALL       # blob capacity
    rc = L.skv_pack(C.byref(shape), 256, 256, 256, C.byref(c), 256, 1 << 30, 256, 16, None)
    assert rc == skv.SKV_ERR_BUFFER_TOO_SMALL       # workspace
    rc = L.skv_importance(C.byref(shape), 256, 256, 101, 1, 0.0, 256, 256, 1 << 30, None)
    assert rc == skv.SKV_ERR_INVALID_ARG            # window > n
    shape3 = skv.make_shape(2, 5, 2, 128, 100)
    rc = L.skv_importance(C.byref(shape3), 256, 256, 8, 1, 0.0, 256, 256, 1 << 30, None)
    assert rc == skv.SKV_ERR_INVALID_ARG            # Hq % Hkv != 0
    assert skv.skv_strerror(skv.SKV_ERR_BAD_BLOB).startswith("malformed")
    # the NEXT-row entry points validate the same way
    rc = L.skv_unpack_patch(C.byref(shape), 0, 0, C.byref(c), 0, 0, None, 0, 0, None)
    assert rc == skv.SKV_ERR_INVALID_ARG
    rc = L.skv_unpack_patch(C.byref(shape), 256, 12345, C.byref(c), 256, 256, None, 256, 1 << 30, None)
    assert rc == skv.SKV_ERR_BAD_BLOB               # blob_bytes disagrees with the layout of `counts`
    shape_dt = skv.make_shape(2, 4, 2, 128, 100)
    shape_dt.dtype = 7
    rc = L.skv_pack(C.byref(shape_dt), 256, 256, 256, C.byref(c), 256, 1 << 30, 256, 1 << 30, None)
    assert rc == skv.SKV_ERR_INVALID_ARG            # unknown element type
    with pytest.raises(skv.SkvError):               # populations exceed n
        skv.skv_counts_from_populations(shape, 60, 50, 0)
    with pytest.raises(skv.SkvError):               # low tier populated but not allowed
        skv.skv_counts_from_populations(shape, 1, 1, 5, allow_int4=False)
    cp = skv.skv_counts_from_populations(shape, 10, 20, 30, allow_int4=2)
    assert cp.as_tuple() == (10, 20, 30, 40) and cp.allow_int4 == 2 and cp.spent_q4 == 8 * 10 + 4 * 20 + 30
    rc = L.skv_assign_tiers_counts(C.byref(shape), C.byref(cp), 11, 0, None, 256, 256, 0, 0, None)
    assert rc == skv.SKV_ERR_BUDGET_INFEASIBLE      # 11 protected positions but only 10 FP16 slots
    rc = L.skv_assign_tiers_counts(C.byref(shape), C.byref(cp), 2, 0, None, 0, 256, 0, 0, None)
    assert rc == skv.SKV_ERR_INVALID_ARG            # null importance


def test_workspace_alignment_broadcast_strides_and_importance_plan_limits():
    """Round-2 review items: a workspace that is not 16-byte aligned, a zero (broadcast) layer / request stride handed to
    skv_importance, and an importance work decomposition that does not fit 32-bit counters all come back as a status
    code before anything is launched (no GPU needed)."""
    import ctypes as C
    L = skv.lib()
    shape = skv.make_shape(2, 4, 2, 128, 100)
    c = skv.skv_tier_counts(shape, skv.make_policy(0.5, 4))
    big = 1 << 40
    for ws in (256 + 8, 256 + 4, 257):
        assert L.skv_pack(C.byref(shape), 256, 256, 256, C.byref(c), 256, big, ws, big, None) == skv.SKV_ERR_UNSUPPORTED
        bb = skv.skv_blob_bytes(shape, c)
        assert L.skv_unpack(C.byref(shape), 256, bb, C.byref(c), 256, 256, None, ws, big, None) == skv.SKV_ERR_UNSUPPORTED
        assert L.skv_unpack_patch(C.byref(shape), 256, bb, C.byref(c), 256, 256, None, ws, big, None) == skv.SKV_ERR_UNSUPPORTED
        assert L.skv_importance(C.byref(shape), 256, 256, 8, 1, 0.0, 256, ws, big, None) == skv.SKV_ERR_UNSUPPORTED
        assert L.skv_importance_kvnorm(C.byref(shape), 256, 0.0, 256, ws, big, None) == skv.SKV_ERR_UNSUPPORTED
        pol = skv.make_policy(0.5, 4)
        assert L.skv_assign_tiers(C.byref(shape), C.byref(pol), 256, 256, None, ws, big, None) == skv.SKV_ERR_UNSUPPORTED
    # broadcast strides: fine for the other readers of K, not expressible in the importance kernel's tensor map
    for field in ("stride_layer", "stride_request"):
        sb = skv.make_shape(2, 4, 2, 128, 100, 2)
        setattr(sb, field, 0)
        assert L.skv_importance(C.byref(sb), 256, 256, 8, 1, 0.0, 256, 256, big, None) == skv.SKV_ERR_UNSUPPORTED
    one = skv.make_shape(1, 4, 2, 128, 100, 1)
    one.stride_layer = one.stride_request = 0                       # a single layer / request: the stride is never used
    assert skv.skv_workspace_bytes(one, 8) > 0
    # 65535 layers x 8 KV heads x 8192 key tiles = 4.3e9 work items: more than a 32-bit counter holds
    huge = skv.make_shape(65535, 8, 8, 128, 1 << 20, 1)
    assert skv.skv_workspace_bytes(huge, 0) > 0
    assert skv.skv_workspace_bytes(huge, 1) == 0
    assert L.skv_importance(C.byref(huge), 256, 256, 1, 1, 0.0, 256, 256, big, None) == skv.SKV_ERR_UNSUPPORTED
    ok = skv.make_shape(65535, 8, 8, 128, 1 << 14, 1)               # 65535 x 8 x 128 tiles = 6.7e7 items: fits
    assert skv.skv_workspace_bytes(ok, 1) > 0


def test_blob_check_accepts_oracle_blob_and_rejects_corruption():
    L_, n, Hkv, d = 2, 50, 2, 64
    rng = np.random.default_rng(1)
    K = rng.standard_normal((L_, n, Hkv, d)).astype(np.float16)
    V = rng.standard_normal((L_, n, Hkv, d)).astype(np.float16)
    c, prot = oracle.tier_counts(n, 0.4, 4, [], True)
    tier = oracle.assign(rng.random((L_, n)).astype(np.float32), prot, c)
    blob = oracle.pack(K, V, tier, c)
    s, cc = skv.skv_blob_check(blob[:256].tobytes(), blob.size)
    assert (s.n_layers, s.n_kv_heads, s.head_dim, s.n_tokens) == (L_, Hkv, d, n)
    assert cc.as_tuple() == (c.n16, c.n8, c.n4, c.n0) and cc.budget_q4 == c.budget_q4 and cc.allow_int4 == 1
    for off in (0, 3, 4, 8, 12, 16, 20, 24, 28, 32, 36, 40, 44, 56, 64, 72, 80, 152, 160, 200, 255):
        h = bytearray(blob[:256].tobytes()); h[off] ^= 0x01
        with pytest.raises(skv.SkvError) as ei:
            skv.skv_blob_check(bytes(h), blob.size)
        assert ei.value.status == skv.SKV_ERR_BAD_BLOB, off
    with pytest.raises(skv.SkvError):
        skv.skv_blob_check(blob[:256].tobytes(), blob.size - 256)
    # NEXT-4: a blob whose low tier is 2-bit (flags = 3, budget in eighths)
    c2, prot = oracle.tier_counts(n, 0.2, 4, [], 2)
    tier2 = oracle.assign(rng.random((L_, n)).astype(np.float32), prot, c2)
    assert set(np.unique(tier2)) <= {16, 8, 2, 0} and (tier2 == 2).any()
    blob2 = oracle.pack(K, V, tier2, c2, 2)
    s2, cc2 = skv.skv_blob_check(blob2[:256].tobytes(), blob2.size)
    assert cc2.as_tuple() == (c2.n16, c2.n8, c2.n4, c2.n0) and cc2.allow_int4 == 2
    assert (cc2.budget_q4, cc2.spent_q4) == (c2.budget_q4, c2.spent_q4)
    assert skv.skv_blob_bytes(s2_shape := skv.make_shape(L_, Hkv, Hkv, d, n), cc2) == blob2.size


def test_workspace_covers_every_entry_point():
    for (L_, Hq, Hkv, d, n, R, w) in [(1, 2, 2, 128, 256, 1, 16), (32, 32, 8, 128, 32768, 4, 64), (42, 16, 8, 256, 4096, 1, 32)]:
        shape = skv.make_shape(L_, Hq, Hkv, d, n, R)
        ws = skv.skv_workspace_bytes(shape, w)
        assert ws % 256 == 0
        assert ws >= R * L_ * ((n + 31) // 32) * 16          # tile prefix table of pack / unpack
        assert ws >= R * L_ * n * 4                           # selection keys when they do not fit shared memory
        assert ws >= R * L_ * Hq * w * 4                      # per-row log-sum-exp of the importance pass


def test_limits_documented_in_the_header_are_the_ones_enforced():
    """include/skv.h lists: n_tokens <= 2^20, n_layers * n_requests <= 65535, counts that a receiver would refuse,
    zero output strides; the workspace query returns 0 instead of dividing by zero."""
    import ctypes as C
    L = skv.lib()
    hdr = open(os.path.join(ROOT, "include", "skv.h")).read()
    assert "n_tokens > 2^20" in hdr and "n_tokens > 2^24" not in hdr and "65535" in hdr
    c0 = skv.skv_counts()
    big = skv.make_shape(1, 2, 2, 128, (1 << 20) + 1)
    ok = skv.make_shape(1, 2, 2, 128, 1 << 20)
    pol = skv.make_policy(0.5)
    assert L.skv_assign_tiers(C.byref(big), C.byref(pol), 256, 256, C.byref(c0), 256, 1 << 40, None) == skv.SKV_ERR_UNSUPPORTED
    assert L.skv_tier_counts(C.byref(ok), C.byref(pol), C.byref(c0)) == skv.SKV_OK
    grid = skv.make_shape(256, 2, 2, 128, 64, 256)                       # L * R = 65536
    assert L.skv_assign_tiers(C.byref(grid), C.byref(pol), 256, 256, C.byref(c0), 256, 1 << 40, None) == skv.SKV_ERR_UNSUPPORTED
    # workspace query: Hq < Hkv or Hq % Hkv != 0 with a window used to divide by zero
    assert skv.skv_workspace_bytes(skv.make_shape(2, 2, 4, 128, 100), 8) == 0
    assert skv.skv_workspace_bytes(skv.make_shape(2, 6, 4, 128, 100), 8) == 0
    assert skv.skv_workspace_bytes(skv.make_shape(2, 4, 4, 128, 100), 101) == 0
    assert skv.skv_workspace_bytes(skv.make_shape(2, 2, 4, 128, 100), 0) > 0
    # counts a receiver would refuse are refused by the sender
    shape = skv.make_shape(2, 4, 2, 128, 100)
    good = skv.skv_counts_from_populations(shape, 10, 20, 30)
    for mutate in (lambda c: setattr(c, "allow_int4", 0),               # low tier populated without the flag
                   lambda c: setattr(c, "budget_q4", c.spent_q4 - 1),    # over budget
                   lambda c: setattr(c, "budget_q4", 4 * 100 + 1),       # budget above all-FP16
                   lambda c: setattr(c, "n0", c.n0 + 1),                 # populations do not add up
                   lambda c: setattr(c, "allow_int4", 3)):
        c = skv.skv_counts_from_populations(shape, 10, 20, 30)
        mutate(c)
        assert L.skv_pack(C.byref(shape), 256, 256, 256, C.byref(c), 256, 1 << 30, 256, 1 << 30, None) == skv.SKV_ERR_INVALID_ARG
        assert L.skv_unpack(C.byref(shape), 256, 1 << 20, C.byref(c), 256, 256, None, 256, 1 << 30, None) == skv.SKV_ERR_INVALID_ARG
    # overlapping output rows: layer stride 0 with two layers
    zs = skv.make_shape(2, 4, 2, 128, 100, strides=(0, 0, 256, 128))
    assert L.skv_unpack(C.byref(zs), 256, skv.skv_blob_bytes(shape, good), C.byref(good), 256, 256, None, 256, 1 << 30, None) == skv.SKV_ERR_INVALID_ARG
