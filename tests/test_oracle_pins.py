"""Pins for the CPU oracle (oracle/skv_oracle.c) against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible mistake in the
oracle (dropped term, wrong sign/index, transposed operand, wrong rounding) fails it.
"""
import math
import os

import numpy as np
import pytest
import torch

import oracle
from conftest import read_golden

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


# ----------------------------------------------------------------------------------------------
# fp16 <-> fp32 conversion: pinned exhaustively against numpy's float16 (an independent library)
# ----------------------------------------------------------------------------------------------
def test_half_to_float_exhaustive():
    bits = np.arange(65536, dtype=np.uint16)
    ref = bits.view(np.float16).astype(np.float32)
    got = np.array([oracle.half_to_float(int(b)) for b in bits], dtype=np.float32)
    nan = np.isnan(ref)
    assert np.array_equal(np.isnan(got), nan)
    assert np.array_equal(got[~nan].view(np.uint32), ref[~nan].view(np.uint32))


def test_float_to_half_rne_against_numpy():
    rng = np.random.default_rng(0)
    halves = np.arange(0, 0x7C00, dtype=np.uint16).view(np.float16).astype(np.float64)
    mids = ((halves[:-1] + halves[1:]) / 2).astype(np.float32)          # exact ties between neighbours
    near = np.concatenate([np.nextafter(mids, np.float32(np.inf)), np.nextafter(mids, np.float32(-np.inf))])
    rand = np.concatenate([rng.standard_normal(20000) * s for s in (1e-7, 1e-4, 1.0, 100.0, 3e4)]).astype(np.float32)
    edge = np.array([0.0, -0.0, 65504.0, 65519.0, 5.96e-8, 2.98e-8, 2.9802322e-8, 6.1e-5, 6.1035156e-5], dtype=np.float32)
    xs = np.concatenate([mids, near, rand, edge, -mids[::7]])
    xs = xs[np.abs(xs) < 65520.0]
    ref = xs.astype(np.float16).view(np.uint16)
    got = np.array([oracle.float_to_half(float(x)) for x in xs], dtype=np.uint16)
    assert np.array_equal(got, ref)


# ----------------------------------------------------------------------------------------------
# O2 tier counts
# ----------------------------------------------------------------------------------------------
def test_tier_fractions_from_paper():
    for b, a4, n16, n8, n4, n0 in read_golden(os.path.join(GOLD, "tier_fractions.txt")):
        c, prot = oracle.tier_counts(10000, float(b), 0, [], bool(int(a4)))
        assert (c.n16, c.n8, c.n4, c.n0) == (int(n16), int(n8), int(n4), int(n0)), b
        assert prot.sum() == 0


def test_tier_counts_invariants_sweep():
    rng = np.random.default_rng(1)
    for _ in range(3000):
        n = int(rng.integers(1, 5000))
        b = float(rng.choice([rng.uniform(0.01, 1.2), rng.integers(1, 41) / 40.0]))
        s = int(rng.integers(0, min(n, 9)))
        rngs = []
        for _r in range(int(rng.integers(0, 3))):
            a = int(rng.integers(0, n + 1)); e = int(rng.integers(a, n + 1)); rngs.append((a, e))
        a4 = bool(rng.integers(0, 2))
        prot_ref = np.zeros(n, bool); prot_ref[:s] = True
        for a, e in rngs:
            prot_ref[a:e] = True
        P = int(prot_ref.sum())
        Q = int(np.floor(4 * min(b, 1.0) * n + 1e-6))
        try:
            c, prot = oracle.tier_counts(n, b, s, rngs, a4)
        except ValueError:
            assert 4 * P > Q            # only infeasible budgets are refused
            continue
        assert 4 * P <= Q
        assert np.array_equal(prot.astype(bool), prot_ref)
        assert c.budget_q4 == Q
        assert c.n16 + c.n8 + c.n4 + c.n0 == n and min(c.n16, c.n8, c.n4, c.n0) >= 0
        assert c.spent_q4 == 4 * c.n16 + 2 * c.n8 + c.n4 <= Q          # Eq. 3: never over budget
        assert c.n16 >= P
        if c.n16 < n:
            assert Q - c.spent_q4 <= 1                                  # budget used up to rounding
        # at most two ADJACENT tiers among the non-protected tokens (Eq. 14-15 structure)
        pops = [c.n16 - P > 0, c.n8 > 0, c.n4 > 0, c.n0 > 0]
        idx = [i for i, p in enumerate(pops) if p]
        assert len(idx) <= 2 and (len(idx) < 2 or idx[1] - idx[0] == 1 or (not a4 and idx == [1, 3]))
        if not a4:
            assert c.n4 == 0


def test_tier_counts_config_table():
    # (n, b, s, ranges, allow_int4) -> counts; closed form of DESIGN.md reading P5 evaluated by hand
    # e.g. C3 b=0.3: Q=floor(4*.3*4096)=4915, P=68, m=4028, R=4915-272=4643 in [m,2m): n8=R-m=615, n4=2m-R=3413
    table = [
        (256, 0.5, 4, [], True, (4, 244, 8, 0)),
        (4096, 0.3, 4, [], False, (4, 2449, 0, 1643)),
        (4096, 0.5, 4, [], False, (4, 4088, 0, 4)),
        (4096, 0.3, 4, [(4032, 4096)], True, (68, 615, 3413, 0)),
        (4096, 0.5, 4, [(4032, 4096)], True, (68, 3892, 136, 0)),
        (4096, 0.5, 4, [], True, (4, 4084, 8, 0)),
        (32768, 0.3, 4, [], True, (4, 6541, 26223, 0)),
        (32768, 0.4, 4, [], True, (4, 19648, 13116, 0)),
        (32768, 0.5, 4, [], True, (4, 32756, 8, 0)),
        (32768, 0.75, 4, [], True, (16384, 16384, 0, 0)),
        (32768, 1.0, 4, [], True, (32768, 0, 0, 0)),
    ]
    for n, b, s, r, a4, want in table:
        c, _ = oracle.tier_counts(n, b, s, r, a4)
        assert (c.n16, c.n8, c.n4, c.n0) == want, (n, b)


def test_overlapping_ranges_counted_once_and_b_clamped():
    c, prot = oracle.tier_counts(100, 1.7, 4, [(2, 10), (8, 12), (50, 50)], True)
    assert prot.sum() == 12 and c.n16 == 100 and c.budget_q4 == 400
    with pytest.raises(ValueError):
        oracle.tier_counts(100, 0.1, 20, [], True)          # 4P = 80 > Q = 40
    with pytest.raises(ValueError):
        oracle.tier_counts(100, 0.5, 0, [(10, 101)], True)  # range outside [0, n]


# ----------------------------------------------------------------------------------------------
# O3 selection
# ----------------------------------------------------------------------------------------------
def _brute_force_tiers(I, prot, counts):
    """rank_j = #{k : I_k > I_j or (I_k == I_j and k < j)} over non-protected tokens, O(n^2)."""
    n = len(I)
    key = np.where(I > 0, I, np.float32(0)).astype(np.float32)
    key[np.isnan(I)] = 0
    tier = np.zeros(n, np.uint8)
    P = int(prot.sum())
    for j in range(n):
        if prot[j]:
            tier[j] = 16
            continue
        rank = 0
        for k in range(n):
            if prot[k] or k == j:
                continue
            if key[k] > key[j] or (key[k] == key[j] and k < j):
                rank += 1
        c16 = counts.n16 - P
        tier[j] = 16 if rank < c16 else 8 if rank < c16 + counts.n8 else 4 if rank < c16 + counts.n8 + counts.n4 else 0
    return tier


@pytest.mark.parametrize("n,b,s,ranges,a4", [
    (64, 0.4, 4, [], True), (97, 0.3, 2, [(90, 97)], True), (50, 0.3, 4, [], False),
    (33, 0.75, 0, [(5, 9)], True), (40, 0.2, 1, [], True), (31, 1.0, 4, [], True)])
def test_selection_matches_brute_force(n, b, s, ranges, a4):
    rng = np.random.default_rng(n)
    I = rng.random((2, n)).astype(np.float32)
    I[0, 5] = I[0, 20] = I[0, 21]        # exact ties
    I[1, 3] = np.nan; I[1, 9] = -1.0; I[1, 10] = -0.0; I[1, 11] = 0.0
    c, prot = oracle.tier_counts(n, b, s, ranges, a4)
    tier = oracle.assign(I, prot, c)
    for l in range(2):
        assert np.array_equal(tier[l], _brute_force_tiers(I[l], prot, c))
        assert [(tier[l] == t).sum() for t in (16, 8, 4, 0)] == [c.n16, c.n8, c.n4, c.n0]


def test_selection_monotone_and_sinks_fp16():
    # Prop. 1: higher importance never gets a lower tier; sinks FP16 whatever their score
    rng = np.random.default_rng(7)
    n = 2000
    I = (rng.random((3, n)) ** 6).astype(np.float32)
    I[:, :4] = 0.0                                           # sinks with the lowest possible score
    c, prot = oracle.tier_counts(n, 0.35, 4, [(1900, 1910)], True)
    tier = oracle.assign(I, prot, c).astype(np.int32)
    assert (tier[:, :4] == 16).all() and (tier[:, 1900:1910] == 16).all()
    for l in range(3):
        free = ~prot.astype(bool)
        order = np.argsort(-I[l][free], kind="stable")
        t = tier[l][free][order]
        assert (np.diff(t) <= 0).all()                       # non-increasing tier along decreasing importance


def test_selection_tie_break_lower_position_first():
    I = np.full((1, 10), 0.5, np.float32)
    c, prot = oracle.tier_counts(10, 0.4, 0, [], True)       # Q=16, m=10: n8=6, n4=4
    assert (c.n8, c.n4) == (6, 4)
    tier = oracle.assign(I, prot, c)
    assert tier[0].tolist() == [8] * 6 + [4] * 4


# ----------------------------------------------------------------------------------------------
# O4 quantizer
# ----------------------------------------------------------------------------------------------
def test_quantizer_worked_examples():
    rows = read_golden(os.path.join(GOLD, "quantizer_worked.txt"))
    groups = {}
    for name, qmax, x, code, ybits in rows:
        groups.setdefault((name, int(qmax)), []).append((float(x), int(code), int(ybits, 16)))
    assert len(groups) == 4
    for (name, qmax), items in groups.items():
        x = np.zeros(128, np.float16)
        x[:len(items)] = [it[0] for it in items]
        assert all(float(np.float16(it[0])) == it[0] for it in items)      # fixtures are exact fp16 values
        ab, q = oracle.quantize_vector(x, qmax)
        assert ab == int(np.abs(x).max().view(np.uint16)), name
        assert q[:len(items)].tolist() == [it[1] for it in items], name
        assert (q[len(items):] == 0).all()
        y = oracle.dequantize_vector(q, qmax, ab)
        assert y[:len(items)].view(np.uint16).tolist() == [it[2] for it in items], name


def test_quantizer_special_cases():
    z = np.zeros(64, np.float16); z[3] = -0.0
    ab, q = oracle.quantize_vector(z, 127)
    assert ab == 0 and (q == 0).all()
    assert (oracle.dequantize_vector(q, 127, ab).view(np.uint16) == 0).all()     # +0.0
    big = np.full(64, 65504.0, np.float16); big[1] = -65504.0
    for qmax in (127, 7):
        ab, q = oracle.quantize_vector(big, qmax)
        assert q[0] == qmax and q[1] == -qmax
        assert np.array_equal(oracle.dequantize_vector(q, qmax, ab), big)        # no overflow
    sub = np.zeros(64, np.float16); sub[0] = np.float16(5.96e-8); sub[1] = -sub[0]
    ab, q = oracle.quantize_vector(sub, 127)
    assert ab == 1 and q[0] == 127 and q[1] == -127
    assert np.array_equal(oracle.dequantize_vector(q, 127, ab), sub)


def _exact_code(x16, inv32, qmax):
    """round-half-even of the exact rational product, clamped (independent of the oracle: fractions only)."""
    from fractions import Fraction
    import math
    ex = Fraction(float(x16)) * Fraction(float(inv32))
    fl = math.floor(ex)
    fr = ex - fl
    r = fl if fr < Fraction(1, 2) else fl + 1 if fr > Fraction(1, 2) else (fl if fl % 2 == 0 else fl + 1)
    return max(-qmax, min(qmax, r))


def test_quantizer_single_rounding_of_the_exact_product():
    rows = read_golden(os.path.join(GOLD, "quantizer_single_rounding.txt"))
    assert len(rows) == 6
    for qmax, amax, x, code, code_two_step in rows:
        qmax, amax, x, code, code_two_step = int(qmax), float(amax), float(x), int(code), int(code_two_step)
        assert float(np.float16(amax)) == amax and float(np.float16(x)) == x and code != code_two_step
        inv = np.float32(qmax) / np.float32(amax)
        assert int(np.rint(np.float32(x) * inv)) == code_two_step            # what the rejected reading gives
        assert _exact_code(x, inv, qmax) == code                              # the fixture is self-consistent
        v = np.zeros(64, np.float16); v[0] = amax; v[1] = x
        ab, q = oracle.quantize_vector(v, qmax)
        assert q[0] == qmax and q[1] == code
    # brute force on random vectors: every code equals the exactly-rounded rational product
    rng = np.random.default_rng(11)
    for qmax in (127, 7):
        for _ in range(20):
            v = (rng.standard_normal(128) * rng.uniform(0.01, 30)).astype(np.float16)
            ab, q = oracle.quantize_vector(v, qmax)
            inv = np.float32(qmax) / np.float32(np.uint16(ab).view(np.float16))
            assert q.tolist() == [_exact_code(e, inv, qmax) for e in v]


@pytest.mark.parametrize("qmax", [127, 7])
def test_quantizer_error_bound(qmax):
    # BASELINE north_star: per-element dequantization error <= scale/2 (on the fp32 product, with the
    # reciprocal-multiply slack derived in DESIGN.md; + half an fp16 ulp on the stored output).
    rng = np.random.default_rng(3)
    for scale_mag in (1e-3, 1.0, 50.0):
        x = (rng.standard_normal((200, 128)) * scale_mag).astype(np.float16)
        x[:, :6] *= 10
        x = np.clip(x, -65504, 65504).astype(np.float16)
        for v in x:
            ab, q = oracle.quantize_vector(v, qmax)
            amax = float(np.uint16(ab).view(np.float16))
            assert amax == float(np.abs(v).max())
            scale = amax / qmax
            assert np.abs(q).max() == qmax                                     # the amax element hits +-qmax
            err = np.abs(q.astype(np.float64) * scale - v.astype(np.float64))
            assert err.max() <= scale / 2 * (1 + 1e-4)
            y = oracle.dequantize_vector(q, qmax, ab).astype(np.float64)
            ulp = np.spacing(np.abs(y).astype(np.float16)).astype(np.float64)
            assert (np.abs(y - v.astype(np.float64)) <= scale / 2 * (1 + 1e-4) + ulp / 2 + 1e-12).all()
            assert (np.sign(q) * np.sign(v.astype(np.float64)) >= 0).all()     # symmetric: sign preserved


def test_quantizer_cosine_band():
    # Table 8: INT8 cosine > 0.9999, INT4 0.96-0.99 on real KV; on N(0,1) vectors the
    # same quantizer must land in the same regime (statistical sanity, not a bit-level pin).
    rng = np.random.default_rng(4)
    x = rng.standard_normal((500, 128)).astype(np.float16)
    for qmax, lo, hi in ((127, 0.9999, 1.0), (7, 0.985, 0.998)):
        cs = []
        for v in x:
            ab, q = oracle.quantize_vector(v, qmax)
            y = oracle.dequantize_vector(q, qmax, ab).astype(np.float64)
            v64 = v.astype(np.float64)
            cs.append(y @ v64 / np.linalg.norm(y) / np.linalg.norm(v64))
        assert lo < np.mean(cs) <= hi, (qmax, np.mean(cs))


# ----------------------------------------------------------------------------------------------
# O5 wire format
# ----------------------------------------------------------------------------------------------
def _u32(b, off):
    return int.from_bytes(bytes(b[off:off + 4]), "little")


def _u64(b, off):
    return int.from_bytes(bytes(b[off:off + 8]), "little")


def _w6_inputs():
    rows = read_golden(os.path.join(GOLD, "quantizer_worked.txt"))
    w1 = [r for r in rows if r[0] == "W1"]
    w3 = [r for r in rows if r[0] == "W3"]
    K = np.zeros((1, 4, 1, 64), np.float16)
    V = np.zeros((1, 4, 1, 64), np.float16)
    K[0, 0, 0, :] = np.arange(64) / 8.0 - 3.0                 # FP16 token: copied verbatim
    V[0, 0, 0, :] = -np.arange(64) / 16.0
    K[0, 1, 0, :len(w1)] = [float(r[2]) for r in w1]          # INT8 token, W1 vector
    V[0, 1, 0, :2] = [1.0, 0.5]                               # W2: amax 1.0 -> codes 127, 64
    K[0, 2, 0, :len(w3)] = [float(r[2]) for r in w3]          # INT4 token, W3 vector
    V[0, 2, 0, :3] = [1.0, 0.5, -0.25]                        # W4: codes 7, 4, -2
    K[0, 3] = 9.0; V[0, 3] = -9.0                             # dropped token: leaves no bytes
    tier = np.array([[16, 8, 4, 0]], np.uint8)
    return K, V, tier, w1, w3


def test_w6_layout_and_hand_written_blob():
    g = {r[0]: r[1:] for r in read_golden(os.path.join(GOLD, "w6_layout.txt"))}
    K, V, tier, w1, w3 = _w6_inputs()
    counts = oracle.Counts(1, 1, 1, 1, 7, 7)
    blob = oracle.pack(K, V, tier, counts, allow_int4=True)
    assert blob.size == int(g["total_bytes"][0]) == oracle.blob_bytes(1, 1, 64, 4, counts)
    # header, field by field
    assert bytes(blob[0:4]) == b"SKV1" and _u32(blob, 4) == 1
    assert [_u32(blob, o) for o in (8, 12, 16, 20)] == [1, 1, 64, 4]
    assert [_u32(blob, o) for o in (24, 28, 32, 36)] == [1, 1, 1, 1]
    assert _u32(blob, 40) == 1 and _u32(blob, 44) == 0 and _u64(blob, 48) == 7
    assert _u64(blob, 56) == int(g["tier_map_off"][0]) and _u64(blob, 64) == int(g["layer0_off"][0])
    assert _u64(blob, 72) == int(g["layer_stride"][0]) and _u64(blob, 160) == int(g["total_bytes"][0])
    seg = [int(v) for v in g["seg_off"]]
    assert [_u64(blob, 80 + 8 * i) for i in range(10)] == seg
    assert not blob[168:256].any()
    # expected blob written by hand from the format text and the worked codes
    want = np.zeros(3072, np.uint8)
    want[:256] = blob[:256]                                    # header checked field by field above
    want[256:260] = [16, 8, 4, 0]
    base = 512
    want[base + seg[0]: base + seg[0] + 128] = K[0, 0, 0].view(np.uint8)
    want[base + seg[1]: base + seg[1] + 128] = V[0, 0, 0].view(np.uint8)
    k8 = np.zeros(64, np.int8); k8[:len(w1)] = [int(r[3]) for r in w1]
    v8 = np.zeros(64, np.int8); v8[:2] = [127, 64]
    want[base + seg[2]: base + seg[2] + 64] = k8.view(np.uint8)
    want[base + seg[3]: base + seg[3] + 64] = v8.view(np.uint8)
    k4 = [int(r[3]) for r in w3] + [0] * (64 - len(w3))
    v4 = [7, 4, -2] + [0] * 61
    for s, codes in ((4, k4), (5, v4)):
        want[base + seg[s]: base + seg[s] + 32] = [(codes[2 * i] & 0xF) | ((codes[2 * i + 1] & 0xF) << 4) for i in range(32)]
    for s, amax in ((6, 1.984375), (7, 1.0), (8, 1.75), (9, 1.0)):
        want[base + seg[s]: base + seg[s] + 2] = np.array([amax], np.float16).view(np.uint8)
    assert np.array_equal(blob, want)
    # W5 nibble packing
    vec = np.zeros(64, np.float16); vec[:6] = [1.75, -1.0, 0.0, -0.25, 0.5, -1.75]   # codes 7,-4,0,-1,2,-7
    ab, q = oracle.quantize_vector(vec, 7)
    assert q[:6].tolist() == [7, -4, 0, -1, 2, -7]
    K2 = np.zeros((1, 1, 1, 64), np.float16); K2[0, 0, 0] = vec
    b2 = oracle.pack(K2, K2, np.array([[4]], np.uint8), oracle.Counts(0, 0, 1, 0, 1, 1))
    off = _u64(b2, 64) + _u64(b2, 80 + 8 * 4)
    assert bytes(b2[off:off + 3]).hex().upper() == "".join(g["nibbles"])
    # decode side: unpack reproduces FP16 row, dequantised rows, zeros for the dropped token
    K3, V3, t3 = oracle.unpack(blob, 1, 1, 64, 4)
    assert np.array_equal(t3, tier)
    assert np.array_equal(K3[0, 0], K[0, 0]) and np.array_equal(V3[0, 0], V[0, 0])
    assert K3[0, 1, 0, :len(w1)].view(np.uint16).tolist() == [int(r[4], 16) for r in w1]
    assert K3[0, 2, 0, :len(w3)].view(np.uint16).tolist() == [int(r[4], 16) for r in w3]
    assert not K3[0, 3].view(np.uint16).any() and not V3[0, 3].view(np.uint16).any()


def test_blob_bytes_closed_form_and_eq1_identity():
    # payload bytes (segments without pads/scales/map/header) == Bytes_FP16 * spent / (4 n)   (Eq. 1-3)
    for (L, Hkv, d, n, b, s, a4) in [(3, 4, 128, 1000, 0.3, 4, True), (2, 8, 256, 257, 0.5, 4, True),
                                     (5, 4, 128, 4096, 0.3, 4, False), (1, 2, 64, 250, 0.8, 0, True)]:
        c, prot = oracle.tier_counts(n, b, s, [], a4)
        bytes_fp16 = 2 * L * Hkv * d * n * 2
        payload = L * 2 * Hkv * d * (2 * c.n16 + c.n8 + c.n4 // 2) if c.n4 % 2 == 0 else None
        if payload is not None:
            assert payload * 4 * n == bytes_fp16 * c.spent_q4
        pad = lambda x: (x + 255) // 256 * 256
        segs = [c.n16 * Hkv * d * 2] * 2 + [c.n8 * Hkv * d] * 2 + [c.n4 * Hkv * d // 2] * 2 + \
               [c.n8 * Hkv * 2] * 2 + [c.n4 * Hkv * 2] * 2
        total = 256 + pad(L * n) + L * sum(pad(x) for x in segs)
        assert oracle.blob_bytes(L, Hkv, d, n, c) == total


# ----------------------------------------------------------------------------------------------
# O5/O6 pack + unpack
# ----------------------------------------------------------------------------------------------
def _rand_kv(L, n, Hkv, d, seed):
    rng = np.random.default_rng(seed)
    K = rng.standard_normal((L, n, Hkv, d)).astype(np.float16)
    K[..., :3] *= 10
    V = rng.standard_normal((L, n, Hkv, d)).astype(np.float16)
    return K, V


def test_b1_identity_round_trip():
    L, n, Hkv, d = 2, 77, 2, 64
    K, V = _rand_kv(L, n, Hkv, d, 5)
    c, prot = oracle.tier_counts(n, 1.0, 4, [], True)
    I = np.random.default_rng(0).random((L, n)).astype(np.float32)
    tier = oracle.assign(I, prot, c)
    assert (tier == 16).all()
    blob = oracle.pack(K, V, tier, c)
    K2, V2, t2 = oracle.unpack(blob, L, Hkv, d, n)
    assert np.array_equal(K2.view(np.uint16), K.view(np.uint16)) and np.array_equal(V2.view(np.uint16), V.view(np.uint16))
    # Eq. 1: payload of an all-FP16 blob is exactly Bytes_FP16
    assert blob.size >= 2 * L * Hkv * d * n * 2


def test_round_trip_matches_vector_quantizer_and_positions():
    L, n, Hkv, d = 2, 130, 2, 128
    K, V = _rand_kv(L, n, Hkv, d, 6)
    c, prot = oracle.tier_counts(n, 0.22, 3, [(100, 104)], True)     # exercises 16 / 4 / drop
    c2, _ = oracle.tier_counts(n, 0.45, 3, [(100, 104)], True)       # exercises 16 / 8 / 4
    I = np.random.default_rng(1).random((L, n)).astype(np.float32)
    for cc in (c, c2):
        tier = oracle.assign(I, prot, cc)
        blob = oracle.pack(K, V, tier, cc)
        K2, V2, t2 = oracle.unpack(blob, L, Hkv, d, n)
        assert np.array_equal(t2, tier)
        for X, X2 in ((K, K2), (V, V2)):
            for l in range(L):
                for j in range(n):
                    t = tier[l, j]
                    if t == 16:
                        assert np.array_equal(X2[l, j].view(np.uint16), X[l, j].view(np.uint16))
                    elif t == 0:
                        assert not X2[l, j].view(np.uint16).any()
                    else:
                        qmax = 127 if t == 8 else 7
                        for h in range(Hkv):
                            ab, q = oracle.quantize_vector(X[l, j, h], qmax)
                            assert np.array_equal(X2[l, j, h].view(np.uint16),
                                                  oracle.dequantize_vector(q, qmax, ab).view(np.uint16))


def test_pack_rejects_mismatched_counts_and_unpack_rejects_bad_header():
    L, n, Hkv, d = 1, 16, 1, 64
    K, V = _rand_kv(L, n, Hkv, d, 8)
    c, prot = oracle.tier_counts(n, 0.5, 0, [], True)
    tier = np.full((L, n), 8, np.uint8)
    blob = oracle.pack(K, V, tier, c)
    bad_tier = tier.copy(); bad_tier[0, 0] = 4
    with pytest.raises(ValueError):
        oracle.pack(K, V, bad_tier, c)
    for off in (0, 4, 8, 20, 24, 64, 160):
        b = blob.copy(); b[off] ^= 1
        with pytest.raises(ValueError):
            oracle.unpack(b, L, Hkv, d, n)


def test_value_error_bound_eq5_and_logit_bound_eq10():
    # Eq. 5: ||y - y~|| <= sum_j p_j ||e_j||;  Eq. 10: e^{-2 eta} p <= p~ <= e^{2 eta} p.
    # Sanity that unpacked rows land at the right positions with the right magnitudes.
    L, n, Hkv, d = 1, 300, 1, 128
    K, V = _rand_kv(L, n, Hkv, d, 9)
    c, prot = oracle.tier_counts(n, 0.3, 4, [], True)
    I = np.random.default_rng(2).random((L, n)).astype(np.float32)
    tier = oracle.assign(I, prot, c)
    K2, V2, _ = oracle.unpack(oracle.pack(K, V, tier, c), L, Hkv, d, n)
    q = np.random.default_rng(3).standard_normal(d)
    k, k2 = K[0, :, 0].astype(np.float64), K2[0, :, 0].astype(np.float64)
    v, v2 = V[0, :, 0].astype(np.float64), V2[0, :, 0].astype(np.float64)
    z, z2 = k @ q / np.sqrt(d), k2 @ q / np.sqrt(d)
    p = np.exp(z - z.max()); p /= p.sum()
    p2 = np.exp(z2 - z2.max()); p2 /= p2.sum()
    eta = np.abs(z2 - z).max()
    assert (p2 <= np.exp(2 * eta) * p * (1 + 1e-9)).all() and (p2 >= np.exp(-2 * eta) * p * (1 - 1e-9)).all()
    e = np.linalg.norm(v - v2, axis=1)
    assert np.linalg.norm(p @ v - p @ v2) <= (p * e).sum() * (1 + 1e-9)
    assert (e[tier[0] == 16] == 0).all() and e[tier[0] == 4].mean() > e[tier[0] == 8].mean() > 0


def test_drop_tail_mass_lemma1():
    # Lemma 1: dropping a set of mass eps with renormalisation moves y by <= 2 eps V.
    L, n, Hkv, d = 1, 200, 1, 64
    K, V = _rand_kv(L, n, Hkv, d, 10)
    c, prot = oracle.tier_counts(n, 0.3, 4, [], False)          # 2-tier: INT8 + drop
    assert c.n0 > 0
    rng = np.random.default_rng(4)
    p = rng.random(n) ** 8; p /= p.sum()
    I = p[None].astype(np.float32)
    tier = oracle.assign(I, prot, c)
    keep = tier[0] != 0
    eps = p[~keep].sum()
    v = V[0, :, 0].astype(np.float64)
    y = p @ v
    yhat = (p[keep] / (1 - eps)) @ v[keep]
    Vmax = np.linalg.norm(v, axis=1).max()
    assert np.linalg.norm(y - yhat) <= 2 * eps * Vmax
    # the dropped set is the lowest-importance one: its mass is below the mass of any equal-size kept set
    assert eps <= np.sort(p[~prot.astype(bool)])[: c.n0].sum() * (1 + 1e-6)


# ----------------------------------------------------------------------------------------------
# O1 importance
# ----------------------------------------------------------------------------------------------
def _rand_qk(L, Hq, Hkv, d, n, w, seed):
    rng = np.random.default_rng(seed)
    K = rng.standard_normal((L, n, Hkv, d)).astype(np.float16)
    Q = rng.standard_normal((L, Hq, w, d)).astype(np.float16)
    return K, Q


@pytest.mark.parametrize("causal", [True, False])
def test_importance_sums_to_one(causal):
    K, Q = _rand_qk(2, 4, 2, 64, 90, 7, 11)
    I = oracle.importance(K, Q, causal=causal, lam=0.0)
    assert I.shape == (2, 90) and (I >= 0).all()
    assert np.allclose(I.astype(np.float64).sum(axis=1), 1.0, atol=1e-6)


def test_importance_zero_keys_closed_forms():
    L, Hq, Hkv, d, n, w = 1, 2, 1, 64, 40, 8
    K = np.zeros((L, n, Hkv, d), np.float16)
    Q = np.random.default_rng(0).standard_normal((L, Hq, w, d)).astype(np.float16)
    I = oracle.importance(K, Q, causal=False)
    assert np.allclose(I, 1.0 / n, rtol=1e-6)
    I = oracle.importance(K, Q, causal=True)
    pos = np.arange(n - w, n)
    want = np.array([(1.0 / (pos[pos >= j] + 1)).sum() / w for j in range(n)])
    assert np.allclose(I[0], want, rtol=1e-6)


def test_importance_dominant_key_and_gqa_mapping():
    # KV head g serves query heads [g*G, (g+1)*G) (integer division, HF repeat_kv convention).
    L, Hq, Hkv, d, n, w = 1, 4, 2, 64, 50, 4
    K = np.zeros((L, n, Hkv, d), np.float16)
    Q = np.zeros((L, Hq, w, d), np.float16)
    Q[..., 0] = 8.0
    K[0, 10, 0, 0] = 30.0           # KV head 0: key 10 dominates  (logit 8*30/8 = 30)
    K[0, 20, 1, 0] = 30.0           # KV head 1: key 20 dominates
    I = oracle.importance(K, Q, causal=True)
    assert abs(I[0, 10] - 0.5) < 1e-6 and abs(I[0, 20] - 0.5) < 1e-6
    Q[0, 2:, :, 0] = 0.0            # query heads 2,3 (-> KV head 1) become uniform
    I = oracle.importance(K, Q, causal=False)
    assert abs(I[0, 10] - (0.5 + 0.5 / n)) < 1e-4 and abs(I[0, 20] - 0.5 / n) < 1e-4


def test_importance_decay_closed_form():
    K, Q = _rand_qk(1, 2, 1, 64, 120, 5, 12)
    I0 = oracle.importance(K, Q, lam=0.0).astype(np.float64)
    for lam in (0.001, 0.005, 0.010):                       # the values the paper prints (Table 15)
        I = oracle.importance(K, Q, lam=lam).astype(np.float64)
        ratio = I[0] / I0[0]
        want = np.exp(-lam * (120 - 1 - np.arange(120)))    # newest token: Delta = 0
        assert np.allclose(ratio, want, rtol=1e-5)
    assert abs(ratio[-1] - 1.0) < 1e-6


@pytest.mark.parametrize("causal", [True, False])
def test_importance_matches_textbook_softmax(causal):
    L, Hq, Hkv, d, n, w = 2, 6, 2, 128, 150, 9
    K, Q = _rand_qk(L, Hq, Hkv, d, n, w, 13)
    I = oracle.importance(K, Q, causal=causal)
    Kt = torch.from_numpy(K).double().permute(0, 2, 1, 3)              # [L][Hkv][n][d]
    Kt = Kt.repeat_interleave(Hq // Hkv, dim=1)                        # repeat_kv
    Qt = torch.from_numpy(Q).double()                                  # [L][Hq][w][d]
    z = torch.matmul(Qt, Kt.transpose(-1, -2)) / d ** 0.5              # [L][Hq][w][n]
    if causal:
        pos = torch.arange(n - w, n)[:, None]
        z = z.masked_fill(torch.arange(n)[None, :] > pos, float("-inf"))
    A = torch.softmax(z, dim=-1).mean(dim=(1, 2))
    assert np.allclose(I, A.numpy(), rtol=1e-6, atol=1e-12)


def _kvnorm_golden(golden_dir):
    rows = read_golden(os.path.join(golden_dir, "kvnorm_worked.txt"))
    keys = [r for r in rows if r[0] == "key"]
    n, Hkv, d = 1 + max(int(r[1]) for r in keys), 1 + max(int(r[2]) for r in keys), 4
    K = np.zeros((1, n, Hkv, d), np.float16)
    norms = np.zeros((n, Hkv))
    for r in keys:
        K[0, int(r[1]), int(r[2])] = [float(x) for x in r[3:7]]
        norms[int(r[1]), int(r[2])] = float(r[7])
    scores = {}
    for r in rows:
        if r[0] == "score":
            scores.setdefault(r[1], {})[int(r[2])] = float(r[3])
    return K, norms, scores


def test_kvnorm_hand_worked_example(golden_dir):
    """tests/golden/kvnorm_worked.txt: Pythagorean key vectors whose norms are integers, scores worked by hand for
    lambda = 0, ln 2 (decay factors 1/8, 1/4, 1/2, 1) and 0.005 (Eq. 13)."""
    K, norms, scores = _kvnorm_golden(golden_dir)
    # the fixture's own norms are integers a reader can check: sum of squares of each row
    assert np.array_equal((K.astype(np.float64) ** 2).sum(axis=-1)[0], norms ** 2)
    for name, lam in (("0", 0.0), ("ln2", math.log(2.0)), ("0.005", 0.005)):
        I = oracle.importance_kvnorm(K, lam=lam)[0].astype(np.float64)
        want = np.array([scores[name][j] for j in range(K.shape[1])])
        assert np.all(np.abs(I - want) <= 1e-7 * want), (name, I, want)          # float32 output: half an ulp = 6e-8
        assert I[1] == 0.0                                                       # the zero token


def test_kvnorm_scaling_permutation_and_normalisation_properties():
    """Properties the definition fixes (no formula retyped): scaling one token's keys by c scales its UNNORMALISED
    score by c (so every ratio to another token's score scales by c); permuting the KV heads or the elements inside a
    head vector changes nothing; an all-zero layer falls back to the uniform 1/n; scores sum to 1 at lambda = 0."""
    rng = np.random.default_rng(14)
    L, n, Hkv, d = 2, 33, 3, 64
    K = rng.standard_normal((L, n, Hkv, d)).astype(np.float16)
    I0 = oracle.importance_kvnorm(K).astype(np.float64)
    assert np.allclose(I0.sum(axis=1), 1.0, atol=1e-6)
    t, c = 7, 4.0                                                                # power of two: exact in fp16
    K2 = K.copy(); K2[:, t] *= np.float16(c)
    I2 = oracle.importance_kvnorm(K2).astype(np.float64)
    others = np.array([j for j in range(n) if j != t])
    assert np.allclose(I2[:, t:t + 1] / I2[:, others], c * I0[:, t:t + 1] / I0[:, others], rtol=1e-5)
    assert np.allclose(I2[:, others] / I2[:, others[:1]], I0[:, others] / I0[:, others[:1]], rtol=1e-5)
    Kp = K[:, :, ::-1, :][:, :, :, rng.permutation(d)].copy()
    assert np.allclose(oracle.importance_kvnorm(Kp), I0, rtol=2e-6)
    Z = np.zeros((1, 5, 2, 64), np.float16)
    assert np.allclose(oracle.importance_kvnorm(Z), 0.2, rtol=1e-7)
    # decay closed form on top of any scores: I_j(lambda) / I_j(0) = exp(-lambda (n-1-j))
    lam = 0.01
    Il = oracle.importance_kvnorm(K, lam=lam).astype(np.float64)
    assert np.allclose(Il / I0, np.exp(-lam * (n - 1 - np.arange(n)))[None, :], rtol=1e-6)


# ----------------------------------------------------------------------------------------------
# NEXT-3 cold-tier precision upgrade
# ----------------------------------------------------------------------------------------------
def test_upgrade_patch_restores_exact_rows_and_touches_nothing_else():
    """Pins that need no implementation: (i) an upgraded token's K/V rows equal the original FP16 rows bit for bit,
    (ii) every other row and tier entry is untouched, (iii) upgrading every non-FP16 token reaches the b = 1 identity
    in two hops, (iv) the upgrade payload is 2 B per element (Eq. 1 restricted to the upgraded tokens)."""
    L, n, Hkv, d = 3, 200, 2, 64
    rng = np.random.default_rng(5)
    K = rng.standard_normal((L, n, Hkv, d)).astype(np.float16)
    V = rng.standard_normal((L, n, Hkv, d)).astype(np.float16)
    counts, prot = oracle.tier_counts(n, 0.3, 4, [], True)
    I = rng.random((L, n)).astype(np.float32)
    tier = oracle.assign(I, prot, counts)
    K1, V1, t1 = oracle.unpack(oracle.pack(K, V, tier, counts, True), L, Hkv, d, n)
    # upgrade the k highest-scored INT4 tokens of every layer to FP16
    k = 17
    up = np.zeros((L, n), np.uint8)
    for l in range(L):
        cand = np.flatnonzero(tier[l] == 4)
        up[l, cand[np.argsort(-I[l, cand], kind="stable")[:k]]] = 16
    uc = oracle.Counts(k, 0, 0, n - k, 4 * k, 4 * k)
    ublob = oracle.pack(K, V, up, uc, True)
    payload = 2 * L * k * Hkv * d * 2
    assert payload <= ublob.size <= payload + 256 + (L * n + 255) // 256 * 256 + L * 10 * 256     # 2 B/elem + framing
    K2, V2, t2 = oracle.unpack_patch(ublob, K1, V1, t1)
    m = up == 16
    assert np.array_equal(K2[m].view(np.uint16), K[m].view(np.uint16)) and np.array_equal(V2[m].view(np.uint16), V[m].view(np.uint16))
    assert np.array_equal(K2[~m].view(np.uint16), K1[~m].view(np.uint16)) and np.array_equal(V2[~m].view(np.uint16), V1[~m].view(np.uint16))
    assert (t2[m] == 16).all() and np.array_equal(t2[~m], t1[~m])
    assert not np.array_equal(K2[m].view(np.uint16), K1[m].view(np.uint16))                  # the INT4 rows really differed
    # upgrade everything that is not FP16 yet -> identity
    up_all = np.where(tier != 16, 16, 0).astype(np.uint8)
    k_all = int((up_all[0] == 16).sum())
    ac = oracle.Counts(k_all, 0, 0, n - k_all, 4 * k_all, 4 * k_all)
    K3, V3, t3 = oracle.unpack_patch(oracle.pack(K, V, up_all, ac, True), K1, V1, t1)
    assert np.array_equal(K3.view(np.uint16), K.view(np.uint16)) and np.array_equal(V3.view(np.uint16), V.view(np.uint16))
    assert (t3 == 16).all()


# ----------------------------------------------------------------------------------------------
# NEXT-4: asymmetric 2-bit low tier
# ----------------------------------------------------------------------------------------------
def test_quantizer2_worked_examples_and_special_cases():
    rows = read_golden(os.path.join(GOLD, "quantizer2_worked.txt"))
    groups = {}
    for name, x, code, ybits in rows:
        groups.setdefault(name, []).append((float(x), int(code), int(ybits, 16)))
    assert len(groups) == 3
    for name, items in groups.items():
        xs = [it[0] for it in items]
        v = np.full(64, min(xs), np.float16)
        v[:len(items)] = xs
        lo, hi, q = oracle.quantize2_vector(v)
        assert lo == int(np.float16(min(xs)).view(np.uint16)) and hi == int(np.float16(max(xs)).view(np.uint16)), name
        assert q[:len(items)].tolist() == [it[1] for it in items], name
        assert (q[len(items):] == 0).all()
        y = oracle.dequantize2_vector(q, lo, hi)
        assert y[:len(items)].view(np.uint16).tolist() == [it[2] for it in items], name
    # constant vector: r = 0 -> codes 0, reconstruction exact; signed zeros are recorded as +0
    c = np.full(64, -3.5, np.float16)
    lo, hi, q = oracle.quantize2_vector(c)
    assert lo == hi == int(np.float16(-3.5).view(np.uint16)) and (q == 0).all()
    assert np.array_equal(oracle.dequantize2_vector(q, lo, hi), c)
    z = np.zeros(64, np.float16); z[5] = -0.0
    lo, hi, q = oracle.quantize2_vector(z)
    assert lo == 0 and hi == 0 and (oracle.dequantize2_vector(q, lo, hi).view(np.uint16) == 0).all()
    big = np.full(64, -65504.0, np.float16); big[1] = 65504.0
    lo, hi, q = oracle.quantize2_vector(big)
    assert q[0] == 0 and q[1] == 3
    assert np.array_equal(oracle.dequantize2_vector(q, lo, hi), big)            # no overflow at the fp16 extremes


def test_quantizer2_codes_are_exactly_rounded_and_error_is_half_a_step():
    from fractions import Fraction
    import math
    rng = np.random.default_rng(12)
    for _ in range(40):
        v = (rng.standard_normal(128) * rng.uniform(0.01, 30) + rng.uniform(-5, 5)).astype(np.float16)
        lo_b, hi_b, q = oracle.quantize2_vector(v)
        lo = np.float32(np.uint16(lo_b).view(np.float16)); hi = np.float32(np.uint16(hi_b).view(np.float16))
        assert float(lo) == float(v.min()) and float(hi) == float(v.max())
        r = np.float32(hi - lo)
        inv = np.float32(3.0) / r
        for e, code in zip(v, q):
            dx = np.float32(np.float32(e) - lo)
            ex = Fraction(float(dx)) * Fraction(float(inv))
            fl = math.floor(ex); fr = ex - fl
            want = fl if fr < Fraction(1, 2) else fl + 1 if fr > Fraction(1, 2) else (fl if fl % 2 == 0 else fl + 1)
            assert int(code) == max(0, min(3, want))
        assert q.min() == 0 and q.max() == 3                                      # the extremes hit codes 0 and 3
        step = float(r) / 3.0
        y = oracle.dequantize2_vector(q, lo_b, hi_b).astype(np.float64)
        ulp = np.spacing(np.abs(y).astype(np.float16)).astype(np.float64)
        assert (np.abs(y - v.astype(np.float64)) <= step / 2 * (1 + 1e-3) + ulp / 2 + 1e-12).all()


def test_tier_counts_two_bit_low_tier():
    # c(2-bit) = 1/8: b = 1/8 -> everything 2-bit; b = 0.5 -> everything INT8; b = 5/16 -> half and half; b = 1 -> FP16
    for b, want in ((0.125, (0, 0, 1000, 0)), (0.5, (0, 1000, 0, 0)), (0.3125, (0, 500, 500, 0)), (1.0, (1000, 0, 0, 0)),
                    (0.75, (500, 500, 0, 0)), (0.0625, (0, 0, 500, 500))):
        c, _ = oracle.tier_counts(1000, b, 0, [], 2)
        assert (c.n16, c.n8, c.n4, c.n0) == want and c.low_bits == 2, (b, c)
    rng = np.random.default_rng(2)
    for _ in range(300):
        n = int(rng.integers(8, 5000)); s = int(rng.integers(0, 5)); b = float(rng.uniform(0.02, 1.0))
        try:
            c, prot = oracle.tier_counts(n, b, s, [], 2)
        except ValueError:
            assert 8 * s > int(np.floor(8 * b * n + 1e-6))
            continue
        assert c.n16 + c.n8 + c.n4 + c.n0 == n and c.n16 >= s
        assert c.spent_q4 == 8 * c.n16 + 4 * c.n8 + c.n4 <= c.budget_q4 == int(np.floor(8 * b * n + 1e-6))
        if c.n16 < n:
            assert c.budget_q4 - c.spent_q4 < 4                                   # less than the cheapest upgrade left over
        assert sum(x > 0 for x in (c.n16 - int(prot.sum()), c.n8, c.n4, c.n0)) <= 2   # two adjacent tiers at most


def test_two_bit_blob_layout_round_trip_and_hand_written_bytes():
    L, n, Hkv, d = 1, 3, 1, 64
    rows = [r for r in read_golden(os.path.join(GOLD, "quantizer2_worked.txt")) if r[0] == "Z1"]
    K = np.zeros((L, n, Hkv, d), np.float16); V = np.zeros((L, n, Hkv, d), np.float16)
    K[0, 0, 0, :] = np.arange(64) / 4.0                       # FP16 token
    K[0, 1, 0, :] = -1.0; K[0, 1, 0, :len(rows)] = [float(r[1]) for r in rows]          # 2-bit token, Z1 vector
    V[0, 1, 0, :] = 0.0; V[0, 1, 0, :2] = [0.75, 0.375]                                # Z2: codes 3, 2, 0, 0 ...
    K[0, 2] = 5.0; V[0, 2] = -5.0                             # dropped
    tier = np.array([[16, 2, 0]], np.uint8)
    counts = oracle.Counts(1, 0, 1, 1, 9, 9, low_bits=2)
    blob = oracle.pack(K, V, tier, counts, 2)
    assert int.from_bytes(bytes(blob[40:44]), "little") == 3                          # flags: low tier allowed, 2-bit
    seg = [int.from_bytes(bytes(blob[80 + 8 * i:88 + 8 * i]), "little") for i in range(10)]
    # raw sizes: K16,V16 128; K8,V8 0; K2,V2 16 (64 codes / 4); SK8,SV8 0; SK2,SV2 4 -> offsets step by 256 where non-empty
    assert seg == [0, 256, 512, 512, 512, 768, 1024, 1024, 1024, 1280]
    base = 256 + 256
    codes = [int(r[2]) for r in rows] + [0] * (64 - len(rows))
    want_k = bytes((codes[4 * i] | codes[4 * i + 1] << 2 | codes[4 * i + 2] << 4 | codes[4 * i + 3] << 6) for i in range(16))
    assert bytes(blob[base + 512:base + 528]) == want_k
    assert bytes(blob[base + 768:base + 784]) == bytes([3 | 2 << 2]) + bytes(15)
    assert bytes(blob[base + 1024:base + 1028]) == bytes([0x00, 0xBC, 0x00, 0x40])    # lo = -1 (0xBC00), hi = 2 (0x4000)
    assert bytes(blob[base + 1280:base + 1284]) == bytes([0x00, 0x00, 0x00, 0x3A])    # lo = 0, hi = 0.75 (0x3A00)
    K2, V2, t2 = oracle.unpack(blob, L, Hkv, d, n)
    assert np.array_equal(t2, tier) and np.array_equal(K2[0, 0], K[0, 0]) and (K2[0, 2] == 0).all()
    assert K2[0, 1, 0, :len(rows)].view(np.uint16).tolist() == [int(r[3], 16) for r in rows]
    assert V2[0, 1, 0, :3].tolist() == [0.75, 0.5, 0.0]


# ----------------------------------------------------------------------------------------------
# NEXT-4: bfloat16 caches (reading P20)
# ----------------------------------------------------------------------------------------------
def _bf16_bits(t):
    import torch
    return t.to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)


def test_bf16_conversions_against_torch():
    import torch
    allbits = np.arange(65536, dtype=np.uint16)
    f = oracle.bf16_to_float(allbits)
    want = torch.from_numpy(allbits.view(np.int16)).view(torch.bfloat16).float().numpy()
    fin = np.isfinite(want)
    assert np.array_equal(f[fin].view(np.uint32), want[fin].view(np.uint32))            # exhaustive, exact
    rng = np.random.default_rng(7)
    x = np.concatenate([rng.standard_normal(4000) * 10.0 ** rng.uniform(-30, 30, 4000),
                        oracle.bf16_to_float(rng.integers(0, 0x7F00, 2000).astype(np.uint16)) * (1 + 2.0 ** -9),   # near ties
                        [0.0, -0.0, 1.0, 3.3895313892515355e38]]).astype(np.float32)
    got = oracle.float_to_bf16(x)
    assert np.array_equal(got, _bf16_bits(torch.from_numpy(x)))                           # RNE, as torch rounds


def test_bf16_quantizer_identities_and_error_bound():
    from fractions import Fraction
    import torch
    rng = np.random.default_rng(13)
    for qmax in (127, 7):
        for _ in range(25):
            xb = _bf16_bits(torch.from_numpy((rng.standard_normal(128) * rng.uniform(1e-3, 100)).astype(np.float32)))
            x = oracle.bf16_to_float(xb).astype(np.float64)
            ab, q = oracle.quantize_vector(xb, qmax, bf16=True)
            amax = float(oracle.bf16_to_float(np.uint16(ab)))
            assert amax == np.abs(x).max() and np.abs(q).max() == qmax
            inv = np.float32(qmax) / np.float32(amax)
            for e, code in zip(x[:32], q[:32]):                                           # exact rational rounding
                assert int(code) == _exact_code(np.float32(e), inv, qmax)
            scale = amax / qmax
            assert np.abs(q * scale - x).max() <= scale / 2 * (1 + 1e-4)
            y = oracle.bf16_to_float(oracle.dequantize_vector(q, qmax, ab, bf16=True)).astype(np.float64)
            assert (np.abs(y - x) <= scale / 2 * (1 + 1e-4) + np.abs(y) * 2.0 ** -8 + 1e-30).all()
    # P20: an amax so small that qmax/amax overflows binary32 -> all codes 0, record kept
    tiny = np.full(64, 0x0001, np.uint16)                                                 # smallest bf16 subnormal, 9.2e-41
    ab, q = oracle.quantize_vector(tiny, 127, bf16=True)
    assert ab == 1 and (q == 0).all()
    # 2-bit on bf16: extremes hit 0 and 3, constant vector exact
    xb = _bf16_bits(torch.from_numpy(rng.standard_normal(64).astype(np.float32)))
    lo, hi, q2 = oracle.quantize2_vector(xb, bf16=True)
    x = oracle.bf16_to_float(xb)
    assert float(oracle.bf16_to_float(np.uint16(lo))) == x.min() and float(oracle.bf16_to_float(np.uint16(hi))) == x.max()
    assert q2.min() == 0 and q2.max() == 3
    y = oracle.bf16_to_float(oracle.dequantize2_vector(q2, lo, hi, bf16=True)).astype(np.float64)
    step = (float(x.max()) - float(x.min())) / 3
    assert (np.abs(y - x.astype(np.float64)) <= step / 2 * (1 + 1e-3) + np.abs(y) * 2.0 ** -8).all()
    # P20, the other end: finite bf16 elements more than FLT_MAX apart (hi - lo = +Inf in binary32).  Fixed by hand:
    # inv = 3 / Inf = 0 -> every code 0; step is taken as 0 -> every element decodes to lo; nothing is NaN or Inf.
    big = float(oracle.bf16_to_float(np.uint16(0x7F62)))                                  # 3.0e38 as bf16 (finite, < FLT_MAX)
    assert 2.9e38 < big < 3.1e38
    wide = np.array([0x7F62, 0xFF62] + [0x3F80] * 30, np.uint16)                          # +3e38, -3e38, 1.0 ...
    lo, hi, q2 = oracle.quantize2_vector(wide, bf16=True)
    assert lo == 0xFF62 and hi == 0x7F62 and (q2 == 0).all()
    y = oracle.dequantize2_vector(q2, lo, hi, bf16=True)
    assert (y == 0xFF62).all()
    # one binade lower the range is finite again and the rule does not apply: extremes hit codes 0 and 3 and round-trip
    half = np.array([0x7EE2, 0xFEE2] + [0x3F80] * 30, np.uint16)                          # +-1.5e38: range 3e38 is finite
    lo, hi, q2 = oracle.quantize2_vector(half, bf16=True)
    assert q2[0] == 3 and q2[1] == 0
    y = oracle.dequantize2_vector(q2, lo, hi, bf16=True)
    assert y[0] == 0x7EE2 and y[1] == 0xFEE2


def test_bf16_blob_round_trip_and_fp16_tier_is_a_copy():
    import torch
    L, n, Hkv, d = 2, 40, 2, 64
    rng = np.random.default_rng(14)
    K = _bf16_bits(torch.from_numpy(rng.standard_normal((L, n, Hkv, d)).astype(np.float32)))
    V = _bf16_bits(torch.from_numpy(rng.standard_normal((L, n, Hkv, d)).astype(np.float32)))
    c, prot = oracle.tier_counts(n, 0.4, 2, [], True)
    tier = oracle.assign(rng.random((L, n)).astype(np.float32), prot, c)
    blob = oracle.pack(K, V, tier, c, True, bf16=True)
    assert blob[40] == 5                                                                  # flags: low tier allowed | bf16
    assert blob.size == oracle.blob_bytes(L, Hkv, d, n, c)                                 # same byte model as FP16 (2 B)
    K2, V2, t2 = oracle.unpack(blob, L, Hkv, d, n, bf16=True)
    assert np.array_equal(t2, tier) and np.array_equal(K2[tier == 16], K[tier == 16])
    for l, j in ((0, 5), (1, 17), (1, 39)):
        for h in range(Hkv):
            t = int(tier[l, j])
            if t in (8, 4):
                ab, q = oracle.quantize_vector(K[l, j, h], 127 if t == 8 else 7, bf16=True)
                assert np.array_equal(K2[l, j, h], oracle.dequantize_vector(q, 127 if t == 8 else 7, ab, bf16=True))
    c1, _ = oracle.tier_counts(n, 1.0, 0, [], True)
    b1 = oracle.pack(K, V, np.full((L, n), 16, np.uint8), c1, True, bf16=True)
    K3, V3, _ = oracle.unpack(b1, L, Hkv, d, n, bf16=True)
    assert np.array_equal(K3, K) and np.array_equal(V3, V)                                 # b = 1 identity


# ----------------------------------------------------------------------------------------------
# NEXT-4: INT8 hot tier (reading P21)
# ----------------------------------------------------------------------------------------------
def test_hot_int8_counts_golden_and_invariants():
    for n, b, s, rb, re_, a4, n16, n8, n4, n0 in read_golden(os.path.join(GOLD, "hot_int8_counts.txt")):
        ranges = [] if int(rb) == int(re_) else [(int(rb), int(re_))]
        a = int(a4)
        c, prot = oracle.tier_counts(int(n), float(b), int(s), ranges, a if a == 2 else bool(a), mode=oracle.MODE_HOT_INT8)
        assert (c.n16, c.n8, c.n4, c.n0) == (int(n16), int(n8), int(n4), int(n0)), (n, b, s, a4, c)
    rng = np.random.default_rng(21)
    for _ in range(2000):
        n = int(rng.integers(1, 5000)); s = int(rng.integers(0, min(n, 9))); b = float(rng.uniform(0.01, 1.2))
        a4 = [False, True, 2][int(rng.integers(0, 3))]
        unit = 8 if a4 == 2 else 4
        try:
            c, prot = oracle.tier_counts(n, b, s, [], a4, mode=oracle.MODE_HOT_INT8)
        except ValueError:
            assert (unit // 2) * s > int(np.floor(unit * min(b, 1.0) * n + 1e-6))       # the INT8 sinks alone do not fit
            continue
        P = int(prot.sum())
        assert c.n16 == 0 and c.n8 >= P and c.n16 + c.n8 + c.n4 + c.n0 == n
        assert c.budget_q4 == int(np.floor(unit * min(b, 1.0) * n + 1e-6))
        assert c.spent_q4 == (unit // 2) * c.n8 + c.n4 <= c.budget_q4
        if c.n8 < n:
            assert c.budget_q4 - c.spent_q4 < max(1, unit // 2 - 1) or (not a4 and c.budget_q4 - c.spent_q4 < unit // 2)
        if not a4:
            assert c.n4 == 0
        assert sum(x > 0 for x in (c.n8 - P, c.n4, c.n0)) <= 2                           # two adjacent tiers at most
        # s = 0 and b <= 1/2: identical to the default ladder (Eq. 14 has no FP16 term there)
        if s == 0 and b <= 0.5:
            d, _ = oracle.tier_counts(n, b, 0, [], a4)
            assert (d.n16, d.n8, d.n4, d.n0) == (c.n16, c.n8, c.n4, c.n0)


def test_hot_int8_selection_brute_force_and_pinned_positions():
    rng = np.random.default_rng(22)
    for n, b, s, ranges, a4 in ((97, 0.3, 3, [(40, 47)], True), (200, 0.2, 4, [], True), (64, 0.4, 2, [(10, 12)], False),
                                (130, 0.22, 5, [(100, 130)], 2)):
        c, prot = oracle.tier_counts(n, b, s, ranges, a4, mode=oracle.MODE_HOT_INT8)
        I = rng.random((2, n)).astype(np.float32)
        I[0, :s] = 0.0                                                  # sinks with the lowest score still ship INT8
        I[1, 7::9] = I[1, 5]                                            # ties
        tier = oracle.assign(I, prot, c)
        low = 2 if a4 == 2 else 4
        for l in range(2):
            free = np.flatnonzero(prot == 0)
            key = np.where(I[l] > 0, I[l], 0.0)
            rank = {int(j): sum(1 for k in free if key[k] > key[j] or (key[k] == key[j] and k < j)) for j in free}
            P = int(prot.sum())
            for j in range(n):
                if prot[j]:
                    want = 8
                else:
                    r = rank[j]
                    want = 8 if r < c.n8 - P else low if r < c.n8 - P + c.n4 else 0
                assert tier[l, j] == want, (n, l, j)
            assert (tier[l] == 16).sum() == 0 and (tier[l] == 8).sum() == c.n8 and (tier[l] == low).sum() == c.n4


def test_hot_int8_blob_has_no_fp16_segment_and_round_trips():
    L, n, Hkv, d = 2, 40, 2, 64
    rng = np.random.default_rng(23)
    K = (rng.standard_normal((L, n, Hkv, d)) * 3).astype(np.float16); V = rng.standard_normal((L, n, Hkv, d)).astype(np.float16)
    c, prot = oracle.tier_counts(n, 0.35, 4, [], True, mode=oracle.MODE_HOT_INT8)
    tier = oracle.assign(rng.random((L, n)).astype(np.float32), prot, c)
    assert (tier[:, :4] == 8).all()
    blob = oracle.pack(K, V, tier, c, True)
    assert int.from_bytes(bytes(blob[40:44]), "little") == 1 | 8                      # low tier allowed + INT8 hot tier
    assert int.from_bytes(bytes(blob[24:28]), "little") == 0                          # n16
    seg = [int.from_bytes(bytes(blob[80 + 8 * i:88 + 8 * i]), "little") for i in range(10)]
    assert seg[0] == seg[1] == seg[2] == 0                                            # K16 and V16 occupy no bytes
    # payload identity (Eq. 3 with c(8) = 1/2, c(4) = 1/4): code bytes = Bytes_FP16 * spent / (4 n)
    code_bytes = 2 * L * Hkv * d * (c.n8 + c.n4 // 2 + (c.n4 % 2) * 0.5)
    assert code_bytes == 2 * L * Hkv * d * n * 2 * c.spent_q4 / (4 * n)
    K2, V2, t2 = oracle.unpack(blob, L, Hkv, d, n)
    assert np.array_equal(t2, tier)
    for l in range(L):
        for j in range(n):
            qm = {8: 127, 4: 7}.get(int(tier[l, j]))
            for h in range(Hkv):
                if qm is None:
                    assert (K2[l, j, h] == 0).all()
                else:
                    ab, q = oracle.quantize_vector(K[l, j, h], qm)
                    assert np.array_equal(K2[l, j, h].view(np.uint16), oracle.dequantize_vector(q, qm, ab).view(np.uint16))
    # a blob that claims the INT8 hot tier but carries FP16 tokens is refused
    bad = blob.copy(); bad[24] = 1; bad[28] -= 1
    with pytest.raises(ValueError):
        oracle.unpack(bad, L, Hkv, d, n)


# ----------------------------------------------------------------------------------------------
# NEXT-4: group-wise 2-bit low tier (reading P22)
# ----------------------------------------------------------------------------------------------
def test_group2_hand_worked_blob_and_what_grouping_buys():
    rows = {r[0]: r for r in read_golden(os.path.join(GOLD, "group2_worked.txt"))}
    L, n, Hkv, d = 1, 1, 1, 64
    K = np.zeros((L, n, Hkv, d), np.float16)
    K[0, 0, 0, :32] = np.tile([float(v) for v in rows["G0"][1:5]], 8)
    K[0, 0, 0, 32:] = np.tile([float(v) for v in rows["G1"][1:5]], 8)
    V = K[..., ::-1].copy()                                                           # groups swapped and reversed
    tier = np.array([[2]], np.uint8)
    cg = oracle.Counts(0, 0, 1, 0, 1, 1, low_bits=2, mode=oracle.MODE_GROUP2)
    blob = oracle.pack(K, V, tier, cg, 2)
    assert int.from_bytes(bytes(blob[40:44]), "little") == 1 | 2 | 16
    seg = [int.from_bytes(bytes(blob[80 + 8 * i:88 + 8 * i]), "little") for i in range(10)]
    # raw sizes: K2,V2 16 bytes of codes; SK2,SV2 two groups x 4 bytes = 8
    assert seg == [0, 0, 0, 0, 0, 256, 512, 512, 512, 768]
    base = 256 + 256
    assert bytes(blob[base:base + 16]) == bytes([int(rows["G0"][7], 16)] * 8 + [int(rows["G1"][7], 16)] * 8)
    rec = bytes(blob[base + 512:base + 520])
    want = b"".join(int(rows[g][k], 16).to_bytes(2, "little") for g in ("G0", "G1") for k in (5, 6))
    assert rec == want
    # V: reversed pattern 6 2 -2 -6 | 3 2 1 0 -> codes 3 2 1 0 in both groups: 0b00011011 = 0x1B; records swapped
    assert bytes(blob[base + 256:base + 272]) == bytes([0x1B] * 16)
    assert bytes(blob[base + 768:base + 776]) == want[4:] + want[:4]
    K2, V2, t2 = oracle.unpack(blob, L, Hkv, d, n)
    assert np.array_equal(K2, K) and np.array_equal(V2, V)                            # every value sits on its group's grid
    # the same vector without grouping: one (lo, hi) = (-6, 6) for all 64 values, group 0 collapses to the code of 2
    cw = oracle.Counts(0, 0, 1, 0, 1, 1, low_bits=2)
    blobw = oracle.pack(K, V, tier, cw, 2)
    assert bytes(blobw[base:base + 8]) == bytes([int(rows["W"][7], 16)] * 8)
    Kw, _, _ = oracle.unpack(blobw, L, Hkv, d, n)
    assert (Kw[0, 0, 0, :32] == 2.0).all() and np.array_equal(Kw[0, 0, 0, 32:], K[0, 0, 0, 32:])


def test_group2_layout_closed_form_error_bound_and_reduction_to_the_ungrouped_quantiser():
    rng = np.random.default_rng(24)
    pad = lambda x: (x + 255) // 256 * 256
    for L, n, Hkv, d, n8, n2 in ((1, 9, 2, 64, 3, 4), (2, 33, 4, 128, 0, 33), (1, 17, 8, 256, 5, 7)):
        cg = oracle.Counts(0, n8, n2, n - n8 - n2, 4 * n8 + n2, 4 * n8 + n2, low_bits=2, mode=oracle.MODE_GROUP2)
        cw = oracle.Counts(0, n8, n2, n - n8 - n2, 4 * n8 + n2, 4 * n8 + n2, low_bits=2)
        # only the record segments differ: d/32 (lo, hi) pairs per head vector instead of one
        diff = L * 2 * (pad(n2 * Hkv * (d // 32) * 4) - pad(n2 * Hkv * 4))
        assert oracle.blob_bytes(L, Hkv, d, n, cg) - oracle.blob_bytes(L, Hkv, d, n, cw) == diff
        K = (rng.standard_normal((L, n, Hkv, d)) * rng.uniform(0.1, 20, (L, n, Hkv, 1))).astype(np.float16)
        K[..., 5] *= 10                                                               # an outlier channel in group 0
        V = rng.standard_normal((L, n, Hkv, d)).astype(np.float16)
        tier = np.zeros((L, n), np.uint8); tier[:, :n8] = 8; tier[:, n8:n8 + n2] = 2
        blob = oracle.pack(K, V, tier, cg, 2)
        K2, V2, t2 = oracle.unpack(blob, L, Hkv, d, n)
        assert np.array_equal(t2, tier)
        X = K[:, n8:n8 + n2].astype(np.float64).reshape(L, n2, Hkv, d // 32, 32)
        Y = K2[:, n8:n8 + n2].astype(np.float64).reshape(L, n2, Hkv, d // 32, 32)
        step = (X.max(-1, keepdims=True) - X.min(-1, keepdims=True)) / 3.0               # per GROUP, from the definition
        ulp = np.spacing(np.abs(Y).astype(np.float16)).astype(np.float64)
        assert (np.abs(Y - X) <= step / 2 * (1 + 1e-3) + ulp / 2 + 1e-12).all()
        # groups without the outlier are coded on their own, finer grid: their error is far below the ungrouped one
        Kw, _, _ = oracle.unpack(oracle.pack(K, V, tier, cw, 2), L, Hkv, d, n)
        eg = np.abs(Y - X)[..., 1:, :].mean(); ew = np.abs(Kw[:, n8:n8 + n2].astype(np.float64).reshape(X.shape) - X)[..., 1:, :].mean()
        assert eg < 0.6 * ew
    # special case that reduces to the ungrouped quantiser: every group of a vector spans the same (min, max)
    L, n, Hkv, d = 1, 4, 2, 128
    g = (rng.standard_normal((L, n, Hkv, 1, 32)) * 2).astype(np.float16)
    K = np.tile(g, (1, 1, 1, d // 32, 1)).reshape(L, n, Hkv, d)
    K = np.take_along_axis(K.reshape(L, n, Hkv, d // 32, 32), rng.permuted(np.tile(np.arange(32), (L, n, Hkv, d // 32, 1)), axis=-1), -1).reshape(L, n, Hkv, d)
    tier = np.full((L, n), 2, np.uint8)
    cg = oracle.Counts(0, 0, n, 0, n, n, low_bits=2, mode=oracle.MODE_GROUP2)
    cw = oracle.Counts(0, 0, n, 0, n, n, low_bits=2)
    bg, bw = oracle.pack(K, K, tier, cg, 2), oracle.pack(K, K, tier, cw, 2)
    lay = lambda b: [int.from_bytes(bytes(b[80 + 8 * i:88 + 8 * i]), "little") for i in range(10)]
    base = int.from_bytes(bytes(bg[64:72]), "little")
    ncode = n * Hkv * d // 4
    assert bytes(bg[base + lay(bg)[4]:base + lay(bg)[4] + ncode]) == bytes(bw[base + lay(bw)[4]:base + lay(bw)[4] + ncode])
    assert np.array_equal(oracle.unpack(bg, L, Hkv, d, n)[0], oracle.unpack(bw, L, Hkv, d, n)[0])
