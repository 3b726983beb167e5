"""Shared plumbing for the GPU parity tests: runs the oracle and the CUDA path on the same seeded inputs.
No arithmetic of the method lives here."""
import numpy as np
import torch

import oracle
import paper_2606_08635_b200 as skv
import skv_synth


def to_layout(x_tm, layout):
    """x_tm: torch [R][L][n][Hkv][d] token-major -> contiguous tensor in `layout` ("token_major" | "hf")."""
    if layout == "token_major":
        return x_tm.contiguous()
    return x_tm.permute(0, 1, 3, 2, 4).contiguous()      # [R][L][Hkv][n][d]


def from_layout(x, layout):
    if layout == "token_major":
        return x
    return x.permute(0, 1, 3, 2, 4).contiguous()


def near_tie_mask(I, tier, rel=2e-3):
    """P14: a token is a near-tie if its score is within rel of a tier threshold (the score of the last
    token admitted to a tier).  I, tier: numpy [L][n]."""
    mask = np.zeros(I.shape, bool)
    for l in range(I.shape[0]):
        for t in (16, 8, 4):
            sel = tier[l] == t
            if sel.any():
                T = I[l][sel].min()
                mask[l] |= np.abs(I[l] - T) <= rel * T + 1e-30
    return mask


class Case:
    """One (config, budget) problem: inputs on host (numpy, canonical token-major) and oracle results."""

    def __init__(self, cfg, b, requests=None, layers=None, with_importance=True, causal=True, lam=0.0,
                 importance_override=None, tier_mode=0):
        self.cfg, self.b, self.causal, self.lam = cfg, b, causal, lam
        self.tier_mode = tier_mode            # NEXT-4 flags: 1 = INT8 hot tier, 2 = group-wise 2-bit (same bits on both sides)
        R = cfg.R if requests is None else requests
        self.R = R
        Ks, Vs, Qs = [], [], []
        for r in range(R):
            K, V = skv_synth.make_kv(cfg, r, layers=layers)
            Ks.append(K); Vs.append(V)
            Qs.append(skv_synth.make_q(cfg, r, layers=layers))
        self.K = torch.stack(Ks); self.V = torch.stack(Vs); self.Q = torch.stack(Qs)   # [R][L][n][Hkv][d]
        self.L = self.K.shape[1]
        self.counts, self.prot = oracle.tier_counts(cfg.n, b, cfg.n_sink, cfg.ranges, cfg.allow_int4, mode=tier_mode)
        self.I, self.tier, self.blob, self.K2, self.V2 = [], [], [], [], []
        for r in range(R):
            if importance_override is not None:
                I = importance_override[r]
            elif with_importance:
                I = oracle.importance(self.K[r].numpy(), self.Q[r].numpy(), causal=causal, lam=lam)
            else:
                I = skv_synth.make_importance(cfg.scaled(L=self.L), r).numpy()
            tier = oracle.assign(I, self.prot, self.counts)
            blob = oracle.pack(self.K[r].numpy(), self.V[r].numpy(), tier, self.counts, cfg.allow_int4)
            K2, V2, t2 = oracle.unpack(blob, self.L, cfg.Hkv, cfg.d, cfg.n)
            assert np.array_equal(t2, tier)
            self.I.append(I); self.tier.append(tier); self.blob.append(blob); self.K2.append(K2); self.V2.append(V2)

    def shape(self, layout="token_major"):
        c = self.cfg
        return skv.make_shape(self.L, c.Hq, c.Hkv, c.d, c.n, self.R, layout=layout)

    def policy(self):
        c = self.cfg
        return skv.make_policy(self.b, c.n_sink, c.ranges, c.allow_int4, self.tier_mode)


def gpu_pipeline(case, layout="token_major", use_oracle_importance=True, run_importance=True):
    """Runs the CUDA path through the C ABI.  Returns dict of host numpy results."""
    dev = torch.device("cuda:0")
    cfg = case.cfg
    shape = case.shape(layout)
    pol = case.policy()
    Kd = to_layout(case.K, layout).to(dev)
    Vd = to_layout(case.V, layout).to(dev)
    Qd = case.Q.to(dev).contiguous()
    ws = torch.empty(skv.skv_workspace_bytes(shape, cfg.w), dtype=torch.uint8, device=dev)
    out = {}
    Igpu = torch.full((case.R, case.L, cfg.n), float("nan"), dtype=torch.float32, device=dev)
    if run_importance:
        skv.skv_importance(shape, Kd, Qd, cfg.w, Igpu, ws, causal=case.causal, lam=case.lam)
        out["I"] = Igpu.cpu().numpy()
    Iin = torch.from_numpy(np.stack(case.I)).to(dev) if use_oracle_importance else Igpu
    tier = torch.full((case.R, case.L, cfg.n), 0xEE, dtype=torch.uint8, device=dev)
    counts = skv.skv_assign_tiers(shape, pol, Iin, tier, ws)
    out["counts"] = counts
    out["tier"] = tier.cpu().numpy()
    bb = skv.skv_blob_bytes(shape, counts)
    blob = torch.full((case.R * bb,), 0xAB, dtype=torch.uint8, device=dev)     # poisoned: every byte must be written
    skv.skv_pack(shape, Kd, Vd, tier, counts, blob, ws)
    out["blob"] = blob.cpu().numpy().reshape(case.R, bb)
    # decode side: header check on the host copy, then unpack into a poisoned dense cache
    hs, hc = skv.skv_blob_check(out["blob"][0][:256].tobytes(), bb)
    assert hc.as_tuple() == counts.as_tuple() and hc.tier_mode == counts.tier_mode == case.tier_mode
    Ko = torch.full_like(Kd, float("nan")); Vo = torch.full_like(Vd, float("nan"))
    tm_out = torch.full_like(tier, 0xEE)
    skv.skv_unpack(shape, blob, bb, hc, Ko, Vo, tm_out, ws)
    torch.cuda.synchronize()
    out["K2"] = from_layout(Ko, layout).cpu().numpy()
    out["V2"] = from_layout(Vo, layout).cpu().numpy()
    out["tier_out"] = tm_out.cpu().numpy()
    return out


def assert_bit_exact(case, out):
    c = case.counts
    assert out["counts"].as_tuple() == (c.n16, c.n8, c.n4, c.n0)
    for r in range(case.R):
        assert np.array_equal(out["tier"][r], case.tier[r]), f"tier map differs (request {r})"
        assert out["blob"][r].size == case.blob[r].size
        if not np.array_equal(out["blob"][r], case.blob[r]):
            bad = np.flatnonzero(out["blob"][r] != case.blob[r])
            raise AssertionError(f"blob differs at {bad.size} bytes, first offsets {bad[:8]} (request {r})")
        assert np.array_equal(out["tier_out"][r], case.tier[r])
        assert np.array_equal(out["K2"][r].view(np.uint16), case.K2[r].view(np.uint16)), "unpacked K differs"
        assert np.array_equal(out["V2"][r].view(np.uint16), case.V2[r].view(np.uint16)), "unpacked V differs"


def assert_importance_close(case, out, rel=1e-3):
    for r in range(case.R):
        Io = case.I[r].astype(np.float64)
        Ig = out["I"][r].astype(np.float64)
        err = np.abs(Ig - Io)
        tol = rel * Io + 1e-30                       # P13
        assert (err <= tol).all(), f"importance: max rel err {np.max(err / (Io + 1e-30)):.3e}"
