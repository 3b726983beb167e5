"""Layer-pipelined prefill -> hop -> decode round trip (Fig. 3 placement).

The paper's timing "isolates the transfer path" with no overlap.  SKV1 blobs are layer-major and
every step of the path is per layer, so a request can be shipped as a sequence of layer chunks, each its own
self-contained SKV1 blob:

    A  H2D   K,V,Q of the chunk (pinned host -> device)                      [h2d stream]
    B  skv_importance -> skv_assign_tiers -> skv_pack                         [compute stream]
    C  D2H   blob (the hop, prefill side; pinned host stands in for the network)   [d2h stream]
    -- host: skv_blob_check on the received header --
    D  H2D   blob (the hop, decode side)                                      [h2d stream]
    E  skv_unpack                                                             [compute stream]
    F  D2H   dense K,V of the chunk                                           [d2h stream]

Chunks flow through `depth` device slots; the two copy directions run concurrently (PCIe is full duplex) and the
kernels hide under the copies, so the round trip costs max(bytes in, bytes out) / link rate instead of their sum.
Requests of a batch may have different token counts (a ragged batch): every chunk carries its own shape.
This module is plumbing only (streams, events, pointer offsets): every computation is a libskv kernel.
"""
import torch

from . import (make_policy, make_shape, skv_assign_tiers, skv_blob_bytes, skv_blob_check, skv_importance,
               skv_pack, skv_tier_counts, skv_unpack, skv_workspace_bytes)


class LayerPipelinedTransfer:
    def __init__(self, L, Hq, Hkv, d, n, w, budget, n_sink=0, ranges=(), allow_int4=True, layers_per_chunk=4,
                 depth=3, device="cuda:0", causal=True, lam=0.0, dtype="f16"):
        """n is the LARGEST token count any request will have (device slots are sized for it).  dtype: "f16" | "bf16"
        (element type of the host caches; they must be torch.float16 / torch.bfloat16 tensors accordingly)."""
        assert depth >= 2 and layers_per_chunk >= 1
        self.L, self.Hq, self.Hkv, self.d, self.n, self.w = L, Hq, Hkv, d, n, w
        self.Lc, self.depth, self.causal, self.lam = min(layers_per_chunk, L), depth, causal, lam
        self.dev = torch.device(device)
        self.dtype = "bf16" if dtype in ("bf16", 1) else "f16"
        self._pol_args = (budget, n_sink, tuple(ranges), allow_int4)
        self.policy = make_policy(*self._pol_args)
        # chunks: full chunks of Lc layers and (if L % Lc) one ragged tail chunk
        self.chunks = [(l0, min(self.Lc, L - l0)) for l0 in range(0, L, self.Lc)]
        self._plans = {}
        bb_max = self._plan(n, self.Lc)[2]
        dv, f16, u8 = self.dev, (torch.bfloat16 if self.dtype == "bf16" else torch.float16), torch.uint8
        mk = lambda numel, dt: [torch.empty((numel,), dtype=dt, device=dv) for _ in range(depth)]
        kv = self.Lc * n * Hkv * d
        self.dK, self.dV, self.dKo, self.dVo = mk(kv, f16), mk(kv, f16), mk(kv, f16), mk(kv, f16)
        self.dQ = mk(self.Lc * Hq * w * d, f16)
        self.dI = mk(self.Lc * n, torch.float32)
        self.dT = mk(self.Lc * n, u8)
        self.d_blob, self.d_blob2 = mk(bb_max, u8), mk(bb_max, u8)
        self.h_blob = [torch.empty((bb_max,), dtype=u8, pin_memory=True) for _ in range(depth)]
        self.ws = torch.empty(max(skv_workspace_bytes(self._plan(n, lc)[0], w) for _, lc in self.chunks), dtype=u8, device=dv)
        self.s_h2d, self.s_comp, self.s_d2h = (torch.cuda.Stream(device=dv) for _ in range(3))
        self.blob_bytes_per_request = self.blob_bytes(n)

    def _plan(self, n, lc):
        """(shape, counts, blob bytes) of a chunk of lc layers of a request with n tokens."""
        key = (n, lc)
        if key not in self._plans:
            assert self.w <= n <= self.n
            s = make_shape(lc, self.Hq, self.Hkv, self.d, n, 1, dtype=self.dtype)
            c = skv_tier_counts(s, self.policy)
            self._plans[key] = (s, c, skv_blob_bytes(s, c))
        return self._plans[key]

    def blob_bytes(self, n):
        return sum(self._plan(n, lc)[2] for _, lc in self.chunks)

    def bytes_per_request(self, n=None):
        """(host->device bytes, device->host bytes) moved for one request of n tokens (default: the largest)."""
        n = self.n if n is None else n
        kv = 2 * self.L * n * self.Hkv * self.d * 2
        q = self.L * self.Hq * self.w * self.d * 2
        return kv + q + self.blob_bytes(n), self.blob_bytes(n) + kv

    def run(self, hK, hV, hQ, hKo, hVo, hI=None, hT=None):
        """Equal-length batch.  hK, hV: pinned host fp16 [R][L][n][Hkv][d]; hQ: pinned [R][L][Hq][w][d]; hKo, hVo:
        pinned outputs [Ro][L][n][Hkv][d]; request r lands in slot r % Ro (Ro = R keeps every request, a smaller Ro
        is a ring for a consumer that drains it).  Optional pinned hI f32 [R][L][n] / hT u8 [R][L][n] receive the
        importance scores and tier maps.  Returns after everything has landed in host memory."""
        R, Ro = hK.shape[0], hKo.shape[0]
        reqs = [dict(K=hK[r], V=hV[r], Q=hQ[r], Ko=hKo[r % Ro], Vo=hVo[r % Ro],
                     I=None if hI is None else hI[r], T=None if hT is None else hT[r]) for r in range(R)]
        self.run_ragged(reqs)

    def run_ragged(self, requests):
        """requests: list of dicts of pinned host tensors, one per request, each with its own token count n_r <= n:
        K, V fp16 [L][n_r][Hkv][d]; Q fp16 [L][Hq][w][d]; Ko, Vo outputs like K; optional I f32 [L][n_r], T u8 [L][n_r].
        Returns after everything has landed in host memory."""
        work = [(req, l0, lc) for req in requests for (l0, lc) in self.chunks]
        N, depth = len(work), self.depth
        need = max(skv_workspace_bytes(self._plan(req["K"].shape[1], lc)[0], self.w) for req, _, lc in work)
        if need > self.ws.numel():                                    # nothing is in flight yet: safe to grow
            self.ws = torch.empty(need, dtype=torch.uint8, device=self.dev)
        L, Hq, Hkv, d, w = self.L, self.Hq, self.Hkv, self.d, self.w
        ev = lambda: [torch.cuda.Event() for _ in range(N)]
        eA, eB, eC, eD, eE, eF = ev(), ev(), ev(), ev(), ev(), ev()
        cur = torch.cuda.current_stream(self.dev)
        start = torch.cuda.Event()
        start.record(cur)
        for s in (self.s_h2d, self.s_comp, self.s_d2h):
            s.wait_event(start)

        def views(k, n, lc):
            kv = lambda buf: buf[k][:lc * n * Hkv * d].view(lc, n, Hkv, d)
            return (kv(self.dK), kv(self.dV), kv(self.dKo), kv(self.dVo), self.dQ[k][:lc * Hq * w * d].view(lc, Hq, w, d),
                    self.dI[k][:lc * n].view(lc, n), self.dT[k][:lc * n].view(lc, n))

        def prefill(i):
            req, l0, lc = work[i]
            n = req["K"].shape[1]
            k = i % depth
            sh, counts, bb = self._plan(n, lc)
            dK, dV, _, _, dQ, dI, dT = views(k, n, lc)
            with torch.cuda.stream(self.s_h2d):
                if i >= depth:
                    self.s_h2d.wait_event(eB[i - depth])              # slot inputs consumed by pack
                dK.copy_(req["K"][l0:l0 + lc], non_blocking=True)
                dV.copy_(req["V"][l0:l0 + lc], non_blocking=True)
                dQ.copy_(req["Q"][l0:l0 + lc], non_blocking=True)
                eA[i].record(self.s_h2d)
            with torch.cuda.stream(self.s_comp):
                self.s_comp.wait_event(eA[i])
                if i >= depth:
                    self.s_comp.wait_event(eC[i - depth])             # slot blob shipped
                skv_importance(sh, dK, dQ, w, dI, self.ws, causal=self.causal, lam=self.lam, stream=self.s_comp)
                skv_assign_tiers(sh, self.policy, dI, dT, self.ws, stream=self.s_comp)
                skv_pack(sh, dK, dV, dT, counts, self.d_blob[k][:bb], self.ws, stream=self.s_comp)
                eB[i].record(self.s_comp)
            with torch.cuda.stream(self.s_d2h):
                self.s_d2h.wait_event(eB[i])
                if i >= depth:
                    self.s_d2h.wait_event(eD[i - depth])              # host slot re-sent to the decode side
                self.h_blob[k][:bb].copy_(self.d_blob[k][:bb], non_blocking=True)
                if req.get("I") is not None:
                    req["I"][l0:l0 + lc].copy_(dI, non_blocking=True)
                if req.get("T") is not None:
                    req["T"][l0:l0 + lc].copy_(dT, non_blocking=True)
                eC[i].record(self.s_d2h)

        def decode(i):
            req, l0, lc = work[i]
            n = req["K"].shape[1]
            k = i % depth
            sh, _, bb = self._plan(n, lc)
            _, _, dKo, dVo, _, _, _ = views(k, n, lc)
            eC[i].synchronize()                                       # the blob has "arrived"
            _, hc = skv_blob_check(self.h_blob[k], bb)                # host-side header validation
            with torch.cuda.stream(self.s_h2d):
                if i >= depth:
                    self.s_h2d.wait_event(eE[i - depth])
                self.d_blob2[k][:bb].copy_(self.h_blob[k][:bb], non_blocking=True)
                eD[i].record(self.s_h2d)
            with torch.cuda.stream(self.s_comp):
                self.s_comp.wait_event(eD[i])
                if i >= depth:
                    self.s_comp.wait_event(eF[i - depth])
                skv_unpack(sh, self.d_blob2[k], bb, hc, dKo, dVo, None, self.ws, stream=self.s_comp)
                eE[i].record(self.s_comp)
            with torch.cuda.stream(self.s_d2h):
                self.s_d2h.wait_event(eE[i])
                req["Ko"][l0:l0 + lc].copy_(dKo, non_blocking=True)
                req["Vo"][l0:l0 + lc].copy_(dVo, non_blocking=True)
                eF[i].record(self.s_d2h)

        lag = 1
        for i in range(N + lag):
            if i < N:
                prefill(i)
            if i - lag >= 0:
                decode(i - lag)
        for s in (self.s_h2d, self.s_comp, self.s_d2h):
            cur.wait_stream(s)
        cur.synchronize()
