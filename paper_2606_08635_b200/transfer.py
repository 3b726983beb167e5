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
This module is plumbing only (streams, events, pointer offsets): every computation is a libskv kernel.
"""
import torch

from . import (make_policy, make_shape, skv_assign_tiers, skv_blob_bytes, skv_blob_check, skv_importance,
               skv_pack, skv_tier_counts, skv_unpack, skv_workspace_bytes)


class LayerPipelinedTransfer:
    def __init__(self, L, Hq, Hkv, d, n, w, budget, n_sink=0, ranges=(), allow_int4=True, layers_per_chunk=4,
                 depth=3, device="cuda:0", causal=True, lam=0.0):
        assert depth >= 2 and layers_per_chunk >= 1
        self.L, self.Hq, self.Hkv, self.d, self.n, self.w = L, Hq, Hkv, d, n, w
        self.Lc, self.depth, self.causal, self.lam = min(layers_per_chunk, L), depth, causal, lam
        self.dev = torch.device(device)
        self.policy = make_policy(budget, n_sink, ranges, allow_int4)
        # chunk shapes: full chunks of Lc layers and (if L % Lc) one ragged tail chunk
        self.chunks = [(l0, min(self.Lc, L - l0)) for l0 in range(0, L, self.Lc)]
        self._shape, self._counts, self._bb = {}, {}, {}
        for lc in sorted({c[1] for c in self.chunks}):
            s = make_shape(lc, Hq, Hkv, d, n, 1)
            self._shape[lc] = s
            self._counts[lc] = skv_tier_counts(s, self.policy)
            self._bb[lc] = skv_blob_bytes(s, self._counts[lc])
        bb_max = max(self._bb.values())
        dv, f16, u8 = self.dev, torch.float16, torch.uint8
        mk = lambda shape, dt: [torch.empty(shape, dtype=dt, device=dv) for _ in range(depth)]
        self.dK, self.dV = mk((self.Lc, n, Hkv, d), f16), mk((self.Lc, n, Hkv, d), f16)
        self.dKo, self.dVo = mk((self.Lc, n, Hkv, d), f16), mk((self.Lc, n, Hkv, d), f16)
        self.dQ = mk((self.Lc, Hq, w, d), f16)
        self.dI = mk((self.Lc, n), torch.float32)
        self.dT = mk((self.Lc, n), u8)
        self.d_blob, self.d_blob2 = mk((bb_max,), u8), mk((bb_max,), u8)
        self.h_blob = [torch.empty((bb_max,), dtype=u8, pin_memory=True) for _ in range(depth)]
        self.ws = torch.empty(skv_workspace_bytes(self._shape[self.Lc], w), dtype=u8, device=dv)
        self.s_h2d, self.s_comp, self.s_d2h = (torch.cuda.Stream(device=dv) for _ in range(3))
        self.blob_bytes_per_request = sum(self._bb[lc] for _, lc in self.chunks)

    def run(self, hK, hV, hQ, hKo, hVo, hI=None, hT=None):
        """hK, hV: pinned host fp16 [R][L][n][Hkv][d]; hQ: pinned [R][L][Hq][w][d]; hKo, hVo: pinned outputs
        [Ro][L][n][Hkv][d]; request r lands in slot r % Ro (Ro = R keeps every request, a smaller Ro is a ring for a
        consumer that drains it).  Optional pinned hI f32 [R][L][n] / hT u8 [R][L][n] receive the importance scores and tier
        maps.  Returns after everything has landed in host memory.  Bytes moved: see `bytes_per_request()`."""
        R = hK.shape[0]
        work = [(r, l0, lc) for r in range(R) for (l0, lc) in self.chunks]
        N, depth = len(work), self.depth
        ev = lambda: [torch.cuda.Event() for _ in range(N)]
        eA, eB, eC, eD, eE, eF = ev(), ev(), ev(), ev(), ev(), ev()
        cur = torch.cuda.current_stream(self.dev)
        start = torch.cuda.Event()
        start.record(cur)
        for s in (self.s_h2d, self.s_comp, self.s_d2h):
            s.wait_event(start)

        def prefill(i):
            r, l0, lc = work[i]
            k = i % depth
            sh = self._shape[lc]
            with torch.cuda.stream(self.s_h2d):
                if i >= depth:
                    self.s_h2d.wait_event(eB[i - depth])              # slot inputs consumed by pack
                self.dK[k][:lc].copy_(hK[r, l0:l0 + lc], non_blocking=True)
                self.dV[k][:lc].copy_(hV[r, l0:l0 + lc], non_blocking=True)
                self.dQ[k][:lc].copy_(hQ[r, l0:l0 + lc], non_blocking=True)
                eA[i].record(self.s_h2d)
            with torch.cuda.stream(self.s_comp):
                self.s_comp.wait_event(eA[i])
                if i >= depth:
                    self.s_comp.wait_event(eC[i - depth])             # slot blob shipped
                skv_importance(sh, self.dK[k], self.dQ[k], self.w, self.dI[k], self.ws, causal=self.causal,
                               lam=self.lam, stream=self.s_comp)
                skv_assign_tiers(sh, self.policy, self.dI[k], self.dT[k], self.ws, stream=self.s_comp)
                skv_pack(sh, self.dK[k], self.dV[k], self.dT[k], self._counts[lc], self.d_blob[k][:self._bb[lc]],
                         self.ws, stream=self.s_comp)
                eB[i].record(self.s_comp)
            with torch.cuda.stream(self.s_d2h):
                self.s_d2h.wait_event(eB[i])
                if i >= depth:
                    self.s_d2h.wait_event(eD[i - depth])              # host slot re-sent to the decode side
                self.h_blob[k][:self._bb[lc]].copy_(self.d_blob[k][:self._bb[lc]], non_blocking=True)
                if hI is not None:
                    hI[r, l0:l0 + lc].copy_(self.dI[k][:lc], non_blocking=True)
                if hT is not None:
                    hT[r, l0:l0 + lc].copy_(self.dT[k][:lc], non_blocking=True)
                eC[i].record(self.s_d2h)

        def decode(i):
            r, l0, lc = work[i]
            k = i % depth
            bb = self._bb[lc]
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
                skv_unpack(self._shape[lc], self.d_blob2[k], bb, hc, self.dKo[k], self.dVo[k], None, self.ws,
                           stream=self.s_comp)
                eE[i].record(self.s_comp)
            with torch.cuda.stream(self.s_d2h):
                self.s_d2h.wait_event(eE[i])
                ro = r % hKo.shape[0]
                hKo[ro, l0:l0 + lc].copy_(self.dKo[k][:lc], non_blocking=True)
                hVo[ro, l0:l0 + lc].copy_(self.dVo[k][:lc], non_blocking=True)
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

    def bytes_per_request(self):
        """(host->device bytes, device->host bytes) moved per request."""
        kv = 2 * self.L * self.n * self.Hkv * self.d * 2
        q = self.L * self.Hq * self.w * self.d * 2
        return kv + q + self.blob_bytes_per_request, self.blob_bytes_per_request + kv
