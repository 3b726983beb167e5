#!/usr/bin/env python
"""bench.py -- pack+unpack GB/s of FP16 KV (BASELINE.json metric) on the largest single-GPU config (C5).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl skv|reference] [--workload C5] [--budget 0.5]

A "step" is one pass of the whole hot path over one batch of synthetic requests:
    skv_importance -> skv_assign_tiers -> skv_pack -> skv_unpack      (9 kernel launches)
`value` = FP16 KV bytes of the batch / (time in skv_pack + skv_unpack), inputs resident in HBM, timed with CUDA
events on the launching stream.  `e2e` = the same bytes / the time of the whole path driven from pinned HOST
buffers (H2D of K,V,Q; the pinned-host D2H+H2D hop of the blob that stands in for the network; D2H of the
dense result).  `roofline` is for the dominant kernel (pack_kernel); `cpu_baseline` times the CPU oracle on a
bounded sample of the same workload (the only use of oracle/ in this file, together with --impl reference).

Multi-GPU (--gpus N under torchrun): requests are independent, so every rank runs its own batch (weak
scaling, no data-path collective); the time is the max over ranks, the value the sum of the ranks' bytes.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "pack+unpack GB/s of FP16 KV"
UNIT = "GB/s"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback ("of fallback")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="skv", choices=["skv", "reference"])
    ap.add_argument("--workload", default="C5")
    ap.add_argument("--budget", type=float, default=0.5)
    ap.add_argument("--requests", type=int, default=None)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-next", action="store_true", help="skip the timings of the NEXT rows (kvnorm score, upgrade)")
    ap.add_argument("--e2e-chunk-layers", type=int, default=4, help="layers per pipelined transfer chunk")
    ap.add_argument("--e2e-depth", type=int, default=3, help="device slots of the pipelined transfer")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


def measured_tensor_peak():
    """(sustained dense bf16/fp16 TFLOP/s, source) -- the importance kernels run inside a long step."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["bf16_tflops_sustained"]), "measured (MEASURED_PEAKS.json bf16_tflops_sustained)"
    except Exception:
        return 1400.0, "fallback (B200_PROFILING.md, sustained)"


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(workload, b, R, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` ("pack" | "unpack"), as captured by
    `ncu --set full` and recorded in profiles/r1_traffic.csv (workload,budget,n_requests,kernel,dram_bytes);
    None when no capture of this exact workload is on file."""
    try:
        with open(os.path.join(ROOT, "profiles", "r1_traffic.csv")) as f:
            for ln in f:
                fld = [x.strip() for x in ln.split(",")]
                if len(fld) >= 5 and fld[0] == workload and fld[3] == kernel:
                    if abs(float(fld[1]) - b) < 1e-9 and int(fld[2]) == R:
                        return float(fld[4])
    except Exception:
        pass
    return None


def config_json(cfg, b, R, extra=None):
    c = {"workload": f"{cfg.name}: {cfg.L} layers, {cfg.Hq} q heads / {cfg.Hkv} KV heads, head_dim {cfg.d}, "
                     f"{cfg.n} tokens, batch of {R} requests, window {cfg.w}, b={b}, "
                     f"{'3-tier FP16/INT8/INT4' if cfg.allow_int4 else '2-tier FP16+INT8'}, {cfg.n_sink} sinks",
         "budget": b, "n_requests": R, "bytes_fp16_per_request": cfg.bytes_fp16,
         "l2": "inputs larger than L2 (batch working set >> 126 MB); no flush needed"}
    if extra:
        c.update(extra)
    return c


# ----------------------------------------------------------------------------------------------------
# clocks sampler (nvidia-smi during the timed region)
# ----------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def wait_first_sample(self, timeout=5.0):
        t_end = time.time() + timeout
        while self.proc and not self.lines and time.time() < t_end:
            time.sleep(0.01)

    def stop(self, t0=None, t1=None):
        """Summary of the samples that arrived in [t0, t1] (the timed region; all samples if none did)."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        inside = [ln for (t, ln) in self.lines if t0 is not None and t0 <= t <= t1 + 0.05]
        for ln in (inside or [ln for (_, ln) in self.lines]):
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "samples_in_timed_region": len(inside),
                "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------------------
# multi-rank plumbing (one process per GPU; no data-path collective: requests are independent)
# ----------------------------------------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def dist_init(backend):
    import torch.distributed as dist
    rank, local, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local, world


def aggregate_over_ranks(ms_local, bytes_local, device="cpu"):
    """max over ranks of the times, sum over ranks of the bytes (weak scaling).  ms_local: list of floats."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(ms_local), dtype=torch.float64, device=device)
    b = torch.tensor([float(bytes_local)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(b, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.tolist()], float(b.item())


def rank_request_ids(rank, R):
    """Requests are independent: rank k owns the global request ids [k*R, (k+1)*R) -- its own
    seeds, its own blobs, no exchange with any other rank."""
    return list(range(rank * R, (rank + 1) * R))


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


# ----------------------------------------------------------------------------------------------------
# the CUDA arm
# ----------------------------------------------------------------------------------------------------
STAGES = ("importance", "assign", "pack", "unpack")
LAUNCHES_PER_STEP = 4 + 1 + 2 + 2     # imp_tc<1>, combine, imp_tc<2>, finish | assign | tile_scan, pack | tile_scan, unpack


class DeviceProblem:
    def __init__(self, cfg, b, R, dev, rank=0):
        import torch
        import paper_2606_08635_b200 as skv
        import skv_synth
        self.skv, self.cfg, self.b, self.R, self.dev = skv, cfg, b, R, dev
        L = cfg.L
        self.K = torch.empty((R, L, cfg.n, cfg.Hkv, cfg.d), dtype=torch.float16, device=dev)
        self.V = torch.empty_like(self.K)
        self.Q = torch.empty((R, L, cfg.Hq, cfg.w, cfg.d), dtype=torch.float16, device=dev)
        for r, rid in enumerate(rank_request_ids(rank, R)):
            self.K[r], self.V[r] = skv_synth.make_kv(cfg, rid, device=dev)
            self.Q[r] = skv_synth.make_q(cfg, rid, device=dev)
        self.shape = skv.make_shape(L, cfg.Hq, cfg.Hkv, cfg.d, cfg.n, R)
        self.policy = skv.make_policy(b, cfg.n_sink, cfg.ranges, cfg.allow_int4)
        self.counts = skv.skv_tier_counts(self.shape, self.policy)
        self.blob_bytes = skv.skv_blob_bytes(self.shape, self.counts)
        self.ws = torch.empty(skv.skv_workspace_bytes(self.shape, cfg.w), dtype=torch.uint8, device=dev)
        self.I = torch.empty((R, L, cfg.n), dtype=torch.float32, device=dev)
        self.tier = torch.empty((R, L, cfg.n), dtype=torch.uint8, device=dev)
        self.blob = torch.empty((R, self.blob_bytes), dtype=torch.uint8, device=dev)
        self.Ko = torch.empty_like(self.K)
        self.Vo = torch.empty_like(self.V)
        self.tier_out = torch.empty_like(self.tier)

    def step(self, events=None):
        skv, s = self.skv, self
        rec = (lambda i: events[i].record()) if events is not None else (lambda i: None)
        rec(0)
        skv.skv_importance(s.shape, s.K, s.Q, s.cfg.w, s.I, s.ws)
        rec(1)
        skv.skv_assign_tiers(s.shape, s.policy, s.I, s.tier, s.ws)
        rec(2)
        skv.skv_pack(s.shape, s.K, s.V, s.tier, s.counts, s.blob, s.ws)
        rec(3)
        skv.skv_unpack(s.shape, s.blob, s.blob_bytes, s.counts, s.Ko, s.Vo, s.tier_out, s.ws)
        rec(4)

    def algorithmic_bytes(self):
        """pack reads Bytes_FP16 + tier map, writes the blob; unpack the mirror."""
        fp16 = self.cfg.bytes_fp16 * self.R
        blob = self.blob_bytes * self.R
        tm = self.cfg.L * self.cfg.n * self.R
        return {"pack": fp16 + blob + tm, "unpack": blob + fp16 + tm}


def run_next_rows(prob, steps):
    """SURVEY.md 8(f) rows at the same workload, outside the timed step: NEXT-1 KV-norm fallback score (reads K once)
    and NEXT-3 cold-tier upgrade (FP16 upgrade blob of 1024 tokens per layer: skv_pack + skv_unpack_patch)."""
    import torch
    skv, cfg, R = prob.skv, prob.cfg, prob.R
    ev = lambda: torch.cuda.Event(enable_timing=True)
    out = {}
    a, b_ = ev(), ev()
    skv.skv_importance_kvnorm(prob.shape, prob.K, prob.I, prob.ws)
    a.record()
    for _ in range(steps):
        skv.skv_importance_kvnorm(prob.shape, prob.K, prob.I, prob.ws)
    b_.record(); torch.cuda.synchronize()
    ms = a.elapsed_time(b_) / steps
    kbytes = cfg.bytes_fp16 * R // 2
    out["kvnorm"] = {"ms": ms, "algorithmic_bytes": kbytes, "GBps": kbytes / (ms * 1e-3) / 1e9}
    k = min(1024, cfg.n // 4)
    up = torch.zeros((R, cfg.L, cfg.n), dtype=torch.uint8, device=prob.dev)
    up[:, :, cfg.n // 2:cfg.n // 2 + 2 * k:2] = 16                      # every other token of a 2k window
    uc = skv.skv_counts_from_populations(prob.shape, k)
    bb = skv.skv_blob_bytes(prob.shape, uc)
    ublob = torch.empty((R, bb), dtype=torch.uint8, device=prob.dev)
    def once():
        skv.skv_pack(prob.shape, prob.K, prob.V, up, uc, ublob, prob.ws)
        skv.skv_unpack_patch(prob.shape, ublob, bb, uc, prob.Ko, prob.Vo, prob.tier_out, prob.ws)
    once()
    a.record()
    for _ in range(steps):
        once()
    b_.record(); torch.cuda.synchronize()
    ms = a.elapsed_time(b_) / steps
    moved = 2 * R * bb                                                  # rows read + blob written, blob read + rows written
    out["upgrade"] = {"tokens_per_layer": k, "blob_bytes_per_request": bb, "ms_pack_plus_patch": ms,
                      "GBps": 2 * moved / (ms * 1e-3) / 1e9}
    del ublob, up
    # NEXT-4: the same caches with an asymmetric 2-bit low tier at b = 0.2 (INT8 + 2-bit mix, budget in eighths)
    pol2 = skv.make_policy(0.2, cfg.n_sink, cfg.ranges, 2)
    c2 = skv.skv_assign_tiers(prob.shape, pol2, prob.I, prob.tier, prob.ws)
    bb2 = skv.skv_blob_bytes(prob.shape, c2)
    blob2 = torch.empty((R, bb2), dtype=torch.uint8, device=prob.dev)
    def once2():
        skv.skv_pack(prob.shape, prob.K, prob.V, prob.tier, c2, blob2, prob.ws)
        skv.skv_unpack(prob.shape, blob2, bb2, c2, prob.Ko, prob.Vo, prob.tier_out, prob.ws)
    once2()
    a.record()
    for _ in range(steps):
        once2()
    b_.record(); torch.cuda.synchronize()
    ms = a.elapsed_time(b_) / steps
    moved2 = 2 * (cfg.bytes_fp16 * R + R * bb2 + cfg.L * cfg.n * R)
    out["two_bit_low_tier"] = {"budget": 0.2, "counts": list(c2.as_tuple()), "blob_bytes_per_request": bb2,
                               "ms_pack_plus_unpack": ms, "GBps": moved2 / (ms * 1e-3) / 1e9,
                               "GBps_of_fp16_kv": cfg.bytes_fp16 * R / (ms * 1e-3) / 1e9}
    del blob2
    # NEXT-4: bfloat16 caches (same values rounded to bf16), the headline policy (b of the run), pack + unpack
    for r in range(R):
        prob.Ko[r].copy_(prob.K[r].float().to(torch.bfloat16).view(torch.float16))     # Ko/Vo reused as bf16 inputs
        prob.Vo[r].copy_(prob.V[r].float().to(torch.bfloat16).view(torch.float16))
    shape_b = skv.make_shape(cfg.L, cfg.Hq, cfg.Hkv, cfg.d, cfg.n, R, dtype="bf16")
    cb = skv.skv_assign_tiers(shape_b, prob.policy, prob.I, prob.tier, prob.ws)
    bbb = skv.skv_blob_bytes(shape_b, cb)
    blob3 = torch.empty((R, bbb), dtype=torch.uint8, device=prob.dev)
    Kb, Vb = prob.Ko.clone(), prob.Vo.clone()
    def once3():
        skv.skv_pack(shape_b, Kb, Vb, prob.tier, cb, blob3, prob.ws)
        skv.skv_unpack(shape_b, blob3, bbb, cb, prob.Ko, prob.Vo, prob.tier_out, prob.ws)
    once3()
    a.record()
    for _ in range(steps):
        once3()
    b_.record(); torch.cuda.synchronize()
    ms = a.elapsed_time(b_) / steps
    moved3 = 2 * (cfg.bytes_fp16 * R + R * bbb + cfg.L * cfg.n * R)
    out["bf16_caches"] = {"budget": prob.b, "ms_pack_plus_unpack": ms, "GBps": moved3 / (ms * 1e-3) / 1e9,
                          "GBps_of_16bit_kv": cfg.bytes_fp16 * R / (ms * 1e-3) / 1e9}
    return out


def run_e2e(cfg, b, R, dev, steps, warmup, chunk_layers=4, depth=3):
    """The whole path driven from pinned HOST buffers through the public API (paper_2606_08635_b200.transfer.
    LayerPipelinedTransfer: per layer chunk  H2D K,V,Q -> importance -> assign -> pack -> D2H blob -> skv_blob_check
    (host) -> H2D blob -> unpack -> D2H K,V,  chunks overlapped on three streams).  Also times, once each for
    context, the same path with no overlap (one request at a time on one stream) and the bare hop of one request
    (raw FP16 K,V vs the SKV1 blob, D2H + H2D)."""
    import torch
    import paper_2606_08635_b200 as skv
    from paper_2606_08635_b200.transfer import LayerPipelinedTransfer
    import skv_synth
    L = cfg.L
    pin = dict(pin_memory=True)
    # pinned host footprint is bounded (N ranks share one host): two distinct requests in, a two-request ring out; the
    # R requests of a step alternate between them -- the bytes copied per step are those of R requests
    Rh = min(R, 2)
    hK = torch.empty((Rh, L, cfg.n, cfg.Hkv, cfg.d), dtype=torch.float16, **pin)
    hV = torch.empty_like(hK, **pin)
    hQ = torch.empty((Rh, L, cfg.Hq, cfg.w, cfg.d), dtype=torch.float16, **pin)
    for r in range(Rh):
        k, v = skv_synth.make_kv(cfg, r, device=dev)
        hK[r].copy_(k); hV[r].copy_(v); hQ[r].copy_(skv_synth.make_q(cfg, r, device=dev))
        del k, v
    hKo = torch.empty((Rh, L, cfg.n, cfg.Hkv, cfg.d), dtype=torch.float16, **pin)
    hVo = torch.empty_like(hKo, **pin)
    reqs = [dict(K=hK[r % Rh], V=hV[r % Rh], Q=hQ[r % Rh], Ko=hKo[r % Rh], Vo=hVo[r % Rh]) for r in range(R)]
    lpc = max(1, min(L, chunk_layers))
    pipe = LayerPipelinedTransfer(L, cfg.Hq, cfg.Hkv, cfg.d, cfg.n, cfg.w, b, cfg.n_sink, cfg.ranges, cfg.allow_int4,
                                  layers_per_chunk=lpc, depth=depth, device=dev)
    torch.cuda.synchronize()
    for _ in range(warmup):
        pipe.run_ragged(reqs)
    barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        pipe.run_ragged(reqs)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    h2d_req, d2h_req = pipe.bytes_per_request()
    out = {"ms_per_step": ms, "steps": steps, "h2d": R * h2d_req, "d2h": R * d2h_req, "layers_per_chunk": lpc, "depth": depth}
    del pipe

    # context 1: no overlap -- one request at a time, one stream, whole-request blobs
    shape = skv.make_shape(L, cfg.Hq, cfg.Hkv, cfg.d, cfg.n, 1)
    policy = skv.make_policy(b, cfg.n_sink, cfg.ranges, cfg.allow_int4)
    counts = skv.skv_tier_counts(shape, policy)
    bb = skv.skv_blob_bytes(shape, counts)
    h_blob = torch.empty((bb,), dtype=torch.uint8, **pin)
    dK = torch.empty((L, cfg.n, cfg.Hkv, cfg.d), dtype=torch.float16, device=dev)
    dV, dKo, dVo = torch.empty_like(dK), torch.empty_like(dK), torch.empty_like(dK)
    dQ = torch.empty((L, cfg.Hq, cfg.w, cfg.d), dtype=torch.float16, device=dev)
    dI = torch.empty((L, cfg.n), dtype=torch.float32, device=dev)
    dT = torch.empty((L, cfg.n), dtype=torch.uint8, device=dev)
    d_blob, d_blob2 = torch.empty((bb,), dtype=torch.uint8, device=dev), torch.empty((bb,), dtype=torch.uint8, device=dev)
    ws = torch.empty(skv.skv_workspace_bytes(shape, cfg.w), dtype=torch.uint8, device=dev)

    def sequential_request(r):
        dK.copy_(hK[r], non_blocking=True); dV.copy_(hV[r], non_blocking=True); dQ.copy_(hQ[r], non_blocking=True)
        skv.skv_importance(shape, dK, dQ, cfg.w, dI, ws)
        c = skv.skv_assign_tiers(shape, policy, dI, dT, ws)
        skv.skv_pack(shape, dK, dV, dT, c, d_blob, ws)
        h_blob.copy_(d_blob, non_blocking=True)
        torch.cuda.current_stream().synchronize()
        _, hc = skv.skv_blob_check(h_blob, bb)
        d_blob2.copy_(h_blob, non_blocking=True)
        skv.skv_unpack(shape, d_blob2, bb, hc, dKo, dVo, None, ws)
        hKo[0].copy_(dKo, non_blocking=True); hVo[0].copy_(dVo, non_blocking=True)
        torch.cuda.current_stream().synchronize()

    sequential_request(0)
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s0.record()
    sequential_request(0)
    s1.record()
    # context 2: the bare hop of one request, raw FP16 K,V vs the blob
    r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    r0.record()
    hKo[0].copy_(dK, non_blocking=True); hVo[0].copy_(dV, non_blocking=True)
    dKo.copy_(hKo[0], non_blocking=True); dVo.copy_(hVo[0], non_blocking=True)
    r1.record()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    h_blob.copy_(d_blob, non_blocking=True); d_blob2.copy_(h_blob, non_blocking=True)
    p1.record()
    torch.cuda.synchronize()
    out.update({"sequential_ms_per_request": s0.elapsed_time(s1),
                "raw_fp16_hop_ms_per_request": r0.elapsed_time(r1), "blob_hop_ms_per_request": p0.elapsed_time(p1)})
    return out


# ----------------------------------------------------------------------------------------------------
# the CPU oracle arm (cpu_baseline leg and --impl reference).  The ONLY place bench.py touches oracle/.
# ----------------------------------------------------------------------------------------------------
def oracle_sample(cfg, b, target_seconds):
    """Times oracle pack + unpack (the metric's two stages) on a bounded sample of the workload: the first
    `layers` layers of request 0 (same generator, same bytes as the CUDA arm's request 0 on the CPU generator).
    Returns (GB/s of FP16 KV, cores, sample description, seconds)."""
    import numpy as np
    import oracle
    import skv_synth
    threads = oracle.max_threads()
    counts, prot = oracle.tier_counts(cfg.n, b, cfg.n_sink, cfg.ranges, cfg.allow_int4)

    def run(layers):
        sub = cfg.scaled(L=layers)
        K, V = skv_synth.make_kv(sub, 0)
        I = skv_synth.make_importance(sub, 0).numpy()
        tier = oracle.assign(I, prot, counts)
        Kn, Vn = K.numpy(), V.numpy()
        t0 = time.perf_counter()
        blob = oracle.pack(Kn, Vn, tier, counts, cfg.allow_int4)
        t1 = time.perf_counter()
        oracle.unpack(blob, layers, cfg.Hkv, cfg.d, cfg.n)
        t2 = time.perf_counter()
        return sub.bytes_fp16, t1 - t0, t2 - t1

    layers = min(cfg.L, max(1, threads))
    nbytes, tp, tu = run(layers)
    per_layer = (tp + tu) / layers
    want = int(min(cfg.L, max(layers, target_seconds / max(per_layer, 1e-9))))
    if want >= threads:
        want = (want // threads) * threads
    if want > layers:
        layers = want
        nbytes, tp, tu = run(layers)
    gbs = nbytes / (tp + tu) / 1e9
    sample = (f"oracle pack+unpack of {layers} of {cfg.L} layers of 1 request ({nbytes / 2**20:.0f} MiB FP16 KV), "
              f"tier map from a synthetic importance vector, OpenMP over layers")
    return gbs, threads, sample, tp + tu, {"pack_s": tp, "unpack_s": tu}


def run_reference(args, cfg, b, R):
    """--impl reference: the CPU oracle as it stands, timed on the host cores.  One bounded sample of the workload
    (some layers of request 0) is generated ONCE and sized so that the whole run -- W warm-up + K timed passes of
    oracle pack + unpack over it -- ends within a few minutes."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    import oracle
    import skv_synth
    threads = oracle.max_threads()
    counts, prot = oracle.tier_counts(cfg.n, b, cfg.n_sink, cfg.ranges, cfg.allow_int4)
    passes = args.warmup + args.steps
    target = max(0.3, min(args.cpu_seconds, 120.0 / max(1, passes)))        # seconds per pass

    def make(layers):
        sub = cfg.scaled(L=layers)
        K, V = skv_synth.make_kv(sub, 0)
        tier = oracle.assign(skv_synth.make_importance(sub, 0).numpy(), prot, counts)
        return sub, K.numpy(), V.numpy(), tier

    def one_pass(sub, Kn, Vn, tier):
        t0 = time.perf_counter()
        blob = oracle.pack(Kn, Vn, tier, counts, cfg.allow_int4)
        oracle.unpack(blob, sub.L, cfg.Hkv, cfg.d, cfg.n)
        return time.perf_counter() - t0

    layers = min(cfg.L, max(1, threads))
    data = make(layers)
    per_layer = one_pass(*data) / layers
    want = int(min(cfg.L, max(1, target / max(per_layer, 1e-9))))
    if want >= threads:
        want = (want // threads) * threads
    if want != layers:
        layers = want
        data = make(layers)
    nbytes = data[0].bytes_fp16
    secs = [one_pass(*data) for _ in range(passes)][args.warmup:]
    mean = sum(secs) / len(secs)
    value = nbytes / mean / 1e9
    sample = (f"oracle pack+unpack of {layers} of {cfg.L} layers of 1 request ({nbytes / 2**20:.0f} MiB FP16 KV) per step, "
              f"tier map from a synthetic importance vector, OpenMP over layers")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * mean, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f16 -> i8/i4 codes (exact products, f32 scales)",
            "data": "synthetic", "config": config_json(cfg, b, R),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------
def main():
    args = parse_args()
    import skv_synth
    cfg = skv_synth.CONFIGS[args.workload]
    R = args.requests if args.requests is not None else cfg.R
    b = args.budget
    if args.impl == "reference":
        run_reference(args, cfg, b, R)
        return

    import torch
    rank, local, world = dist_init("nccl")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    from paper_2606_08635_b200 import lib
    lib()                                              # fail loudly if the CUDA library is missing

    prob = DeviceProblem(cfg, b, R, dev, rank)
    for _ in range(max(args.warmup, 3)):
        prob.step()
    torch.cuda.synchronize()
    K = args.steps
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(K)]
    sampler = ClockSampler(local)
    barrier()
    torch.cuda.synchronize()
    sampler.start()
    sampler.wait_first_sample()
    t_wall0 = time.perf_counter()
    t_abs0 = time.time()
    for k in range(K):
        prob.step(ev[k])
    torch.cuda.synchronize()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop(t_abs0, time.time())

    total_ms = ev[0][0].elapsed_time(ev[K - 1][4])
    stage_ms = [sum(ev[k][i].elapsed_time(ev[k][i + 1]) for k in range(K)) / K for i in range(4)]
    stage_min = [min(ev[k][i].elapsed_time(ev[k][i + 1]) for k in range(K)) for i in range(4)]
    bytes_local = cfg.bytes_fp16 * R
    red, bytes_all = aggregate_over_ranks([total_ms / K] + stage_ms, bytes_local, device=dev)
    ms_step, (ms_imp, ms_asg, ms_pack, ms_unpack) = red[0], red[1:]
    value = bytes_all / ((ms_pack + ms_unpack) * 1e-3) / 1e9

    next_rows = None if args.no_next else run_next_rows(prob, min(K, 10))
    e2e = None
    if not args.no_e2e:
        r = run_e2e(cfg, b, R, dev, steps=min(K, 3), warmup=1, chunk_layers=args.e2e_chunk_layers, depth=args.e2e_depth)
        red2, _ = aggregate_over_ranks([r["ms_per_step"]], bytes_local, device=dev)
        e2e = {"value": bytes_all / (red2[0] * 1e-3) / 1e9, "unit": "GB/s of FP16 KV, whole path from pinned host buffers",
               "h2d_bytes_per_step": r["h2d"], "d2h_bytes_per_step": r["d2h"], "ms_per_step": red2[0], "steps": r["steps"],
               "ms_per_request": red2[0] / R, "pipeline": f"layer chunks of {r['layers_per_chunk']}, {r['depth']} slots, 3 streams",
               "sequential_ms_per_request": r["sequential_ms_per_request"],
               "raw_fp16_hop_ms_per_request": r["raw_fp16_hop_ms_per_request"],
               "blob_hop_ms_per_request": r["blob_hop_ms_per_request"]}

    if rank != 0:
        return
    peak, peak_src = measured_peak()
    alg = prob.algorithmic_bytes()
    dom = "pack" if ms_pack >= ms_unpack else "unpack"
    dom_ms = max(ms_pack, ms_unpack)
    achieved = alg[dom] / (dom_ms * 1e-3) / 1e9
    traffic = ncu_traffic(args.workload, b, R, dom)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f16 -> i8/i4 codes (quantiser arithmetic in f32); importance f16 x f16 -> f32",
        "data": "synthetic", "config": config_json(cfg, b, R),
        "stages_ms": {"importance": ms_imp, "assign": ms_asg, "pack": ms_pack, "unpack": ms_unpack},
        "stages_ms_min": dict(zip(STAGES, stage_min)),
        "ms_per_request_on_gpu": ms_step / R,
        "frac_of_hbm_peak_pack_plus_unpack": (alg["pack"] + alg["unpack"]) / ((ms_pack + ms_unpack) * 1e-3) / 1e9 / peak,
        "roofline": {"bound": "hbm", "kernel": dom + "_kernel (+ tile_scan, < 1 % of the stage)", "achieved": achieved,
                     "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak,
                     "algorithmic_bytes_per_launch": alg[dom], "avg_launch_ms": dom_ms, "traffic": traffic,
                     "other": {k: {"achieved": alg[k] / (m * 1e-3) / 1e9, "frac": alg[k] / (m * 1e-3) / 1e9 / peak}
                               for k, m in (("pack", ms_pack), ("unpack", ms_unpack))},
                     "frac_of_nominal_8TBs": achieved / 8000.0},
        "importance": {"ms": ms_imp, "useful_tflops": 2.0 * cfg.L * cfg.Hq * cfg.w * cfg.n * cfg.d * R / (ms_imp * 1e-3) / 1e12,
                       "executed_tflops": 4.0 * cfg.L * cfg.Hq * cfg.w * cfg.n * cfg.d * R / (ms_imp * 1e-3) / 1e12,
                       "note": "two-pass: the contraction and the exponentials run twice; bound by the MUFU ex2 / FMA / "
                               "tensor pipe mix at d_h = 128 (profiles/r1_full_v4_ncu.md), not by the tensor pipe alone",
                       "tensor_peak_tflops": measured_tensor_peak()[0], "tensor_peak_source": measured_tensor_peak()[1],
                       "useful_frac_of_tensor_peak": 2.0 * cfg.L * cfg.Hq * cfg.w * cfg.n * cfg.d * R / (ms_imp * 1e-3) / 1e12 / measured_tensor_peak()[0],
                       "executed_frac_of_tensor_peak": 4.0 * cfg.L * cfg.Hq * cfg.w * cfg.n * cfg.d * R / (ms_imp * 1e-3) / 1e12 / measured_tensor_peak()[0]},
        "clocks": clocks, "gpu_launches": LAUNCHES_PER_STEP * K, "wall_s_timed_region": t_wall,
    }
    if next_rows is not None:
        for v in next_rows.values():
            v["frac_of_hbm_peak"] = v["GBps"] / peak
        line["next_rows"] = next_rows
    if e2e is not None:
        line["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        gbs, threads, sample, secs, parts = oracle_sample(cfg, b, args.cpu_seconds)
        line["cpu_baseline"] = {"value": gbs, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                                "seconds": secs, **parts}
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
