#!/usr/bin/env python
"""bench.py -- pack+unpack GB/s of FP16 KV (BASELINE.json metric) on the largest single-GPU config (C5).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl skv|reference] [--workload C5] [--budget 0.5]

A "step" is one pass of the whole hot path over one batch of synthetic requests:
    skv_importance -> skv_assign_tiers -> skv_pack -> skv_unpack
(6 kernel launches at C5: importance, assign, tile scan + pack, tile scan + unpack; 4 for n <= 8192 tokens, where the
scan is fused into pack / unpack)
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
    ap.add_argument("--l2-flush", default="auto", choices=["auto", "on", "off"],
                    help="read a 512 MiB buffer between stages (outside the stage events) so that no stage finds its "
                         "input in L2; auto = on for batches whose FP16 KV is below 2 GiB (C1-C4)")
    ap.add_argument("--no-sweep", action="store_true", help="skip the C1-C4 / budget sweep reported under 'sweep'")
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


TRAFFIC_FILE = "profiles/r3_traffic.csv"
CODEC_SOURCES = ("paper_2606_08635_b200/csrc/skv_pack.cu", "paper_2606_08635_b200/csrc/skv_unpack.cu",
                 "paper_2606_08635_b200/csrc/skv_codec.cuh")


def codec_sources_hash(root=None):
    """`git hash-object` (sha1 of "blob <len>\0" + contents) of the three files that make the pack / unpack kernels,
    first 10 hex digits each, joined by '+': the revision stamp of a recorded traffic row.  Computed with hashlib so
    that it also works on the GPU box, where the snapshot has no .git."""
    import hashlib
    out = []
    for rel in CODEC_SOURCES:
        with open(os.path.join(root or ROOT, rel), "rb") as f:
            data = f.read()
        out.append(hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()[:10])
    return "+".join(out)


def ncu_traffic(workload, b, R, kernel, path=None, root=None):
    """(dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` ("pack" | "unpack"), provenance) as
    captured by `ncu --set full` and RECORDED in profiles/r3_traffic.csv
    (workload,budget,n_requests,kernel,dram_bytes,codec_hash,captured) -- not measured in this run.  A row counts only
    if its codec_hash equals codec_sources_hash() of the tree that is running: a capture of other kernel sources is
    refused, (None, "stale: ...").  (None, None) when no capture of this exact workload is on file."""
    try:
        with open(path or os.path.join(ROOT, TRAFFIC_FILE)) as f:
            for ln in f:
                if ln.lstrip().startswith("#"):
                    continue
                fld = [x.strip() for x in ln.split(",", 6)]
                if len(fld) >= 6 and fld[0] == workload and fld[3] == kernel:
                    if abs(float(fld[1]) - b) < 1e-9 and int(fld[2]) == R:
                        have = codec_sources_hash(root)
                        if fld[5] != have:
                            return None, f"stale: the row was captured on codec sources {fld[5]}, the tree has {have}"
                        return float(fld[4]), (fld[6] if len(fld) > 6 else None)
    except Exception:
        pass
    return None, None


L2_BYTES = 126 * 2**20
FLUSH_BYTES = 512 * 2**20


def want_flush(args, cfg, R):
    if args.l2_flush == "auto":
        return cfg.bytes_fp16 * R < 2 * 2**30
    return args.l2_flush == "on"


def l2_note(cfg, R, blob_bytes, flush):
    """How the timed steps relate to the 126 MB L2, computed from the working set of one step."""
    kv = cfg.bytes_fp16 * R
    ws = 2 * kv + blob_bytes * R
    if flush:
        return (f"L2 flushed between stages: {FLUSH_BYTES >> 20} MiB read (clean lines) after every stage, outside the stage events "
                f"(step working set {ws / 2**20:.0f} MiB, blob {blob_bytes * R / 2**20:.0f} MiB would otherwise be partly "
                f"L2-resident between pack and unpack); ms_per_step = sum of the four stage times")
    if blob_bytes * R < 4 * L2_BYTES:
        return (f"no flush: step working set {ws / 2**20:.0f} MiB; the blob ({blob_bytes * R / 2**20:.0f} MiB) may be partly "
                f"L2-resident when unpack reads it")
    return (f"inputs larger than L2: every stage streams >= {min(kv, blob_bytes * R) / 2**20:.0f} MiB "
            f"(> 30x the 126 MB L2) between two uses of a line; no flush needed")


def config_json(cfg, b, R, extra=None):
    """The workload, identical for both arms (the driver compares the two `config` objects): nothing arm-specific goes
    in here -- the L2 note of a line is its sibling key `l2`."""
    c = {"workload": f"{cfg.name}: {cfg.L} layers, {cfg.Hq} q heads / {cfg.Hkv} KV heads, head_dim {cfg.d}, "
                     f"{cfg.n} tokens, batch of {R} requests, window {cfg.w}, b={b}, "
                     f"{'3-tier FP16/INT8/INT4' if cfg.allow_int4 else '2-tier FP16+INT8'}, {cfg.n_sink} sinks",
         "budget": b, "n_requests": R, "bytes_fp16_per_request": cfg.bytes_fp16}
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
    if backend == "nccl":
        import torch
        torch.cuda.set_device(local)                  # before the process group exists: NCCL binds to the current device
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local, world


def numa_cpus_of_pci(domain, bus, device, sysfs="/sys/bus/pci/devices"):
    """CPUs local to the PCI device (Linux sysfs `local_cpulist`, e.g. "0-15,32-47"), or None."""
    path = os.path.join(sysfs, f"{domain:04x}:{bus:02x}:{device:02x}.0", "local_cpulist")
    try:
        with open(path) as f:
            txt = f.read().strip()
    except OSError:
        return None
    cpus = set()
    for part in txt.split(","):
        if not part:
            continue
        lo, _, hi = part.partition("-")
        try:
            cpus.update(range(int(lo), int(hi or lo) + 1))
        except ValueError:
            return None
    return cpus or None


def bind_rank_to_gpu_numa_node(local):
    """Under torchrun (N ranks on one host) every rank pins host memory for the e2e leg: run the rank -- and so the
    first touch of its pinned buffers -- on the CPUs of the NUMA node its GPU hangs off, so that eight ranks do not all
    allocate on node 0 and cross the socket link on every copy.  Best effort: any failure leaves the affinity alone."""
    try:
        import torch
        pr = torch.cuda.get_device_properties(local)
        cpus = numa_cpus_of_pci(pr.pci_domain_id, pr.pci_bus_id, pr.pci_device_id)
        if cpus:
            allowed = cpus & os.sched_getaffinity(0)
            if allowed:
                os.sched_setaffinity(0, allowed)
                return sorted(allowed)
    except Exception:
        pass
    return None


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


def dist_finish():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        try:
            dist.destroy_process_group()
        except Exception:
            pass


# ----------------------------------------------------------------------------------------------------
# the CUDA arm
# ----------------------------------------------------------------------------------------------------
STAGES = ("importance", "assign", "pack", "unpack")
FUSE_MAX_TOKENS = 8192                # csrc/skv_common.cuh kFuseMaxTokens: up to here pack / unpack need no scan launch


def launches_per_step(cfg):
    """Kernels of libskv launched by one step: imp_fused_kernel | assign_kernel | [tile_scan,] pack | [tile_scan,] unpack."""
    return 1 + 1 + (1 if cfg.n <= FUSE_MAX_TOKENS else 2) * 2


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
        self.blob_flat = torch.empty((R * self.blob_bytes,), dtype=torch.uint8, device=dev)
        self.blob = self.blob_flat.view(R, self.blob_bytes)
        self.Ko = torch.empty_like(self.K)
        self.Vo = torch.empty_like(self.V)
        self.tier_out = torch.empty_like(self.tier)
        self.flush_buf = None

    def set_budget(self, b):
        """Same caches, another budget (the C5 b-sweep): new policy, counts and blob size; buffers are reused."""
        import torch
        skv = self.skv
        self.b = b
        self.policy = skv.make_policy(b, self.cfg.n_sink, self.cfg.ranges, self.cfg.allow_int4)
        self.counts = skv.skv_tier_counts(self.shape, self.policy)
        self.blob_bytes = skv.skv_blob_bytes(self.shape, self.counts)
        if self.blob_flat.numel() < self.R * self.blob_bytes:
            self.blob = self.blob_flat = None
            self.blob_flat = torch.empty((self.R * self.blob_bytes,), dtype=torch.uint8, device=self.dev)
        self.blob = self.blob_flat[:self.R * self.blob_bytes].view(self.R, self.blob_bytes)

    def enable_flush(self):
        import torch
        self.flush_buf = torch.zeros(FLUSH_BYTES // 8, dtype=torch.int64, device=self.dev)

    def step(self, events=None):
        """events: 8 CUDA events = (start, stop) of each of the four stages.  With an L2 flush enabled the flush runs
        between a stage's stop event and the next stage's start event."""
        skv, s = self.skv, self
        rec = (lambda i: events[i].record()) if events is not None else (lambda i: None)
        blob = s.blob
        # the flush READS 512 MiB (a torch reduction, outside the stage events): the lines it leaves in L2 are clean, so
        # the next stage does not pay for write-backs of somebody else's dirty lines
        fl = (lambda: s.flush_buf.sum()) if s.flush_buf is not None else (lambda: None)
        rec(0)
        skv.skv_importance(s.shape, s.K, s.Q, s.cfg.w, s.I, s.ws)
        rec(1); fl(); rec(2)
        skv.skv_assign_tiers(s.shape, s.policy, s.I, s.tier, s.ws)
        rec(3); fl(); rec(4)
        skv.skv_pack(s.shape, s.K, s.V, s.tier, s.counts, blob, s.ws)
        rec(5); fl(); rec(6)
        skv.skv_unpack(s.shape, blob, s.blob_bytes, s.counts, s.Ko, s.Vo, s.tier_out, s.ws)
        rec(7); fl()

    def algorithmic_bytes(self):
        """pack reads the rows it ships (dropped tokens are never loaded) + the tier map and
        writes the blob; unpack reads the blob and writes every row (dropped ones as zeros) + the tier map."""
        fp16 = self.cfg.bytes_fp16 * self.R
        blob = self.blob_bytes * self.R
        tm = self.cfg.L * self.cfg.n * self.R
        c = self.counts
        shipped = (c.n16 + c.n8 + c.n4) / float(self.cfg.n)
        return {"pack": int(fp16 * shipped) + blob + tm, "unpack": blob + fp16 + tm}


def time_problem(prob, K, W, flush, sampler=None, dev=None):
    """W untimed warm-up steps, then K timed steps bracketed by barrier + synchronize; per-stage CUDA events on the
    launching stream.  Returns per-stage mean / min ms and ms per step (event time of the K steps / K; with an L2
    flush between stages: the sum of the stage means)."""
    import torch
    if flush and prob.flush_buf is None:
        prob.enable_flush()
    if not flush:
        prob.flush_buf = None
    for _ in range(W):
        prob.step()
    torch.cuda.synchronize()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(8)] for _ in range(K)]
    barrier()
    torch.cuda.synchronize()
    if sampler is not None:
        sampler.start()
        sampler.wait_first_sample()
    t_wall0 = time.perf_counter()
    t_abs0 = time.time()
    for k in range(K):
        prob.step(ev[k])
    torch.cuda.synchronize()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop(t_abs0, time.time()) if sampler is not None else None
    stage_ms = [sum(ev[k][2 * i].elapsed_time(ev[k][2 * i + 1]) for k in range(K)) / K for i in range(4)]
    stage_min = [min(ev[k][2 * i].elapsed_time(ev[k][2 * i + 1]) for k in range(K)) for i in range(4)]
    ms_step = sum(stage_ms) if flush else ev[0][0].elapsed_time(ev[K - 1][7]) / K
    return {"stage_ms": stage_ms, "stage_min": stage_min, "ms_step": ms_step, "clocks": clocks, "wall_s": t_wall}


def importance_lower_bound_ms(cfg, R, hbm_gbs, tensor_tflops, sm_count=148, sm_ghz=1.965, ex2_per_clk_sm=16.0):
    """max of (K read once from HBM, the contraction twice at the sustained tensor peak, the exponentials
    twice at 16 MUFU results per clock per SM at the maximum SM clock).  Returns (ms, which term binds)."""
    k_bytes = cfg.bytes_fp16 * R / 2.0
    flop = 2.0 * cfg.L * cfg.Hq * cfg.w * cfg.n * cfg.d * R
    exps = 1.0 * cfg.L * cfg.Hq * cfg.w * cfg.n * R
    terms = {"hbm (K once)": k_bytes / (hbm_gbs * 1e9), "tensor (2 passes)": 2.0 * flop / (tensor_tflops * 1e12),
             "ex2 (2 passes)": 2.0 * exps / (sm_count * ex2_per_clk_sm * sm_ghz * 1e9)}
    which = max(terms, key=terms.get)
    return terms[which] * 1e3, which


def graph_replay_ms(prob, reps=20):
    """The whole path (importance -> assign -> pack -> unpack) captured once into a CUDA graph and replayed: the latency a
    serving loop sees for one request batch, without host launch gaps and without an L2 flush (warm L2, stated so)."""
    import torch
    saved, prob.flush_buf = prob.flush_buf, None
    try:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            prob.step()
        for _ in range(3):
            graph.replay()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            graph.replay()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps
    finally:
        prob.flush_buf = saved


def sweep_row(prob, res, peak, flush):
    cfg = prob.cfg
    alg = prob.algorithmic_bytes()
    imp, asg, pk, up = res["stage_ms"]
    kv = cfg.bytes_fp16 * prob.R
    return {"workload": cfg.name, "budget": prob.b, "n_requests": prob.R, "counts": list(prob.counts.as_tuple()),
            "stages_ms": dict(zip(STAGES, res["stage_ms"])), "stages_ms_min": dict(zip(STAGES, res["stage_min"])),
            "ms_per_step": res["ms_step"], "value": kv / ((pk + up) * 1e-3) / 1e9, "unit": UNIT,
            "pack_frac_of_hbm_peak": alg["pack"] / (pk * 1e-3) / 1e9 / peak,
            "unpack_frac_of_hbm_peak": alg["unpack"] / (up * 1e-3) / 1e9 / peak,
            "pack_plus_unpack_frac_of_hbm_peak": (alg["pack"] + alg["unpack"]) / ((pk + up) * 1e-3) / 1e9 / peak,
            "gpu_launches_per_step": launches_per_step(cfg),
            "importance_lower_bound_ms": importance_lower_bound_ms(cfg, prob.R, peak, measured_tensor_peak()[0])[0],
            "importance_frac_of_lower_bound": importance_lower_bound_ms(cfg, prob.R, peak, measured_tensor_peak()[0])[0] / imp,
            "l2": l2_note(cfg, prob.R, prob.blob_bytes, flush)}


def run_sweep(args, main_prob, dev, peak, steps):
    """BASELINE.json's other configs and budgets through the same timing loop: C1-C4 at their
    budgets with the L2 flushed between stages, and the remaining budgets of the C5 sweep on the main problem's caches."""
    import skv_synth
    rows = []
    main_cfg, main_b = main_prob.cfg, main_prob.b
    for name in ("C1", "C2", "C3", "C4", "C5"):
        cfg = skv_synth.CONFIGS[name]
        if cfg.name == main_cfg.name:
            for b in cfg.budgets:
                if abs(b - main_b) < 1e-9:
                    continue
                main_prob.set_budget(b)
                fl = want_flush(args, cfg, main_prob.R)
                rows.append(sweep_row(main_prob, time_problem(main_prob, steps, 3, fl), peak, fl))
            main_prob.set_budget(main_b)
            main_prob.flush_buf = None
            continue
        if cfg.bytes_fp16 * cfg.R > main_cfg.bytes_fp16 * main_prob.R:
            continue                                         # never sweep anything larger than the main workload
        prob = DeviceProblem(cfg, cfg.budgets[0], cfg.R, dev)
        for b in cfg.budgets:
            prob.set_budget(b)
            fl = want_flush(args, cfg, cfg.R)
            row = sweep_row(prob, time_problem(prob, steps, 3, fl), peak, fl)
            row["cuda_graph_replay_ms_per_step"] = graph_replay_ms(prob)
            row["cuda_graph_note"] = "whole path as ONE captured CUDA graph, back-to-back replays, L2 not flushed"
            rows.append(row)
        del prob
    return rows


def run_next_rows(prob, steps):
    """SURVEY.md 8(f) rows at the same workload, outside the timed step: NEXT-1 KV-norm fallback score (reads K once),
    NEXT-3 cold-tier upgrade (FP16 upgrade blob of 1024 tokens per layer: skv_pack + skv_unpack_patch) and every NEXT-4
    variant (2-bit low tier, group-wise 2-bit, INT8 hot tier, bfloat16 caches), each as pack + unpack on algorithmic
    bytes (main() adds frac_of_hbm_peak)."""
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
    # NEXT-4: the group-wise 2-bit low tier (reading P22) at the same b = 0.2, and the INT8 hot tier
    # (reading P21: nothing ships at FP16) at b = 0.4 (INT8 + low-tier mix; b >= 0.5 would be all INT8)
    for key, bx, polx in (
            ("group2_low_tier", 0.2, skv.make_policy(0.2, cfg.n_sink, cfg.ranges, 2, tier_mode=skv.SKV_MODE_GROUP2)),
            ("hot_int8", 0.4, skv.make_policy(0.4, cfg.n_sink, cfg.ranges, cfg.allow_int4, tier_mode=skv.SKV_MODE_HOT_INT8))):
        cx = skv.skv_assign_tiers(prob.shape, polx, prob.I, prob.tier, prob.ws)
        bbx = skv.skv_blob_bytes(prob.shape, cx)
        blobx = torch.empty((R, bbx), dtype=torch.uint8, device=prob.dev)
        def oncex():
            skv.skv_pack(prob.shape, prob.K, prob.V, prob.tier, cx, blobx, prob.ws)
            skv.skv_unpack(prob.shape, blobx, bbx, cx, prob.Ko, prob.Vo, prob.tier_out, prob.ws)
        oncex()
        a.record()
        for _ in range(steps):
            oncex()
        b_.record(); torch.cuda.synchronize()
        ms = a.elapsed_time(b_) / steps
        movedx = 2 * (cfg.bytes_fp16 * R + R * bbx + cfg.L * cfg.n * R)
        out[key] = {"budget": bx, "counts": list(cx.as_tuple()), "blob_bytes_per_request": bbx,
                    "ms_pack_plus_unpack": ms, "GBps": movedx / (ms * 1e-3) / 1e9,
                    "GBps_of_fp16_kv": cfg.bytes_fp16 * R / (ms * 1e-3) / 1e9}
        del blobx
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


def pcie_duplex_ms(h2d_bytes, d2h_bytes, h_src, h_dst, dev, chunk=256 * 2**20, reps=3):
    """The denominator of the e2e leg, measured in the same run: the time to move exactly `h2d_bytes` host -> device and
    `d2h_bytes` device -> host, both directions at once on two streams, from / to the same pinned buffers, with no
    kernel anywhere -- what the link alone would take for the step's traffic.  Copies go in `chunk`-byte pieces that
    cycle through the pinned tensors `h_src` / `h_dst` and one device staging buffer per direction."""
    import torch
    srcs = [t.view(torch.uint8).reshape(-1) for t in h_src]
    dsts = [t.view(torch.uint8).reshape(-1) for t in h_dst]
    chunk = int(min(chunk, min(t.numel() for t in srcs + dsts)))
    d_in = torch.empty((chunk,), dtype=torch.uint8, device=dev)
    d_out = torch.zeros((chunk,), dtype=torch.uint8, device=dev)
    s_in, s_out = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)

    def pieces(total, bufs):
        left, i = int(total), 0
        while left > 0:
            buf = bufs[i % len(bufs)]
            per = buf.numel() // chunk
            for k in range(per):
                if left <= 0:
                    break
                m = min(chunk, left)
                yield buf[k * chunk:k * chunk + m], m
                left -= m
            i += 1

    def once():
        with torch.cuda.stream(s_in):
            for h, m in pieces(h2d_bytes, srcs):
                d_in[:m].copy_(h, non_blocking=True)
        with torch.cuda.stream(s_out):
            for h, m in pieces(d2h_bytes, dsts):
                h.copy_(d_out[:m], non_blocking=True)

    once()
    torch.cuda.synchronize()
    best = float("inf")
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        cur = torch.cuda.current_stream()
        e0.record(cur)
        s_in.wait_event(e0); s_out.wait_event(e0)
        once()
        cur.wait_stream(s_in); cur.wait_stream(s_out)
        e1.record(cur)
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    return best


def run_e2e(cfg, b, R, dev, steps, warmup, chunk_layers=4, depth=3, host_requests=2):
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
    # pinned host footprint is bounded: `host_requests` distinct requests in and as many out (2 on a single rank, 1 per
    # rank under torchrun, where N ranks share one host's pinned memory); the R requests of a step cycle through them --
    # the bytes copied per step are those of R requests
    Rh = max(1, min(R, host_requests))
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
    out = {"ms_per_step": ms, "steps": steps, "h2d": R * h2d_req, "d2h": R * d2h_req, "layers_per_chunk": lpc, "depth": depth,
           "host_requests": Rh}
    del pipe
    out["pcie_duplex_ms"] = pcie_duplex_ms(R * h2d_req, R * d2h_req, (hK, hV), (hKo, hVo), dev)

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
def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.lower().startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except Exception:
        pass
    import platform
    return platform.processor() or platform.machine()


def oracle_sample(cfg, b, target_seconds):
    """SURVEY.md 8(d) 'Oracle timing': the oracle as it stands on a bounded sample of the workload (the first layers of
    request 0, made by the CPU generator of skv_synth: the same distribution as the CUDA arm's device-generated request
    0, not the same bytes -- the `sample` string says so), about `target_seconds` of
    CPU work in total:
      (b) pack + unpack with OpenMP over layers on every available core -- the headline `value`;
      (a) pack + unpack single-threaded on ONE layer;
      (c) importance (float64 triple loop) and assign (qsort) on a token-truncated slice of one layer, timed separately
          (importance cost is linear in n; the report says what was timed and the per-layer extrapolation).
    Returns the cpu_baseline dict."""
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

    # (a) single thread, one layer
    oracle.set_threads(1)
    nb1, tp1, tu1 = run(1)
    # (c) importance + assign, single layer, OpenMP as the oracle has it; importance on n_imp <= n tokens
    oracle.set_threads(threads)
    n_imp = int(min(cfg.n, 4096))
    sub = cfg.scaled(L=1, n=n_imp, ranges=())
    K1, _ = skv_synth.make_kv(sub, 0)
    Q1 = skv_synth.make_q(sub, 0)
    t0 = time.perf_counter()
    oracle.importance(K1.numpy(), Q1.numpy())
    t_imp = time.perf_counter() - t0
    I1 = skv_synth.make_importance(cfg.scaled(L=1), 0).numpy()
    t0 = time.perf_counter()
    oracle.assign(I1, prot, counts)
    t_asg = time.perf_counter() - t0
    # (b) all cores, as many layers as the time target allows
    budget_s = max(1.0, target_seconds - (tp1 + tu1) - t_imp - t_asg)
    layers = min(cfg.L, max(1, threads))
    nbytes, tp, tu = run(layers)
    per_layer = (tp + tu) / layers
    want = int(min(cfg.L, max(layers, budget_s / max(per_layer, 1e-9))))
    if want >= threads:
        want = (want // threads) * threads
    if want > layers:
        layers = want
        nbytes, tp, tu = run(layers)
    gbs = nbytes / (tp + tu) / 1e9
    sample = (f"oracle pack+unpack of {layers} of {cfg.L} layers of 1 request ({nbytes / 2**20:.0f} MiB FP16 KV), "
              f"tier map from a synthetic importance vector, OpenMP over layers; CPU-generator bytes (skv_synth on the host: "
              f"the same distribution as the CUDA arm's device-generated request 0, not the same bytes)")
    return {"value": gbs, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample, "cpu_model": cpu_model(),
            "seconds": tp + tu, "pack_s": tp, "unpack_s": tu,
            "single_thread": {"value": nb1 / (tp1 + tu1) / 1e9, "unit": UNIT, "cores": 1, "pack_s": tp1, "unpack_s": tu1,
                              "sample": f"oracle pack+unpack of 1 layer of 1 request ({nb1 / 2**20:.0f} MiB FP16 KV), 1 thread"},
            "importance": {"seconds": t_imp, "cores": threads,
                           "sample": f"oracle importance (float64) of 1 layer truncated to {n_imp} of {cfg.n} tokens, "
                                     f"window {cfg.w}, {cfg.Hq} query heads, OpenMP as the oracle has it",
                           "seconds_per_layer_extrapolated": t_imp * cfg.n / n_imp,
                           "seconds_per_request_extrapolated": t_imp * cfg.n / n_imp * cfg.L},
            "assign": {"seconds": t_asg, "cores": 1, "sample": f"oracle assign (qsort) of 1 layer of {cfg.n} tokens",
                       "seconds_per_request_extrapolated": t_asg * cfg.L}}


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
              f"tier map from a synthetic importance vector, OpenMP over layers; CPU-generator bytes (skv_synth on the host)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * mean, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f16 -> i8/i4 codes (exact products, f32 scales)",
            "data": "synthetic", "config": config_json(cfg, b, R), "l2": "CPU arm: not applicable",
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                             "cpu_model": cpu_model()},
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

    numa = bind_rank_to_gpu_numa_node(local) if world > 1 else None
    prob = DeviceProblem(cfg, b, R, dev, rank)
    flush = want_flush(args, cfg, R)
    K = args.steps
    W = max(args.warmup, 3)
    sampler = ClockSampler(local)
    res = time_problem(prob, K, W, flush, sampler=sampler, dev=dev)
    clocks, t_wall = res["clocks"], res["wall_s"]
    bytes_local = cfg.bytes_fp16 * R
    red, bytes_all = aggregate_over_ranks([res["ms_step"]] + res["stage_ms"], bytes_local, device=dev)
    ms_step, (ms_imp, ms_asg, ms_pack, ms_unpack) = red[0], red[1:]
    stage_min = res["stage_min"]
    value = bytes_all / ((ms_pack + ms_unpack) * 1e-3) / 1e9
    peak, peak_src = measured_peak()

    sweep = None
    if not args.no_sweep and world == 1:
        sweep = run_sweep(args, prob, dev, peak, min(K, 10))
    next_rows = None if args.no_next else run_next_rows(prob, min(K, 10))
    e2e = None
    if not args.no_e2e:
        r = run_e2e(cfg, b, R, dev, steps=min(K, 10), warmup=1, chunk_layers=args.e2e_chunk_layers, depth=args.e2e_depth,
                    host_requests=1 if world > 1 else 2)
        red2, _ = aggregate_over_ranks([r["ms_per_step"]], bytes_local, device=dev)
        e2e = {"value": bytes_all / (red2[0] * 1e-3) / 1e9, "unit": UNIT,
               "what": "GB/s of FP16 KV through the whole path from pinned host buffers (H2D K,V,Q; D2H + H2D hop of the blob; D2H result)",
               "h2d_bytes_per_step": r["h2d"], "d2h_bytes_per_step": r["d2h"], "ms_per_step": red2[0], "steps": r["steps"],
               "ms_per_request": red2[0] / R, "pipeline": f"layer chunks of {r['layers_per_chunk']}, {r['depth']} slots, 3 streams",
               "pinned_host_requests": r["host_requests"], "rank0_cpu_affinity": (len(numa) if numa else None),
               "sequential_ms_per_request": r["sequential_ms_per_request"],
               "raw_fp16_hop_ms_per_request": r["raw_fp16_hop_ms_per_request"],
               "blob_hop_ms_per_request": r["blob_hop_ms_per_request"],
               "pcie_duplex_ms": r["pcie_duplex_ms"], "frac_of_pcie": r["pcie_duplex_ms"] / red2[0],
               "pcie_note": "pcie_duplex_ms = the step's H2D and D2H byte counts copied both ways at once from / to the same "
                            "pinned buffers on two streams with no kernels, best of 3, this run, this rank; frac_of_pcie = "
                            "that time / the e2e step time (1.0 = the path is hidden entirely behind the link)"}

    if rank != 0:
        dist_finish()
        return
    alg = prob.algorithmic_bytes()
    dom = "pack" if ms_pack >= ms_unpack else "unpack"
    dom_ms = max(ms_pack, ms_unpack)
    achieved = alg[dom] / (dom_ms * 1e-3) / 1e9
    traffic, traffic_src = ncu_traffic(args.workload, b, R, dom)
    imp_flop = 2.0 * cfg.L * cfg.Hq * cfg.w * cfg.n * cfg.d * R
    tpeak, tpeak_src = measured_tensor_peak()
    fused = cfg.n <= FUSE_MAX_TOKENS
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f16 -> i8/i4 codes (quantiser arithmetic in f32); importance f16 x f16 -> f32",
        "data": "synthetic", "config": config_json(cfg, b, R), "l2": l2_note(cfg, R, prob.blob_bytes, flush),
        "stages_ms": {"importance": ms_imp, "assign": ms_asg, "pack": ms_pack, "unpack": ms_unpack},
        "stages_ms_min": dict(zip(STAGES, stage_min)),
        "ms_per_request_on_gpu": ms_step / R,
        "frac_of_hbm_peak_pack_plus_unpack": (alg["pack"] + alg["unpack"]) / ((ms_pack + ms_unpack) * 1e-3) / 1e9 / peak,
        "roofline": {"bound": "hbm",
                     "kernel": f"{dom}_fast_kernel" + ("" if fused else " (+ tile_scan_kernel, < 1 % of the stage)"),
                     "achieved": achieved,
                     "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak,
                     "algorithmic_bytes_per_launch": alg[dom], "avg_launch_ms": dom_ms,
                     "traffic": traffic, "traffic_source": (f"recorded ncu --set full capture, {TRAFFIC_FILE}: {traffic_src}"
                                                            if traffic is not None else traffic_src),
                     "other": {k: {"achieved": alg[k] / (m * 1e-3) / 1e9, "frac": alg[k] / (m * 1e-3) / 1e9 / peak}
                               for k, m in (("pack", ms_pack), ("unpack", ms_unpack))},
                     "frac_of_nominal_8TBs": achieved / 8000.0},
        "importance": {"ms": ms_imp, "useful_tflops": imp_flop / (ms_imp * 1e-3) / 1e12,
                       "executed_tflops": 2.0 * imp_flop / (ms_imp * 1e-3) / 1e12,
                       "note": "two-pass: the contraction and the exponentials run twice; bound by the MUFU ex2 / FMA / "
                               "tensor pipe mix at d_h = 128 (profiles/r2_importance_ncu.md), not by the tensor pipe alone",
                       "lower_bound_ms": importance_lower_bound_ms(cfg, R, peak, tpeak)[0],
                       "lower_bound_term": importance_lower_bound_ms(cfg, R, peak, tpeak)[1],
                       "frac_of_lower_bound": importance_lower_bound_ms(cfg, R, peak, tpeak)[0] / ms_imp,
                       "tensor_peak_tflops": tpeak, "tensor_peak_source": tpeak_src,
                       "useful_frac_of_tensor_peak": imp_flop / (ms_imp * 1e-3) / 1e12 / tpeak,
                       "executed_frac_of_tensor_peak": 2.0 * imp_flop / (ms_imp * 1e-3) / 1e12 / tpeak},
        "clocks": clocks, "gpu_launches": launches_per_step(cfg) * K, "wall_s_timed_region": t_wall,
    }
    if sweep is not None:
        line["sweep"] = sweep
    if next_rows is not None:
        for v in next_rows.values():
            v["frac_of_hbm_peak"] = v["GBps"] / peak
        line["next_rows"] = next_rows
    if e2e is not None:
        line["e2e"] = e2e
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = oracle_sample(cfg, b, args.cpu_seconds)        # rank 0 only (the other ranks returned above)
    print(json.dumps(line), flush=True)
    dist_finish()


if __name__ == "__main__":
    main()
