"""Host-side logic of bench.py that needs no GPU: the CPU-baseline legs SURVEY.md 8(d) asks for, the L2 labelling
computed from the working set, the launch count per step and the algorithmic-byte model."""
import os
import sys
import types

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench
import skv_synth


def test_cpu_baseline_has_every_leg_of_the_measurement_contract():
    cfg = skv_synth.Config("tiny-bench", L=4, Hq=4, Hkv=2, d=64, n=512, w=8, R=1, seed=3)
    cb = bench.oracle_sample(cfg, 0.5, target_seconds=1.0)
    assert cb["kind"] == "oracle" and cb["unit"] == "GB/s" and cb["value"] > 0 and cb["cores"] >= 1
    assert isinstance(cb["cpu_model"], str) and cb["cpu_model"]
    st = cb["single_thread"]
    assert st["cores"] == 1 and st["value"] > 0 and st["unit"] == "GB/s"
    assert cb["importance"]["seconds"] > 0 and cb["importance"]["seconds_per_request_extrapolated"] > 0
    assert cb["assign"]["seconds"] > 0
    import oracle
    assert oracle.max_threads() == cb["cores"]                       # the single-thread leg restored the thread count


def test_l2_label_follows_the_working_set():
    args = types.SimpleNamespace(l2_flush="auto")
    C = skv_synth.CONFIGS
    assert bench.want_flush(args, C["C2"], 1) and bench.want_flush(args, C["C4"], 1)
    assert not bench.want_flush(args, C["C5"], 4)
    assert "flushed" in bench.l2_note(C["C2"], 1, 119_000_000, True)
    assert "partly" in bench.l2_note(C["C2"], 1, 119_000_000, False)
    assert "larger than L2" in bench.l2_note(C["C5"], 4, 2_182_000_000, False)


def test_launch_count_per_step():
    C = skv_synth.CONFIGS
    assert bench.launches_per_step(C["C2"]) == 4          # importance, assign, pack, unpack (scan fused, n = 4096)
    assert bench.launches_per_step(C["C5"]) == 6          # + one tile scan each for pack and unpack (n = 32768)


def test_numa_cpu_list_parsing(tmp_path):
    d = tmp_path / "0000:1b:00.0"
    d.mkdir()
    (d / "local_cpulist").write_text("0-3,8,10-11\n")
    assert bench.numa_cpus_of_pci(0, 0x1b, 0, sysfs=str(tmp_path)) == {0, 1, 2, 3, 8, 10, 11}
    assert bench.numa_cpus_of_pci(0, 0x1c, 0, sysfs=str(tmp_path)) is None            # no such device: affinity left alone
    (d / "local_cpulist").write_text("garbage")
    assert bench.numa_cpus_of_pci(0, 0x1b, 0, sysfs=str(tmp_path)) is None


def test_recorded_ncu_traffic_is_on_file_for_the_bench_workload():
    for kernel in ("pack", "unpack"):
        traffic, source = bench.ncu_traffic("C5", 0.5, 4, kernel)
        alg = 25_912_476_672                                               # algorithmic bytes of one launch
        assert traffic is not None and abs(traffic - alg) / alg < 0.01     # no re-reads: DRAM traffic = algorithmic bytes
        assert "rev" in source                                             # provenance of the capture travels with the number
    assert bench.ncu_traffic("C5", 0.45, 4, "pack") == (None, None)        # no capture of that workload: null, not a guess
    for w in ("C2", "C3", "C4"):                                           # the single-request configs of the sweep are on file too
        for kernel in ("pack", "unpack"):
            assert bench.ncu_traffic(w, 0.5, 1, kernel)[0] is not None, (w, kernel)


def test_recorded_ncu_traffic_is_refused_when_the_kernel_sources_changed(tmp_path):
    """A traffic row is stamped with `git hash-object` of the three files that make the pack / unpack kernels; bench.py
    uses it only while those files are the ones that were profiled."""
    import hashlib
    import subprocess
    have = bench.codec_sources_hash()
    assert len(have.split("+")) == 3 and all(len(h) == 10 for h in have.split("+"))
    try:                                                                   # the stamp really is git's blob hash
        out = subprocess.run(["git", "hash-object", os.path.join(ROOT, bench.CODEC_SOURCES[0])], capture_output=True, text=True, check=True)
        assert out.stdout.strip()[:10] == have.split("+")[0]
    except (OSError, subprocess.CalledProcessError):
        pass                                                               # no git on this box: the hashlib form stands alone
    csv = tmp_path / "traffic.csv"
    csv.write_text("# comment\n"
                   f"C5,0.5,4,pack,100,{have},2026-01-01 rev abc (x<1; 2>)\n"
                   "C5,0.5,4,unpack,200,0000000000+0000000000+0000000000,2026-01-01 rev old\n")
    assert bench.ncu_traffic("C5", 0.5, 4, "pack", path=str(csv)) == (100.0, "2026-01-01 rev abc (x<1; 2>)")
    traffic, why = bench.ncu_traffic("C5", 0.5, 4, "unpack", path=str(csv))
    assert traffic is None and why.startswith("stale")
    # the same good row is refused by a tree whose codec differs by one byte
    root = tmp_path / "tree"
    for rel in bench.CODEC_SOURCES:
        dst = root / rel
        dst.parent.mkdir(parents=True, exist_ok=True)
        dst.write_bytes(open(os.path.join(ROOT, rel), "rb").read() + (b" " if rel.endswith("skv_codec.cuh") else b""))
    traffic, why = bench.ncu_traffic("C5", 0.5, 4, "pack", path=str(csv), root=str(root))
    assert traffic is None and why.startswith("stale")
    # every row of the committed file carries the stamp of the committed sources
    rows = [ln for ln in open(os.path.join(ROOT, bench.TRAFFIC_FILE)) if ln.strip() and not ln.startswith("#")]
    assert len(rows) >= 8 and all(ln.split(",")[5] == have for ln in rows)


def test_importance_lower_bounds_match_the_survey_table():
    C = skv_synth.CONFIGS
    want = {"C2": 0.044, "C3": 0.058, "C4": 0.108, "C5": 0.92}              # SURVEY.md 8(d), ms per request
    for name, ms in want.items():
        got, which = bench.importance_lower_bound_ms(C[name], 1, 6523.0, 1413.0)
        assert abs(got - ms) / ms < 0.04, (name, got, which)
    assert bench.importance_lower_bound_ms(C["C4"], 1, 6523.0, 1413.0)[1].startswith("hbm")
    assert bench.importance_lower_bound_ms(C["C5"], 1, 6523.0, 1413.0)[1].startswith("ex2")


def test_both_arms_print_the_same_config_object():
    """The driver compares `config` of the CUDA arm and of `--impl reference`: it holds the workload only (the note on
    how the timed steps relate to L2 is a sibling key of the line), so the two are equal for equal arguments."""
    C = skv_synth.CONFIGS
    a = bench.config_json(C["C5"], 0.5, 4)
    assert "l2" not in a and "workload" in a and a["n_requests"] == 4 and a["budget"] == 0.5
    assert a == bench.config_json(C["C5"], 0.5, 4)
    src = open(bench.__file__).read()
    assert src.count('"config": config_json(cfg, b, R), "l2":') == 2        # the two lines: reference arm and CUDA arm
