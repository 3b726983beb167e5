"""N > 1 plumbing of bench.py on CPU: two gloo ranks (world_size 2, 127.0.0.1).  The path shards by request with
no data-path collective; the only cross-rank steps are the barrier and the max-over-ranks /
sum-over-ranks reduction of the timings and byte counts, which is what this covers, plus the request split and
that only rank 0 of the reference arm does any work."""
import json
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, os.environ["SKV_ROOT"])
    import bench
    rank, local, world = bench.dist_init("gloo")
    bench.barrier()
    ms_local = [10.0 + 5.0 * rank, 1.0, 2.0 - rank, 3.0, 4.0 + rank]
    red, total = bench.aggregate_over_ranks(ms_local, 1000 * (rank + 1))
    # the e2e leg: one time per rank (ms of a pipelined step from pinned host buffers), same reduction
    red2, total2 = bench.aggregate_over_ranks([100.0 - 30.0 * rank], 1000 * (rank + 1))
    e2e_value = total2 / (red2[0] * 1e-3) / 1e9
    bench.barrier()
    print(json.dumps({"rank": rank, "world": world, "red": red, "bytes": total, "red2": red2, "e2e_value": e2e_value,
                      "ids": bench.rank_request_ids(rank, 4)}), flush=True)
""")


def _spawn(rank, world, port, tmp):
    env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
               MASTER_PORT=str(port), SKV_ROOT=ROOT, GLOO_SOCKET_IFNAME="lo")
    return subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                            text=True, cwd=str(tmp))


def test_two_rank_gloo_max_time_sum_bytes(tmp_path):
    port = 29600 + os.getpid() % 300
    procs = [_spawn(r, 2, port, tmp_path) for r in range(2)]
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=180)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    for d in outs:
        assert d["world"] == 2
        assert d["red"] == [15.0, 1.0, 2.0, 3.0, 5.0]           # max over ranks, element by element
        assert d["bytes"] == 3000.0                               # sum over ranks (weak scaling)
        assert d["red2"] == [100.0]                               # e2e: the slowest rank's step time ...
        assert abs(d["e2e_value"] - 3000.0 / 0.1 / 1e9) < 1e-18   # ... under the bytes of all ranks
    assert outs[0]["ids"] == [0, 1, 2, 3] and outs[1]["ids"] == [4, 5, 6, 7]   # disjoint requests per rank


def test_reference_arm_runs_on_rank0_only(tmp_path):
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29599")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120, cwd=str(tmp_path))
    assert p.returncode == 0 and p.stdout.strip() == ""        # rank != 0: exits 0 without work or output
