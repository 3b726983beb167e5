"""Build libskv.so (hand-written CUDA for sm_100a + the C ABI of include/skv.h) in-tree with nvcc.

    python -m paper_2606_08635_b200.build [--force] [--verbose] [--define NAME[=VALUE] ...]

--define passes -DNAME[=VALUE] to nvcc.  The switches that exist are SKV_EX2_FMA_PAIRS=k (csrc/skv_importance_tc.cu: how
many of 8 exponential pairs run on the FMA pipe; profiles/r2_importance_ncu.md) and SKV_FUSE_MAX_TOKENS=n
(csrc/skv_common.cuh) -- such a library is for measurements only; rebuild without the switch afterwards.

The shared library sits next to this file so that it travels with the repository snapshot; it links the
CUDA runtime statically and needs no GPU to load (nvcc cross-compiles on a CPU-only box).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libskv.so")
SOURCES = ["skv_host.cu", "skv_scan.cu", "skv_pack.cu", "skv_unpack.cu", "skv_assign.cu", "skv_kvnorm.cu", "skv_importance_tc.cu",
           "skv_noalloc.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--compiler-options", "-fPIC", "-cudart", "static"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "skv.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, defines=()):
    if not force and not defines and not _stale():
        return LIB
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, src.replace(".cu", ".o"))
        cmd = ([_nvcc()] + NVCC_FLAGS + ["-D" + d for d in defines] + (["-Xptxas", "-v"] if verbose else []) +
               ["-c", os.path.join(CSRC, src), "-o", obj])
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for src, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode:
            sys.stderr.write(out)
        if p.returncode:
            raise RuntimeError(f"nvcc failed on {src}")
    cmd = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static", "-o", LIB + ".tmp"] + objs
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    _defs = [sys.argv[i + 1] for i, a in enumerate(sys.argv[:-1]) if a == "--define"]
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, defines=_defs))
