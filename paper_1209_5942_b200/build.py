"""Build liblqcd.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

One object file per source, compiled in parallel, then linked; `python build.py [-DNAME=VALUE ...]` passes
extra nvcc flags (a forced rebuild)."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "liblqcd.so")
SOURCES = ["api.cu", "hopping.cu", "hopping_float.cu", "hopping_staged.cu", "force.cu", "gauge_update.cu", "vector_ops.cu", "pack.cu", "stream_probe.cu"]
HEADERS = [os.path.join(CSRC, "lqcd_internal.h"), os.path.join(CSRC, "site_ops.cuh"), os.path.join(CSRC, "kp_log_table.h"), os.path.join(HERE, "..", "include", "lqcd.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xptxas=-v", "-Xcompiler", "-fPIC",
]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]   # hopping_float.cu includes hopping.cu
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(src, extra_flags):
    obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
    cmd = [_nvcc()] + NVCC_FLAGS + list(extra_flags) + ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    return src, obj, cmd, res


def build(force=False, verbose=False, extra_flags=()):
    """Compile every .cu under csrc/ into paper_1209_5942_b200/liblqcd.so."""
    if not force and not needs_build():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as pool:
        results = list(pool.map(lambda s: _compile(s, extra_flags), SOURCES))
    objs = []
    for src, obj, cmd, res in results:
        if verbose or res.returncode != 0:
            sys.stderr.write(f"==== {src}\n" + res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        objs.append(obj)
    link = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs
    res = subprocess.run(link, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("link failed: " + " ".join(link))
    return LIB


if __name__ == "__main__":
    build(force=True, verbose=True, extra_flags=sys.argv[1:])
    print(LIB)
