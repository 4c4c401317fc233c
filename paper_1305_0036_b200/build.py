"""Build libts_b200.so (the CUDA path) in-tree with nvcc for sm_100a.

    python -m paper_1305_0036_b200.build [--force] [--verbose]

Objects go to paper_1305_0036_b200/build/, the library to paper_1305_0036_b200/libts_b200.so.  nvcc cross-compiles
without a GPU.  Only files under csrc/ and include/ are compiled; nothing from oracle/ is linked.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libts_b200.so")
SOURCES = ["ts_v2_probe.cu", "ts_v2_chunk0.cu", "ts_v2_chunk1.cu", "ts_v2_chunk0_h9.cu", "ts_v2_chunk1_h9.cu", "ts_v2_H9.cu", "ts_v2_H10.cu", "ts_v2_A.cu", "ts_v2_Hs.cu", "ts_v2_Hf.cu", "ts_tile_cfgG.cu", "ts_api.cu", "ts_shard.cu",
           "ts_tile.cu", "ts_naive.cu", "ts_small.cu", "ts_reduce.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"] + os.environ.get("TS_EXTRA_NVCC", "").split()


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _deps():
    d = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "ts_b200.h")]
    return max(os.path.getmtime(p) for p in d)


def build(force: bool = False, verbose: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= _deps():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()

    def compile_one(src):
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_FLAGS + ["-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        with open(obj + ".log", "w") as f:
            f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            print(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    cmd = [nvcc, "-shared", "-o", LIB] + objs + ["-cudart", "static"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
