"""Builds the C-ABI CUDA library in-tree: paper_1605_03262_b200/libpyjac_b200.so (sm_100a only), and the
bench / test helper library libpyjac_b200_tools.so beside it (include/pyjac_b200_tools.h).

    python -m paper_1605_03262_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  kernels.cu is compiled once per S (states a CTA interleaves; in parallel), the
objects go to paper_1605_03262_b200/build/.  The .so is git-ignored but travels to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
SO = os.path.join(HERE, "libpyjac_b200.so")
TOOLS_SO = os.path.join(HERE, "libpyjac_b200_tools.so")          # bench / test helpers, not the product
HOST_SOURCES = ["api.cu", "mech_pack.cu", "dispatch.cu", "fd.cu", "tools.cu"]
# states a CTA interleaves per iteration -- keep in step with csrc/dispatch.cu
KERNEL_S = [1, 2, 3, 4, 6]
HEADERS = ["device_mech.h", "kernels.h", "mech_pack.h", os.path.join("..", "..", "include", "pyjac_b200.h"),
           os.path.join("..", "..", "include", "pyjac_b200_tools.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def is_stale() -> bool:
    if not os.path.exists(SO) or not os.path.exists(TOOLS_SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in HOST_SOURCES + ["kernels.cu"] + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return SO
    os.makedirs(OBJ, exist_ok=True)
    extra = (["-Xptxas", "-v"] if verbose else []) + os.environ.get("PYJAC_NVCC_FLAGS", "").split()
    jobs = []      # (object, command)
    for f in HOST_SOURCES:
        o = os.path.join(OBJ, f[:-3] + ".o")
        jobs.append((o, [_nvcc()] + NVCC_FLAGS + extra + ["-c", os.path.join(CSRC, f), "-o", o]))
    for sv in KERNEL_S:
        o = os.path.join(OBJ, "kernels_s%d.o" % sv)
        jobs.append((o, [_nvcc()] + NVCC_FLAGS + extra + ["-DPYJAC_S=%d" % sv, "-c",
                                                          os.path.join(CSRC, "kernels.cu"), "-o", o]))

    def run(job):
        return subprocess.run(job[1], cwd=CSRC, capture_output=True, text=True)

    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        results = list(ex.map(run, jobs))
    failed = False
    for (o, cmd), res in zip(jobs, results):
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        failed = failed or res.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed building %s" % SO)
    objs = [j[0] for j in jobs]
    tools_obj = os.path.join(OBJ, "tools.o")
    pack_obj = os.path.join(OBJ, "mech_pack.o")
    for so, parts in ((SO, [o for o in objs if o != tools_obj]), (TOOLS_SO, [tools_obj, pack_obj])):
        link = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a"] + parts + ["-o", so]
        res = subprocess.run(link, cwd=CSRC, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("link failed for %s" % so)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
