"""Build libtridsk.so in-tree with nvcc for sm_100a (B200).  `python -m paper_2510_24186_b200.build`."""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtridsk.so")
SOURCES = ["api.cu", "mc_kernel.cu", "mc_lane.cu", "mc_cta.cu", "grid_build.cu", "topk.cu", "score_direct.cu", "microbench.cu", "mdn.cu"]
HEADERS = ["internal.h", "chain.cuh", "mdn.cuh", os.path.join("..", "..", "include", "tridsk.h")]
# TRIDSK_NVCC_EXTRA: extra nvcc flags for experiments (e.g. "-DLANE_F32X2"); part of the content hash
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC,-fopenmp", "--expt-relaxed-constexpr"] + os.environ.get("TRIDSK_NVCC_EXTRA", "").split()


def _digest(paths, extra="") -> str:
    h = hashlib.sha256(extra.encode())
    for p in paths:
        with open(p, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    """Content-hash stamped (mtimes do not survive a copy to the GPU box): rebuilds only if a source changed."""
    nvcc = os.environ.get("NVCC", "nvcc")
    hdrs = [os.path.join(CSRC, h) for h in HEADERS]
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    stamp, want = LIB + ".stamp", _digest(srcs + hdrs, " ".join(NVCC_FLAGS))
    if not force and not verbose and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == want:
        return LIB
    bdir = os.path.join(HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    objs, jobs = [], []
    for s in SOURCES:
        src, obj = os.path.join(CSRC, s), os.path.join(bdir, s.replace(".cu", ".o"))
        objs.append(obj)
        ostamp, owant = obj + ".stamp", _digest([src] + hdrs, " ".join(NVCC_FLAGS))
        if force or verbose or not os.path.exists(obj) or not os.path.exists(ostamp) or open(ostamp).read() != owant:
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
            jobs.append((cmd, ostamp, owant))
    with ThreadPoolExecutor(max_workers=4) as ex:
        for (cmd, ostamp, owant), r in zip(jobs, ex.map(lambda j: subprocess.run(j[0], capture_output=True, text=True), jobs)):
            if verbose or r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode != 0:
                raise RuntimeError("nvcc failed: " + " ".join(cmd))
            with open(ostamp, "w") as f:
                f.write(owant)
    subprocess.check_call([nvcc, "-shared", "-o", LIB] + objs + ["-lgomp", "-lcudart"])
    with open(stamp, "w") as f:
        f.write(want)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
