"""Build step for libts.so: nvcc, sm_100a only, in-tree (the .so travels to the GPU box with the snapshot)."""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libts.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
         "-Xptxas", "-v"]
# The projection decides integers (cull set, pixel rects, depth keys, tile counts) that must equal the float32 oracle's
# bit for bit: its translation unit is compiled WITHOUT implicit multiply-add contraction, so that a plain a * b + c
# written there later cannot silently fuse; the fused operations of DESIGN.md N1-N3 are spelled __fmaf_rn.
FMAD = {"ts_project.cu": "--fmad=false"}


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale():
    if not os.path.exists(SO):
        return True
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "ts.h")]
    return any(os.path.getmtime(d) > os.path.getmtime(SO) for d in deps)


def build_variant(name: str, defines) -> str:
    """Another build of the same sources with extra -D flags (e.g. the job-timeline build of timeline.py): objects under
    build/<name>/, library libts_<name>.so next to libts.so.  The product library is not touched."""
    out_dir = os.path.join(HERE, "..", "build", name)
    os.makedirs(out_dir, exist_ok=True)
    so = os.path.join(HERE, f"libts_{name}.so")
    objs = []
    for src in sources():
        obj = os.path.join(out_dir, os.path.basename(src)[:-3] + ".o")
        fmad = FMAD.get(os.path.basename(src), "--fmad=true")
        flags = [f for f in FLAGS if f not in ("-Xptxas", "-v")]
        r = subprocess.run([NVCC, *flags, *[f"-D{d}" for d in defines], fmad, "-c", src, "-o", obj], capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(obj)
    r = subprocess.run([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", so, *objs, "-lcudart", "-ldl"],
                       capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link failed")
    return so


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return SO
    objs = []
    logs = []
    for src in sources():
        obj = os.path.join(CSRC, os.path.basename(src)[:-3] + ".o")
        fmad = FMAD.get(os.path.basename(src), "--fmad=true")
        r = subprocess.run([NVCC, *FLAGS, fmad, "-c", src, "-o", obj], capture_output=True, text=True)
        logs.append(r.stderr)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(obj)
    r = subprocess.run([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", SO, *objs, "-lcudart", "-ldl"], capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link failed")
    with open(os.path.join(CSRC, "ptxas.log"), "w") as fh:
        fh.write("\n".join(logs))
    if verbose:
        print("\n".join(logs))
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
