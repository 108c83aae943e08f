"""Build libpm2d.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpm2d.so")
SOURCES = ["pm2d_api.cu", "pm2d_particles.cu", "pm2d_lanes.cu", "pm2d_fields.cu", "pm2d_poisson.cu", "pm2d_diag.cu", "pm2d_static.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-diag-suppress", "128", "-Wno-deprecated-gpu-targets"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "pm2d.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build_id() -> str:
    """Hash of the sources the library is built from: pm2d_version() carries it, profiles/ tag their numbers with it."""
    h = hashlib.sha1()
    for f in sorted(os.listdir(CSRC)) + [os.path.join("..", "..", "include", "pm2d.h")]:
        h.update(open(os.path.join(CSRC, f), "rb").read())
    return h.hexdigest()[:10]


STAGE_SOURCES = ["pm2d_lanes.cu", "pm2d_particle_dev.cuh", "pm2d_internal.h"]


def stage_id() -> str:
    """Hash of the sources the fused stage kernel of the lane order (k_stage_lanes) is compiled from: profiles/ tag the
    ncu figures of that kernel with it, bench.py drops them when it differs."""
    h = hashlib.sha1()
    for f in STAGE_SOURCES:
        h.update(open(os.path.join(CSRC, f), "rb").read())
    return h.hexdigest()[:10]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = list(NVCC_FLAGS)
    objs = []
    procs = []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    for src in SOURCES:
        obj = os.path.join(HERE, "build", src.replace(".cu", ".o"))
        cmd = [nvcc, *flags, f'-DPM2D_BUILD_ID="{build_id()}"', "-c", os.path.join(CSRC, src), "-o", obj] + (["-Xptxas", "-v"] if verbose else [])
        procs.append((cmd, subprocess.Popen(cmd)))
        objs.append(obj)
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc, "-shared", "-o", tmp, *objs, "-lcudart"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
