"""Build csrc/ into paper_1410_6685_b200/libsafegpu.so for sm_100a (in-tree, so the .so travels with gpurun).

nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -fmad=false
  -fmad=false: no FMA contraction — every elementwise primitive rounds once (R1); the kernels also
  use explicit _rn intrinsics.  Never --use_fast_math; default -prec-div=true -prec-sqrt=true -ftz=false.
"""
from __future__ import annotations

import concurrent.futures
import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libsafegpu.so")
NSHARDS = 8        # == SG_NSHARDS in csrc/sg_tmpl_launch.cuh: the template instances compile as eight translation units in parallel
SOURCES = [f"sg_vm_shard.cu@{k}" for k in range(4)] + [f"sg_tmpl_shard.cu@{k}" for k in range(NSHARDS)] + ["sg_kernels.cu", "sg_api.cpp", "sg_plan.cpp", "sg_build.cpp", "sg_transpose.cu", "sg_ge.cu", "sg_sort.cu", "sg_noalloc.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-fmad=false", "-std=c++17",
    "-Xcompiler", "-fPIC", "-x", "cu",
]


def _stamp() -> str:
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        with open(os.path.join(CSRC, name), "rb") as f:
            h.update(name.encode())
            h.update(f.read())
    with open(os.path.join(os.path.dirname(HERE), "include", "sg.h"), "rb") as f:
        h.update(f.read())
    h.update(" ".join(FLAGS).encode())
    return h.hexdigest()


def _dep_hash(src: str) -> str:
    """Hash of what an object depends on: its source, the flags, include/sg.h and every header in csrc/ it may include
    (host .cpp files never include the kernel headers .cuh / .inc; sg_transpose.cu includes only sg_kernels.h / sg_prog.h)."""
    light = src.endswith(".cpp") or src in ("sg_transpose.cu", "sg_ge.cu", "sg_sort.cu")
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name == src or name.endswith(".h") or (not light and name.endswith((".cuh", ".inc"))):
            with open(os.path.join(CSRC, name), "rb") as f:
                h.update(name.encode())
                h.update(f.read())
    with open(os.path.join(os.path.dirname(HERE), "include", "sg.h"), "rb") as f:
        h.update(f.read())
    h.update(" ".join(FLAGS).encode())
    return h.hexdigest()


def _compile(item: str) -> str:
    src, _, shard = item.partition("@")             # "file@k": shard k of the template instances (-DSG_SHARD=k)
    obj = os.path.join(OBJ, src + (f".{shard}" if shard else "") + ".o")
    dep_file, dep = obj + ".dep", _dep_hash(src)
    if os.path.exists(obj) and os.path.exists(dep_file) and open(dep_file).read() == dep:
        return obj              # unchanged since it was compiled
    extra = [f"-D{'SG_VM_DTYPE' if src == 'sg_vm_shard.cu' else 'SG_SHARD'}={shard}"] if shard else []
    subprocess.run([NVCC, *FLAGS, *extra, "-c", os.path.join(CSRC, src), "-o", obj], check=True)
    with open(dep_file, "w") as f:
        f.write(dep)
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    if force:
        for name in os.listdir(OBJ):
            if name.endswith(".dep"):
                os.remove(os.path.join(OBJ, name))
    stamp_file = os.path.join(OBJ, "stamp")
    stamp = _stamp()
    if not force and os.path.exists(LIB) and os.path.exists(stamp_file) and open(stamp_file).read() == stamp:
        return LIB
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(_compile, SOURCES))
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.run([NVCC, "-shared", "-o", tmp, *objs, "-gencode", "arch=compute_100a,code=sm_100a"], check=True)
    os.replace(tmp, LIB)
    with open(stamp_file, "w") as f:
        f.write(stamp)
    if verbose:
        print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force=True, verbose=True)
