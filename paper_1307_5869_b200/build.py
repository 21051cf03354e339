"""Build libprand.so (the C-ABI library of include/prand.h) in-tree with nvcc for sm_100a.

Usage: ``python -m paper_1307_5869_b200.build [--force] [--verbose]``.  The library is written next
to this file so that it travels to the GPU box with the repo snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libprand.so")
MT_TABLE = os.path.join(HERE, "mt19937_polys.bin")
SOURCES = ["prand.cu", "skip_ops.cpp", "k_lfsr113.cu", "k_mrg32k3a.cu", "k_mt19937.cu", "k_gmgq.cu",
           "k_fill.cu", "k_devapi.cu", "k_probe.cu", "k_noalloc.cu"]
HEADERS = ["internal.h", "k_common.cuh", "skip_ops.h"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "--fmad=false"]


def _stale(target: str, deps: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    hdrs = [os.path.join(CSRC, h) for h in HEADERS]
    hdrs += [os.path.join(HERE, "..", "include", h)
             for h in ("prand.h", "prand_host.h", "prand_ops.h", "prand_device.cuh", "prand_device_gm.cuh")]
    hdrs.append(os.path.abspath(__file__))
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    objs, procs = [], []
    for src in SOURCES:
        path = os.path.join(CSRC, src)
        obj = os.path.join(objdir, os.path.splitext(src)[0] + ".o")
        objs.append(obj)
        if force or _stale(obj, [path] + hdrs):
            cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", path, "-o", obj]
            if src.endswith(".cpp"):
                cmd = [NVCC] + FLAGS + ["-x", "cu", "-c", path, "-o", obj]
            procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = []
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            failed.append((src, out))
        elif verbose and out:
            print(f"--- {src}\n{out}")
    if failed:
        raise RuntimeError("nvcc failed:\n" + "\n".join(f"--- {s}\n{o}" for s, o in failed))
    if force or procs or _stale(LIB, objs):
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call([NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs + ["-cudart", "shared"])
        os.replace(tmp, LIB)
    build_mt_table(force)
    return LIB


def build_mt_table(force: bool = False) -> str:
    """The MT19937 jump-polynomial table of PAPER.md:378 (x^v mod phi for v = 2^n, n < 512, and v = m 2^i,
    m = 15..24, i < 128; 1792 x 2496 bytes): written once by csrc/mt_table_gen.cpp next to the library."""
    srcs = [os.path.join(CSRC, f) for f in ("mt_table_gen.cpp", "skip_ops.cpp")]
    deps = srcs + [os.path.join(CSRC, f) for f in ("skip_ops.h", "internal.h")]
    if not force and not _stale(MT_TABLE, deps):
        return MT_TABLE
    exe = os.path.join(HERE, "build", "mt_table_gen")
    subprocess.check_call([NVCC, "-O2", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-x", "cu"] + srcs +
                          ["-o", exe, "-cudart", "shared"])
    tmp = MT_TABLE + f".tmp{os.getpid()}"
    subprocess.check_call([exe, tmp])
    os.replace(tmp, MT_TABLE)
    return MT_TABLE


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
