"""Builds libfs.so (the CUDA product library) in-tree with nvcc for sm_100a.

    python -m paper_2505_23940_b200.build [--force] [--verbose]

The library links the CUDA runtime statically and has no torch dependency.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfs.so")
SOURCES = ["fs_api.cu", "fs_kernels_fluid.cu", "fs_kernels_pcg.cu", "fs_kernels_mg.cu", "fs_kernels_mgf.cu", "fs_kernels_ibm.cu", "fs_tma.cu", "fs_beam.cu", "fs_kernels_momv.cu", "fs_kernels_pcgc.cu",
           "noalloc/fs_noalloc.cu"]     # self-contained extra entry point (include/fs_noalloc.h); not part of the hot path
HEADERS = [os.path.join(CSRC, "fs_internal.cuh"), os.path.join(HERE, "..", "include", "fs.h"), os.path.join(HERE, "..", "include", "fs_noalloc.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]


def csrc_hash():
    """sha256 over csrc/*.cu, csrc/*.cuh and include/fs.h (sorted by name): identifies the sources a profile was
    captured from (bench.py refuses a committed ncu capture whose hash differs from the current sources).  These are the
    sources of the hot path; csrc/noalloc/ (one self-contained entry point, its own translation unit and header) is not
    among them."""
    import hashlib
    h = hashlib.sha256()
    files = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh")))
    for f in files + [os.path.normpath(HEADERS[1])]:
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    objs, procs = [], []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(objdir, os.path.basename(src).replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + HEADERS):
            cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
            procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose:
            sys.stderr.write(out)
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    if force or procs or _stale(LIB, objs):
        subprocess.check_call([NVCC, "-shared", "-o", LIB] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
