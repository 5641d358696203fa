"""Build libdem_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

One object per translation unit under csrc/build/ (compiled in parallel, reused while its inputs are unchanged), then
one link.  Whether an object or the library is current is decided by a hash of the sources, not by time stamps: the
hash of everything under csrc/ and include/ is compiled into the library (dem_version()) and checked when it is loaded,
so a prebuilt .so that lags its sources is rebuilt (or refused) instead of being used silently.
"""
from __future__ import annotations

import concurrent.futures
import glob
import hashlib
import os
import shutil
import subprocess
import time

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.normpath(os.path.join(HERE, "..", "include"))
OBJDIR = os.path.join(CSRC, "build")  # object names carry a hash of the flags, so the two builds do not collide
# DEM_CHECKED=1 in the environment selects the checked build (device-side bounds checks of every index into the kernels'
# hand-rolled shared-memory structures, csrc/dem_types.h: DEM_ASSERT): another library file, built from the same
# sources with -DDEM_CHECKED, which binding.lib() then loads instead.  `python -m pytest tests -m gpu` under
# DEM_CHECKED=1 is the repo's substitute for a compute-sanitizer memcheck run (profiles/r02_sanitizers.md).
CHECKED = os.environ.get("DEM_CHECKED") == "1"
LIB = os.path.join(HERE, "libdem_b200_checked.so" if CHECKED else "libdem_b200.so")
HASHFILE = LIB + ".hash"
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
              "-Xptxas", "-v"] + (["-DDEM_CHECKED"] if CHECKED else [])


def _nvcc():
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libdem_b200.so cannot be built (there is no CPU fallback)")


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def headers():
    return sorted(glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h"))
                  + glob.glob(os.path.join(INCLUDE, "*.h")))


def source_hash():
    """Hash of every source and header the library is built from (and of the compiler flags)."""
    h = hashlib.sha1(" ".join(NVCC_FLAGS).encode())
    for f in sources() + headers():
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def built_hash():
    try:
        return open(HASHFILE).read().strip()
    except OSError:
        return None


def stale():
    return not os.path.exists(LIB) or built_hash() != source_hash()


def build(force=False, verbose=False):
    """Compile the library if it is missing or was built from other sources; returns its path."""
    if not (force or stale()):
        return LIB
    nvcc, tag = _nvcc(), source_hash()
    os.makedirs(OBJDIR, exist_ok=True)
    hdr = hashlib.sha1(" ".join(NVCC_FLAGS).encode())
    for f in headers():
        hdr.update(open(f, "rb").read())
    jobs = []
    for src in sources():
        key = hashlib.sha1(hdr.digest() + open(src, "rb").read()).hexdigest()[:16]
        base = os.path.splitext(os.path.basename(src))[0]
        obj = os.path.join(OBJDIR, "%s.%s.o" % (base, key))
        if force or not os.path.exists(obj):
            for old in glob.glob(os.path.join(OBJDIR, base + ".*.o")):
                if time.time() - os.path.getmtime(old) > 600:  # objects of abandoned source states
                    os.remove(old)
            jobs.append((src, obj))
        else:
            jobs.append((None, obj))

    def compile_one(job):
        src, obj = job
        if src is None:
            return obj, ""
        # dem_version() reports the hash of the sources the library was built from
        extra = ["-DDEM_SOURCE_HASH=\"%s\"" % tag] if os.path.basename(src) == "dem_lib.cu" else []
        res = subprocess.run([nvcc] + NVCC_FLAGS + extra + ["-c", src, "-o", obj + ".tmp"], capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s%s" % (src, res.stdout, res.stderr))
        os.replace(obj + ".tmp", obj)
        return obj, res.stdout + res.stderr

    with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as pool:
        done = list(pool.map(compile_one, jobs))
    if verbose:
        for _, log in done:
            print(log)
    tmp = LIB + ".tmp%d" % os.getpid()
    res = subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a"] + [o for o, _ in done] + ["-o", tmp],
                         capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + res.stdout + res.stderr)
    os.replace(tmp, LIB)
    with open(HASHFILE, "w") as f:
        f.write(tag + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
