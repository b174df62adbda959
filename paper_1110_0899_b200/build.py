"""Build libwolff_b200.so (sm_100a only) in-tree with nvcc.  `python -m paper_1110_0899_b200.build [--force]`."""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB_NAME = "libwolff_b200.so"
LIB_PATH = os.path.join(HERE, LIB_NAME)
CHECKED_LIB_PATH = os.path.join(HERE, "libwolff_b200_checked.so")
JITTER_LIB_PATH = os.path.join(HERE, "libwolff_b200_jitter.so")
PROFILE_LIB_PATH = os.path.join(HERE, "libwolff_b200_profile.so")
SOURCES = ["api.cu", "batch_api.cu", "growth.cu", "growth_batch.cu", "growth_cluster.cu", "growth_tiles.cu", "measure.cu", "microbench.cu", "noalloc.cu"]
HEADERS = ["internal.h", "device_common.cuh", "expand.cuh", os.path.join(ROOT, "include", "wolff.h")]
NVCC_COMPILE_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC,-fvisibility=hidden,-Wall",
]
NVCC_LINK_FLAGS = ["--shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a"]
OBJ_DIR = os.path.join(HERE, "build")


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libwolff_b200.so cannot be built (there is no CPU fallback)")


def _header_paths():
    return [h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]


def needs_build(lib_path: str = LIB_PATH) -> bool:
    if not os.path.exists(lib_path):
        return True
    deps = [os.path.join(CSRC, s) for s in SOURCES] + _header_paths()
    return os.path.getmtime(lib_path) < max(os.path.getmtime(d) for d in deps)


def build(force: bool = False, verbose: bool = False, checked: bool = False, jitter: bool = False, profile: bool = False) -> str:
    """One nvcc per source file, side by side (the files share no device code, so there is no device link), then one
    link.  Objects are kept under paper_1110_0899_b200/build/ (git-ignored) and reused while they are newer than
    their source and every header.

    checked=True builds libwolff_b200_checked.so with -DWOLFF_CHECKED (every queue, list, tile and bit-plane index is
    compared with its bound before use: device_common.cuh); load it with WOLFF_B200_LIB=<path> (binding.py).
    jitter=True builds libwolff_b200_jitter.so with -DWOLFF_CHECKED -DWOLFF_JITTER (random sleeps between the steps of the
    lock-free protocols, device_common.cuh).
    profile=True builds libwolff_b200_profile.so with -DWOLFF_PROFILE (cycle and pass counters inside the barrier-free growth
    kernels, read through wolff_get_stats; `bench.py --profile-counters` prints them).  Never the measured path."""
    lib_path = PROFILE_LIB_PATH if profile else (JITTER_LIB_PATH if jitter else (CHECKED_LIB_PATH if checked else LIB_PATH))
    if not force and not needs_build(lib_path):
        return lib_path
    nvcc = nvcc_path()
    extra = os.environ.get("WOLFF_NVCC_EXTRA", "").split()      # e.g. -DWOLFF_PROFILE (per-section cycle counters)
    if checked or jitter:
        extra.append("-DWOLFF_CHECKED")
    if jitter:
        extra.append("-DWOLFF_JITTER")
    if profile:
        extra.append("-DWOLFF_PROFILE")
    os.makedirs(OBJ_DIR, exist_ok=True)
    tag = ("_" + "".join(c if c.isalnum() else "_" for c in " ".join(extra))) if extra else ""
    newest_header = max(os.path.getmtime(h) for h in _header_paths())
    jobs = []
    objs = []
    for src in SOURCES:
        path = os.path.join(CSRC, src)
        obj = os.path.join(OBJ_DIR, os.path.splitext(src)[0] + tag + ".o")
        objs.append(obj)
        fresh = os.path.exists(obj) and os.path.getmtime(obj) >= max(os.path.getmtime(path), newest_header)
        if fresh and not force:
            continue
        cmd = [nvcc] + NVCC_COMPILE_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj + ".tmp", path]
        jobs.append((cmd, obj, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)))
    failed = []
    for cmd, obj, proc in jobs:
        _, err = proc.communicate()
        if proc.returncode != 0:
            failed.append("%s\n%s" % (" ".join(cmd), err))
        else:
            os.replace(obj + ".tmp", obj)
            if verbose:
                sys.stderr.write(err)
    if failed:
        raise RuntimeError("nvcc failed:\n" + "\n".join(failed))
    tmp = lib_path + ".tmp.%d" % os.getpid()
    cmd = [nvcc] + NVCC_LINK_FLAGS + ["-o", tmp] + objs
    proc = subprocess.run(cmd, capture_output=True, text=True)
    if proc.returncode != 0:
        raise RuntimeError("link failed:\n%s\n%s" % (" ".join(cmd), proc.stderr))
    os.replace(tmp, lib_path)
    return lib_path


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv, jitter="--jitter" in sys.argv,
                profile="--profile" in sys.argv))
