"""Compile the CUDA library in-tree: paper_2104_00537_b200/libsph_b200.so (sm_100a only).

Usage: python -m paper_2104_00537_b200.build [--force]
nvcc cross-compiles without a GPU.  Object files go to csrc/build/ (git-ignored).
"""
import hashlib
import json
import os
import socket
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libsph_b200.so")
STAMP = LIB + ".stamp"     # what the library was built from, where and with which flags (git-ignored, travels with the .so)
SOURCES = ["sph_api.cu", "nl_kernels.cu", "pi_kernels.cu", "pi_tiled.cu", "pi_quad.cu", "su_kernels.cu", "bx_kernels.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
# No -use_fast_math: the canonical predicate (C2) and conversions (C1) need IEEE mul/fma/div.
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC,-fvisibility=hidden", "-Xptxas", "-v"]
FLAGS += os.environ.get("SPH_NVCC_EXTRA", "").split()      # e.g. -DQ_STATS (development counters; never in a release build)


def _deps():
    d = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh"))]
    d.append(os.path.join(os.path.dirname(HERE), "include", "sph.h"))
    return d


def source_digest() -> str:
    """SHA-256 over the names and contents of every source the library is built from, plus the compiler flags."""
    h = hashlib.sha256(" ".join(FLAGS).encode())
    for p in sorted(_deps()):
        h.update(os.path.basename(p).encode())
        with open(p, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def host_id() -> str:
    """Host name plus the kernel's boot id: two machines started from the same image share the former only."""
    try:
        with open("/proc/sys/kernel/random/boot_id") as f:
            boot = f.read().strip()
    except OSError:
        boot = "?"
    return f"{socket.gethostname()}/{boot}"


def read_stamp() -> dict:
    try:
        with open(STAMP) as f:
            return json.load(f)
    except Exception:
        return {}


def built_on_this_host() -> bool:
    """True when the library in the tree was compiled on this machine from the sources as they are now."""
    st = read_stamp()
    return os.path.exists(LIB) and st.get("sources") == source_digest() and st.get("host") == host_id()


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile unless the library in the tree was built from exactly these sources and flags (content digest in the
    stamp file; file times do not survive a copy of the tree to another machine)."""
    srcs = [s for s in SOURCES if os.path.exists(os.path.join(CSRC, s))]
    digest = source_digest()
    if not force and os.path.exists(LIB) and read_stamp().get("sources") == digest:
        return LIB
    os.makedirs(OBJ, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        cmd = [NVCC, *FLAGS, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
        with open(obj + ".ptxas.txt", "w") as f:
            f.write(r.stderr)
        if verbose:
            print(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=len(srcs)) as ex:
        objs = list(ex.map(compile_one, srcs))
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call([NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp, *objs])
    os.replace(tmp, LIB)
    nvcc_version = subprocess.run([NVCC, "--version"], capture_output=True, text=True).stdout.strip().splitlines()[-1:]
    with open(STAMP, "w") as f:
        json.dump({"sources": digest, "host": host_id(), "nvcc": " ".join(nvcc_version),
                   "flags": FLAGS}, f, indent=1)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
