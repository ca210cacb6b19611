"""Build libmuca_b200.so (hand-written CUDA for sm_100a + the C ABI of include/muca.h) in-tree.

Usage: python -m paper_1707_00919_b200.build [--force]   (also called by __graft_entry__.build()).
nvcc cross-compiles without a GPU.  The built library sits next to this file so that it travels
with the repository snapshot to the GPU box; it is git-ignored.
"""
import fcntl
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = [os.path.join(CSRC, "muca.cu")]
DEPS = SOURCES + sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cuh")) + \
    [os.path.join(os.path.dirname(HERE), "include", "muca.h")]
LIB = os.path.join(HERE, "libmuca_b200.so")
# the same sources with -DMUCA_CHECKED: the kernels check their ring hand-overs and state addresses themselves
# (csrc/muca_device.cuh "Self-checks"); loaded instead of LIB when the environment has MUCA_CHECKED=1
LIB_CHECKED = os.path.join(HERE, "libmuca_b200_checked.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def nvcc() -> str:
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    cand = os.path.join(cuda, "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(d) > t for d in DEPS)


def csrc_sha256() -> str:
    """sha256 over csrc/ (names and contents, sorted): identifies the kernels a profile under profiles/ was captured from
    (bench.py marks the ncu counters it quotes as stale when this no longer matches the stamp in the summary file)."""
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh")):
            h.update(name.encode())
            with open(os.path.join(CSRC, name), "rb") as f:
                h.update(f.read())
    return h.hexdigest()


class NvccMissing(RuntimeError):
    """No nvcc on this machine (the only case in which an existing library may be used as it is)."""


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    lib = LIB_CHECKED if checked else LIB
    if not force and not stale(lib):
        return lib
    # Several processes may get here at once (one rank per GPU under torchrun, the two-process tests): one builds, the
    # others wait for the lock and then find the library fresh.  Each build writes a file of its own and renames it.
    with open(lib + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not force and not stale(lib):
            return lib
        tmp = f"{lib}.{os.getpid()}.tmp"
        cmd = [nvcc()] + NVCC_FLAGS + (["-DMUCA_CHECKED"] if checked else []) + ["-o", tmp] + SOURCES
        try:
            res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        except FileNotFoundError as e:
            raise NvccMissing(str(e)) from e
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout)
        if res.returncode != 0:
            if os.path.exists(tmp):
                os.remove(tmp)
            raise RuntimeError("nvcc failed building " + os.path.basename(lib))
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    if "--hash" in sys.argv:
        print(csrc_sha256())
        sys.exit(0)
    print(build(force="--force" in sys.argv, verbose=True))
    print(build(force="--force" in sys.argv, verbose=True, checked=True))
