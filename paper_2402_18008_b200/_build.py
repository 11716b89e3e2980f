"""Build libhg.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import os
import shutil
import subprocess
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libhg.so"
SOURCES = ["hg_api.cu", "hg_batched.cu", "hg_grid.cu", "hg_ransac.cu", "hg_rect.cu", "hg_variants.cu"]
HEADERS = [CSRC / "hg_device.cuh", CSRC / "hg_host.h", PKG.parent / "include" / "hg.h"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "-Xptxas", "-v"]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libhg cannot be built")
    return exe


def is_stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = [CSRC / s for s in SOURCES] + HEADERS + [Path(__file__)]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    """Compile every .cu of csrc/ into one shared library (static cudart).  Safe when several processes call it at once
    (one rank per GPU under torchrun): the build runs under an exclusive file lock, objects go to a per-process
    directory and the library is moved into place atomically, so no rank ever dlopens a half-written file."""
    if not force and not is_stale():
        return LIB
    build_dir = PKG / "build"
    build_dir.mkdir(exist_ok=True)
    import fcntl
    with open(build_dir / ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not is_stale():            # another process built it while this one waited
                return LIB
            objs, log = [], []
            for s in SOURCES:
                obj = build_dir / (s + ".o")
                cmd = [_nvcc(), *NVCC_FLAGS, "-c", str(CSRC / s), "-o", str(obj)]
                r = subprocess.run(cmd, capture_output=True, text=True)
                log.append(r.stderr)
                if r.returncode != 0:
                    raise RuntimeError("nvcc failed for %s:\n%s" % (s, r.stderr))
                objs.append(str(obj))
            tmp = PKG / ("libhg.so.tmp.%d" % os.getpid())
            cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", str(tmp), *objs, "-cudart", "static"]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if r.returncode != 0:
                raise RuntimeError("link failed:\n" + r.stderr)
            os.replace(tmp, LIB)
            (build_dir / "ptxas.log").write_text("\n".join(log))
            if verbose:
                print("\n".join(log))
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
