"""Build libkara.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2607_01237_b200.build [--force] [--verbose]

One nvcc -c per csrc/*.cu (skipped when the object is newer than every source/header), then a
shared link with the static CUDA runtime, so the library loads on a machine without a driver
(symbols resolve; calls fail with a CUDA error).  The driver API entry point the TMA descriptors
need is fetched at run time through cudaGetDriverEntryPoint, so there is no link against libcuda.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
OBJ = HERE / "build"
SO = HERE / "libkara.so"
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC,-Wall,-Wextra", "-Xptxas", "-v", "--expt-relaxed-constexpr",
         *os.environ.get("KARA_NVCC_EXTRA", "").split()]   # e.g. -DKARA_TC_DEBUG (mbarrier watchdog)


def build(force: bool = False, verbose: bool = False) -> Path:
    OBJ.mkdir(exist_ok=True)
    hdrs = list(CSRC.glob("*.h")) + list(CSRC.glob("*.cuh")) + [HERE.parent / "include" / "kara.h"]
    newest_hdr = max(p.stat().st_mtime for p in hdrs)
    # objects are only reused if they were compiled with the same flags (-D switches change the code)
    flags_file, flags_now = OBJ / "FLAGS.txt", " ".join(FLAGS)
    if not flags_file.exists() or flags_file.read_text() != flags_now:
        force = True
    objs, rebuilt = [], False
    for stale in OBJ.glob("*.o"):                      # objects of sources that no longer exist
        if not (CSRC / (stale.stem + ".cu")).exists():
            stale.unlink()
            rebuilt = True
    for cu in sorted(CSRC.glob("*.cu")):
        o = OBJ / (cu.stem + ".o")
        objs.append(o)
        if force or not o.exists() or o.stat().st_mtime < max(cu.stat().st_mtime, newest_hdr):
            cmd = [NVCC, *FLAGS, "-c", str(cu), "-o", str(o)]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if verbose or r.returncode:
                sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            if r.returncode:
                raise RuntimeError(f"nvcc failed on {cu.name}")
            (OBJ / (cu.stem + ".ptxas.txt")).write_text(r.stderr)
            rebuilt = True
    flags_file.write_text(flags_now)
    if rebuilt or not SO.exists():
        tmp = SO.with_suffix(f".tmp{os.getpid()}.so")
        cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static",
               *map(str, objs), "-o", str(tmp)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            raise RuntimeError("link failed")
        os.replace(tmp, SO)
    return SO


def build_variant(extra_flags, out: Path) -> Path:
    """Compiles every csrc/*.cu with FLAGS + extra_flags into a scratch directory next to `out` and links them to `out`
    (a diagnostic build, e.g. -DKARA_TC_DEBUG: the mbarrier watchdog; the product library in-tree is not touched)."""
    out = Path(out)
    objdir = out.parent / (out.stem + "_obj")
    objdir.mkdir(parents=True, exist_ok=True)
    objs = []
    for cu in sorted(CSRC.glob("*.cu")):
        o = objdir / (cu.stem + ".o")
        r = subprocess.run([NVCC, *FLAGS, *extra_flags, "-c", str(cu), "-o", str(o)], capture_output=True, text=True)
        if r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError(f"nvcc failed on {cu.name}")
        objs.append(o)
    r = subprocess.run([NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static",
                        *map(str, objs), "-o", str(out)], capture_output=True, text=True)
    if r.returncode:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link failed")
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
