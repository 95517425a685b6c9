"""Builds the C-ABI shared library libcupymag_b200.so in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libcupymag_b200.so"
SOURCES = ["cm_mesh.cu", "cm_assemble.cu", "cm_spmv_cg.cu", "cm_fields.cu", "cm_api.cu", "cm_noalloc.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC,-fopenmp",
              "--expt-relaxed-constexpr"]


def _nvcc() -> str:
    return os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.h")) + [HERE.parent / "include" / "cupymag_b200.h"]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines: tuple = (), out: Path | None = None) -> Path:
    """Compiles csrc/*.cu and links the shared library.  `defines` (e.g. ("CM_U_CSR1=4",)) and `out` build a tuning
    variant beside the default library (set `binding.LIB_PATH` before the first call to load it)."""
    if out is None and not defines and not force and not needs_build():
        return LIB
    lib = Path(out) if out is not None else LIB
    objdir = HERE / "build" / (lib.stem if out is not None else "default")
    objdir.mkdir(parents=True, exist_ok=True)
    dflags = [f"-D{d}" for d in defines]

    def compile_one(src: str) -> Path:
        obj = objdir / (src + ".o")
        cmd = [_nvcc(), *NVCC_FLAGS, *dflags, *(["-Xptxas", "-v"] if verbose else []), "-c", str(CSRC / src), "-o", str(obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError(f"nvcc failed on {src}")
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    cmd = [_nvcc(), "-shared", "-o", str(lib), *map(str, objs), "-Xcompiler", "-fopenmp", "-lgomp"]
    subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    defs = tuple(a[2:] for a in sys.argv[1:] if a.startswith("-D"))
    outs = [a.split("=", 1)[1] for a in sys.argv[1:] if a.startswith("--out=")]
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, defines=defs, out=Path(outs[0]) if outs else None))
