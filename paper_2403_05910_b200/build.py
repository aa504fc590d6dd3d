"""Builds libxf.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.  `python -m paper_2403_05910_b200.build`."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
INCLUDE = HERE.parent / "include"
OBJ = CSRC / "build"
LIB = HERE / "libxf.so"
SOURCES = ["xf_api.cu", "xf_prim.cu", "xf_ghost.cu", "xf_sweep_x.cu", "xf_sweep_y.cu", "xf_sweep_z.cu", "xf_probe.cu", "xf_visc.cu", "xf_halo.cu", "xf_react.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", f"-I{INCLUDE}"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or Path(cand).exists()):
            return cand
    raise RuntimeError("nvcc not found")


def _stale(target: Path, deps) -> bool:
    if not target.exists():
        return True
    t = target.stat().st_mtime
    return any(Path(d).stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    OBJ.mkdir(exist_ok=True)
    headers = list(CSRC.glob("*.cuh")) + list(INCLUDE.glob("*.h")) + [Path(__file__)]
    nvcc = _nvcc()

    def compile_one(src: str):
        obj = OBJ / (src[:-3] + ".o")
        if force or _stale(obj, [CSRC / src] + headers):
            r = subprocess.run([nvcc, *NVCC_FLAGS, "-c", str(CSRC / src), "-o", str(obj)], capture_output=True, text=True)
            (OBJ / (src[:-3] + ".ptxas.log")).write_text(r.stderr)
            if r.returncode != 0:
                raise RuntimeError(f"nvcc failed on {src}:\n{r.stderr}")
            if verbose:
                sys.stderr.write(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=min(8, len(SOURCES))) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    if force or _stale(LIB, objs):
        tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.run([nvcc, "-shared", "-arch=sm_100a", "-o", str(tmp), *map(str, objs), "-ldl"], check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
