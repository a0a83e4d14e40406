"""Builds libhhrr.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2510_13726_b200.build [--force]

geometry.cu is compiled with -fmad=false: the integer cell classification is defined by its
fp64 operation order.  Everything else uses default
contraction.  cudart is linked statically so the library does not depend on which
libcudart the host process (PyTorch) has loaded.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
INCLUDE = HERE.parent / "include"
LIB = HERE / "libhhrr.so"
OBJ = HERE / "build"
# one build per velocity set (HHRR_Q): D3Q27 (BASELINE.json's configs) and D3Q19 (the paper's own)
LIBS = {27: LIB, 19: HERE / "libhhrr_q19.so"}

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v", f"-I{INCLUDE}"]
SOURCES = {
    "api.cu": [],
    "collide.cu": [],
    "fused_ws.cu": [],
    "fused_xpull.cu": [],
    "wallmodel.cu": [],
    "geometry.cu": ["-fmad=false"],
}


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (Path(cand).exists() or cand == "nvcc"):
            return cand
    raise RuntimeError("nvcc not found")


def _newest_dep() -> float:
    deps = list(CSRC.glob("*.cu*")) + list(CSRC.glob("*.h")) + list(INCLUDE.glob("*.h")) + [Path(__file__)]
    return max(p.stat().st_mtime for p in deps)


def _compile(q: int, name: str, extra: list[str]) -> Path:
    tag = "" if q == 27 else f".q{q}"
    obj = OBJ / (name + tag + ".o")
    cmd = [nvcc(), *ARCH, *COMMON, f"-DHHRR_Q={q}", *extra, "-c", str(CSRC / name), "-o", str(obj)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    (OBJ / (name + tag + ".log")).write_text(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode:
        raise RuntimeError(f"nvcc failed on {name} (D3Q{q}):\n{r.stdout}\n{r.stderr}")
    return obj


def build(force: bool = False) -> Path:
    """Builds libhhrr.so (D3Q27) and libhhrr_q19.so (D3Q19); returns the path of the former."""
    if not force and all(p.exists() and p.stat().st_mtime >= _newest_dep() for p in LIBS.values()):
        return LIB
    OBJ.mkdir(exist_ok=True)
    jobs = [(q, name, extra) for q in LIBS for name, extra in SOURCES.items()]
    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(lambda j: _compile(*j), jobs))
    for q, out in LIBS.items():
        mine = [str(o) for (jq, _, _), o in zip(jobs, objs) if jq == q]
        cmd = [nvcc(), *ARCH, "-shared", "-o", str(out), *mine, "-cudart", "static"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode:
            raise RuntimeError(f"link failed (D3Q{q}):\n{r.stdout}\n{r.stderr}")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
