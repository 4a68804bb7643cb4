"""Build of the C-ABI shared library ``libraptor_b200.so`` (in-tree, next to this file) with nvcc for sm_100a.

The ray kernel (csrc/raptor_render.cu) is compiled once per (plasma model, integrator)
(-DRAPTOR_MODEL=0..6 -DRAPTOR_INTEG=0..3) in parallel;
objects go to ``build/`` (git-ignored) and are linked with the API and the satellite kernels.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libraptor_b200.so")
N_MODELS = 7
N_INTEG = 4
HEADERS = ["raptor_device.cuh", "raptor_kernels.h", os.path.join("..", "..", "include", "raptor.h")]
SOURCES = ["raptor_render.cu", "raptor_render_f32.cu", "raptor_kernels.cu", "raptor_flux_static.cu", "raptor_api.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--fmad=true", "-Xcompiler", "-fPIC"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, extra: list[str] | None = None, out: str | None = None) -> str:
    """Compiles and links the library; ``extra`` = additional nvcc flags (e.g. -DRAPTOR_MIN_BLOCKS=4),
    ``out`` = alternative output path."""
    lib = out or LIB
    if not force and out is None and not needs_build():
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tag = os.path.splitext(os.path.basename(lib))[0]
    objdir = os.path.join(OBJ, tag)
    os.makedirs(objdir, exist_ok=True)
    base = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + (extra or [])
    jobs = []
    for m in range(N_MODELS):
        for i in range(N_INTEG):
            o = os.path.join(objdir, f"raptor_render_m{m}_i{i}.o")
            jobs.append((base + [f"-DRAPTOR_MODEL={m}", f"-DRAPTOR_INTEG={i}", "-c",
                                 os.path.join(CSRC, "raptor_render.cu"), "-o", o], o))
    for src in ("raptor_kernels.cu", "raptor_flux_static.cu", "raptor_api.cu", "raptor_render_f32.cu"):
        o = os.path.join(objdir, src.replace(".cu", ".o"))
        jobs.append((base + ["-c", os.path.join(CSRC, src), "-o", o], o))
    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as pool:
        list(pool.map(lambda j: subprocess.check_call(j[0]), jobs))
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", lib] + [j[1] for j in jobs])
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
