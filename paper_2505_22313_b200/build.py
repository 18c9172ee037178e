"""Build the CUDA path (csrc/*.cu) into paper_2505_22313_b200/libdop.so for sm_100a with nvcc.

In-tree on purpose: the .so travels to the GPU box with the repo snapshot and is what the tests,
bench.py and __graft_entry__ load through ctypes.  nvcc cross-compiles without a GPU.
The register-blocked kernels are instantiated per (tile type, digit length) in separate objects
(pow2_inst.cu, once per entry of POW2_INST) so that they compile in parallel.
"""
from __future__ import annotations

import concurrent.futures
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdop.so")
OBJDIR = os.path.join(HERE, "build")
SOURCES = ["api.cu", "plan.cu", "kernels_generic.cu", "kernels_pow2.cu", "blur.cu", "noalloc.cu", "smooth.cu"]
# (column-type?, digit length) -- must match the DOP_DECL list in kernels_pow2.cu
POW2_INST = [(1, L) for L in (16, 32, 64, 128, 256, 512)] + \
            [(0, L) for L in (64, 128, 256, 512, 1024, 2048, 4096, 8192)]
POW2_X3 = (16, 32, 64, 128)  # digits 3 * LP
# (digit length, bundle width, pipeline depth) of the TMA column kernels -- must match DOP_TMA_LIST in kernels_pow2.cu
TMA_INST = [(16, 32, 3), (32, 32, 3), (64, 32, 3), (64, 16, 3), (128, 32, 3), (128, 16, 3), (256, 32, 2), (256, 16, 3), (256, 16, 2), (512, 16, 2),
            (96, 32, 3), (192, 32, 3), (384, 32, 2)]
CLUSTER_INST = [(4096, 2), (4096, 1), (2048, 4), (1024, 8)]  # (local transform length M, lines per CTA S): rows of 16 M
HEADERS = ["dop_internal.h", "bfly.cuh", "fft_regs.cuh", "pow2_impl.cuh", "cluster_row.cuh", "tma_col.cuh", os.path.join("..", "..", "include", "dop.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _units():
    """(object path, source path, extra flags) of every translation unit."""
    units = [(os.path.join(OBJDIR, s.replace(".cu", ".o")), os.path.join(CSRC, s), []) for s in SOURCES]
    for m, sl in CLUSTER_INST:
        units.append((os.path.join(OBJDIR, f"cluster_{m}_{sl}.o"), os.path.join(CSRC, "cluster_inst.cu"),
                      [f"-DDOP_INST_CLUSTER_M={m}", f"-DDOP_INST_CLUSTER_S={sl}"]))
    for L, nb, nst in TMA_INST:
        units.append((os.path.join(OBJDIR, f"tma_{L}_{nb}_{nst}.o"), os.path.join(CSRC, "tma_inst.cu"),
                      [f"-DDOP_INST_TMA_L={L}", f"-DDOP_INST_TMA_NB={nb}", f"-DDOP_INST_TMA_NST={nst}"]))
    for lp in POW2_X3:
        units.append((os.path.join(OBJDIR, f"pow2_x3_{lp}.o"), os.path.join(CSRC, "pow2_inst.cu"),
                      [f"-DDOP_INST_X3={lp}"]))
    for col, L in POW2_INST:
        units.append((os.path.join(OBJDIR, f"pow2_{'col' if col else 'row'}_{L}.o"),
                      os.path.join(CSRC, "pow2_inst.cu"), [f"-DDOP_INST_COL={col}", f"-DDOP_INST_L={L}"]))
    return units


def _dep_stamp() -> str:
    h = hashlib.sha256()
    for d in [os.path.join(CSRC, s) for s in SOURCES + HEADERS + ["pow2_inst.cu", "cluster_inst.cu", "tma_inst.cu"]] + [os.path.abspath(__file__)]:
        with open(d, "rb") as f:
            h.update(f.read())
    h.update((" ".join(NVCC_FLAGS) + os.environ.get("DOP_NVCC_EXTRA", "")).encode())
    return h.hexdigest()


def source_stamp() -> str:
    """Hash of the kernel sources only (csrc/ + include/dop.h): what an ncu capture is valid for."""
    h = hashlib.sha256()
    for d in sorted(os.listdir(CSRC)) + [os.path.join("..", "..", "include", "dop.h")]:
        with open(os.path.join(CSRC, d), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def _stale() -> bool:
    stamp = os.path.join(OBJDIR, "stamp")
    if not os.path.exists(LIB) or not os.path.exists(stamp):
        return True
    with open(stamp) as f:
        return f.read().strip() != _dep_stamp()


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if libdop.so is missing or its sources changed; return its path."""
    if not force and not _stale():
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    nvcc = _nvcc()
    extra = ["-Xptxas", "-v"] if verbose else []
    extra += os.environ.get("DOP_NVCC_EXTRA", "").split()  # tuning experiments, e.g. -DDOP_RESIDENT_THREADS=1024

    def compile_one(u):
        obj, src, flags = u
        r = subprocess.run([nvcc] + NVCC_FLAGS + extra + flags + ["-c", src, "-o", obj],
                           capture_output=True, text=True)
        return u, r

    units = _units()
    workers = max(1, min(len(units), os.cpu_count() or 4))
    with concurrent.futures.ThreadPoolExecutor(workers) as ex:
        for u, r in ex.map(compile_one, units):
            if verbose or r.returncode != 0:
                sys.stderr.write(f"== {os.path.basename(u[0])}\n{r.stdout}{r.stderr}")
            if r.returncode != 0:
                raise RuntimeError(f"nvcc failed for {u[0]}")
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.run([nvcc, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a",
                    "-o", tmp] + [u[0] for u in units], check=True)
    os.replace(tmp, LIB)
    with open(os.path.join(OBJDIR, "stamp"), "w") as f:
        f.write(_dep_stamp())
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
