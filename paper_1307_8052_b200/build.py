"""Compile the CUDA libraries in-tree (sm_100a only, nvcc cross-compiles without a GPU):
paper_1307_8052_b200/librpa_chi0.so (the product, include/rpa_chi0.h) and paper_1307_8052_b200/librpa_probes.so (the
issue-rate probes bench.py divides by, include/rpa_probes.h).  Run as ``python -m paper_1307_8052_b200.build [--force]``."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librpa_chi0.so")
PROBES_LIB = os.path.join(HERE, "librpa_probes.so")
SOURCES = ["rpa_chi0.cu"]
HEADERS = ["common.cuh", "fft.cuh", "pair_density.cuh", "pair_density_zy.cuh", "orbitals.cuh", "optical.cuh", "paw.cuh", "rank_k.cuh", "rank_k3m.cuh", "energy.cuh", "probe_i8.cuh", "rank_k_i8.cuh",
           os.path.join("..", "..", "include", "rpa_chi0.h")]
PROBES_SOURCES = ["probes.cu"]
PROBES_HEADERS = ["probe_i8.cuh", os.path.join("..", "..", "include", "rpa_probes.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC",
              "-shared", "-Xptxas", "-v", "-diag-suppress", "20011,20013,20014,20015"]


def _stale(lib, deps) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in deps)


def _compile(lib, sources, headers, force, verbose) -> str:
    if not force and not _stale(lib, sources + headers):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", lib] + [os.path.join(CSRC, f) for f in sources]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building " + os.path.basename(lib))
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    return _compile(LIB, SOURCES, HEADERS, force, verbose)


def build_probes(force: bool = False, verbose: bool = False) -> str:
    return _compile(PROBES_LIB, PROBES_SOURCES, PROBES_HEADERS, force, verbose)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
    print(build_probes(force="--force" in sys.argv, verbose=True))
