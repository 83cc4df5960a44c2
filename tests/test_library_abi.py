"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/rpa_chi0.h
declares; argument validation that needs no GPU; the product path refuses to run without CUDA."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1307_8052_b200 import binding as B
from paper_1307_8052_b200 import build as cuda_build
from paper_1307_8052_b200 import workload as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols(header="rpa_chi0.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rpa_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    path = cuda_build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    names = _declared_symbols()
    assert len(names) >= 14
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/rpa_chi0.h but not exported"
    assert sorted(B.EXPORTS) == names, "binding.EXPORTS out of sync with the header"


def test_probe_library_builds_and_exports_every_declared_symbol():
    """include/rpa_probes.h is the bench-only helper library: its symbols live in librpa_probes.so, none in the product."""
    from paper_1307_8052_b200 import probes
    path = cuda_build.build_probes()
    lib = ctypes.CDLL(path)
    names = _declared_symbols("rpa_probes.h")
    assert names == sorted(probes.EXPORTS)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/rpa_probes.h but not exported"
    product = ctypes.CDLL(cuda_build.build())
    for n in names:
        assert not hasattr(product, n), f"{n} must not be exported by librpa_chi0.so"


def test_library_keeps_no_process_global_switches():
    """no global state except the thread-local error string -- kernel choice is an explicit setter
    (rpa_chi0_set_rank_k_mode, rpa_chi0_set_ec_lanes), never an environment variable."""
    csrc = os.path.join(ROOT, "paper_1307_8052_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f


def test_total_energy_is_the_weighted_q_sum():
    """rpa_total_energy (Eq. 1): host arithmetic behind the C ABI, so it runs without a GPU."""
    assert B.rpa_total_energy([-0.5, -0.25, 1.0], [0.125, 0.375, 0.5]) == -0.5 * 0.125 - 0.25 * 0.375 + 0.5
    assert B.rpa_total_energy([], []) == 0.0
    out = ctypes.c_double(7.0)
    assert B.lib().rpa_total_energy(2, None, None, ctypes.byref(out)) == B.RPA_ERR_INVALID_ARG
    assert B.lib().rpa_total_energy(-1, None, None, ctypes.byref(out)) == B.RPA_ERR_INVALID_ARG
    with pytest.raises(ValueError):
        B.rpa_total_energy([1.0], [0.5, 0.5])


def test_library_is_sm100a_with_dmma_and_bulk_copies():
    """The rank-K kernel must carry FP64 tensor-core and TMA-engine instructions in its sm_100a SASS."""
    import subprocess
    try:
        out = subprocess.run(["cuobjdump", "-sass", cuda_build.build()], capture_output=True, text=True)
    except OSError:
        pytest.skip("cuobjdump unavailable")
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in out.stdout
    body = out.stdout.split("rank_k_kernel", 1)[1].split("Function :", 1)[0]
    assert body.count("DMMA") >= 256   # 8 k-steps x 32 DMMA.8x8x4, fully unrolled
    assert "UBLKCP" in body            # cp.async.bulk on the TMA engine
    k3m = out.stdout.split("rank_k3m_kernel", 1)[1].split("Function :", 1)[0]
    assert k3m.count("DMMA") >= 4 * 24   # the chi0 accumulation: 4 k-steps x 24 DMMA.8x8x4 per 16-pair chunk, unrolled
    assert "UTMALDG" in k3m            # cp.async.bulk.tensor: the N tiles arrive through a 2-D tensor map
    i8 = out.stdout.split("rank_k_i8_kernel", 1)[1].split("Function :", 1)[0]
    assert i8.count("UTCIMMA") >= 8    # tcgen05.mma.kind::i8: 8 (6 digits) or 10 (7 digits) wide MMAs per K block
    assert "UBLKCP" in i8


def test_workspace_bytes_host_only():
    cfg = W.CONFIGS[0]
    n = B.rpa_chi0_workspace_bytes(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), cfg.n_omega, 0, 8)
    ng = 155
    assert n >= cfg.n_omega * ng * ng * 16
    # more omega, more batch, more projectors: never smaller
    assert B.rpa_chi0_workspace_bytes(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), 16, 0, 8) > n
    assert B.rpa_chi0_workspace_bytes(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), cfg.n_omega, 16384, 8) > n
    assert B.rpa_chi0_workspace_bytes(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), cfg.n_omega, 0, 64) > n


@pytest.mark.parametrize("bad", ["grid", "ecut", "omega", "cell", "proj"])
def test_workspace_bytes_rejects_invalid(bad):
    cfg = W.CONFIGS[0]
    grid, cell, ecut, nw, proj = list(cfg.grid), cfg.cell.copy(), W.tuned_ecut(cfg), 8, 8
    if bad == "grid":
        grid[1] = 0
    elif bad == "ecut":
        ecut = -1.0
    elif bad == "omega":
        nw = 0
    elif bad == "cell":
        cell[2] = cell[1]
    else:
        proj = -3
    with pytest.raises(B.RpaError) as ei:
        B.rpa_chi0_workspace_bytes(grid, cell, cfg.q_red, ecut, nw, 0, proj)
    assert ei.value.code == B.RPA_ERR_INVALID_ARG
    assert "rpa_chi0_workspace_bytes" in B.rpa_last_error()


def test_null_handle_calls_return_invalid_arg():
    lib = B.lib()
    n = ctypes.c_int32()
    assert lib.rpa_chi0_ng(None, ctypes.byref(n)) == B.RPA_ERR_INVALID_ARG
    assert lib.rpa_chi0_reset(None) == B.RPA_ERR_INVALID_ARG
    assert lib.rpa_chi0_sync(None) == B.RPA_ERR_INVALID_ARG
    assert lib.rpa_chi0_get(None, 0, None) == B.RPA_ERR_INVALID_ARG
    lib.rpa_chi0_destroy(None)  # no-op
    assert isinstance(B.rpa_last_error(), str)


def test_create_rejects_bad_workspace_and_omega_without_gpu():
    """Validation happens before any CUDA call, so these run on the CPU box."""
    lib = B.lib()
    cfg = W.CONFIGS[0]
    g = np.asarray(cfg.grid, dtype=np.int32)
    c = np.ascontiguousarray(cfg.cell).reshape(9)
    om, wt = W.omega_grid(4)
    out = ctypes.c_void_p()

    def create(q, ws, nbytes, omega=om):
        qa = np.asarray(q, dtype=np.float64)
        return lib.rpa_chi0_create(ctypes.byref(out), g.ctypes.data_as(ctypes.c_void_p), c.ctypes.data_as(ctypes.c_void_p),
                                   qa.ctypes.data_as(ctypes.c_void_p), W.tuned_ecut(cfg), 4,
                                   omega.ctypes.data_as(ctypes.c_void_p), wt.ctypes.data_as(ctypes.c_void_p), 0, 0, ws,
                                   ctypes.c_size_t(nbytes), None)

    # q = 0 is accepted since the optical limit (NEXT-2) exists: the same workspace checks apply to it
    assert create((0.0, 0.0, 0.0), None, 1 << 40) == B.RPA_ERR_WORKSPACE
    assert create(cfg.q_red, None, 1 << 40) == B.RPA_ERR_WORKSPACE
    assert create(cfg.q_red, ctypes.c_void_p(8), 1 << 40) == B.RPA_ERR_WORKSPACE  # misaligned
    assert create(cfg.q_red, ctypes.c_void_p(256), 16) == B.RPA_ERR_WORKSPACE     # too small
    bad_om = om.copy()
    bad_om[2] = 0.0
    assert create(cfg.q_red, ctypes.c_void_p(256), 1 << 40, bad_om) == B.RPA_ERR_INVALID_ARG
    assert out.value is None


def test_product_path_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    cfg = W.CONFIGS[0]
    om, wt = W.omega_grid(cfg.n_omega)
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)


def test_product_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package may import or load it."""
    pkg = os.path.join(ROOT, "paper_1307_8052_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "rpa_oracle" not in txt, f
