"""Host logic of the CUDA path: the register butterflies (radix 2-8, 12) and the mixed-radix Stockham passes of
csrc/fft.cuh are __host__ __device__; tests/host/fft_host_check.cu runs them on the CPU against a direct DFT in
long double (Eq. 12, P:L104-106 needs a forward transform with exp(-2 pi i jk/N))."""
import os
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


@pytest.mark.skipif(not (os.path.exists(NVCC) or shutil.which("nvcc")), reason="nvcc not available")
def test_butterflies_and_lines_match_direct_dft(tmp_path):
    exe = str(tmp_path / "fft_host_check")
    src = os.path.join(HERE, "host", "fft_host_check.cu")
    r = subprocess.run([NVCC, "-O1", "-std=c++17", "--extended-lambda", "-o", exe, src], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    out = subprocess.run([exe], capture_output=True, text=True, check=True).stdout
    rows = [ln.split() for ln in out.strip().splitlines()]
    assert len(rows) == 8 + 13
    for kind, n, err in rows:
        err = float(err)
        assert err >= 0.0, (kind, n)
        tol = 1e-14 * max(4.0, float(n))
        assert err < tol, (kind, n, err)


@pytest.mark.skipif(not (os.path.exists(NVCC) or shutil.which("nvcc")), reason="nvcc not available")
def test_work_item_map_of_the_pair_density_kernel_matches_a_plain_walk(tmp_path):
    """pdzy_plan_units / pdzy_unit / pdzy_fastdiv (csrc/pair_density_zy.cuh): closed-form unit -> (row, first pair, count)
    map with magic-number divisions, against a walk over the pairs, for 60 000 random launches (starting mid-row, ending
    mid-row, single pairs, G = 1, 2, 4) and the launch shapes of the BASELINE configs."""
    exe = str(tmp_path / "unit_map_check")
    src = os.path.join(HERE, "host", "unit_map_check.cu")
    r = subprocess.run([NVCC, "-O1", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-diag-suppress", "20208", "-o", exe, src],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    out = subprocess.run([exe], capture_output=True, text=True)
    cases, bad = (int(x) for x in out.stdout.split())
    assert out.returncode == 0 and bad == 0 and cases == 60000, out.stdout


@pytest.mark.skipif(not (os.path.exists(NVCC) or shutil.which("nvcc")), reason="nvcc not available")
def test_tile_order_of_the_rank_k_kernel_is_a_permutation_sorted_by_work(tmp_path):
    """rk3_tile_order / rk3_tile_units (csrc/rank_k3m.cuh): every lower-triangle tile exactly once, work never increasing,
    the block count of a tile never below a plain walk over its elements; matrix sizes 1 ... 700 and those of the configs."""
    exe = str(tmp_path / "tile_order_check")
    src = os.path.join(HERE, "host", "tile_order_check.cu")
    r = subprocess.run([NVCC, "-O1", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-diag-suppress", "20208", "-o", exe, src],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    out = subprocess.run([exe], capture_output=True, text=True)
    sizes, bad = (int(x) for x in out.stdout.split())
    assert out.returncode == 0 and bad == 0 and sizes == 705, out.stdout
