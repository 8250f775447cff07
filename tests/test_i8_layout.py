"""The tensor-core engine's operand images and MMA sequence, checked on the host (no GPU).

tests/i8_layout_harness.cu is compiled by nvcc as a HOST program: it builds the A and B images with the very functions
i8_prep_kernel uses (paper_1302_4000_b200/csrc/i8_layout.cuh), plays gram_i8tc_kernel's MMA sequence on a plain model of
the instruction and compares every accumulator entry, at the place the epilogue reads it, with the level sums taken
directly from the integers -- for every k-step count, on ragged N."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


@pytest.fixture(scope="module")
def harness(tmp_path_factory):
    if not (os.path.exists(NVCC) or shutil.which("nvcc")):
        pytest.fail("nvcc not found: the layout harness is compiled from the product's own header")
    exe = str(tmp_path_factory.mktemp("i8h") / "i8_layout_harness")
    cmd = [NVCC if os.path.exists(NVCC) else "nvcc", "-std=c++17", "-O2", "--expt-relaxed-constexpr",
           "-Wno-deprecated-gpu-targets", "-o", exe, os.path.join(ROOT, "tests", "i8_layout_harness.cu")]
    r = subprocess.run(cmd, capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
    return exe


# (N, L): every k-step count 1..8, full and ragged last k-steps; ragged N so that the last row and column tiles are partial;
# 100 = C4's chain length, 36 / 71 / 108 / 140 / 215 / 250 appear in the paper
CASES = [(40, 1), (50, 4), (45, 32), (33, 36), (33, 64), (45, 71), (40, 96), (70, 100), (33, 108), (37, 128), (37, 129),
         (33, 140), (35, 160), (34, 161), (33, 193), (33, 215), (33, 225), (40, 250), (35, 256)]


@pytest.mark.parametrize("N,L", CASES)
def test_images_and_mma_sequence_give_the_level_sums(harness, N, L):
    r = subprocess.run([harness, str(N), str(L), str(7 * N + L)], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.startswith("OK") and f"ksteps={(L + 31) // 32} " in r.stdout, r.stdout
