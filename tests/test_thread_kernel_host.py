"""Host logic of the CUDA path: the bit-parallel trial arithmetic of the thread-per-cell kernel
(gather by byte permutes, population counts, coefficient table, two-level acceptance filter, swap)
compiled for the host and checked against a brute-force energy difference on random tiles.
Independent of oracle/ (the check recomputes dE from unpacked species)."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "host_checks", "thread_trial_check.cu")


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", shutil.which("nvcc")):
        if cand and os.path.exists(cand):
            return cand
    return None


@pytest.mark.skipif(_nvcc() is None, reason="nvcc not available")
def test_trial_arithmetic_matches_brute_force(tmp_path):
    exe = str(tmp_path / "thread_trial_check")
    build = subprocess.run([_nvcc(), "-O1", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-o", exe, SRC],
                           capture_output=True, text=True, timeout=600)
    assert build.returncode == 0, build.stdout + build.stderr
    run = subprocess.run([exe], capture_output=True, text=True, timeout=600)
    assert run.returncode == 0, run.stdout + run.stderr
    last = run.stdout.strip().splitlines()[-1]
    assert "mismatches 0" in last, run.stdout
    # the run must have exercised acceptances, the near-threshold path and the unfiltered variant
    fields = dict(zip(["checked", "accepted", "near"], [int(s.split()[-1]) for s in
                  [last.split("checked ")[1].split(" trials")[0],
                   last.split("accepted ")[1].split(",")[0],
                   last.split("forced-near-threshold ")[1].split(",")[0]]]))
    assert fields["checked"] >= 1_000_000 and fields["accepted"] > 100_000 and fields["near"] > 10_000


@pytest.mark.skipif(_nvcc() is None, reason="nvcc not available")
def test_fcc_trial_arithmetic_matches_brute_force(tmp_path):
    """The packed FCC kernel's trial (sweep_fcc.cuh: sublattice-planar 4-bit tile, neighbours gathered by rotations and
    bit-selects, EPI differences by byte-permute look-ups) for every basis index, column, direction, 2..8 species, two
    and three shells, against a brute-force energy difference from the species at their positions."""
    src = os.path.join(ROOT, "tests", "host_checks", "fcc_trial_check.cu")
    exe = str(tmp_path / "fcc_trial_check")
    build = subprocess.run([_nvcc(), "-O1", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-o", exe, src],
                           capture_output=True, text=True, timeout=600)
    assert build.returncode == 0, build.stdout + build.stderr
    run = subprocess.run([exe], capture_output=True, text=True, timeout=600)
    assert run.returncode == 0, run.stdout + run.stderr
    last = run.stdout.strip().splitlines()[-1]
    assert "mismatches 0" in last, run.stdout
    checked = int(last.split("checked ")[1].split(" trials")[0])
    accepted = int(last.split("accepted ")[1].split(",")[0])
    near = int(last.split("forced-near-threshold ")[1].split(",")[0])
    assert checked >= 900_000 and accepted > 100_000 and near > 10_000


@pytest.mark.skipif(_nvcc() is None, reason="nvcc not available")
def test_bcc4_trial_arithmetic_matches_brute_force(tmp_path):
    """The packed BCC kernel for up to 8 species (sweep_bcc4.cuh: sublattice-planar 4-bit tile, nine row loads per site,
    byte-permute look-ups) for both sublattices, every column, direction, 2..8 species, one and two shells, against a
    brute-force energy difference from the species at their positions."""
    src = os.path.join(ROOT, "tests", "host_checks", "bcc4_trial_check.cu")
    exe = str(tmp_path / "bcc4_trial_check")
    build = subprocess.run([_nvcc(), "-O1", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-o", exe, src],
                           capture_output=True, text=True, timeout=600)
    assert build.returncode == 0, build.stdout + build.stderr
    run = subprocess.run([exe], capture_output=True, text=True, timeout=600)
    assert run.returncode == 0, run.stdout + run.stderr
    last = run.stdout.strip().splitlines()[-1]
    assert "mismatches 0" in last, run.stdout
    assert int(last.split("checked ")[1].split(" trials")[0]) >= 1_000_000
    assert int(last.split("accepted ")[1].split(",")[0]) > 100_000
