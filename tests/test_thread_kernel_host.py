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
