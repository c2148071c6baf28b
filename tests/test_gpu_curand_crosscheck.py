"""Pin P1's optional cross-check: the oracle's Philox4x32-10 against cuRAND's Philox device generator,
a third implementation neither side of the parity contract was written from.  cuRAND's state is (key = seed,
counter = 128-bit block number advanced by offset / 4 within subsequence): curand_init(seed, subsequence, offset) followed
by curand4 returns block  ctr = {offset/4 lo, offset/4 hi, subsequence lo, subsequence hi},  key = {seed lo, seed hi}  --
exactly the layout of DESIGN.md R6 with subsequence = step and offset = 4 * storage index."""
import os
import shutil
import subprocess

import pytest

import oracle

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_philox_equals_curand_philox4_32_10(tmp_path):
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available on this box")
    exe = str(tmp_path / "curand_probe")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-o", exe,
                    os.path.join(HERE, "curand_philox_probe.cu")], check=True)
    cases = [(0, 0, 0), (0, 0, 4), (7, 3, 4 * 12345), (0xDEADBEEFCAFEF00D, 3599, 4 * (2 ** 26 - 1)),
             (2 ** 64 - 1, 2 ** 40 + 17, 4 * (2 ** 33 + 5))]
    args = [str(x) for c in cases for x in c]
    out = subprocess.run([exe] + args, check=True, capture_output=True, text=True).stdout.strip().splitlines()
    assert len(out) == len(cases)
    for (seed, sub, off), line in zip(cases, out):
        words = [int(w, 16) for w in line.split()[3:]]
        i = off // 4
        ctr = [i & 0xFFFFFFFF, i >> 32, sub & 0xFFFFFFFF, (sub >> 32) & 0xFFFFFFFF]
        key = [seed & 0xFFFFFFFF, seed >> 32]
        assert [int(x) for x in oracle.philox4x32_10(ctr, key)] == words, (seed, sub, off)
