"""Index arithmetic of the FFT tile kernel bodies, run on the host (one std::thread per CUDA thread)
against a naive double-precision DFT.  See tests/host_emulation_test.cpp (the kernel bodies are included from paper_2410_02395_b200/csrc)."""
import os
import shutil
import subprocess
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2410_02395_b200", "csrc")


@pytest.mark.skipif(shutil.which("g++") is None, reason="no host compiler")
def test_fft_bodies_on_host():
    with tempfile.TemporaryDirectory() as tmp:
        exe = os.path.join(tmp, "mbs_host_emu")
        r = subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-I", CSRC,
                            os.path.join(ROOT, "tests", "host_emulation_test.cpp"), "-o", exe],
                           capture_output=True, text=True)
        assert r.returncode == 0, r.stderr[-4000:]
        r = subprocess.run([exe], capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stdout[-4000:]
        assert "HOST EMULATION PASSED" in r.stdout
