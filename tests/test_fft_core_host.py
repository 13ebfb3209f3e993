"""The FFT building blocks of the CUDA path, exercised on the CPU (no GPU needed): csrc/fft_core.cuh compiles as plain
C++, so fft32 (the 32-point register DFT) is checked against a naive fp64 DFT, and the index maps of the
register-resident transform kernels (mk_fft_fast.cu: four-step 1024 = 32 x 32 through a padded transposition, radix-2
split for nt = 4096) are replayed lane by lane against the definition of the DFT.  This is host logic of the product,
not the oracle: the oracle has no FFT at all."""
import subprocess
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent


def test_fft32_and_four_step_index_maps(tmp_path):
    exe = tmp_path / "fft_core_host"
    src = ROOT / "tests" / "host" / "fft_core_host.cpp"
    inc = ROOT / "paper_2106_04649_b200" / "csrc"
    subprocess.run(["g++", "-O1", "-std=c++17", f"-I{inc}", "-o", str(exe), str(src)], check=True)
    r = subprocess.run([str(exe)], capture_output=True, text=True)
    print(r.stdout)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "HF=2 forward(inverse) roundtrip" in r.stdout
