"""The C ABI from plain C: tests/c_client/abi_client.c (no Python, no torch; the CUDA runtime only for device memory)
is compiled with gcc against include/gdrr.h and libgdrr_b200.so, run on the GPU, and its printed signals are compared
with the oracle on the same formula-built inputs."""
import os
import shutil
import subprocess

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from parity_util import check_signal  # noqa: E402
from test_oracle_pins import tiny_workload  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_plain_c_client_matches_the_oracle(tmp_path):
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_1204_6367_b200 as g                      # (builds the library if it is missing)
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    exe = str(tmp_path / "abi_client")
    libdir = os.path.dirname(g.LIBRARY_PATH)
    cmd = [shutil.which("gcc") or "gcc", "-std=c99", "-O1", "-o", exe, os.path.join(ROOT, "tests", "c_client", "abi_client.c"),
           "-I", os.path.join(ROOT, "include"), "-I", os.path.join(cuda, "include"),
           "-L", libdir, "-lgdrr_b200", "-L", os.path.join(cuda, "lib64"), "-lcudart", "-lm",
           f"-Wl,-rpath,{libdir}", f"-Wl,-rpath,{os.path.join(cuda, 'lib64')}"]
    subprocess.run(cmd, check=True)
    out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout.splitlines()
    assert out[0].startswith("launches 2 sampler") and out[0].endswith("version " + g.gdrr_version())
    assert out[-1] == "host path identical 1"
    got = np.array([float(x) for x in out[1:-1]]).reshape(3, 30, 40)

    z, y, x = np.meshgrid(np.arange(16), np.arange(20), np.arange(24), indexing="ij")
    rho = (0.25 * ((x * 7 + y * 3 + z * 5) % 9)).astype(np.float32)
    mat = (((x + 2 * y + 3 * z) % 7) < 3).astype(np.uint8)
    w = tiny_workload(rho, mat, n_materials=2, spacing=(1.5, 1.5, 2.0), nu=40, nv=30, du=1.2, dv=1.2,
                      phis=[0.0, 0.7, 3.3], step=0.6, energies=np.array([40.0, 60.0, 80.0]),
                      mu_hat=np.array([[0.030, 0.022, 0.018], [0.060, 0.035, 0.025]]),
                      phi_weight=np.array([0.2, 0.5, 0.3]), response=np.array([0.6, 1.0, 1.4]))
    check_signal(got, oracle.project(w)["signal"], "C client")
