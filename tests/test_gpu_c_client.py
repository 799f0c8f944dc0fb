"""The C ABI used from C: tests/c_client/lm_client.c is compiled with gcc against include/lm.h and liblm.so (plus the
CUDA runtime for cudaMalloc / cudaMemcpy) and run as its own process -- no Python, no torch on the path.  It checks the
closed forms the paper and the textbook fix (self mobilities, two-sphere sedimentation, M^{1/2} of one sphere) and the
error codes."""
import json
import os
import subprocess

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_c_client(tmp_path):
    from paper_2510_02135_b200 import build
    lib = build.build()
    exe = str(tmp_path / "lm_client")
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    subprocess.run(["gcc", "-O1", "-std=c99", "-o", exe, os.path.join(ROOT, "tests", "c_client", "lm_client.c"), "-I", os.path.join(cuda, "include"),
                    lib, "-L", os.path.join(cuda, "lib64"), "-lcudart", "-lm", "-Wl,-rpath," + os.path.dirname(lib), "-Wl,-rpath," + os.path.join(cuda, "lib64")],
                   check=True)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "lm_client: OK" in r.stdout
    # the same client times lm_mdot called back to back from C (what the library costs without Python marshalling)
    t = subprocess.run([exe, "--time"], capture_output=True, text=True, timeout=300)
    assert t.returncode == 0, t.stdout + t.stderr
    rows = [json.loads(line) for line in t.stdout.splitlines() if line.startswith("{")]
    assert len(rows) == 10 and all(0.5 < row["us_per_mdot_from_c"] < 500 for row in rows), rows
    print("\n".join(json.dumps(row) for row in rows))
