"""Host logic of libge on the CPU: the tiling arithmetic of the blocked kernels (tiles, strips, units,
meetings) is compiled as host code from the kernels' own headers and checked exhaustively -- every output
node written by exactly one tile, every window inside the rod, every halo at least as wide as the nodes
that go stale.  No GPU needed."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_tiling_arithmetic(tmp_path):
    exe = str(tmp_path / "geometry_check")
    cmd = [os.environ.get("NVCC", "nvcc"), "-std=c++17", "-O1", "-gencode", "arch=compute_100a,code=sm_100a",
           "-I", os.path.join(ROOT, "include"), "-o", exe, os.path.join(ROOT, "tests", "geometry_check.cu")]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=900)
    assert r.returncode == 0, r.stdout[-3000:]
    r = subprocess.run([exe], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=300)
    sys.stdout.write(r.stdout[-2000:])
    assert r.returncode == 0 and "GEOMETRY OK" in r.stdout, r.stdout[-3000:]
