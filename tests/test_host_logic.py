"""CPU-only checks of host logic that the kernels share with the launcher (no GPU, no compute calls)."""
import os
import subprocess
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_gqa_ranges_partition_the_tile_list():
    """GqaPlan (host + device struct of the GQA decode kernel): static ranges, then the small dynamically
    claimed ones, must tile [0, total) exactly and range_of() must invert them; brute force on 20 000
    seeded (total, CTA count) pairs, compiled with nvcc as a host program."""
    src = os.path.join(ROOT, "tests", "native", "gqa_plan_check.cu")
    with tempfile.TemporaryDirectory() as d:
        exe = os.path.join(d, "gqa_plan_check")
        subprocess.run([os.environ.get("NVCC", "nvcc"), "-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O1",
                        "-o", exe, src], check=True)
        out = subprocess.run([exe], capture_output=True, text=True)
        assert out.returncode == 0, out.stdout + out.stderr
        assert "0 bad" in out.stdout
