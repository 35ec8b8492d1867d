"""CPU-only checks of the boundary: the C-ABI library builds, loads, and exports every symbol
include/*.h declare (no compute calls without a GPU)."""
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_02640_b200 import build
    build.build_library()
    from paper_2607_02640_b200 import binding
    return binding.load()


def _declared():
    text = "".join(open(os.path.join(ROOT, "include", f)).read() for f in sorted(os.listdir(os.path.join(ROOT, "include")))
                   if f.endswith(".h"))
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(metronome_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2607_02640_b200 import binding
    declared = _declared()
    assert set(declared) == set(binding.EXPORTS), (declared, binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    out = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    for name in declared:
        assert re.search(rf"\bT {name}\b", out), f"{name} is not an exported C symbol"


def test_host_only_entry_points(lib):
    from paper_2607_02640_b200 import binding
    assert lib.metronome_abi_version() == 3
    assert lib.metronome_strerror(5) == b"POOL_EXHAUSTED"
    # closed form of the per-session cap for the five configs
    for (S, W, n), want in {(4, 128, 8): 11, (4, 750, 1): 49, (4, 2048, 25): 132, (4, 1024, 25): 68,
                            (4, 2048, 13): 131}.items():
        assert binding.max_blocks_per_session(S, W, 16, n) == want
    assert binding.max_blocks_per_session(4, 0, 16, 1) == -1
    cfg = binding.PoolConfig(2, 32, 4, 128, 16, 4, 2048, 128, 25, 1000, 0.0, 0, 0, None, 0)
    assert lib.metronome_kv_storage_bytes(cfg) == 2 * 1000 * 4 * 2 * 16 * 128 * 2
    bad = binding.PoolConfig(1, 32, 5, 128, 16, 4, 2048, 128, 25, 1000, 0.0, 0, 0, None, 0)
    assert lib.metronome_kv_storage_bytes(bad) == 0


def test_sass_is_sm100a_only():
    from paper_2607_02640_b200 import binding
    out = subprocess.run(["cuobjdump", "--list-elf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out and "sm_90" not in out and "sm_80" not in out


def test_sass_census_shows_the_hardware_paths_each_kernel_claims():
    """the chunk kernel is tcgen05 (UTCHMMA) with TMEM loads / stores (LDTM / STTM) and bulk
    async copies (UBLKCP); the GQA decode kernel is mma.sync (HMMA) + ldmatrix + bulk copies; the row kernel
    is CUDA cores only (packed FFMA2, no tensor instruction)."""
    from paper_2607_02640_b200 import build
    build.build_library()
    c = build.sass_census()
    for D in (64, 128):
        u, g, r = c[f"attend_umma_kernel<{D}, false>"], c[f"attend_gqa_kernel<{D}, false>"], c[f"attend_rows_kernel<{D}, false>"]
        assert u.get("UTCHMMA", 0) > 0 and u.get("LDTM", 0) > 0 and u.get("STTM", 0) > 0 and u.get("UBLKCP", 0) > 0, u
        assert g.get("HMMA", 0) > 0 and g.get("LDSM", 0) > 0 and g.get("UBLKCP", 0) > 0 and "UTCHMMA" not in g, g
        uh = c[f"attend_umma_kernel<{D}, true>"]          # half-size variant (R <= 128 rows, two CTAs per SM): the same tcgen05 path
        assert uh.get("UTCHMMA", 0) > 0 and uh.get("LDTM", 0) > 0 and uh.get("STTM", 0) > 0 and uh.get("UBLKCP", 0) > 0, uh
        g8 = c[f"attend_gqa_kernel<{D}, true>"]         # fp8 KV tile: E4M3 -> fp16 conversions feed the same mma.sync path
        assert g8.get("HMMA", 0) > 0 and g8.get("LDSM", 0) > 0 and g8.get("UBLKCP", 0) > 0 and g8.get("F2FP.F16.E4M3", 0) > 0, g8
        assert r.get("FFMA2", 0) > 0 and "HMMA" not in r and "UTCHMMA" not in r, r


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_02640_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2607_02640_b200", text, flags=re.M), f
