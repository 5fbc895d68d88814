"""The C-ABI library builds, loads and exports every symbol include/dmrgk.h declares (no compute
calls without a GPU); the product path fails loudly when no CUDA device is present."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "dmrgk.h")
HARNESS_HEADER = os.path.join(ROOT, "include", "dmrgk_harness.h")      # test / measurement aids of the same library


@pytest.fixture(scope="module")
def lib():
    from paper_2311_14106_b200 import build, dmrgk
    build.build()
    return dmrgk.load()


def declared_symbols():
    src = open(HEADER, encoding="utf-8").read() + open(HARNESS_HEADER, encoding="utf-8").read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dmrgk_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert len(names) >= 40
    for n in names:
        assert hasattr(lib, n), f"{n} declared in dmrgk.h but not exported by libdmrgk.so"


def test_binding_covers_the_header(lib):
    from paper_2311_14106_b200 import dmrgk
    assert sorted(dmrgk.SIGNATURES) == declared_symbols()


def test_version_and_status_codes(lib):
    from paper_2311_14106_b200 import dmrgk
    assert b"sm_100a" in lib.dmrgk_version()
    src = open(HEADER, encoding="utf-8").read()
    for name in ("EINVAL", "ESHAPE", "ECHARGE", "EALIGN", "ENOMEM", "ECUDA", "ENOTCONV", "ESTATE"):
        m = re.search(rf"DMRGK_{name}\s*=\s*(-?\d+)", src)
        assert int(m.group(1)) == getattr(dmrgk, name)


def test_no_cpu_fallback(lib):
    """Without a CUDA device ctx_create reports DMRGK_ECUDA; nothing computes on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2311_14106_b200 import dmrgk
    with pytest.raises(dmrgk.DmrgkError) as e:
        dmrgk.Ctx(0)
    assert e.value.status == dmrgk.ECUDA
    assert "no CPU fallback" in e.value.message


def test_null_handles_are_rejected(lib):
    """Argument validation that needs no device."""
    from paper_2311_14106_b200 import dmrgk
    assert lib.dmrgk_space_create(None, 1, 0, None, None, ctypes.byref(ctypes.c_void_p())) == dmrgk.EINVAL
    assert lib.dmrgk_heff_apply(None, None, None, None, None, None) == dmrgk.EINVAL
    assert lib.dmrgk_davidson_step(None, None, None, None) == dmrgk.EINVAL
    assert b"NULL" in lib.dmrgk_last_error()
    lib.dmrgk_heff_destroy(None)
    lib.dmrgk_davidson_destroy(None)
    assert lib.dmrgk_vec_scratch_bytes(4) % 128 == 0


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2311_14106_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f), encoding="utf-8").read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            text = open(os.path.join(ROOT, "oracle", f), encoding="utf-8").read()
            assert "paper_2311_14106_b200" not in re.sub(r'""".*?"""', "", text, flags=re.S), f


def test_balanced_tile_plan_host_rules():
    """The planner's tiling rules (DESIGN.md §4.1 "balanced tiles"), host only: ceil(extent/tile_max) tiles that
    cover the extent exactly, origins at multiples of 16, extents ≤ tile_max that differ by at most 16 with the
    larger ones first; the cost of a tile = fragment products of its fullest warp × 4 with a floor."""
    from paper_2311_14106_b200 import dmrgk
    for tile_max in (64, 128):
        for extent in list(range(0, 300)) + [573, 640, 650, 794, 1000, 4096]:
            cuts = dmrgk.plan_tile_cuts(extent, tile_max)
            n = len(cuts) - 1
            assert n == -(-extent // tile_max) and cuts[0] == 0 and cuts[-1] == extent
            ext = [b - a for a, b in zip(cuts[:-1], cuts[1:])]
            assert all(0 < e <= tile_max for e in ext) and all(c % 16 == 0 for c in cuts[:-1])
            if n:
                full = [-(-e // 16) for e in ext]                       # in 16-row panels
                assert max(full) - min(full) <= 1 and full == sorted(full, reverse=True)
    assert dmrgk.plan_tile_cuts(650) == [0, 64, 128, 192, 256, 320, 384, 448, 512, 560, 608, 650]
    assert dmrgk.plan_tile_cost(64, 64) == 64 and dmrgk.plan_tile_cost(48, 64) == 48 and dmrgk.plan_tile_cost(52, 64) == 64
    assert dmrgk.plan_tile_cost(128, 64) == 128 and dmrgk.plan_tile_cost(8, 8) == dmrgk.plan_tile_cost(1, 1) == 24   # the floor
    with pytest.raises(dmrgk.DmrgkError):
        dmrgk.plan_tile_cuts(10, 32)


def test_build_is_serialised_by_a_file_lock():
    """Several processes may call build() at once (torchrun ranks, parallel test workers): it runs under an
    exclusive lock on _build/.lock.  While this process holds that lock a second process's build() waits; once
    released it returns the library path (nothing to recompile: the stamps are current)."""
    import fcntl
    import subprocess
    import sys
    import time
    from paper_2311_14106_b200 import build as b
    b.build()
    with open(os.path.join(b.OUT, ".lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        p = subprocess.Popen([sys.executable, "-c", "from paper_2311_14106_b200 import build as b; print(b.build())"],
                             cwd=ROOT, stdout=subprocess.PIPE, text=True)
        time.sleep(3.0)
        assert p.poll() is None                     # still waiting for the lock
        fcntl.flock(lock, fcntl.LOCK_UN)
    out, _ = p.communicate(timeout=120)
    assert p.returncode == 0 and out.strip().endswith("libdmrgk.so")
    assert b.built_hash() == b.source_hash()
    assert not [f for f in os.listdir(b.OUT) if ".tmp" in f]
