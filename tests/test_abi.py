"""Host-side checks that need no GPU: the C-ABI library builds for sm_100a, loads, and exports
every symbol include/ps_poisson.h declares; argument validation that happens before any CUDA
call; the product package never touches the oracle."""
import ctypes
import os
import re

import pytest

from paper_2104_01636_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def declared_symbols():
    with open(os.path.join(ROOT, "include", "ps_poisson.h")) as f:
        text = f.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ps_[a-z_]+)\s*\(", text)))


def test_header_and_binding_agree():
    assert declared_symbols() == sorted(binding.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_sass_is_sm100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", build.LIB], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_strerror(lib):
    assert lib.ps_strerror(0) == b"ok"
    assert b"invalid" in lib.ps_strerror(binding.PS_EINVAL)
    assert b"ps_set_fraction" in lib.ps_strerror(binding.PS_ESTATE)


@pytest.mark.parametrize("args", [
    (0, 4, 4, 1.0, 1.0, 1.0),          # nx < 1
    (4, 0, 4, 1.0, 1.0, 1.0),          # ny < 1
    (4, 4, 0, 1.0, 1.0, 1.0),          # nz < 2
    (4, 4, 5, 1.0, 1.0, 1.0),          # odd nz: colouring breaks across the periodic wrap
    (4, 4, 4, 0.0, 1.0, 1.0),          # dx <= 0
    (4, 4, 4, 1.0, -1.0, 1.0),
    (4, 4, 4, 1.0, 1.0, float("nan")),
    (4, 4, 4, 1.0, float("inf"), 1.0),
])
def test_create_rejects_bad_arguments_before_touching_cuda(lib, args):
    h = ctypes.c_void_p()
    assert lib.ps_create(ctypes.byref(h), *args) == binding.PS_EINVAL
    assert not h.value


def test_null_handles(lib):
    assert lib.ps_create(None, 4, 4, 4, 1.0, 1.0, 1.0) == binding.PS_EINVAL
    assert lib.ps_destroy(None) == binding.PS_OK
    assert lib.ps_workspace_bytes(None) == 0
    assert lib.ps_set_check_interval(None, 10) == binding.PS_EINVAL
    assert lib.ps_solve(None, None, None, 1.5, 1, 0.0, None) == binding.PS_EINVAL
    assert lib.ps_launch_count(None) == 0


def test_no_gpu_means_error_not_fallback(lib):
    """Without a device ps_create must fail with PS_ECUDA (never silently compute on the CPU)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = ctypes.c_void_p()
    assert lib.ps_create(ctypes.byref(h), 8, 8, 8, 1.0, 1.0, 1.0) == binding.PS_ECUDA
    assert b"CUDA error" in lib.ps_strerror(binding.PS_ECUDA)


def test_binding_raises_without_library(tmp_path):
    with pytest.raises(RuntimeError, match="no fallback"):
        binding.load(str(tmp_path / "libps_poisson.so"))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2104_01636_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, fn)) as f:
                    src = f.read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), fn
                assert "ps_oracle" not in src and "ora_" not in src, fn
    with open(os.path.join(ROOT, "include", "ps_poisson.h")) as f:
        assert "ps_oracle" not in f.read()


@pytest.mark.parametrize("shape", [(256, 256, 512), (128, 128, 256), (384, 384, 1024), (64, 64, 128),
                                   (32, 32, 64), (186, 46, 8), (130, 44, 4), (2, 2, 2), (66, 17, 6)])
@pytest.mark.parametrize("z_chunks", [0, 1, 3])
def test_fused_work_split_covers_every_plane_once_and_is_balanced(lib, shape, z_chunks):
    """Host logic of the fused kernel's launch (ps_fused_plan, no GPU): the tiles partition the
    cross-section within the box capacities; the items cover every (tile, plane) exactly once, are
    grouped per CTA in launch order, have at least 2 planes; and with the automatic split
    (z_chunks = 0: lockstep rounds of tile x chunk items, the leftover of the last round cut again
    into one range per CTA) no CTA marches more than a few percent above the mean."""
    nx, ny, nz = shape
    if z_chunks > nz // 2:
        pytest.skip("more chunks than plane pairs")
    tiles, items = binding.fused_plan(nx, ny, nz, 148, z_chunks)
    cover = {}
    for xs, xe, ys, ye in tiles:
        assert 0 <= xs < xe <= nx and xs % 2 == 0 and xe % 2 == 0 and xe - xs <= 64
        assert 0 <= ys < ye <= ny
        rows = (ye - ys) + (ys > 0) + (ye < ny)              # owned rows + red-ring rows
        assert rows <= 16
        for i in range(xs, xe, 2):
            for j in range(ys, ye):
                assert (i, j) not in cover
                cover[(i, j)] = 1
    assert len(cover) == (nx // 2) * ny
    seen = [[0] * nz for _ in tiles]
    steps = {}
    last_cta = -1
    for cta, tile, ks, ke in items:
        assert cta in (last_cta, last_cta + 1)               # grouped per CTA, CTAs in order
        last_cta = cta
        assert 0 <= ks < ke <= nz and ke - ks >= 2
        for k in range(ks, ke):
            seen[tile][k] += 1
        steps[cta] = steps.get(cta, 0) + (ke - ks) + 3
    assert all(v == 1 for row in seen for v in row)
    assert 1 <= len(steps) <= 148
    if z_chunks == 0:
        mean = len(tiles) * nz / len(steps)
        assert max(steps.values()) <= 1.04 * mean + 9, (max(steps.values()), mean)


def test_fused_plan_rejects_odd_nx(lib):
    import ctypes as ct
    n = [ct.c_int() for _ in range(3)]
    assert lib.ps_fused_plan(5, 7, 6, 148, 0, None, 0, None, 0, *[ct.byref(x) for x in n]) == binding.PS_EINVAL
