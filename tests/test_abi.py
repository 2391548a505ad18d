"""CPU-side checks of the C-ABI boundary (include/corr.h): the library builds, loads and exports
every declared symbol; the host logic (baseline index, triangular tile schedule, argument
validation) behaves as the header says.  No kernel is launched here (-m "not gpu").
"""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "corr.h")


@pytest.fixture(scope="module")
def binding():
    from paper_1305_5639_b200 import binding as b
    b.lib()          # nvcc cross-compiles here if the .so is stale
    return b


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)          # strip comments
    return sorted(set(re.findall(r"\b(corr_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported_and_bound(binding):
    names = declared_symbols()
    assert "corr_create" in names and "corr_xengine" in names and "corr_destroy" in names
    raw = ctypes.CDLL(binding.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), "libcorr.so does not export %s" % n
        assert n in binding.SYMBOLS, "binding.py does not bind %s" % n
    # and the binding binds nothing the header does not declare
    assert sorted(binding.SYMBOLS) == names


def test_baseline_index_matches_header(binding):
    # b(i,j) = i(i+1)/2 + j for 0 <= j <= i, else -1 (corr.h)
    b = 0
    for i in range(40):
        for j in range(i + 1):
            assert binding.baseline_index(i, j) == b
            b += 1
    assert binding.baseline_index(3, 4) == -1
    assert binding.baseline_index(3, -1) == -1
    assert binding.baseline_index(65535, 65535) == 65535 * 65536 // 2 + 65535


@pytest.mark.parametrize("N,P,dtype", [(1, 1, "ci8"), (1, 2, "cf16"), (16, 2, "ci8"), (33, 2, "ci8"),
                                       (64, 2, "ci8"), (100, 1, "cf16"), (128, 2, "cf16"),
                                       (256, 2, "ci8"), (300, 2, "ci8"), (1024, 2, "ci8")])
def test_tile_schedule_covers_lower_triangle_exactly_once(binding, N, P, dtype):
    """Every needed real-component product (u, v) -- u on the conjugated side, station(u) >= station(v) --
    lies in exactly one tile, and no tile is entirely above the block diagonal."""
    tiles = binding.tile_schedule(N, P, dtype, "single")
    M2 = 2 * N * P
    cover = np.zeros((M2, M2), dtype=np.int16) if M2 <= 2048 else None
    for row0, col0, ncols in tiles:
        assert row0 % 128 == 0 and col0 % 16 == 0 and 16 <= ncols <= 256 and ncols % 16 == 0
        assert row0 < M2 and col0 < M2
        last_station_of_rows = (min(row0 + 128, M2) - 1) // (2 * P)
        assert col0 // (2 * P) <= last_station_of_rows          # the tile touches the triangle
        if cover is not None:
            cover[row0:row0 + 128, col0:col0 + ncols] += 1
    if cover is not None:
        st = np.arange(M2) // (2 * P)
        need = st[:, None] >= st[None, :]
        assert (cover[need] == 1).all()
        assert cover.max() <= 1
    # executed area is at most ~2.2x the needed area for any N >= 64, and tends to 1
    if N >= 64:
        executed = sum(128 * n for _, _, n in tiles)
        needed = (2 * P) ** 2 * N * (N + 1) // 2
        assert executed < 2.2 * needed


@pytest.mark.parametrize("N,P", [(1, 1), (16, 2), (33, 2), (64, 2), (96, 2), (100, 1), (256, 2), (300, 2), (512, 2), (1024, 2)])
def test_pair_tile_schedule_covers_lower_triangle_exactly_once(binding, N, P):
    """256 x 256 pair tiles: every 256-block of the Gram matrix touching the lower station triangle appears exactly once,
    column-block major (tiles that share their columns are neighbours in the feed order)."""
    tiles = binding.tile_schedule(N, P, "ci8", "pair")
    M2 = 2 * N * P
    R = -(-M2 // 256)
    assert [(r, c) for r, c, _ in tiles] == [(256 * rb, 256 * cb) for cb in range(R) for rb in range(cb, R)]
    assert all(n == 256 for _, _, n in tiles)


def test_tile_schedule_rejects_bad_arguments(binding):
    L = binding.lib()
    assert L.corr_tile_schedule(0, 2, 0, 1, None, 0) == binding.CORR_EINVAL
    assert L.corr_tile_schedule(4, 3, 0, 1, None, 0) == binding.CORR_EINVAL
    assert L.corr_tile_schedule(4, 2, 7, 1, None, 0) == binding.CORR_EINVAL
    assert L.corr_tile_schedule(4, 2, 0, 1, None, 5) == binding.CORR_EINVAL   # max_tiles > 0 with NULL
    assert L.corr_tile_schedule(4, 2, 0, 0, None, 0) == binding.CORR_EINVAL   # AUTO / SIMT have no tile schedule
    assert L.corr_tile_schedule(4, 2, 0, 3, None, 0) == binding.CORR_EINVAL


def test_null_handle_helpers_are_safe(binding):
    L = binding.lib()
    assert L.corr_input_bytes(None) == 0
    assert L.corr_output_bytes(None) == 0
    assert L.corr_workspace_bytes(None) == 0
    assert L.corr_xengine(None, None, None, 0, None) == binding.CORR_EINVAL
    assert L.corr_xengine_host(None, None, None, 0) == binding.CORR_EINVAL
    assert L.corr_set_kernel(None, 0) == binding.CORR_EINVAL
    assert L.corr_get_kernel(None) == binding.CORR_EINVAL
    L.corr_destroy(None)     # no-op


def test_create_rejects_bad_geometry_without_touching_the_gpu(binding):
    L = binding.lib()
    for args in [(0, 2, 4, 4, 0), (4, 3, 4, 4, 0), (4, 2, 0, 4, 0), (4, 2, 4, 0, 0), (4, 2, 4, 4, 9),
                 (-1, 1, 1, 1, 0)]:
        assert not L.corr_create(*args)
        assert b"invalid geometry" in L.corr_last_error(None)


def test_product_fails_loudly_without_a_gpu(binding):
    """No CPU fallback: on a box without a B200, corr_create returns NULL and the binding raises."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present; the failure path is exercised on the CPU box")
    with pytest.raises(binding.CorrError):
        binding.Correlator(4, 2, 4, 4, "ci8")


def test_product_does_not_import_the_oracle():
    """The product path and the oracle share no code and neither imports the other."""
    imp = re.compile(r"^\s*(import|from)\s+(\S+)", re.M)
    inc = re.compile(r'#\s*include\s+"([^"]+)"')
    pkg = os.path.join(ROOT, "paper_1305_5639_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            src = open(os.path.join(dirpath, f), errors="ignore").read()
            if f.endswith(".py"):
                assert not [m for m in imp.findall(src) if m[1].split(".")[0] == "oracle"], f
            if f.endswith((".cu", ".cuh", ".h")):
                assert not [m for m in inc.findall(src) if "oracle" in m], f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        src = open(os.path.join(ROOT, "oracle", f), errors="ignore").read() if f.endswith((".py", ".c", ".h")) else ""
        assert not [m for m in imp.findall(src) if m[1].split(".")[0] == "paper_1305_5639_b200"], f
        assert not [m for m in inc.findall(src) if "csrc" in m or "corr.h" in m], f
