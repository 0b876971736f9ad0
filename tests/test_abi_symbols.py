"""No GPU: the C-ABI library builds (nvcc cross-compiles sm_100a), loads, and exports every symbol that
include/gsnfs.h declares; the Python binding covers the same names; pure host entry points work."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2606_05650_b200 import build
    return build.build()


def _declared():
    src = open(os.path.join(ROOT, "include", "gsnfs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gsnfs_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported_and_bound(libpath):
    names = _declared()
    assert {"gsnfs_octree_encode", "gsnfs_octree_decode", "gsnfs_raht_forward", "gsnfs_raht_inverse",
            "gsnfs_voxel_merge", "gsnfs_create", "gsnfs_destroy"} <= set(names)
    L = ctypes.CDLL(libpath)
    for n in names:
        assert hasattr(L, n), n
    from paper_2606_05650_b200 import binding
    assert set(binding.exported_symbols()) == set(names)


def test_host_only_entry_points(libpath):
    from paper_2606_05650_b200 import binding
    assert "sm_100a" in binding.gsnfs_version()
    # sum_{d<depth} min(8^d, n), rounded up to 16
    assert binding.gsnfs_occ_capacity(1_000_000, 16) == (sum(min(8 ** d, 1_000_000) for d in range(16)) + 15) // 16 * 16
    assert binding.gsnfs_occ_capacity(10, 0) == 0 and binding.gsnfs_occ_capacity(10, 22) == 0
    assert binding.lib().gsnfs_strerror(-4) == b"corrupt occupancy stream"


def test_no_cpu_fallback_without_gpu(libpath):
    import torch
    from paper_2606_05650_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.Context(max_points=1000)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_05650_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("oracle tests", ""), f
