"""The C-ABI library builds, loads without a GPU and exports every symbol include/omnimem.h declares;
host-only argument checks (no compute calls)."""
import ctypes
import os
import re

import pytest

from paper_2605_30519_b200 import binding as om
from paper_2605_30519_b200 import build as om_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    om_build.build()
    return om.load()


def test_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "omnimem.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = sorted(set(re.findall(r"\b(omnimem_[a-z_0-9]+)\s*\(", header)))
    assert len(declared) >= 15
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(om.EXPORTS) == declared
    assert lib.omnimem_version() >= 100


def test_struct_layouts_match_header():
    assert ctypes.sizeof(om.CacheDesc) == 40 and ctypes.sizeof(om.SelectParams) == 32
    assert ctypes.sizeof(om.AweInfo) == 32 and ctypes.sizeof(om.AttnParams) == 32


def test_host_side_validation(lib):
    sizes = [ctypes.c_size_t() for _ in range(4)]
    d = om.CacheDesc(12, 128, 64, om.DTYPE_BF16, 93600 + 4680)
    assert lib.omnimem_cache_sizes(ctypes.byref(d), *[ctypes.byref(s) for s in sizes]) == om.OK
    max_blocks = -(-(93600 + 4680) // 64)
    assert sizes[0].value == 12 * max_blocks * 64 * 128 * 2 == sizes[1].value
    assert sizes[2].value == 12 * max_blocks * 128 * 2 and sizes[3].value == 12 * max_blocks * 4
    for bad in (om.CacheDesc(12, 96, 64, 1, 1000), om.CacheDesc(12, 128, 30, 1, 1000), om.CacheDesc(12, 128, 64, 7, 1000), om.CacheDesc(12, 128, 30, 1, 1000, 48, 0)):
        assert lib.omnimem_cache_sizes(ctypes.byref(bad), *[ctypes.byref(s) for s in sizes]) == om.EUNSUPPORTED
        assert lib.omnimem_last_error()
    # the paper's geometry: 30-token blocks in 32-row pages, 156 blocks per chunk
    pd = om.CacheDesc(12, 128, 30, om.DTYPE_BF16, 21 * 4680, 32, 156)
    assert lib.omnimem_cache_sizes(ctypes.byref(pd), *[ctypes.byref(s) for s in sizes]) == om.OK
    assert sizes[0].value == 12 * (21 * 156) * 32 * 128 * 2
    assert lib.omnimem_cache_sizes(ctypes.byref(om.CacheDesc(12, 128, 60, 1, 1000, 32, 0)), *[ctypes.byref(s) for s in sizes]) == om.EINVAL
    assert lib.omnimem_cache_sizes(ctypes.byref(om.CacheDesc(0, 128, 64, 1, 1000)), *[ctypes.byref(s) for s in sizes]) == om.EINVAL
    # workspace query is host-only arithmetic
    a, b = ctypes.c_size_t(), ctypes.c_size_t()
    sp = om.SelectParams(64, 16, 4680, 220, 0.088)
    ap = om.AttnParams(64, 16, 4680, 0.088, om.FUSE_JOINT, 0)
    assert lib.omnimem_workspace_bytes(ctypes.byref(d), 4680, ctypes.byref(sp), ctypes.byref(ap), ctypes.byref(a), ctypes.byref(b)) == om.OK
    assert a.value >= 12 * 74 * max_blocks * 4
    bad_sp = om.SelectParams(64, 65, 4680, 220, 0.088)
    assert lib.omnimem_workspace_bytes(ctypes.byref(d), 4680, ctypes.byref(bad_sp), None, ctypes.byref(a), ctypes.byref(b)) == om.EUNSUPPORTED
    # NULL handles are rejected, not dereferenced
    assert lib.omnimem_append_chunk(None, None, None, 1, 128, 128, None) == om.EINVAL
    assert lib.omnimem_pool_keys(None, 0, 1, None) == om.EINVAL
    assert lib.omnimem_cache_tokens(None) == om.EINVAL
