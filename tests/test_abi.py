"""CPU-only checks of the boundary: libqbvh.so loads without a GPU and exports every symbol include/qbvh.h
declares; host-side argument validation that needs no device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_functions():
    src = open(os.path.join(ROOT, "include", "qbvh.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(qbvh_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_1901_08088_b200 import build
    return ctypes.CDLL(build.build())


def test_library_exports_every_declared_symbol(lib):
    names = header_functions()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), n
    from paper_1901_08088_b200 import qbvh
    assert sorted(qbvh.SYMBOLS) == names            # the binding carries the same names
    for n in names:
        assert callable(getattr(qbvh, n))


def test_host_side_validation_without_gpu(lib):
    from paper_1901_08088_b200 import qbvh
    assert qbvh.qbvh_workspace_bytes(0, 1) > 0
    b1, b2 = qbvh.qbvh_workspace_bytes(1 << 20, 1), qbvh.qbvh_workspace_bytes(1 << 21, 1)
    assert b1 % 256 == 0 and 1.85 < b2 / b1 < 2.1 and b1 < 180 * (1 << 20)   # ~150 B / particle + the cell tables
    for bad in [(-1, 1), (1 << 30, 1), (10, 0), (10, 5)]:
        with pytest.raises(qbvh.QbvhError):
            qbvh.qbvh_workspace_bytes(*bad)
    with pytest.raises(qbvh.QbvhError):
        qbvh.qbvh_set_num_types(5)
    with pytest.raises(qbvh.QbvhError):
        qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 33)
    with pytest.raises(qbvh.QbvhError):
        qbvh.qbvh_set_option(99, 0)
    qbvh.qbvh_set_option(qbvh.OPT_LEAF_COLLAPSE, 4)
    assert qbvh.qbvh_get_option(qbvh.OPT_LEAF_COLLAPSE) == 4
    # no tree yet: neighbors / export refuse; build without a workspace refuses; misaligned workspace refuses
    import numpy as np
    qbvh.qbvh_set_workspace(None)
    r = np.ones((1, 1), np.float32)
    with pytest.raises(qbvh.QbvhError) as e:
        qbvh.qbvh_neighbors(r, None, None, 4)
    assert e.value.code == qbvh.ERR_NOT_BUILT
    with pytest.raises(qbvh.QbvhError) as e:
        qbvh.qbvh_build(1234 * 256, None, 10, np.array([0, 0, 0, 1, 1, 1], np.float32))
    assert e.value.code == qbvh.ERR_WORKSPACE
    with pytest.raises(qbvh.QbvhError) as e:
        qbvh.qbvh_set_workspace(257, 1 << 20)
    assert e.value.code == qbvh.ERR_WORKSPACE
    with pytest.raises(qbvh.QbvhError) as e:
        qbvh.qbvh_build(1234 * 256, None, 10, np.array([0, 0, 0, 1, -1, 1], np.float32))
    assert e.value.code == qbvh.ERR_INVALID_ARG
    assert "workspace" in qbvh.qbvh_error_string(qbvh.ERR_WORKSPACE)
    assert qbvh.qbvh_staging_bytes(1000, 64) >= 1000 * (12 + 4 + 4 + 256)
