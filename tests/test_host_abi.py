"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol include/lgf.h
declares; host-side argument logic that needs no GPU."""
import ctypes

import pytest

import paper_1208_1186_b200 as lgf


def test_library_exports_every_declared_symbol():
    lib = lgf.load_library()
    names = lgf.declared_symbols()
    assert {"lgf_create", "lgf_load", "lgf_iterate", "lgf_fix", "lgf_store", "lgf_measure", "lgf_destroy",
            "lgf_workspace_bytes", "lgf_strerror"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_workspace_bytes_host_logic():
    V = 32 ** 4
    b18 = lgf.workspace_bytes((32, 32, 32, 32), lgf.LGF_F64, lgf.LGF_REAL18)
    b12 = lgf.workspace_bytes((32, 32, 32, 32), lgf.LGF_F64, lgf.LGF_REAL12)
    f18 = lgf.workspace_bytes((32, 32, 32, 32), lgf.LGF_F32, lgf.LGF_REAL18)
    assert b18 - b12 == 4 * 6 * V * 8                      # 6 reals per link saved
    assert 4 * 18 * V * 8 + 2 * 8 * V * 8 <= b18 < 4 * 18 * V * 8 + 2.7 * 8 * V * 8   # links + Delta + padded layout-B spectrum + two 19 MB staging buffers
    assert f18 < b18
    assert lgf.workspace_bytes((5, 8, 8, 8), lgf.LGF_F64, lgf.LGF_REAL18) == 0     # 5 is not 2^a 3^b
    assert lgf.workspace_bytes((1, 8, 8, 8), lgf.LGF_F64, lgf.LGF_REAL18) == 0
    assert lgf.workspace_bytes((8, 8, 8, 8), 7, lgf.LGF_REAL18) == 0
    assert lgf.workspace_bytes((8, 8, 8, 8), lgf.LGF_F64, 10) == 0
    assert lgf.workspace_bytes((48, 48, 48, 8), lgf.LGF_F64, lgf.LGF_REAL12) > 0
    assert lgf.workspace_bytes((4096, 4096, 2, 2), lgf.LGF_F64, lgf.LGF_REAL12) == 0      # V < 2^31, (x,y) plane too large for a tile
    assert lgf.workspace_bytes((512, 512, 2, 2), lgf.LGF_F64, lgf.LGF_REAL12) == 0        # factorises, but no tile fits on chip


def test_strerror_and_null_handling():
    lib = lgf.load_library()
    assert lib.lgf_strerror(0) == b"ok"
    assert b"invalid" in lib.lgf_strerror(-1)
    assert b"host allocation" in lib.lgf_strerror(-5)
    assert lib.lgf_destroy(None) == -1
    assert lib.lgf_launch_count(None) == 0
    h = ctypes.c_void_p()
    L = (ctypes.c_int32 * 4)(8, 8, 8, 8)
    assert lib.lgf_create(L, 1, 18, None, 0, None, ctypes.byref(h)) == -1          # null workspace


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((8, 8, 8, 8))
