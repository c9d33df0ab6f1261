"""lgf_measure_static (include/lgf.h): step 1 (theta, F) with its scratch in a static __device__ array, for callers that
cannot call cudaMalloc.  Checked against the existing path (a context's lgf_measure on the same links, LGF_REAL18 so
both read the same 18 reals per link) on two calls in a row that share the static array, the second on a SMALLER lattice
so that the array still holds the first call's partials beyond the ones the second call writes.
Tolerance: that of test_k1_delta_theta_F (1e-13 relative, fp64 sums of the same per-site terms in a different order; in
fp32 the per-site terms are additions in the same order too, so the same bound holds).
This file is named to be collected last: the run uses `pytest -x`."""
import ctypes

import pytest
import torch

import lgf_inputs as gi
import paper_1208_1186_b200 as lgf

CASES = [  # (first lattice, second lattice): several CTAs of 256 sites with a ragged tail, then fewer CTAs
    ((16, 16, 16, 16), (6, 6, 6, 4)),
    ((12, 6, 8, 4), (8, 8, 8, 8)),
]


def _existing_path(L, prec, links):
    gf = lgf.GaugeFixer(L, prec, lgf.LGF_REAL18)
    gf.load(links)
    r = gf.measure()
    gf.close()
    return r


@pytest.mark.gpu
@pytest.mark.parametrize("prec", [lgf.LGF_F64, lgf.LGF_F32])
@pytest.mark.parametrize("La,Lb", CASES)
def test_measure_static_matches_context_measure_twice(La, Lb, prec):
    dt = torch.float64 if prec == lgf.LGF_F64 else torch.float32
    lgf.static_init()
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    for L, seed in ((La, 31), (Lb, 32)):
        links = gi.as_real(gi.make_config(L, seed, 0.59), dt).cuda().contiguous()
        ref = _existing_path(L, prec, links)
        got = lgf.measure_static(L, links, out=out)
        assert got is out
        theta, F = (float(v) for v in out.cpu())          # the copy synchronises with the stream the kernels ran on
        assert ref.theta > 1e-3                            # a rough field: the comparison is not vacuous
        assert abs(theta - ref.theta) <= 1e-13 * ref.theta, (L, theta, ref.theta)
        assert abs(F - ref.F) <= 1e-13 * max(abs(ref.F), 1e-3), (L, F, ref.F)


@pytest.mark.gpu
def test_measure_static_is_repeatable_and_leaves_links_alone():
    L = (8, 8, 8, 8)
    links = gi.as_real(gi.make_config(L, 33, 0.59), torch.float64).cuda().contiguous()
    keep = links.clone()
    a = lgf.measure_static(L, links).cpu()
    b = lgf.measure_static(L, links).cpu()
    assert torch.equal(a, b)                               # fixed summation order: bit-identical
    assert torch.equal(links, keep)


def test_measure_static_limits():
    """Size and argument checks happen before any CUDA call (no GPU needed): the static array is 1 MiB, one 16-byte
    partial per 256 sites, i.e. LGF_STATIC_MAX_SITES = 64^4 sites."""
    lib = lgf.load_library()
    assert lib.lgf_static_scratch_bytes() == 1 << 20
    assert lgf.STATIC_MAX_SITES == 64 ** 4 == (lib.lgf_static_scratch_bytes() // 16) * 256
    fake = ctypes.c_void_p(256)                            # never dereferenced: the call is refused first
    too_big = (ctypes.c_int32 * 4)(128, 64, 64, 64)
    assert lib.lgf_measure_static(too_big, lgf.LGF_F64, fake, None, fake) == -1
    assert b"LGF_STATIC_MAX_SITES" in lib.lgf_static_last_error()
    ok_L = (ctypes.c_int32 * 4)(8, 8, 8, 8)
    assert lib.lgf_measure_static(ok_L, 7, fake, None, fake) == -1            # bad precision
    assert lib.lgf_measure_static(ok_L, lgf.LGF_F64, None, None, fake) == -1  # null links
    assert lib.lgf_measure_static((ctypes.c_int32 * 4)(8, 8, 1, 8), lgf.LGF_F64, fake, None, fake) == -1
