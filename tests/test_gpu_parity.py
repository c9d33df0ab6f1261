"""GPU parity: the CUDA path (through the C ABI) against the oracle on the same seeded inputs.
Tolerances are north_star's: fp64 links after 1 iteration max|dU| <= 1e-12; theta, F at convergence
relative 1e-10 and identical iteration counts; fp32 per-iteration links <= 2e-5, F relative 1e-5."""
import numpy as np
import pytest
import torch

import lgf_inputs as gi
import oracle
import paper_1208_1186_b200 as lgf

pytestmark = pytest.mark.gpu
ALPHA = 0.08

# compile-time-sized FFT kernels: (8,8,8,8), (16,16,8,8), (16,16,16,16); mixed / generic runtime-radix kernels: the rest
SHAPES = [(8, 8, 8, 8), (16, 16, 8, 8), (6, 4, 12, 8), (4, 6, 3, 2), (16, 8, 4, 12), (12, 12, 6, 4), (2, 2, 2, 2),
          (24, 18, 4, 8), (8, 8, 16, 16)]
MODES = [(lgf.LGF_F64, lgf.LGF_REAL18), (lgf.LGF_F64, lgf.LGF_REAL12)]


def _pack(D):
    """oracle Delta [V,3,3] -> packed [V,4] complex."""
    return np.stack([D[:, 0, 1], D[:, 0, 2], D[:, 1, 2], D[:, 0, 0].imag + 1j * D[:, 1, 1].imag], 1)


def _cplx(t):
    return torch.view_as_complex(t.to(torch.float64).contiguous()).numpy()


def _max_abs_diff(a, b, chunk=1 << 20):
    """max |a - b| over two equally shaped complex arrays, in chunks (64^4: no 10 GB temporaries)."""
    a = a.reshape(-1)
    b = b.reshape(-1)
    m = 0.0
    for i in range(0, a.size, chunk * 36):
        m = max(m, float(np.max(np.abs(a[i:i + chunk * 36] - b[i:i + chunk * 36]))))
    return m


ULP = 2.0 ** -52          # spacing of fp64 numbers in [1, 2): the size of one rounding of an O(1) link entry


def _theta_floor(theta, V, d):
    """DESIGN.md §3 "theta near the rounding floor": theta = (1/3V) sum |Delta_ij|^2 and every Delta entry is a sum of 16
    link entries of size O(1).  If those entries carry independent errors of rms size e, theta moves by
    (2/3V) sqrt(sum |Delta|^2) e = 2 sqrt(theta/(3V)) e (random signs over the 9V entries); link fields that differ by
    rms d give e = sqrt(8) d (8 links enter a Delta entry with weight 1 each, up to the h.c.)."""
    return 2.0 * np.sqrt(8.0 * theta / (3.0 * V)) * d


def _check_theta_reduction(gf, L, r):
    """Noise-free check of the GPU's theta / F reduction: the oracle's measurement of the GPU's OWN final links.  No
    trajectory noise enters; what is left is the evaluation order of the 16-term sums behind each Delta entry, one
    rounding (1 ulp of 1.0) per entry: 1e-13 relative plus 4 x that fixed floor (it only matters below theta ~ 1e-13)."""
    _, theta_o, F_o = oracle.measure(L, gf.store())
    assert abs(r.theta - theta_o) <= 1e-13 * theta_o + 4.0 * _theta_floor(theta_o, gi.volume(L), ULP / np.sqrt(8.0)), (r.theta, theta_o)
    assert abs(r.F - F_o) <= 1e-13 * abs(F_o)


def _fixer(L, prec, stor, U):
    dt = torch.float64 if prec == lgf.LGF_F64 else torch.float32
    gf = lgf.GaugeFixer(L, prec, stor)
    gf.load(gi.as_real(U, dt))
    return gf


@pytest.mark.parametrize("L", SHAPES)
@pytest.mark.parametrize("prec,stor", MODES)
def test_k1_delta_theta_F(L, prec, stor):
    U = gi.make_config(L, 21, 0.59)
    D, theta, F = oracle.measure(L, U)
    gf = _fixer(L, prec, stor, U)
    r = gf.measure()
    got = _cplx(gf.debug_delta())
    assert np.max(np.abs(got - _pack(D))) <= 2e-14
    assert abs(r.theta - theta) <= 1e-13 * theta
    assert abs(r.F - F) <= 1e-13 * max(abs(F), 1e-3)
    assert r.iterations == 0
    gf.close()


@pytest.mark.parametrize("L", SHAPES)
def test_k2_k3_k4_fourier_acceleration(L):
    U = gi.make_config(L, 22, 0.59)
    D, _, _ = oracle.measure(L, U)
    Dt = _pack(oracle.fourier_accelerate(L, D))      # oracle transforms all 9 elements (pin P10)
    gf = _fixer(L, lgf.LGF_F64, lgf.LGF_REAL18, U)
    gf.measure()
    gf.debug_fourier_accelerate()
    got = _cplx(gf.debug_delta())
    assert np.max(np.abs(got - Dt)) <= 1e-13 * max(1.0, np.max(np.abs(Dt)))
    gf.close()


@pytest.mark.parametrize("L", SHAPES + [(8, 8, 64, 64), (48, 48, 8, 8), (8, 8, 48, 8), (32, 32, 8, 8), (8, 8, 32, 32)])
def test_k2_k3_k4_fourier_acceleration_fp32(L):
    """fp32 K2-K4 against the fp64 oracle fed the same fp32-rounded links.  Tolerance: fp32 unit roundoff 6e-8 x
    sqrt(log2 V) butterfly levels x the filter's rms gain (sqrt(mean S^2) ~ 4 in 4D, S <= p2max/p2min) gives ~1e-6 of
    max|Delta~| per entry; 1e-5 x max(1, max|Delta~|) is asserted (Delta from fp32 links carries 1e-7 itself)."""
    U32 = gi.as_real(gi.make_config(L, 22, 0.59), torch.float32)
    D, _, _ = oracle.measure(L, gi.from_real(U32))
    Dt = _pack(oracle.fourier_accelerate(L, D))
    gf = lgf.GaugeFixer(L, lgf.LGF_F32, lgf.LGF_REAL18)
    gf.load(U32)
    gf.measure()
    assert np.max(np.abs(_cplx(gf.debug_delta()) - _pack(D))) <= 4e-6          # K1 in fp32: 16-term sums of O(1) entries
    gf.debug_fourier_accelerate()
    got = _cplx(gf.debug_delta())
    assert np.max(np.abs(got - Dt)) <= 1e-5 * max(1.0, np.max(np.abs(Dt)))
    gf.close()


@pytest.mark.parametrize("L", SHAPES)
@pytest.mark.parametrize("prec,stor", MODES)
def test_one_iteration_links_fp64(L, prec, stor):
    U = gi.make_config(L, 23, 0.59)
    ref, thh, Fh = oracle.iterate(L, U, 1, ALPHA)
    gf = _fixer(L, prec, stor, U)
    r = gf.iterate(1, ALPHA)
    got = _cplx(gf.store())
    assert np.max(np.abs(got - ref)) <= 1e-12
    assert r.iterations == 1
    assert abs(r.theta - thh[1]) <= 1e-11 * thh[1]
    assert abs(r.F - Fh[1]) <= 1e-12
    gf.close()


@pytest.mark.parametrize("L", [(8, 8, 8, 8), (6, 4, 12, 8)])
@pytest.mark.parametrize("prec,stor", MODES)
def test_five_iterations_track_oracle(L, prec, stor):
    U = gi.make_config(L, 24, 0.59)
    ref, thh, Fh = oracle.iterate(L, U, 5, ALPHA)
    gf = _fixer(L, prec, stor, U)
    r = gf.iterate(5, ALPHA)
    got = _cplx(gf.store())
    assert np.max(np.abs(got - ref)) <= 1e-11
    assert abs(r.theta - thh[5]) <= 1e-10 * thh[5]
    # unitarity, det = 1 (P4)
    g = torch.from_numpy(got)
    eye = torch.eye(3, dtype=torch.complex128)
    assert float((g @ g.conj().transpose(-1, -2) - eye).abs().max()) < 1e-13
    assert float((torch.linalg.det(g) - 1).abs().max()) < 1e-13
    # plaquette invariance (P5), via lgf_inputs' independent code
    assert abs(gi.mean_plaquette(g, L) - gi.mean_plaquette(U, L)) < 1e-13
    gf.close()


def test_config0_convergence_8x4_fp64_18():
    """configs[0]: 8^4 fp64 18-real, plaquette 0.59, alpha 0.08, theta < 1e-12 or 5000 iterations."""
    L = (8, 8, 8, 8)
    U = gi.make_config(L, gi.CONFIG_SEED + 0, 0.59)
    ref, n, theta, F, thh, Fh = oracle.fix(L, U, ALPHA, 1e-12, 5000)
    gf = _fixer(L, lgf.LGF_F64, lgf.LGF_REAL18, U)
    r = gf.fix(ALPHA, 1e-12, 5000)
    assert r.iterations == n and r.converged
    assert abs(r.theta - theta) <= 1e-10 * theta            # north_star's bar, plain
    assert abs(r.F - F) <= 1e-10 * F
    assert np.max(np.abs(_cplx(gf.store()) - ref)) <= 1e-11
    _check_theta_reduction(gf, L, r)
    gf.close()


def test_config1_convergence_16x4_fp64_12_and_pure_gauge():
    """configs[1]: 16^4 fp64 12-real to theta < 1e-15; pure-gauge copy of the unit field reaches F = 1."""
    L = (16, 16, 16, 16)
    U = gi.make_config(L, gi.CONFIG_SEED + 1, 0.59)
    ref, n, theta, F, thh, Fh = oracle.fix(L, U, ALPHA, 1e-15, 5000)
    gf = _fixer(L, lgf.LGF_F64, lgf.LGF_REAL12, U)
    r = gf.fix(ALPHA, 1e-15, 5000)
    assert r.iterations == n and r.converged
    # theta at the crossing (5e-16) is a sum of squares of Delta entries ~2e-8 that are differences of O(1) link
    # entries: two correct fp64 runs whose links differ by rounding (rms d) disagree in theta by
    # sigma = 2 sqrt(8 theta / (3V)) d.  d is FIXED here, not measured: 8 ulp of 1.0, i.e. ~1.25 ulp of
    # rounding per update (two 3x3 complex products per link) accumulated as a random walk over the ~40 updates of this
    # run.  north_star's relative 1e-10 plus 3 sigma of that floor (3e-9 relative at this crossing, theta = 5e-16 on
    # 65 536 sites); the measured link difference must itself stay inside the assumed 8 ulp (measured: 4.6).
    d_fixed = 8.0 * ULP
    d_rms = float(np.sqrt(np.mean(np.abs(_cplx(gf.store()) - ref) ** 2)))
    assert d_rms <= d_fixed, d_rms
    sigma = _theta_floor(theta, gi.volume(L), d_fixed)
    assert abs(r.theta - theta) <= 1e-10 * theta + 3.0 * sigma, (r.theta, theta, d_rms, sigma)
    _check_theta_reduction(gf, L, r)
    assert abs(r.F - F) <= 1e-10 * F
    # well above the floor the plain relative bar holds: theta after 25 updates (~1e-9)
    gf.load(gi.as_real(U))
    r25 = gf.fix(ALPHA, 1e-30, 25)
    assert r25.iterations == 25 and abs(r25.theta - thh[25]) <= 1e-10 * thh[25]
    Up = gi.make_config(L, gi.CONFIG_SEED + 1, kind="pure_gauge")
    _, n2, th2, F2, _, _ = oracle.fix(L, Up, ALPHA, 1e-15, 5000)
    gf.load(gi.as_real(Up))
    r2 = gf.fix(ALPHA, 1e-15, 5000)
    assert r2.iterations == n2 and r2.converged
    assert abs(1 - r2.F) < 1e-13 and abs(r2.F - F2) < 1e-13
    gf.close()


@pytest.mark.parametrize("L", [(8, 8, 8, 8), (6, 4, 12, 8), (16, 8, 4, 12)])
@pytest.mark.parametrize("stor", [lgf.LGF_REAL18, lgf.LGF_REAL12])
def test_fp32_iterations(L, stor):
    """fp32: generate in fp64, round once, feed the same rounded values to both sides."""
    U = gi.make_config(L, 25, 0.59)
    U32 = gi.as_real(U, torch.float32)
    Ur = gi.from_real(U32)
    gf = lgf.GaugeFixer(L, lgf.LGF_F32, stor)
    gf.load(U32)
    cur = Ur
    for it in range(1, 4):
        ref, thh, Fh = oracle.iterate(L, Ur, it, ALPHA)
        r = gf.iterate(1, ALPHA)
        got = _cplx(gf.store())
        assert np.max(np.abs(got - ref)) <= 2e-5
        assert abs(r.F - Fh[it]) <= 1e-5 * abs(Fh[it])
    gf.close()


@pytest.mark.parametrize("prec", [lgf.LGF_F64, lgf.LGF_F32])
def test_load_store_roundtrip(prec):
    L = (6, 4, 12, 8)
    dt = torch.float64 if prec == lgf.LGF_F64 else torch.float32
    U = gi.as_real(gi.make_config(L, 26, 0.59), dt)
    gf = lgf.GaugeFixer(L, prec, lgf.LGF_REAL18)
    gf.load(U)
    assert torch.equal(gf.store(), U)                                  # bitwise for 18-real
    assert torch.equal(gf.store(device="cuda").cpu(), U)
    gf.load(U.cuda())
    assert torch.equal(gf.store(), U)
    gf.close()
    gf = lgf.GaugeFixer(L, prec, lgf.LGF_REAL12)
    gf.load(U)
    out = gf.store()
    assert torch.equal(out[:, :, :2], U[:, :, :2])                     # rows 0,1 bitwise
    if prec == lgf.LGF_F64:
        ref = oracle.two_row_roundtrip(U)
        assert np.max(np.abs(_cplx(out) - ref)) <= 4e-16
    else:
        assert float((out - U).abs().max()) < 1e-6
    gf.close()


def test_fix_semantics_and_errors():
    L = (4, 4, 4, 4)
    U = gi.make_config(L, 27, 0.59)
    gf = lgf.GaugeFixer(L, lgf.LGF_F64, lgf.LGF_REAL18)
    with pytest.raises(lgf.LgfError):
        gf.measure()                                                   # LGF_ESTATE before load
    gf.load(gi.as_real(U))
    r0 = gf.measure()
    r = gf.fix(ALPHA, 1e30, 100)                                       # already below tol
    assert r.iterations == 0 and r.converged and r.theta == r0.theta
    r = gf.fix(ALPHA, 1e-30, 7)                                        # hits max_iter
    assert r.iterations == 7 and not r.converged
    ref, thh, Fh = oracle.iterate(L, U, 7, ALPHA)
    assert abs(r.theta - thh[7]) <= 1e-10 * thh[7]
    r = gf.iterate(0, ALPHA)
    assert r.iterations == 0 and abs(r.theta - thh[7]) <= 1e-10 * thh[7]
    with pytest.raises(lgf.LgfError):
        gf.iterate(1, -1.0)
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((5, 4, 4, 4))                                   # prime factor 5
    gf.close()


def test_run_to_run_determinism():
    L = (8, 8, 8, 8)
    U = gi.as_real(gi.make_config(L, 28, 0.59))
    outs = []
    for _ in range(2):
        gf = lgf.GaugeFixer(L, lgf.LGF_F64, lgf.LGF_REAL12)
        gf.load(U)
        r = gf.iterate(10, ALPHA)
        outs.append((r.theta, r.F, gf.store()))
        gf.close()
    assert outs[0][0] == outs[1][0] and outs[0][1] == outs[1][1] and torch.equal(outs[0][2], outs[1][2])


@pytest.mark.parametrize("L,prec,stor", [((48, 48, 48, 8), lgf.LGF_F32, lgf.LGF_REAL12), ((32, 32, 32, 32), lgf.LGF_F64, lgf.LGF_REAL12),
                                         ((64, 64, 8, 8), lgf.LGF_F64, lgf.LGF_REAL18), ((8, 8, 64, 64), lgf.LGF_F64, lgf.LGF_REAL12)])
def test_run_to_run_determinism_of_the_pipelined_kernels(L, prec, stor):
    """compute-sanitizer is closed on this pool: a race in an mbarrier ring, a named-barrier group or a
    TMA-store drain of the pipelined FFT kernels would show up as run-to-run differences long before it shows up as a
    parity failure.  Five runs of seven iterations from the same links, many tiles per CTA: one bit pattern."""
    dt = torch.float64 if prec == lgf.LGF_F64 else torch.float32
    U = gi.as_real(gi.make_config(L, 29, 0.59, device="cuda"), dt)
    gf = lgf.GaugeFixer(L, prec, stor)
    assert "pipelined" in gf.describe()
    first = None
    for _ in range(5):
        gf.load(U)
        r = gf.iterate(7, ALPHA)
        out = gf.store(device="cuda")
        if first is None:
            first = (r.theta, r.F, out.clone())
        else:
            assert (r.theta, r.F) == first[:2] and torch.equal(out, first[2])
    gf.close()


@pytest.mark.parametrize("L,prec,stor", [((32, 32, 32, 32), lgf.LGF_F64, lgf.LGF_REAL12),
                                         ((32, 32, 32, 32), lgf.LGF_F64, lgf.LGF_REAL18),
                                         ((48, 48, 48, 8), lgf.LGF_F64, lgf.LGF_REAL12),
                                         ((48, 48, 48, 8), lgf.LGF_F64, lgf.LGF_REAL18),
                                         ((48, 48, 48, 12), lgf.LGF_F64, lgf.LGF_REAL12),
                                         ((48, 48, 48, 4), lgf.LGF_F64, lgf.LGF_REAL12),
                                         ((48, 48, 48, 6), lgf.LGF_F64, lgf.LGF_REAL12)])
def test_full_size_one_iteration(L, prec, stor):
    """BASELINE.json's full sizes (configs[2], configs[3]) in the launch configuration bench.py times:
    every link after one iteration against the oracle, element by element."""
    U = gi.make_config(L, gi.CONFIG_SEED + 2, 0.59, device="cuda").cpu()
    ref, thh, Fh = oracle.iterate(L, U, 1, ALPHA)
    gf = _fixer(L, prec, stor, U)
    r0 = gf.measure()
    assert abs(r0.theta - thh[0]) <= 1e-12 * thh[0]
    r = gf.iterate(1, ALPHA)
    got = _cplx(gf.store())
    assert np.max(np.abs(got - ref)) <= 1e-12
    assert abs(r.theta - thh[1]) <= 1e-11 * thh[1] and abs(r.F - Fh[1]) <= 1e-12
    gf.close()


@pytest.mark.parametrize("L", [(32, 32, 32, 32), (48, 48, 48, 8)])
def test_full_size_fp32(L):
    U32 = gi.as_real(gi.make_config(L, gi.CONFIG_SEED + 2, 0.59, device="cuda").cpu(), torch.float32)
    ref, thh, Fh = oracle.iterate(L, gi.from_real(U32), 2, ALPHA)
    for stor in (lgf.LGF_REAL12, lgf.LGF_REAL18):
        gf = lgf.GaugeFixer(L, lgf.LGF_F32, stor)
        gf.load(U32)
        r = gf.iterate(2, ALPHA)
        assert np.max(np.abs(_cplx(gf.store()) - ref)) <= 2e-5
        assert abs(r.F - Fh[2]) <= 1e-5 * abs(Fh[2])
        gf.close()


def test_generic_and_compile_time_fft_paths_agree(monkeypatch):
    """The runtime-radix kernels (forced by LGF_FORCE_GENERIC_FFT) and the compile-time-sized kernels
    must both match the oracle on a shape that has both."""
    L = (16, 16, 8, 8)
    U = gi.make_config(L, 29, 0.59)
    ref, thh, _ = oracle.iterate(L, U, 2, ALPHA)
    for force in (False, True):
        if force:
            monkeypatch.setenv("LGF_DEVKNOBS", "1")
            monkeypatch.setenv("LGF_FORCE_GENERIC_FFT", "1")
        gf = _fixer(L, lgf.LGF_F64, lgf.LGF_REAL18, U)
        gf.iterate(2, ALPHA)
        assert np.max(np.abs(_cplx(gf.store()) - ref)) <= 1e-12
        gf.close()


@pytest.mark.parametrize("zb", ["1", "2"])
@pytest.mark.parametrize("L", [(16, 16, 8, 8), (8, 8, 16, 16), (6, 4, 12, 8)])
def test_zblock_walk_order(monkeypatch, L, zb):
    """The site kernels' z-blocked (z-block outer, t inner) CTA order used on lattices whose t-slice outgrows
    the L2 (LGF_ZBLOCK forces it on small ones): same links, theta and F as the oracle, in every mode."""
    monkeypatch.setenv("LGF_DEVKNOBS", "1")
    monkeypatch.setenv("LGF_ZBLOCK", zb)
    U = gi.make_config(L, 37, 0.59)
    ref, thh, Fh = oracle.iterate(L, U, 2, ALPHA)
    for prec, stor in MODES:
        gf = _fixer(L, prec, stor, U)
        r = gf.iterate(2, ALPHA)
        assert np.max(np.abs(_cplx(gf.store()) - ref)) <= 1e-12
        assert abs(r.theta - thh[2]) <= 1e-10 * thh[2] and abs(r.F - Fh[2]) <= 1e-12
        gf.close()
    U32 = gi.as_real(U, torch.float32)
    ref32, _, Fh32 = oracle.iterate(L, gi.from_real(U32), 2, ALPHA)
    for stor in (lgf.LGF_REAL12, lgf.LGF_REAL18):
        gf = lgf.GaugeFixer(L, lgf.LGF_F32, stor)
        gf.load(U32)
        r = gf.iterate(2, ALPHA)
        assert np.max(np.abs(_cplx(gf.store()) - ref32)) <= 2e-5
        assert abs(r.F - Fh32[2]) <= 1e-5 * abs(Fh32[2])
        gf.close()


@pytest.mark.parametrize("L", [(8, 8, 8, 8), (16, 16, 8, 8), (32, 8, 4, 8)])
@pytest.mark.parametrize("prec,stor", MODES)
def test_fused_update_kernel(monkeypatch, L, prec, stor):
    """K5 + K1 fused into the marching kernel (LGF_FUSED=1): out-of-place update with swapped link
    buffers; links after 1, 2 (odd/even buffer) and 5 iterations, theta/F and the fix count vs the oracle."""
    monkeypatch.setenv("LGF_DEVKNOBS", "1")
    monkeypatch.setenv("LGF_FUSED", "1")
    U = gi.make_config(L, 31, 0.59)
    gf = _fixer(L, prec, stor, U)
    if L != (32, 8, 4, 8):                                 # (32, 8) has no pipelined FFT entry: unfused path
        assert gf.path_info()["fused"]
    for n in (1, 2, 5):
        ref, thh, Fh = oracle.iterate(L, U, n, ALPHA)
        gf.load(gi.as_real(U))
        r = gf.iterate(n, ALPHA)
        assert r.iterations == n
        assert np.max(np.abs(_cplx(gf.store()) - ref)) <= (1e-12 if n == 1 else 1e-11)
        assert abs(r.theta - thh[n]) <= 1e-10 * thh[n] and abs(r.F - Fh[n]) <= 1e-12
        m = gf.measure()                                   # stand-alone K1 on the swapped buffer agrees with the fused Delta
        assert abs(m.theta - r.theta) <= 1e-12 * r.theta and abs(m.F - r.F) <= 1e-14
    _, nfix, th, F, _, _ = oracle.fix(L, U, ALPHA, 1e-12, 5000)
    gf.load(gi.as_real(U))
    rf = gf.fix(ALPHA, 1e-12, 5000)
    assert rf.iterations == nfix and rf.converged and abs(rf.F - F) <= 1e-10 * F
    gf.close()


@pytest.mark.parametrize("L", [(8, 8, 64, 64), (64, 64, 8, 8), (48, 48, 8, 8), (8, 8, 48, 8), (8, 8, 48, 4), (8, 8, 48, 6),
                               (16, 16, 48, 12)])
def test_large_extent_fft_kernels(L):
    """The 48- and 64-point two-stage line kernels (64^4's K3 runs on the half-tile ring) on lattices the
    oracle still finishes in seconds: two iterations in fp64 12-real and fp32 18-real."""
    U = gi.make_config(L, 33, 0.59)
    ref, thh, Fh = oracle.iterate(L, U, 2, ALPHA)
    gf = _fixer(L, lgf.LGF_F64, lgf.LGF_REAL12, U)
    assert gf.path_info()["fft_path"] == "pipelined"
    r = gf.iterate(2, ALPHA)
    assert np.max(np.abs(_cplx(gf.store()) - ref)) <= 1e-12
    assert abs(r.theta - thh[2]) <= 1e-10 * thh[2] and abs(r.F - Fh[2]) <= 1e-12
    gf.close()
    U32 = gi.as_real(U, torch.float32)
    ref32, _, Fh32 = oracle.iterate(L, gi.from_real(U32), 2, ALPHA)
    gf = lgf.GaugeFixer(L, lgf.LGF_F32, lgf.LGF_REAL18)
    gf.load(U32)
    r = gf.iterate(2, ALPHA)
    assert np.max(np.abs(_cplx(gf.store()) - ref32)) <= 2e-5
    assert abs(r.F - Fh32[2]) <= 1e-5 * abs(Fh32[2])
    gf.close()


def test_full_size_64x4_one_iteration():
    """configs[4] at its full size, 64^4 (16.8 M sites, 9.7 GB of fp64 links), in the launch configuration bench.py
    times there and nowhere smaller: K3 on the half-tile ring, K2/K4 on 64x64 two-stage planes, the site kernels in
    the z-blocked walk order.  Every link after one iteration against the oracle, element by element (fp64, both
    storage modes), the initial theta and F, and the fp32 paths (12- and 18-real) against the oracle fed the rounded field.
    About a minute of host time: the oracle transforms 9 x 16.8 M complex numbers."""
    L = (64, 64, 64, 64)
    U = gi.make_config(L, gi.CONFIG_SEED + 4, 0.59, device="cuda")
    Ur = gi.as_real(U).cpu()
    ref, thh, Fh = oracle.iterate(L, Ur, 1, ALPHA)
    for stor in (lgf.LGF_REAL12, lgf.LGF_REAL18):
        gf = lgf.GaugeFixer(L, lgf.LGF_F64, stor)
        gf.load(Ur)
        r0 = gf.measure()
        assert abs(r0.theta - thh[0]) <= 1e-12 * thh[0] and abs(r0.F - Fh[0]) <= 1e-12
        r = gf.iterate(1, ALPHA)
        got = _cplx(gf.store())
        assert _max_abs_diff(got, ref) <= 1e-12
        assert abs(r.theta - thh[1]) <= 1e-11 * thh[1] and abs(r.F - Fh[1]) <= 1e-12
        gf.close()
        del got
    del ref
    U32 = Ur.to(torch.float32)
    del Ur, U
    torch.cuda.empty_cache()
    ref32, _, Fh32 = oracle.iterate(L, U32.to(torch.float64), 1, ALPHA)
    for stor in (lgf.LGF_REAL12, lgf.LGF_REAL18):
        gf = lgf.GaugeFixer(L, lgf.LGF_F32, stor)
        gf.load(U32)
        r = gf.iterate(1, ALPHA)
        assert _max_abs_diff(_cplx(gf.store()), ref32) <= 2e-5
        assert abs(r.F - Fh32[1]) <= 1e-5 * abs(Fh32[1])
        gf.close()


def _fix_vs_oracle(L, seed, prec, stor, plaq):
    """lgf_fix to theta < 1e-15 at a full-size config against oracle.fix on the same field: identical iteration
    count, theta and F within north_star's relative 1e-10, links; and the GPU's theta / F reduction against the oracle's
    measurement of the GPU's own final links (no trajectory noise)."""
    U = gi.make_config(L, seed, plaq, device="cuda").cpu()
    ref, n, theta, F, thh, Fh = oracle.fix(L, U, ALPHA, 1e-15, 5000)
    gf = _fixer(L, prec, stor, U)
    r = gf.fix(ALPHA, 1e-15, 5000)
    assert r.iterations == n and r.converged, (r.iterations, n)
    got = _cplx(gf.store())
    assert abs(r.theta - theta) <= 1e-10 * theta, (r.theta, theta)        # north_star's bar, plain (V is large enough here)
    _check_theta_reduction(gf, L, r)
    assert abs(r.F - F) <= 1e-10 * F
    assert _max_abs_diff(got, ref) <= 1e-11
    # F never decreases along the way (pin P6 on the GPU trajectory), theta well above the floor tracks the oracle
    gf.load(gi.as_real(U))
    k = min(20, n - 1)
    rk = gf.fix(ALPHA, 1e-30, k)
    assert rk.iterations == k and abs(rk.theta - thh[k]) <= 1e-10 * thh[k] and abs(rk.F - Fh[k]) <= 1e-12
    gf.close()


def test_config2_fix_32x4_fp64_12():
    """configs[2]: the 32^4 fp64 run to theta < 1e-15 (12-real, the headline mode), full size, vs the oracle."""
    _fix_vs_oracle((32, 32, 32, 32), gi.CONFIG_SEED + 2, lgf.LGF_F64, lgf.LGF_REAL12, 0.59)


def test_config3_fix_48x3x8_fp64_12():
    """configs[3]: 48^3 x 8 (radix-3 lines along x, y, z), fp64 12-real, plaquette 0.58, to theta < 1e-15, full size."""
    _fix_vs_oracle((48, 48, 48, 8), gi.CONFIG_SEED + 3, lgf.LGF_F64, lgf.LGF_REAL12, 0.58)


def test_config2_fp32_1000_iterations_properties():
    """configs[2]'s fixed 1000-iteration fp32 run at 32^4 in both storage modes: what must hold at any size without
    an oracle run of that length -- every link still unitary with det 1 to the fp32 bar (2e-5, no re-projection:
    reading #14), the mean plaquette of the result equal to the input's (gauge invariance, pin P5), F not below
    the fp64 value reached by the converged fp64 run minus the fp32 bar, theta at the fp32 floor."""
    L = (32, 32, 32, 32)
    U = gi.make_config(L, gi.CONFIG_SEED + 2, 0.59, device="cuda")
    plaq0 = gi.mean_plaquette(U, L)
    U32 = gi.as_real(U, torch.float32)
    gf64 = lgf.GaugeFixer(L, lgf.LGF_F64, lgf.LGF_REAL12)
    gf64.load(gi.as_real(U))
    r64 = gf64.fix(ALPHA, 1e-15, 5000)
    gf64.close()
    for stor in (lgf.LGF_REAL12, lgf.LGF_REAL18):
        gf = lgf.GaugeFixer(L, lgf.LGF_F32, stor)
        gf.load(U32)
        r = gf.iterate(1000, ALPHA)
        out = gi.from_real(gf.store(device="cuda").to(torch.float64))
        gf.close()
        eye = torch.eye(3, dtype=out.dtype, device=out.device)
        uni = (out @ out.conj().transpose(-1, -2) - eye).abs().max().item()
        det = (torch.linalg.det(out) - 1).abs().max().item()
        assert uni <= 2e-5 and det <= 2e-5, (uni, det)
        assert abs(gi.mean_plaquette(out, L) - plaq0) <= 2e-5
        assert abs(r.F - r64.F) <= 1e-5 * r64.F
        assert r.theta < 1e-12
        del out


@pytest.mark.parametrize("L", [(8, 8, 8, 8), (6, 4, 12, 8), (16, 8, 4, 12), (16, 16, 8, 8)])
def test_iterate_after_fix_without_reload(L):
    """lgf_fix converges in the middle of a batch of enqueued iterations; the no-op iterations behind the crossing
    must leave Delta of the final links intact, because a following lgf_iterate reuses it (pipelined, one-tile-per-CTA
    and generic FFT paths).  Reference: a fresh context loaded with the stored links."""
    U = gi.make_config(L, 43, 0.59)
    gf = _fixer(L, lgf.LGF_F64, lgf.LGF_REAL12, U)
    for tol in (1e-6, 3e-7, 1e-7):                        # a tolerance whose crossing falls inside a batch of 8
        gf.load(gi.as_real(U))
        r = gf.fix(ALPHA, tol, 5000)
        if r.iterations % 8 != 0:
            break
    assert r.converged and r.iterations % 8 != 0
    mid = gf.store()
    ra = gf.iterate(3, ALPHA)
    after = gf.store()
    gf.close()
    gf2 = lgf.GaugeFixer(L, lgf.LGF_F64, lgf.LGF_REAL12)
    gf2.load(mid)
    rb = gf2.iterate(3, ALPHA)
    assert ra.theta == rb.theta and ra.F == rb.F and torch.equal(after, gf2.store())
    gf2.close()


@pytest.mark.parametrize("L", [(8, 8, 8, 8), (6, 4, 12, 8), (4, 6, 3, 2), (16, 16, 16, 4), (24, 18, 4, 8), (32, 32, 32, 8)])
def test_wilson_lines_and_singlet_correlator(L):
    """The step after the path (eq. (1)): Wilson lines and the singlet correlator of the GPU's links against
    the oracle's written-out definition on the same links, fp64 (12- and 18-real) and fp32; then the same after a fix,
    on the gauge-fixed links of both sides; the links, theta and F of the context are untouched by the measurement."""
    U = gi.make_config(L, 61, 0.59)
    Wo = oracle.wilson_lines(L, U)
    Co = oracle.singlet_correlator(L, U) if gi.volume(L) // L[3] <= 8192 else None
    for prec, stor in MODES:
        gf = _fixer(L, prec, stor, U)
        W = torch.view_as_complex(gf.wilson_lines()).numpy()
        assert np.max(np.abs(W - Wo)) <= 1e-13
        if Co is not None:
            C = torch.view_as_complex(gf.singlet_correlator()).numpy()
            assert np.max(np.abs(C - Co)) <= 1e-13
            Cd = torch.view_as_complex(gf.singlet_correlator(device="cuda")).cpu().numpy()
            assert np.array_equal(C, Cd)
        r0 = gf.measure()
        r = gf.iterate(3, ALPHA)
        C3 = torch.view_as_complex(gf.singlet_correlator()).numpy()
        assert abs(C3[0] - 1) <= 1e-13 and np.max(np.abs(C3)) <= 1 + 1e-13
        r1 = gf.iterate(1, ALPHA)                          # the scratch use did not disturb the iteration
        ref, thh, Fh = oracle.iterate(L, U, 4, ALPHA)
        assert abs(r1.theta - thh[4]) <= 1e-10 * thh[4] and np.max(np.abs(_cplx(gf.store()) - ref)) <= 1e-11
        if Co is not None:
            Cfix = oracle.singlet_correlator(L, gf.store())
            assert np.max(np.abs(torch.view_as_complex(gf.singlet_correlator()).numpy() - Cfix)) <= 1e-13
        gf.close()
    U32 = gi.as_real(U, torch.float32)
    gf = lgf.GaugeFixer(L, lgf.LGF_F32, lgf.LGF_REAL12)
    gf.load(U32)
    Wo32 = oracle.wilson_lines(L, gi.from_real(U32))
    assert np.max(np.abs(torch.view_as_complex(gf.wilson_lines().to(torch.float64)).numpy() - Wo32)) <= 2e-5
    if Co is not None:
        Co32 = oracle.singlet_correlator(L, gi.from_real(U32))
        assert np.max(np.abs(torch.view_as_complex(gf.singlet_correlator().to(torch.float64)).numpy() - Co32)) <= 2e-5
    gf.close()


@pytest.mark.parametrize("L,nbatch", [((8, 8, 8, 8), 5), ((16, 16, 16, 16), 3), ((6, 4, 12, 8), 2), ((16, 16, 8, 8), 4)])
@pytest.mark.parametrize("prec,stor", MODES)
def test_batched_context_equals_single_lattice_contexts(monkeypatch, L, nbatch, prec, stor):
    """lgf_create_batch: nbatch different lattices fixed by the same launches.  Each lattice must
    come out exactly as from a context of its own (same kernels, same per-lattice reduction order: bitwise), with its
    own iteration count -- the lattices converge at different iterations -- and lattice 0 must match the oracle.
    (A single 8^4 lattice would otherwise run the single-cluster kernel, which rounds Delta in another order: the
    comparison contexts are kept on the five-kernel graph, the kernels the batched context runs.)"""
    monkeypatch.setenv("LGF_DEVKNOBS", "1")
    monkeypatch.setenv("LGF_CLUSTER", "0")
    Us = [gi.make_config(L, 80 + b, 0.59 if b % 2 == 0 else 0.57) for b in range(nbatch)]
    stack = torch.cat([gi.as_real(u) for u in Us], 0)
    gb = lgf.GaugeFixer(L, prec, stor, nbatch=nbatch)
    gb.load(stack)
    m = gb.measure()
    rb = gb.iterate(2, ALPHA)
    after2 = gb.store().reshape(nbatch, -1, 4, 3, 3, 2)
    gb.load(stack.cuda())
    rf = gb.fix(ALPHA, 1e-10, 500)
    fixed = gb.store(device="cuda").cpu().reshape(nbatch, -1, 4, 3, 3, 2)
    assert len({r.iterations for r in rf}) > 1 or nbatch < 3          # the crossings differ between the lattices
    for b in range(nbatch):
        g1 = _fixer(L, prec, stor, Us[b])
        m1 = g1.measure()
        assert (m[b].theta, m[b].F) == (m1.theta, m1.F)
        r1 = g1.iterate(2, ALPHA)
        assert (rb[b].theta, rb[b].F, rb[b].iterations) == (r1.theta, r1.F, 2)
        assert torch.equal(after2[b], g1.store())
        g1.load(gi.as_real(Us[b]))
        f1 = g1.fix(ALPHA, 1e-10, 500)
        assert (rf[b].iterations, rf[b].theta, rf[b].F, rf[b].converged) == (f1.iterations, f1.theta, f1.F, True)
        assert torch.equal(fixed[b], g1.store())
        g1.close()
    ref, n, theta, F, _, _ = oracle.fix(L, Us[0], ALPHA, 1e-10, 500)
    assert rf[0].iterations == n and abs(rf[0].theta - theta) <= 1e-10 * theta and abs(rf[0].F - F) <= 1e-10 * F
    assert np.max(np.abs(_cplx(fixed[0]) - ref)) <= 1e-11
    r3 = gb.iterate(3, ALPHA)                                          # a batched fix leaves Delta stale: iterate re-measures
    assert all(r.iterations == 3 for r in r3) and all(r.theta < 1e-10 for r in r3)
    gb.close()


def test_batched_context_fp32_and_limits():
    L = (8, 8, 8, 8)
    Us = [gi.as_real(gi.make_config(L, 90 + b, 0.59), torch.float32) for b in range(4)]
    gb = lgf.GaugeFixer(L, lgf.LGF_F32, lgf.LGF_REAL12, nbatch=4)
    gb.load(torch.cat(Us, 0))
    rb = gb.iterate(3, ALPHA)
    out = gb.store().reshape(4, -1, 4, 3, 3, 2)
    for b in range(4):
        ref, thh, Fh = oracle.iterate(L, gi.from_real(Us[b]), 3, ALPHA)
        assert np.max(np.abs(_cplx(out[b]) - ref)) <= 2e-5 and abs(rb[b].F - Fh[3]) <= 1e-5 * abs(Fh[3])
    with pytest.raises(lgf.LgfError):
        gb.singlet_correlator()                                         # single-lattice contexts only
    gb.close()
    # every further lattice adds its links (12 reals) and its two Delta-sized fields; tables and the staging buffers do not scale
    per_lattice = 4 * 12 * 8 ** 4 * 4 + 2 * 8 * 8 ** 4 * 4
    assert lgf.workspace_bytes(L, lgf.LGF_F32, lgf.LGF_REAL12, nbatch=4) - lgf.workspace_bytes(L, lgf.LGF_F32, lgf.LGF_REAL12) >= 3 * per_lattice
    assert lgf.workspace_bytes(L, lgf.LGF_F32, lgf.LGF_REAL12, nbatch=5000) == 0      # grid z = nbatch x (z,t) tiles < 2^16


def test_describe_reports_the_kernels_a_lattice_fell_onto():
    U = gi.make_config((8, 8, 64, 64), 95, 0.59)
    gf = _fixer((8, 8, 64, 64), lgf.LGF_F64, lgf.LGF_REAL12, U)
    gf.iterate(1, ALPHA)
    d = gf.describe()
    assert "pipelined" in d and "fft_zt_pipe3q" in d and "12-real" in d and "fp64" in d and "6 launches" in d
    gf.close()
    gf = lgf.GaugeFixer((6, 4, 12, 8))
    assert "runtime-radix" in gf.describe()                # extents that are not instantiated: the generic kernels, and it says so
    gf.close()
    gf = lgf.GaugeFixer((64, 64, 8, 8), lgf.LGF_F32, lgf.LGF_REAL18, nbatch=2)
    assert "fft_xy_pipe_io" in gf.describe() and "x 2," in gf.describe()
    gf.close()


ALL_MODES = [(lgf.LGF_F64, lgf.LGF_REAL18), (lgf.LGF_F64, lgf.LGF_REAL12), (lgf.LGF_F32, lgf.LGF_REAL18), (lgf.LGF_F32, lgf.LGF_REAL12)]


@pytest.mark.parametrize("prec,stor", ALL_MODES)
def test_cluster8_path_against_oracle_and_graph_path(monkeypatch, prec, stor):
    """8^4 (configs[0]'s shape): lgf_iterate / lgf_fix run the single-cluster kernel (lgf_cluster8.cuh: the field stays
    in the distributed shared memory of 16 CTAs, one launch per call).  Element by element against the oracle, and
    against the five-kernel graph path of the same library (LGF_CLUSTER=0); state carries over between calls."""
    L = (8, 8, 8, 8)
    U = gi.make_config(L, 23, 0.59)
    tol_u, tol_rel = (1e-12, 1e-12) if prec == lgf.LGF_F64 else (2e-5, 1e-5)
    ref, thh, Fh = oracle.iterate(L, U, 6, ALPHA)
    gf = _fixer(L, prec, stor, U)
    assert "k_cluster8_iterate" in gf.describe()
    r0 = gf.iterate(0, ALPHA)                                  # measure only
    assert r0.iterations == 0 and abs(r0.theta - thh[0]) <= tol_rel * thh[0]
    r1 = gf.iterate(2, ALPHA)
    r2 = gf.iterate(4, ALPHA)                                  # 2 + 4 updates in two launches = the oracle's 6
    assert (r1.iterations, r2.iterations) == (2, 4)
    got = _cplx(gf.store())
    assert np.max(np.abs(got - ref)) <= tol_u * 6
    assert abs(r1.theta - thh[2]) <= 10 * tol_rel * thh[2] and abs(r2.theta - thh[6]) <= 10 * tol_rel * thh[6]
    assert abs(r2.F - Fh[6]) <= tol_rel * 6
    rm = gf.measure()                                          # K1 of the five-kernel path on the links the cluster kernel wrote back
    assert abs(rm.theta - r2.theta) <= (1e-13 if prec == lgf.LGF_F64 else 1e-5) * r2.theta
    d_cluster = _cplx(gf.debug_delta())
    gf.close()
    monkeypatch.setenv("LGF_DEVKNOBS", "1")
    monkeypatch.setenv("LGF_CLUSTER", "0")
    gg = _fixer(L, prec, stor, U)
    assert "k_cluster8_iterate" not in gg.describe()
    rg = gg.iterate(6, ALPHA)
    assert np.max(np.abs(_cplx(gg.store()) - got)) <= tol_u
    assert abs(rg.theta - r2.theta) <= 10 * tol_rel * r2.theta
    assert np.max(np.abs(_cplx(gg.debug_delta()) - d_cluster)) <= (1e-13 if prec == lgf.LGF_F64 else 2e-5)
    gg.close()


def test_cluster8_fix_counts_iterations_like_the_oracle():
    """lgf_fix on the cluster path: the stopping test runs on the device after EVERY update; same count as the oracle,
    0 iterations on a field already below tolerance, max_iter respected."""
    L = (8, 8, 8, 8)
    U = gi.make_config(L, 24, 0.59)
    ref, n, theta, F, thh, Fh = oracle.fix(L, U, ALPHA, 1e-10, 5000)
    gf = _fixer(L, lgf.LGF_F64, lgf.LGF_REAL12, U)
    assert "k_cluster8_iterate" in gf.describe()
    r = gf.fix(ALPHA, 1e-10, 5000)
    assert r.iterations == n and r.converged and abs(r.theta - theta) <= 1e-9 * theta
    assert np.max(np.abs(_cplx(gf.store()) - ref)) <= 1e-11
    again = gf.fix(ALPHA, 1e-10, 5000)                         # already below the tolerance
    assert again.iterations == 0 and again.converged
    gf.load(gi.as_real(U, torch.float64))
    capped = gf.fix(ALPHA, 1e-10, 5)
    assert capped.iterations == 5 and not capped.converged and abs(capped.theta - thh[5]) <= 1e-11 * thh[5]
    gf.close()


@pytest.mark.parametrize("prec,stor", [(lgf.LGF_F64, lgf.LGF_REAL18), (lgf.LGF_F32, lgf.LGF_REAL12)])
def test_cluster8_batched_context_runs_one_cluster_per_lattice(prec, stor):
    """A batched 8^4 context launches one 16-CTA cluster per lattice (more lattices than the GPU hosts clusters at a
    time: the rest queue).  Every lattice comes out bitwise as from a single-lattice context, with its own iteration
    count, and lattice 0 matches the oracle."""
    L, nbatch = (8, 8, 8, 8), 11
    dt = torch.float64 if prec == lgf.LGF_F64 else torch.float32
    tol = 1e-10 if prec == lgf.LGF_F64 else 1e-9
    Us = [gi.make_config(L, 60 + b, 0.59 if b % 2 == 0 else 0.57) for b in range(nbatch)]
    stack = torch.cat([gi.as_real(u, dt) for u in Us], 0)
    gb = lgf.GaugeFixer(L, prec, stor, nbatch=nbatch)
    assert "k_cluster8_iterate" in gb.describe()
    gb.load(stack)
    rb = gb.iterate(3, ALPHA)
    after3 = gb.store().reshape(nbatch, -1, 4, 3, 3, 2)
    gb.load(stack)
    rf = gb.fix(ALPHA, tol, 300)
    fixed = gb.store().reshape(nbatch, -1, 4, 3, 3, 2)
    assert len({r.iterations for r in rf}) > 1
    for b in range(nbatch):
        g1 = _fixer(L, prec, stor, Us[b])
        r1 = g1.iterate(3, ALPHA)
        assert (rb[b].theta, rb[b].F, rb[b].iterations) == (r1.theta, r1.F, 3)
        assert torch.equal(after3[b], g1.store())
        g1.load(gi.as_real(Us[b], dt))
        f1 = g1.fix(ALPHA, tol, 300)
        assert (rf[b].iterations, rf[b].theta, rf[b].F, rf[b].converged) == (f1.iterations, f1.theta, f1.F, f1.converged)
        assert torch.equal(fixed[b], g1.store())
        g1.close()
    if prec == lgf.LGF_F64:
        ref, n, theta, F, _, _ = oracle.fix(L, Us[0], ALPHA, tol, 300)
        assert rf[0].iterations == n and abs(rf[0].theta - theta) <= 1e-9 * theta
        assert np.max(np.abs(_cplx(fixed[0]) - ref)) <= 1e-11
    gb.close()


def test_cluster8_many_clusters_in_flight_stay_bitwise_repeatable():
    """Regression guard for the cluster barriers (relaxed arrives read stale shared memory in 18 of 3300
    runs of exactly this shape -- fp32, two CTAs per SM, 11 clusters in flight -- while every other test stayed green):
    60 batched runs, every lattice bitwise equal to its single-lattice reference."""
    L, nbatch, prec, stor = (8, 8, 8, 8), 11, lgf.LGF_F32, lgf.LGF_REAL12
    Us = [gi.make_config(L, 60 + b, 0.59 if b % 2 == 0 else 0.57) for b in range(nbatch)]
    ref = []
    for b in range(nbatch):
        g1 = _fixer(L, prec, stor, Us[b])
        r = g1.iterate(3, ALPHA)
        ref.append((r.theta, r.F, g1.store().clone()))
        g1.close()
    stack = torch.cat([gi.as_real(u, torch.float32) for u in Us], 0).cuda()
    gb = lgf.GaugeFixer(L, prec, stor, nbatch=nbatch)
    assert "k_cluster8_iterate" in gb.describe()
    bad = 0
    for rep in range(60):
        gb.load(stack)
        rb = gb.iterate(3, ALPHA)
        out = gb.store().reshape(nbatch, -1, 4, 3, 3, 2)
        for b in range(nbatch):
            if (rb[b].theta, rb[b].F) != ref[b][:2] or not torch.equal(out[b], ref[b][2]):
                bad += 1
    gb.close()
    assert bad == 0
