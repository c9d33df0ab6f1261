"""Pins for the oracle: every check here compares the oracle with
something that is NOT the oracle -- numpy.fft / a direct O(N^2) sum typed here, closed forms,
invariants computed by lgf_inputs' independent plaquette code, brute-force convolution.
CPU only (`-m "not gpu"`)."""
import math

import numpy as np
import pytest
import torch

import lgf_inputs as gi
import oracle

ALPHA = 0.08


def _rng(seed):
    return np.random.default_rng(seed)


def _coords(L):
    V = gi.volume(L)
    s = np.arange(V)
    x = s % L[0]
    y = (s // L[0]) % L[1]
    z = (s // (L[0] * L[1])) % L[2]
    t = s // (L[0] * L[1] * L[2])
    return np.stack([x, y, z, t], 1)


# ---------------------------------------------------------------- P1: FFT
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7, 8, 9, 12, 16, 18, 24, 32, 48, 64])
def test_fft1d_vs_direct_sum_and_numpy(n):
    z = _rng(n).normal(size=n) + 1j * _rng(n + 100).normal(size=n)
    k = np.arange(n)
    for sign in (-1, +1):
        W = np.exp(sign * 2j * np.pi * np.outer(k, k) / n)        # typed-out definition
        ref = W @ z
        lib = np.fft.fft(z) if sign < 0 else np.fft.ifft(z) * n   # library routine
        for got in (oracle.fft1d(z, sign), oracle.dft1d(z, sign)):
            assert np.max(np.abs(got - ref)) <= 1e-13 * n * np.max(np.abs(z))
            assert np.max(np.abs(got - lib)) <= 1e-13 * n * np.max(np.abs(z))


@pytest.mark.parametrize("L", [(4, 6, 3, 2), (2, 2, 2, 2), (8, 4, 6, 3)])
def test_transform4d_vs_numpy_and_direct(L):
    V = gi.volume(L)
    f = _rng(1).normal(size=V) + 1j * _rng(2).normal(size=V)
    grid = f.reshape(L[3], L[2], L[1], L[0])
    ref_f = np.fft.fftn(grid).reshape(-1)
    ref_i = np.fft.ifftn(grid).reshape(-1)
    for direct in (False, True):
        assert np.max(np.abs(oracle.transform4d(L, f, -1, direct) - ref_f)) <= 1e-12 * np.max(np.abs(ref_f))
        assert np.max(np.abs(oracle.transform4d(L, f, +1, direct) - ref_i)) <= 1e-13
    # inverse(forward(f)) = f, Parseval
    F = oracle.transform4d(L, f, -1)
    assert np.max(np.abs(oracle.transform4d(L, F, +1) - f)) <= 1e-13
    assert abs(np.sum(np.abs(F) ** 2) / V - np.sum(np.abs(f) ** 2)) <= 1e-11 * np.sum(np.abs(f) ** 2)


def test_transform4d_axis_order_and_plane_wave():
    """A single plane wave exp(+2 pi i q.x/L) lands on mode q only: pins the axis <-> index map
    (x fastest) and the forward sign."""
    L = (4, 6, 3, 2)
    V = gi.volume(L)
    q = (1, 4, 2, 1)
    c = _coords(L)
    phase = sum(q[m] * c[:, m] / L[m] for m in range(4))
    f = np.exp(2j * np.pi * phase)
    F = oracle.transform4d(L, f, -1)
    sq = q[0] + L[0] * (q[1] + L[1] * (q[2] + L[2] * q[3]))
    assert abs(F[sq] - V) < 1e-10
    F[sq] = 0
    assert np.max(np.abs(F)) < 1e-10
    # impulse <-> constant
    d = np.zeros(V, complex)
    d[0] = 1
    assert np.max(np.abs(oracle.transform4d(L, d, -1) - 1)) < 1e-14


# ---------------------------------------------------------------- P2: p^2 table
@pytest.mark.parametrize("L", [(8, 8, 8, 8), (6, 4, 12, 8), (9, 9, 9, 4), (4, 6, 3, 2)])
def test_psq_table(L):
    p2, pmax = oracle.psq(L)
    c = _coords(L)
    ref = sum(4 * np.sin(np.pi * c[:, m] / L[m]) ** 2 for m in range(4))
    assert np.max(np.abs(p2 - ref)) < 1e-14
    assert p2[0] == 0.0
    assert abs(p2.mean() - 8.0) < 1e-13                 # mean over k of p^2 = 2 N_d
    assert abs(pmax - p2.max()) < 1e-14
    if all(l % 2 == 0 for l in L):
        assert abs(pmax - 16.0) < 1e-14
    else:
        assert pmax < 16.0
    # p^2(k) = p^2(-k)
    neg = [(-c[:, m]) % L[m] for m in range(4)]
    sneg = neg[0] + L[0] * (neg[1] + L[1] * (neg[2] + L[2] * neg[3]))
    assert np.max(np.abs(p2 - p2[sneg])) < 1e-14


def test_psq_max_odd_value():
    _, pmax = oracle.psq((9, 9, 9, 4))
    assert abs(pmax - (3 * 4 * math.sin(math.pi * 4 / 9) ** 2 + 4.0)) < 1e-13
    assert abs(pmax - 15.638) < 1e-3                    # SURVEY.md §8(c) reading #7


# ---------------------------------------------------------------- P3, P9: Delta
def _delta_numpy(U, L):
    """Typed-out definition with torch.roll neighbours (independent of the oracle's indexing)."""
    M = torch.zeros(gi.volume(L), 3, 3, dtype=torch.complex128)
    for mu in range(4):
        back = torch.roll(gi._grid(U[:, mu], L), shifts=+1, dims=gi._AXIS[mu]).reshape(-1, 3, 3)
        M += back - U[:, mu]
    A = M - M.conj().transpose(-1, -2)
    tr = torch.einsum("nii->n", A) / 3
    A = A - tr[:, None, None] * torch.eye(3, dtype=torch.complex128)
    return A.numpy()


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (6, 4, 3, 2), (8, 8, 8, 8)])
def test_delta_definition_and_properties(L):
    U = gi.make_config(L, 11, 0.59)
    D, theta, F = oracle.measure(L, U)
    ref = _delta_numpy(U, L)
    assert np.max(np.abs(D - ref)) < 1e-14
    assert np.max(np.abs(D + D.conj().transpose(0, 2, 1))) == 0.0        # anti-Hermitian, exactly
    assert np.max(np.abs(np.einsum("nii->n", D))) < 4e-15                # traceless (rounding of Tr/3)
    assert np.max(np.abs(D.sum(0))) < 1e-11                              # sum_x Delta = 0 (telescopes)
    V = gi.volume(L)
    assert abs(theta - np.sum(np.abs(ref) ** 2) / (3 * V)) < 1e-12 * theta
    Fref = float(torch.einsum("nmii->", U).real) / (12 * V)
    assert abs(F - Fref) < 1e-14


def test_delta_zero_on_constant_fields():
    L = (4, 6, 3, 2)
    V = gi.volume(L)
    D, theta, F = oracle.measure(L, gi.unit_links(L))
    assert np.max(np.abs(D)) == 0 and theta == 0 and F == 1.0
    Vmu = gi.haar_su3(1, 5, 0, 4)                       # x-independent U_mu(x) = V_mu
    U = Vmu[None].expand(V, 4, 3, 3).contiguous()
    D, theta, _ = oracle.measure(L, U)
    assert np.max(np.abs(D)) < 1e-15 and theta < 1e-29


def test_measure_global_rotation_invariance():
    """P9: U -> G U G^+ (constant G) leaves theta, F unchanged and maps Delta -> G Delta G^+."""
    L = (4, 4, 4, 4)
    U = gi.make_config(L, 12, 0.59)
    G = gi.haar_su3(2, 6, 0, 1)[0]
    UG = G @ U @ G.conj().T
    D0, t0, F0 = oracle.measure(L, U)
    D1, t1, F1 = oracle.measure(L, UG)
    assert abs(t0 - t1) < 1e-12 and abs(F0 - F1) < 1e-15
    Gn = G.numpy()
    assert np.max(np.abs(D1 - Gn @ D0 @ Gn.conj().T)) < 1e-13


def test_theta_haar_expectation():
    """P8: independent Haar links: E[theta] = 128/9, E[F] = 0."""
    L = (8, 8, 8, 8)
    _, theta, F = oracle.measure(L, gi.make_config(L, 9, kind="haar_links"))
    assert abs(theta - 128.0 / 9.0) < 0.15              # sigma ~ 0.05 at V = 4096
    assert abs(F) < 0.01


# ---------------------------------------------------------------- P4: SU(3) algebra
def test_reunitarise_properties():
    rng = _rng(5)
    for _ in range(20):
        m = np.eye(3) + 0.3 * (rng.normal(size=(3, 3)) + 1j * rng.normal(size=(3, 3)))
        g = oracle.reunitarise(m)
        assert np.max(np.abs(g @ g.conj().T - np.eye(3))) < 1e-15 * 4
        assert abs(np.linalg.det(g) - 1) < 1e-15 * 4
        # row 0 keeps its direction; row 1 stays in span(row0, row1) with positive overlap
        assert abs(np.vdot(g[0], m[0]) - np.linalg.norm(m[0])) < 1e-14
        assert np.vdot(g[1], m[1]).real > 0 and abs(np.vdot(g[1], m[1]).imag) < 1e-14
        # equals QR-based construction: rows of m^T's QR (library routine)
        q, r = np.linalg.qr(m.T.copy())
        q = q * (np.diag(r) / np.abs(np.diag(r)))[None, :].conj()   # make diag(r) real positive
        assert np.max(np.abs(g[:2] - q.T[:2])) < 1e-14
    su = gi.haar_su3(3, 7, 0, 4).numpy()
    for u in su:
        assert np.max(np.abs(oracle.reunitarise(u) - u)) < 4e-16


def test_two_row_roundtrip():
    L = (4, 4, 4, 4)
    U = gi.make_config(L, 13, 0.59)
    R = oracle.two_row_roundtrip(U)
    assert np.array_equal(R[:, :, :2], U.numpy()[:, :, :2])
    assert np.max(np.abs(R - U.numpy())) < 4e-15     # gauge-transformed links are unitary to a few ulp


# ---------------------------------------------------------------- P5: update orientation
def _polyakov_traces(U, L, mu):
    g = gi._grid(U[:, mu], L)                           # [Lt,Lz,Ly,Lx,3,3]
    ax = gi._AXIS[mu]
    P = None
    for i in range(L[mu]):
        sl = g.select(ax, i)
        P = sl if P is None else P @ sl
    return torch.einsum("...ii->...", P)


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (6, 4, 3, 2)])
def test_update_preserves_plaquettes_and_polyakov_loops(L):
    U = gi.make_config(L, 14, 0.58)
    U1, th, Fh = oracle.iterate(L, U, 3, ALPHA)
    U1 = torch.from_numpy(U1)
    p0, p1 = gi.plaquette_traces(U, L), gi.plaquette_traces(U1, L)
    assert float((p0 - p1).abs().max()) < 1e-13
    for mu in range(4):
        assert float((_polyakov_traces(U, L, mu) - _polyakov_traces(U1, L, mu)).abs().max()) < 1e-13
    eye = torch.eye(3, dtype=torch.complex128)
    assert float((U1 @ U1.conj().transpose(-1, -2) - eye).abs().max()) < 1e-13
    assert float((torch.linalg.det(U1) - 1).abs().max()) < 1e-13
    assert abs(gi.mean_plaquette(U, L) - gi.mean_plaquette(U1, L)) < 1e-14


def test_update_is_the_stated_gauge_transform():
    """U' = g(x) U g(x+mu)^+ checked against lgf_inputs.gauge_transform (independent torch code)."""
    L = (4, 6, 3, 2)
    U = gi.make_config(L, 15, 0.59)
    g = gi.haar_su3(4, 8, 0, gi.volume(L))
    got = oracle.update_links(L, U, g)
    ref = gi.gauge_transform(U, g, L).numpy()
    assert np.max(np.abs(got - ref)) < 1e-14


# ---------------------------------------------------------------- P6, P7: direction, 1/V, alpha/2, p^2
@pytest.mark.parametrize("L", [(8, 8, 8, 8), (6, 4, 12, 8)])
def test_pure_gauge_reaches_F_one(L):
    U = gi.make_config(L, 16, kind="pure_gauge")
    _, n, theta, F, thh, Fh = oracle.fix(L, U, ALPHA, 1e-15, 500)
    assert theta < 1e-15 and n < 60
    assert abs(1 - F) < 1e-13
    assert np.all(np.diff(Fh) > -1e-15)                 # F non-decreasing (reading #18)
    tail = thh[-4:-1] / thh[-5:-2]
    assert np.all(np.abs(tail - (1 - 16 * ALPHA) ** 2) < 0.02)   # tail ratio -> 0.0784


@pytest.mark.parametrize("L,alpha", [((8, 8, 8, 8), 0.08), ((8, 8, 8, 8), 0.05), ((6, 4, 12, 8), 0.08)])
def test_closed_form_first_step_ratio(L, alpha):
    """P7: infinitesimal gauge copy of the unit field: theta1/theta0 = (1 - alpha p2max)^2."""
    U = gi.small_gauge_copy_of_unit(L, 3, 1e-5)
    _, thh, Fh = oracle.iterate(L, U, 1, alpha)
    assert abs(thh[1] / thh[0] - (1 - 16 * alpha) ** 2) < 5e-6
    assert Fh[1] >= Fh[0]


def test_closed_form_one_step_convergence():
    L = (8, 8, 8, 8)
    U = gi.small_gauge_copy_of_unit(L, 3, 1e-5)
    _, thh, _ = oracle.iterate(L, U, 1, 1.0 / 16.0)
    assert thh[1] / thh[0] < 1e-8


def test_rough_config_F_monotone_and_counts():
    """configs[0]: 8^4, plaquette 0.59, alpha 0.08, theta < 1e-12 (~31 iterations)."""
    L = (8, 8, 8, 8)
    U = gi.make_config(L, gi.CONFIG_SEED, 0.59)
    assert abs(gi.mean_plaquette(U, L) - 0.59) < 0.005
    _, n, theta, F, thh, Fh = oracle.fix(L, U, ALPHA, 1e-12, 5000)
    assert 25 <= n <= 40 and theta < 1e-12
    assert np.all(np.diff(Fh) > -1e-15)
    small = thh < 1e-3
    assert np.all(np.diff(thh[small]) < 0)              # strictly decreasing in the linear regime
    assert 0.85 < F < 0.95
    # without Fourier acceleration it would need ~10x more: the scale must be active
    assert thh[20] < 1e-3


def test_fix_count_semantics():
    """Reading #12: strict theta < tol tested after each update on the updated links;
    `iterations` = number of updates applied; a field already below tolerance takes 0 updates; max_iter caps."""
    L = (4, 6, 3, 2)
    U = gi.make_config(L, 20, 0.59)
    tol = 1e-8
    _, n, theta, F, thh, Fh = oracle.fix(L, U, ALPHA, tol, 5000)
    assert len(thh) == n + 1 and len(Fh) == n + 1 and n >= 2
    assert thh[n] < tol <= thh[n - 1]                   # first crossing, strict
    assert np.all(thh[:n] >= tol)                       # no earlier iterate was already below
    assert theta == thh[n] and F == Fh[n]
    # the history is the trajectory of `iterate`: same updates, nothing skipped or repeated
    ref, thi, Fi = oracle.iterate(L, U, n, ALPHA)
    assert np.array_equal(thi, thh) and np.array_equal(Fi, Fh)
    # strictness: a tolerance equal to a value on the trajectory does not stop there
    _, n_eq, _, _, _, _ = oracle.fix(L, U, ALPHA, float(thh[n - 1]), 5000)
    assert n_eq == n                                    # theta[n-1] == tol continues, theta[n] < tol stops
    _, n_eq2, _, _, _, _ = oracle.fix(L, U, ALPHA, float(thh[n]), 5000)
    assert n_eq2 > n                                    # theta == tol is NOT converged
    # max_iter caps the count; the result is the k-th iterate
    for k in (0, 1, 3):
        out, nk, thk, Fk, hk, _ = oracle.fix(L, U, ALPHA, 1e-300, k)
        assert nk == k and len(hk) == k + 1 and thk == thh[k]
    # already below tolerance: zero updates, links untouched
    out, n0, th0, _, h0, _ = oracle.fix(L, U, ALPHA, 1e30, 5000)
    assert n0 == 0 and th0 == thh[0] and len(h0) == 1
    assert np.array_equal(out, gi.from_real(gi.as_real(U)).numpy().reshape(out.shape))


# ---------------------------------------------------------------- P11: brute-force convolution
def test_fourier_acceleration_equals_position_space_convolution():
    L = (4, 4, 2, 2)
    V = gi.volume(L)
    U = gi.make_config(L, 17, 0.59)
    D, _, _ = oracle.measure(L, U)
    Dt = oracle.fourier_accelerate(L, D)
    Dt_direct = oracle.fourier_accelerate(L, D, direct=True)
    assert np.max(np.abs(Dt - Dt_direct)) < 1e-13
    # kernel K(r) = (1/V) sum_{k != 0} (p2max/p2(k)) cos(2 pi k.r/L), typed out here
    c = _coords(L)
    p2 = sum(4 * np.sin(np.pi * c[:, m] / L[m]) ** 2 for m in range(4))
    S = np.zeros(V)
    S[1:] = p2.max() / p2[1:]
    Kr = np.zeros(V)
    for r in range(V):
        ph = sum(c[:, m] * c[r, m] / L[m] for m in range(4))
        Kr[r] = np.sum(S * np.cos(2 * np.pi * ph)) / V
    out = np.zeros_like(D)
    for x in range(V):
        diff = [(c[x, m] - c[:, m]) % L[m] for m in range(4)]
        sidx = diff[0] + L[0] * (diff[1] + L[1] * (diff[2] + L[2] * diff[3]))
        out[x] = np.einsum("y,yij->ij", Kr[sidx], D)
    assert np.max(np.abs(out - Dt)) < 1e-12
    # the filtered field stays anti-Hermitian and traceless (K real)
    assert np.max(np.abs(Dt + Dt.conj().transpose(0, 2, 1))) < 1e-13
    assert np.max(np.abs(np.einsum("nii->n", Dt))) < 1e-13


def test_build_g_first_order():
    L = (4, 4, 2, 2)
    U = gi.make_config(L, 18, 0.59)
    D, _, _ = oracle.measure(L, U)
    Dt = oracle.fourier_accelerate(L, D)
    g = oracle.build_g(L, Dt, ALPHA)
    for s in (0, 5, 63):
        assert np.max(np.abs(g[s] - oracle.reunitarise(np.eye(3) + 0.5 * ALPHA * Dt[s]))) == 0
    assert np.max(np.abs(g @ g.conj().transpose(0, 2, 1) - np.eye(3))) < 1e-14


def test_oracle_thread_count_does_not_change_bits():
    L = (4, 6, 3, 2)
    U = gi.make_config(L, 19, 0.59)
    n0 = oracle.threads()
    a = oracle.iterate(L, U, 3, ALPHA)
    oracle.set_threads(1)
    b = oracle.iterate(L, U, 3, ALPHA)
    oracle.set_threads(n0)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
