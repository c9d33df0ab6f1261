"""Pins of the oracle's temporal Wilson lines and singlet correlator (eq. (1)):
closed forms, symmetries, a torch restatement and gauge covariance -- nothing here calls the CUDA path."""
import numpy as np
import pytest
import torch

import lgf_inputs as gi
import oracle

SHAPES = [(4, 4, 4, 4), (6, 4, 3, 8), (4, 6, 2, 3), (8, 4, 4, 2)]


def _vs(L):
    return L[0] * L[1] * L[2]


def _field(U, L):
    """links [V,4,3,3] -> numpy [t,z,y,x,mu,3,3]."""
    return U.numpy().reshape(L[3], L[2], L[1], L[0], 4, 3, 3)


@pytest.mark.parametrize("L", SHAPES)
def test_unit_field_gives_unit_lines_and_unit_correlator(L):
    U = gi.unit_links(L)
    W = oracle.wilson_lines(L, U)
    assert np.array_equal(W, np.broadcast_to(np.eye(3), W.shape))
    C = oracle.singlet_correlator(L, U)
    assert np.max(np.abs(C - 1.0)) == 0


@pytest.mark.parametrize("L", SHAPES)
def test_wilson_lines_equal_typed_out_ordered_product(L):
    U = gi.make_config(L, 51, 0.59)
    W = oracle.wilson_lines(L, U)
    f = _field(U, L)
    ref = np.broadcast_to(np.eye(3, dtype=complex), (L[2], L[1], L[0], 3, 3)).copy()
    for t in range(L[3]):                                   # U_t(x,0) U_t(x,1) ... in this order
        ref = ref @ f[t, :, :, :, 3]
    assert np.max(np.abs(W - ref.reshape(-1, 3, 3))) < 1e-14
    assert np.max(np.abs(W @ W.conj().transpose(0, 2, 1) - np.eye(3))) < 1e-13      # a product of SU(3) matrices
    assert np.max(np.abs(np.linalg.det(W) - 1)) < 1e-13
    if L[3] > 2:                                            # the order matters: the reversed product is another matrix
        rev = np.broadcast_to(np.eye(3, dtype=complex), ref.shape).copy()
        for t in reversed(range(L[3])):
            rev = rev @ f[t, :, :, :, 3]
        assert np.max(np.abs(W - rev.reshape(-1, 3, 3))) > 1e-3


@pytest.mark.parametrize("L", SHAPES)
def test_correlator_closed_forms_and_symmetry(L):
    U = gi.make_config(L, 52, 0.59)
    W = oracle.wilson_lines(L, U)
    C = oracle.singlet_correlator(L, U)
    Vs = _vs(L)
    assert abs(C[0] - 1.0) < 1e-14                          # C(0) = (1/3Vs) sum Tr W W^+ = 1
    S = W.sum(0)                                            # sum_r C(r) = Tr[(sum_x W)(sum_y W)^+] / (3 Vs)
    assert abs(C.sum() - np.sum(np.abs(S) ** 2) / (3 * Vs)) < 1e-12 * Vs
    c = C.reshape(L[2], L[1], L[0])
    neg = np.roll(c[::-1, ::-1, ::-1], 1, axis=(0, 1, 2))   # C(-r)
    assert np.max(np.abs(neg - c.conj())) < 1e-14
    assert np.max(np.abs(C)) <= 1 + 1e-14                   # Cauchy-Schwarz, |Tr a b^+| <= 3


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (6, 4, 3, 8)])
def test_correlator_equals_roll_restatement(L):
    U = gi.make_config(L, 53, 0.59)
    W = oracle.wilson_lines(L, U).reshape(L[2], L[1], L[0], 3, 3)
    C = oracle.singlet_correlator(L, U).reshape(L[2], L[1], L[0])
    for r in [(0, 0, 1), (1, 0, 0), (2, 3, 1), (L[2] - 1, 1, L[0] - 1)]:       # (rz, ry, rx)
        shifted = np.roll(W, shift=(-r[0], -r[1], -r[2]), axis=(0, 1, 2))       # W(x + r)
        ref = np.einsum("zyxij,zyxij->", shifted, W.conj()) / (3 * _vs(L))
        assert abs(C[r] - ref) < 1e-14


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (4, 6, 2, 3)])
def test_gauge_covariance(L):
    """U_mu(x) -> g(x) U_mu(x) g(x+mu)^+ maps W(x) -> g(x,0) W(x) g(x,0)^+ (the product along periodic t telescopes):
    Tr W (the Polyakov loop) is invariant, and so is C when g does not depend on the spatial position."""
    U = gi.make_config(L, 54, 0.59)
    V = gi.volume(L)
    g = gi.haar_su3(99, 2, 0, V)
    Ug = gi.gauge_transform(U, g, L)
    W, Wg = oracle.wilson_lines(L, U), oracle.wilson_lines(L, Ug)
    g0 = g.numpy()[:_vs(L)]                                 # t = 0 slice: sites x + Lx (y + Ly z)
    assert np.max(np.abs(Wg - g0 @ W @ g0.conj().transpose(0, 2, 1))) < 1e-13
    assert np.max(np.abs(np.einsum("nii->n", W) - np.einsum("nii->n", Wg))) < 1e-13
    # spatially constant transform h(t): C unchanged
    h = gi.haar_su3(7, 2, 0, L[3])
    gt = h.repeat_interleave(_vs(L), dim=0)                 # site s = xs + Vs t -> h[t]
    C, Ch = oracle.singlet_correlator(L, U), oracle.singlet_correlator(L, gi.gauge_transform(U, gt, L))
    assert np.max(np.abs(C - Ch)) < 1e-13
    # a position-dependent transform changes C(r != 0): the quantity is NOT gauge invariant
    Cg = oracle.singlet_correlator(L, Ug)
    assert abs(Cg[0] - 1) < 1e-13 and np.max(np.abs(C - Cg)) > 1e-3
