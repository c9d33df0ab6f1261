"""Seeded synthetic SU(3) lattice inputs (shared by the oracle tests, the GPU tests and bench.py).

This module is the ONLY code that both sides of the parity check see.  It holds no step of the
gauge-fixing ITERATION (no Delta, no FFT, no p^2 table, no g-build from Delta~); it only makes the
*inputs* named by BASELINE.json `configs` (SURVEY.md §8(d) "Inputs").  Two of its tools do restate
formulas the method also uses, for the generator's own purposes: `su3_project` is a row Gram-Schmidt
(SURVEY.md §8(c) reading #9's formula, used here to MAKE SU(3) matrices) and `gauge_transform` is
U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger (step 5's formula, used here to scramble the gauge).  Neither the
oracle nor the CUDA path calls them; tests use the second as an independent pin of the update's
orientation.  The inputs:

* rough links  U = SU3-projection of exp(i eps H),  H = sum_a xi_a lambda_a / 2,  xi_a ~ N(0,1),
  eps chosen so the mean plaquette hits a target (0.55 - 0.60, "beta ~ 6.0-like roughness");
* a Haar-random SU(3) gauge transform per site, applied as U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger;
* the "pure gauge copy of the unit configuration" (configs[1]): the same transform applied to U = 1;
* a *small* gauge transform g = SU3(exp(i eps H)) of the unit field (pin P7).

Random numbers come from a counter-based generator (splitmix64 finaliser of (seed, stream, index)),
so a field does not depend on chunking, loop order or device.  Everything is plain torch tensor
code and runs on CPU or on a CUDA device (`device=`), in float64 / complex128.

Layout of a link field (the C-ABI boundary layout): site-major
`links[s, mu, row, col]` complex, s = x + Lx*(y + Ly*(z + Lz*t)), L = (Lx, Ly, Lz, Lt), mu = 0..3
<-> x, y, z, t.  `as_real(links)` views it as the `[s][mu][row][col][re,im]` real array.
"""
from __future__ import annotations

import math
from typing import Sequence, Tuple

import torch

__all__ = [
    "volume", "gaussian", "uniform53", "random_algebra", "su3_project", "haar_su3",
    "rough_links", "gauge_transform", "unit_links", "epsilon_for_plaquette", "mean_plaquette",
    "make_config", "small_gauge_copy_of_unit", "as_real", "from_real", "CONFIG_SEED",
]

CONFIG_SEED = 12081186  # + config index (SURVEY.md §8(d) "Seeds")

_M64 = (1 << 64) - 1


def _s64(v: int) -> int:
    """Python int (mod 2^64) -> the same bit pattern as a signed 64-bit value."""
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


_GOLDEN = _s64(0x9E3779B97F4A7C15)
_C1 = _s64(0xBF58476D1CE4E5B9)
_C2 = _s64(0x94D049BB133111EB)


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right of int64 bit patterns."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def _mix64(z: torch.Tensor) -> torch.Tensor:
    """splitmix64 output function on int64 tensors (two's complement wrap = arithmetic mod 2^64)."""
    z = z + _GOLDEN
    z = (z ^ _lsr(z, 30)) * _C1
    z = (z ^ _lsr(z, 27)) * _C2
    return z ^ _lsr(z, 31)


def _mix64_int(v: int) -> int:
    v = (v + 0x9E3779B97F4A7C15) & _M64
    v = ((v ^ (v >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    v = ((v ^ (v >> 27)) * 0x94D049BB133111EB) & _M64
    return v ^ (v >> 31)


def _bits(seed: int, stream: int, index: torch.Tensor) -> torch.Tensor:
    key = _mix64_int((seed & _M64) ^ _mix64_int(stream & _M64))
    return _mix64(index + _s64(key))


def uniform53(seed: int, stream: int, index: torch.Tensor) -> torch.Tensor:
    """Uniform in (0, 1]: (top 53 bits + 1) * 2^-53, one value per int64 counter in `index`."""
    return (_lsr(_bits(seed, stream, index), 11).to(torch.float64) + 1.0) * (2.0 ** -53)


def gaussian(seed: int, stream: int, index: torch.Tensor) -> torch.Tensor:
    """N(0,1) by Box-Muller from counters (2*index, 2*index+1) of the given stream."""
    u1 = uniform53(seed, stream, 2 * index)
    u2 = uniform53(seed, stream, 2 * index + 1)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)


def volume(L: Sequence[int]) -> int:
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3])


def _gell_mann(device) -> torch.Tensor:
    lam = torch.zeros(8, 3, 3, dtype=torch.complex128)
    lam[0, 0, 1] = lam[0, 1, 0] = 1
    lam[1, 0, 1] = -1j
    lam[1, 1, 0] = 1j
    lam[2, 0, 0] = 1
    lam[2, 1, 1] = -1
    lam[3, 0, 2] = lam[3, 2, 0] = 1
    lam[4, 0, 2] = -1j
    lam[4, 2, 0] = 1j
    lam[5, 1, 2] = lam[5, 2, 1] = 1
    lam[6, 1, 2] = -1j
    lam[6, 2, 1] = 1j
    s3 = 1.0 / math.sqrt(3.0)
    lam[7, 0, 0] = lam[7, 1, 1] = s3
    lam[7, 2, 2] = -2 * s3
    return lam.to(device)


def random_algebra(seed: int, stream: int, first: int, count: int, device="cpu") -> torch.Tensor:
    """H[n] = sum_a xi_a lambda_a / 2 for n = first .. first+count-1 (traceless Hermitian, [count,3,3])."""
    n = torch.arange(first, first + count, dtype=torch.int64, device=device)
    idx = n[:, None] * 8 + torch.arange(8, dtype=torch.int64, device=device)[None, :]
    xi = gaussian(seed, stream, idx)                       # [count, 8]
    return torch.einsum("na,aij->nij", xi.to(torch.complex128), _gell_mann(device)) * 0.5


def su3_project(m: torch.Tensor) -> torch.Tensor:
    """Rows 0,1 orthonormalised in order, row 2 = conj(row0 x row1).  m: [..., 3, 3] complex."""
    r0 = m[..., 0, :]
    r1 = m[..., 1, :]
    r0 = r0 / torch.linalg.vector_norm(r0, dim=-1, keepdim=True)
    r1 = r1 - (r0.conj() * r1).sum(-1, keepdim=True) * r0
    r1 = r1 / torch.linalg.vector_norm(r1, dim=-1, keepdim=True)
    r2 = torch.linalg.cross(r0, r1, dim=-1).conj()
    return torch.stack([r0, r1, r2], dim=-2)


def haar_su3(seed: int, stream: int, first: int, count: int, device="cpu") -> torch.Tensor:
    """Haar-distributed SU(3): 3x3 complex Gaussian matrix -> su3_project.  [count, 3, 3]."""
    n = torch.arange(first, first + count, dtype=torch.int64, device=device)
    idx = n[:, None] * 18 + torch.arange(18, dtype=torch.int64, device=device)[None, :]
    z = gaussian(seed, stream, idx).reshape(count, 3, 3, 2)
    return su3_project(torch.complex(z[..., 0], z[..., 1]))


_CHUNK = 1 << 18


def rough_links(L: Sequence[int], eps: float, seed: int, device="cpu") -> torch.Tensor:
    """links[s, mu] = su3_project(matrix_exp(i eps H)), independent per link.  [V, 4, 3, 3]."""
    nlinks = volume(L) * 4
    out = torch.empty(nlinks, 3, 3, dtype=torch.complex128, device=device)
    for first in range(0, nlinks, _CHUNK):
        cnt = min(_CHUNK, nlinks - first)
        H = random_algebra(seed, 1, first, cnt, device)
        out[first:first + cnt] = su3_project(torch.linalg.matrix_exp(1j * eps * H))
    return out.reshape(volume(L), 4, 3, 3)


def unit_links(L: Sequence[int], device="cpu") -> torch.Tensor:
    eye = torch.eye(3, dtype=torch.complex128, device=device)
    return eye.expand(volume(L), 4, 3, 3).clone()


def _grid(field: torch.Tensor, L: Sequence[int]) -> torch.Tensor:
    """[V, ...] -> [Lt, Lz, Ly, Lx, ...] (x fastest)."""
    return field.reshape(L[3], L[2], L[1], L[0], *field.shape[1:])


_AXIS = (3, 2, 1, 0)  # mu -> grid axis


def shift_fwd(field: torch.Tensor, L: Sequence[int], mu: int) -> torch.Tensor:
    """f(x) -> f(x + mu_hat), periodic.  field: [V, ...]."""
    return torch.roll(_grid(field, L), shifts=-1, dims=_AXIS[mu]).reshape(field.shape)


def gauge_transform(links: torch.Tensor, g: torch.Tensor, L: Sequence[int]) -> torch.Tensor:
    """U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger.  links [V,4,3,3], g [V,3,3]."""
    out = torch.empty_like(links)
    for mu in range(4):
        gf = shift_fwd(g, L, mu)
        out[:, mu] = g @ links[:, mu] @ gf.conj().transpose(-1, -2)
    return out


def mean_plaquette(links: torch.Tensor, L: Sequence[int]) -> float:
    """(1/(6V)) sum_x sum_{mu<nu} Re Tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+] / 3."""
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            a = links[:, mu] @ shift_fwd(links[:, nu], L, mu)
            b = links[:, nu] @ shift_fwd(links[:, mu], L, nu)
            tot += float(torch.einsum("nij,nij->", a, b.conj()).real)
    return tot / (6.0 * 3.0 * volume(L))


def plaquette_traces(links: torch.Tensor, L: Sequence[int]) -> torch.Tensor:
    """Tr of every plaquette, [6, V] complex (gauge-invariant; used by the invariance pins)."""
    out = []
    for mu in range(4):
        for nu in range(mu + 1, 4):
            a = links[:, mu] @ shift_fwd(links[:, nu], L, mu)
            b = links[:, nu] @ shift_fwd(links[:, mu], L, nu)
            out.append(torch.einsum("nij,nij->n", a, b.conj()))
    return torch.stack(out)


_EPS_CACHE: dict = {}


def epsilon_for_plaquette(target: float, seed: int = 7, nsample: int = 1 << 16) -> float:
    """eps with E[plaquette] = target for independent links: plaquette = c(eps)^4,
    c = E[Re Tr U]/3; c is estimated on a fixed sample and eps is bisected."""
    key = (round(target, 6), seed, nsample)
    if key in _EPS_CACHE:
        return _EPS_CACHE[key]
    H = random_algebra(seed, 99, 0, nsample)

    def plaq(eps: float) -> float:
        U = su3_project(torch.linalg.matrix_exp(1j * eps * H))
        c = float(torch.einsum("nii->", U).real) / (3.0 * nsample)
        return c ** 4

    lo, hi = 0.05, 1.2
    for _ in range(40):
        mid = 0.5 * (lo + hi)
        if plaq(mid) > target:
            lo = mid
        else:
            hi = mid
    _EPS_CACHE[key] = 0.5 * (lo + hi)
    return _EPS_CACHE[key]


def make_config(L: Sequence[int], seed: int, plaquette: float = 0.59, kind: str = "rough",
                device="cpu") -> torch.Tensor:
    """The configs' generator.  kind = "rough": rough links at the target plaquette + Haar gauge
    transform;  kind = "pure_gauge": Haar gauge transform of the unit field;  kind = "haar_links":
    independent Haar-random links (pin P8).  Returns complex128 [V, 4, 3, 3]."""
    V = volume(L)
    if kind == "haar_links":
        return haar_su3(seed, 3, 0, 4 * V, device).reshape(V, 4, 3, 3)
    g = haar_su3(seed, 2, 0, V, device)
    if kind == "pure_gauge":
        base = unit_links(L, device)
    elif kind == "rough":
        base = rough_links(L, epsilon_for_plaquette(plaquette), seed, device)
    else:
        raise ValueError(kind)
    return gauge_transform(base, g, L)


def small_gauge_copy_of_unit(L: Sequence[int], seed: int, eps: float = 1e-5, device="cpu") -> torch.Tensor:
    """U_mu(x) = g(x) g(x+mu)^+, g = su3_project(exp(i eps H)) (pin P7)."""
    V = volume(L)
    g = su3_project(torch.linalg.matrix_exp(1j * eps * random_algebra(seed, 4, 0, V, device)))
    return gauge_transform(unit_links(L, device), g, L)


def as_real(links: torch.Tensor, dtype=torch.float64) -> torch.Tensor:
    """complex [V,4,3,3] -> contiguous real [V,4,3,3,2] of `dtype` (fp32: rounded once)."""
    return torch.view_as_real(links.contiguous()).to(dtype).contiguous()


def from_real(arr: torch.Tensor) -> torch.Tensor:
    return torch.view_as_complex(arr.to(torch.float64).contiguous())
