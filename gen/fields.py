"""Seeded, index-addressable synthetic inputs (gauge links, Gaussian spinors).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library
(``paper_2407_08092_b200/``) with identical bits.  It holds none of the
method's arithmetic: no Dirac operator, no gamma matrices, no clover term.
It only draws random numbers and builds SU(3) matrices.

Every value is a pure function of ``(seed, global index)`` through a
counter-based hash (splitmix64 finaliser), so any site range of any lattice
can be generated in chunks, on the CPU or on a CUDA device, without storing a
generator state.  (Box-Muller uses log/sin/cos, whose last bit may differ
between CPU and CUDA libm; parity tests therefore always hand the *same
array* to both sides.)

Recipe (BASELINE.json configs; SURVEY.md section 8(c) readings R17, R18 --
the paper itself, Table 5, only names the CLQCD ensemble,
which is not available; these fields stand in for it):

* ``G``: 3x3, iid N(0,1) real and imaginary parts.
* ``H = (G + G^H)/2 - tr(.)/3 * 1``  (traceless Hermitian).
* ``U = exp(i * eps * H)`` by scaling-and-squaring Taylor series in fp64.
* optional re-unitarisation (R17): normalise row 0; Gram-Schmidt row 1
  against row 0 and normalise; row 2 = conj(row 0 x row 1).
* spinors: iid N(0,1) real and imaginary parts, 12 complex per site.

Natural (external) layouts, C order, x fastest among sites:

* gauge  ``[t][z][y][x][mu][row][col]`` complex  -> shape (T, L, L, L, 4, 3, 3)
* spinor ``[t][z][y][x][spin][colour]`` complex  -> shape (T, L, L, L, 4, 3)
"""
from __future__ import annotations

import math

import torch

_MASK64 = (1 << 64) - 1


def _s64(c: int) -> int:
    """Two's-complement reinterpretation of an unsigned 64-bit constant."""
    c &= _MASK64
    return c - (1 << 64) if c >= (1 << 63) else c


_C1 = _s64(0xBF58476D1CE4E5B9)
_C2 = _s64(0x94D049BB133111EB)
_GOLD = _s64(0x9E3779B97F4A7C15)
_STREAM = _s64(0xD1B54A32D192ED03)


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right on int64 tensors (torch's >> is arithmetic)."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def _mix64(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _C1
    z = (z ^ _lsr(z, 27)) * _C2
    return z ^ _lsr(z, 31)


def hash_u64(seed: int, counter: torch.Tensor) -> torch.Tensor:
    """64 pseudo-random bits per counter value (int64 tensor, wraps mod 2^64)."""
    key = _s64((seed + 1) * 0x9E3779B97F4A7C15)
    z = counter * _STREAM + key
    return _mix64(_mix64(z) + _GOLD)


def uniform01(seed: int, counter: torch.Tensor) -> torch.Tensor:
    """Uniform in the open interval (0, 1), fp64, 53 bits."""
    bits = _lsr(hash_u64(seed, counter), 11)
    return (bits.to(torch.float64) + 0.5) * (2.0 ** -53)


def gaussian(seed: int, start: int, count: int, device="cpu") -> torch.Tensor:
    """``count`` iid N(0,1) fp64 values with global indices start..start+count-1."""
    idx = torch.arange(start, start + count, dtype=torch.int64, device=device)
    pair = idx >> 1
    u1 = uniform01(seed, 2 * pair)
    u2 = uniform01(seed, 2 * pair + 1)
    r = torch.sqrt(-2.0 * torch.log(u1))
    ang = (2.0 * math.pi) * u2
    return torch.where((idx & 1) == 0, r * torch.cos(ang), r * torch.sin(ang))


def complex_gaussian(seed: int, start: int, count: int, device="cpu") -> torch.Tensor:
    """``count`` complex values, re and im iid N(0,1); global complex index start.."""
    g = gaussian(seed, 2 * start, 2 * count, device=device).view(count, 2)
    return torch.view_as_complex(g.contiguous())


def _expm_i_eps_h(H: torch.Tensor, eps: float) -> torch.Tensor:
    """exp(i*eps*H) for a batch of 3x3 Hermitian matrices, fp64 to ~1e-16."""
    A = (1j * eps) * H
    # scale so that ||A/2^s|| <= 0.25, Taylor to order 14, square s times
    nrm = torch.linalg.matrix_norm(A, ord="fro").max().item() if A.numel() else 0.0
    s = max(0, int(math.ceil(math.log2(max(nrm, 1e-300) / 0.25)))) if nrm > 0.25 else 0
    A = A / (2.0 ** s)
    eye = torch.eye(3, dtype=A.dtype, device=A.device).expand_as(A)
    term = eye.clone()
    acc = eye.clone()
    for k in range(1, 15):
        term = torch.matmul(term, A) / k
        acc = acc + term
    for _ in range(s):
        acc = torch.matmul(acc, acc)
    return acc


def reunitarise(U: torch.Tensor) -> torch.Tensor:
    """Project a batch of 3x3 matrices onto SU(3) row by row (reading R17)."""
    r0 = U[..., 0, :]
    r1 = U[..., 1, :]
    r0 = r0 / torch.linalg.vector_norm(r0, dim=-1, keepdim=True)
    r1 = r1 - (torch.conj(r0) * r1).sum(-1, keepdim=True) * r0
    r1 = r1 / torch.linalg.vector_norm(r1, dim=-1, keepdim=True)
    r2 = torch.conj(torch.linalg.cross(r0, r1, dim=-1))
    return torch.stack([r0, r1, r2], dim=-2)


def gauge_links(seed: int, link_start: int, link_count: int, eps: float,
                reunit: bool = False, device="cpu") -> torch.Tensor:
    """Links with global link indices ``4*site + mu`` in [link_start, +link_count).

    Returns complex128 of shape (link_count, 3, 3).
    """
    G = complex_gaussian(seed, 9 * link_start, 9 * link_count, device=device)
    G = G.view(link_count, 3, 3)
    H = 0.5 * (G + G.conj().transpose(-1, -2))
    tr = torch.diagonal(H, dim1=-2, dim2=-1).sum(-1) / 3.0
    H = H - tr[:, None, None] * torch.eye(3, dtype=H.dtype, device=H.device)
    U = _expm_i_eps_h(H, eps)
    if reunit:
        U = reunitarise(U)
    return U


def gauge_field(L: int, T: int, seed: int, eps: float, reunit: bool = False,
                device="cpu", dtype=torch.complex128,
                chunk_links: int = 1 << 22) -> torch.Tensor:
    """Whole gauge field, natural layout (T, L, L, L, 4, 3, 3), in ``dtype``.

    Generated in fp64 chunk by chunk and rounded once to ``dtype``.
    """
    nlinks = 4 * L * L * L * T
    out = torch.empty((nlinks, 3, 3), dtype=dtype, device=device)
    for s in range(0, nlinks, chunk_links):
        n = min(chunk_links, nlinks - s)
        out[s:s + n] = gauge_links(seed, s, n, eps, reunit, device).to(dtype)
    return out.view(T, L, L, L, 4, 3, 3)


def unit_gauge_field(L: int, T: int, device="cpu", dtype=torch.complex128) -> torch.Tensor:
    """Free field: every link is the 3x3 identity."""
    U = torch.zeros((T, L, L, L, 4, 3, 3), dtype=dtype, device=device)
    for c in range(3):
        U[..., c, c] = 1.0
    return U


def spinor_field(L: int, T: int, seed: int, device="cpu", dtype=torch.complex128,
                 chunk_sites: int = 1 << 22) -> torch.Tensor:
    """Complex Gaussian spinor, natural layout (T, L, L, L, 4, 3), in ``dtype``."""
    V = L * L * L * T
    out = torch.empty((V, 12), dtype=dtype, device=device)
    for s in range(0, V, chunk_sites):
        n = min(chunk_sites, V - s)
        out[s:s + n] = complex_gaussian(seed, 12 * s, 12 * n, device).view(n, 12).to(dtype)
    return out.view(T, L, L, L, 4, 3)


def site_parity(L: int, T: int, device="cpu") -> torch.Tensor:
    """(T, L, L, L) int64 tensor of (x+y+z+t) mod 2 (even = 0)."""
    t = torch.arange(T, device=device).view(T, 1, 1, 1)
    z = torch.arange(L, device=device).view(1, L, 1, 1)
    y = torch.arange(L, device=device).view(1, 1, L, 1)
    x = torch.arange(L, device=device).view(1, 1, 1, L)
    return (x + y + z + t) & 1


def random_su3_per_site(L: int, T: int, seed: int, device="cpu") -> torch.Tensor:
    """One Haar-ish SU(3) matrix per site (for gauge-covariance tests), (T,L,L,L,3,3)."""
    V = L * L * L * T
    G = complex_gaussian(seed, 0, 9 * V, device=device).view(V, 3, 3)
    W = reunitarise(G)
    return W.view(T, L, L, L, 3, 3)
