"""Seeded synthetic input generators on a torch device (for the paper-scale configs).

Same recipes and the same counter hash as ``inputs.py`` (numpy), written with torch ops so that
the 32^3x64 / 48^3x96 gauge fields and the 500 packed Z4 sources of BASELINE.json c4/c5 can be
produced on the GPU in seconds.  Like ``inputs.py`` this module holds INPUT generation only: no
Dirac operator, no gamma matrices, no solver, no contraction.  Z4 exponents are bit-identical to
``inputs.z4_exponents``; gauge links agree with ``inputs.gauge_field`` to rounding (the matrix
exponential is taken with ``torch.linalg.matrix_exp`` instead of an eigendecomposition).
"""
from __future__ import annotations

import math

import torch

from .inputs import GAUGE_STREAM, volume

_MASK64 = (1 << 64) - 1


def _s64(v: int) -> int:
    """Python int (mod 2^64) -> the signed 64-bit value with the same bits."""
    v &= _MASK64
    return v - (1 << 64) if v >= (1 << 63) else v


_GOLDEN = 0x9E3779B97F4A7C15
_M1 = _s64(0xBF58476D1CE4E5B9)
_M2 = _s64(0x94D049BB133111EB)


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    """logical shift right of int64 bit patterns"""
    return (z >> k) & ((1 << (64 - k)) - 1)


def mix64(z: torch.Tensor) -> torch.Tensor:
    z = z ^ _lsr(z, 30)
    z = z * _M1
    z = z ^ _lsr(z, 27)
    z = z * _M2
    z = z ^ _lsr(z, 31)
    return z


def _mix64_int(z: int) -> int:
    z &= _MASK64
    z ^= z >> 30
    z = (z * 0xBF58476D1CE4E5B9) & _MASK64
    z ^= z >> 27
    z = (z * 0x94D049BB133111EB) & _MASK64
    z ^= z >> 31
    return z


def hash_i64(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """h(seed, stream, idx) as int64 bit patterns; idx int64."""
    k = _mix64_int(int(seed) * _GOLDEN + int(stream))
    return mix64(idx + _s64(k))


def z4_packed(dims, seed: int, r: int, device) -> torch.Tensor:
    """Packed Z4 exponents of source r: uint8 [3V], byte j = k[4j] | k[4j+1]<<2 | k[4j+2]<<4 | k[4j+3]<<6."""
    n = volume(dims) * 12
    out = torch.empty(n // 4, dtype=torch.uint8, device=device)
    step = 1 << 24
    for a in range(0, n, step):
        b = min(n, a + step)
        k = (hash_i64(seed, r, torch.arange(a, b, dtype=torch.int64, device=device)) & 3).view(-1, 4)
        out[a // 4:b // 4] = (k[:, 0] | (k[:, 1] << 2) | (k[:, 2] << 4) | (k[:, 3] << 6)).to(torch.uint8)
    return out


def z4_source(dims, seed: int, r: int, device) -> torch.Tensor:
    """Z4 volume source eta_r, complex128 [T,Lz,Ly,Lx,4,3] on device."""
    lx, ly, lz, lt = (int(d) for d in dims)
    n = volume(dims) * 12
    k = hash_i64(seed, r, torch.arange(n, dtype=torch.int64, device=device)) & 3
    table = torch.tensor([1, 1j, -1, -1j], dtype=torch.complex128, device=device)
    return table[k].view(lt, lz, ly, lx, 4, 3)


def gaussians(seed: int, stream: int, first: int, count: int, device) -> torch.Tensor:
    j = torch.arange(first, first + count, dtype=torch.int64, device=device)
    h1 = _lsr(hash_i64(seed, stream, j * 2), 11).to(torch.float64)
    h2 = _lsr(hash_i64(seed, stream, j * 2 + 1), 11).to(torch.float64)
    u1 = (h1 + 1.0) * (1.0 / 9007199254740992.0)
    u2 = h2 * (1.0 / 9007199254740992.0)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)


def su3_project(u: torch.Tensor) -> torch.Tensor:
    r0 = u[..., 0, :]
    r0 = r0 / torch.linalg.vector_norm(r0, dim=-1, keepdim=True)
    r1 = u[..., 1, :]
    r1 = r1 - r0 * torch.sum(torch.conj(r0) * r1, dim=-1, keepdim=True)
    r1 = r1 / torch.linalg.vector_norm(r1, dim=-1, keepdim=True)
    r2 = torch.conj(torch.linalg.cross(r0, r1, dim=-1))
    return torch.stack([r0, r1, r2], dim=-2)


def gauge_field(dims, eps: float, seed: int, device) -> torch.Tensor:
    """Synthetic SU(3) gauge field, complex128 [T,Lz,Ly,Lx,4,3,3] on device (BASELINE.json recipe)."""
    lx, ly, lz, lt = (int(d) for d in dims)
    nlink = volume(dims) * 4
    out = torch.empty((nlink, 3, 3), dtype=torch.complex128, device=device)
    eye = torch.eye(3, dtype=torch.complex128, device=device)
    step = 1 << 20
    for a in range(0, nlink, step):
        b = min(nlink, a + step)
        g = gaussians(seed, GAUGE_STREAM, a * 18, (b - a) * 18, device).view(-1, 18)
        m = torch.complex(g[:, 0::2], g[:, 1::2]).reshape(-1, 3, 3)
        h = 0.5 * (m + m.conj().transpose(-1, -2))
        tr = torch.diagonal(h, dim1=-2, dim2=-1).sum(-1) / 3.0
        h = h - tr[:, None, None] * eye
        out[a:b] = su3_project(torch.linalg.matrix_exp(1j * eps * h))
    return out.view(lt, lz, ly, lx, 4, 3, 3)
