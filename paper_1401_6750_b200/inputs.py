"""Seeded synthetic input generators (numpy only).

This module is the ONE piece shared by the CPU oracle's tests and the CUDA
path's tests/bench: it produces *inputs* (gauge links, Z4 noise, random spinors,
momentum lists) and contains none of the method's arithmetic (no Dirac operator,
no gamma matrices, no solver, no contraction).  It imports nothing from the rest
of the package and nothing from ``oracle/``.

Recipes (BASELINE.json configs c1..c5):

* counter-based hash   ``mix`` = splitmix64 finaliser,
  ``h(seed, stream, idx) = mix(mix(seed*0x9E3779B97F4A7C15 + stream) + idx)``
* Z4 noise   ``eta[site][spin][col] = i**(h(seed, r, (site*4+spin)*3+col) & 3)``
  ("random stochastic sources"; BASELINE.json c1 "Z4 volume source")
* gauge      18 Box-Muller Gaussians per link -> A (3x3 complex),
  ``H = (A + A^dag)/2 - tr/3``, ``U = exp(i*eps*H)`` by Hermitian
  eigendecomposition, then SU(3) projection (Gram-Schmidt rows 0,1; row 2 =
  conj(row0 x row1))  (BASELINE.json c1 recipe)

Canonical array shapes (site order x fastest, t slowest; dims = (Lx, Ly, Lz, T)):
  spinor  complex128 [T, Lz, Ly, Lx, 4, 3]      (spin, colour)
  gauge   complex128 [T, Lz, Ly, Lx, 4, 3, 3]   (mu = x,y,z,t ; row ; col)
"""
from __future__ import annotations

import numpy as np

_U64 = np.uint64
GAUGE_STREAM = 0x6761756765  # ascii "gauge"
_GOLDEN = 0x9E3779B97F4A7C15
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB


def mix64(z):
    """splitmix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    z = np.asarray(z, dtype=_U64).copy()
    with np.errstate(over="ignore"):
        z ^= z >> _U64(30)
        z *= _U64(_M1)
        z ^= z >> _U64(27)
        z *= _U64(_M2)
        z ^= z >> _U64(31)
    return z


def hash_u64(seed: int, stream: int, idx):
    """h(seed, stream, idx) for an array of counters idx (uint64)."""
    base = (int(seed) * _GOLDEN + int(stream)) & 0xFFFFFFFFFFFFFFFF
    k = mix64(np.array([base], dtype=_U64))[0]
    with np.errstate(over="ignore"):
        return mix64(np.asarray(idx, dtype=_U64) + k)


def volume(dims) -> int:
    lx, ly, lz, lt = (int(d) for d in dims)
    return lx * ly * lz * lt


def z4_exponents(dims, seed: int, r: int) -> np.ndarray:
    """Exponents k in {0,1,2,3} (uint8, flat [V*12]) of Z4 source number r."""
    n = volume(dims) * 12
    out = np.empty(n, dtype=np.uint8)
    step = 1 << 22
    for a in range(0, n, step):
        b = min(n, a + step)
        out[a:b] = (hash_u64(seed, r, np.arange(a, b, dtype=_U64)) & _U64(3)).astype(np.uint8)
    return out


_Z4 = np.array([1, 1j, -1, -1j], dtype=np.complex128)


def z4_from_exponents(dims, k: np.ndarray) -> np.ndarray:
    lx, ly, lz, lt = (int(d) for d in dims)
    return _Z4[k].reshape(lt, lz, ly, lx, 4, 3)


def z4_source(dims, seed: int, r: int) -> np.ndarray:
    """Z4 volume source eta_r, complex128 [T,Lz,Ly,Lx,4,3]."""
    return z4_from_exponents(dims, z4_exponents(dims, seed, r))


def pack_z4(k: np.ndarray) -> np.ndarray:
    """Pack exponents 4 per byte: byte j holds k[4j+m] in bits 2m..2m+1."""
    k = np.asarray(k, dtype=np.uint8).reshape(-1, 4)
    return (k[:, 0] | (k[:, 1] << 2) | (k[:, 2] << 4) | (k[:, 3] << 6)).astype(np.uint8)


def _uniform_open(hv):
    """(0,1] double from the top 53 bits."""
    return ((hv >> _U64(11)).astype(np.float64) + 1.0) * (1.0 / 9007199254740992.0)


def _uniform_half_open(hv):
    """[0,1) double from the top 53 bits."""
    return (hv >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def gaussians(seed: int, stream: int, first: int, count: int) -> np.ndarray:
    """count unit Gaussians: Box-Muller (cos branch) from counters 2j, 2j+1."""
    j = np.arange(first, first + count, dtype=_U64)
    u1 = _uniform_open(hash_u64(seed, stream, j * _U64(2)))
    u2 = _uniform_half_open(hash_u64(seed, stream, j * _U64(2) + _U64(1)))
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def su3_project(u: np.ndarray) -> np.ndarray:
    """Gram-Schmidt rows 0,1; row 2 = conj(row0 x row1).  u: [...,3,3]."""
    r0 = u[..., 0, :]
    r0 = r0 / np.linalg.norm(r0, axis=-1, keepdims=True)
    r1 = u[..., 1, :]
    r1 = r1 - r0 * np.sum(np.conj(r0) * r1, axis=-1, keepdims=True)
    r1 = r1 / np.linalg.norm(r1, axis=-1, keepdims=True)
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)


def _links_from_gaussians(g: np.ndarray, eps: float) -> np.ndarray:
    """g: [n,18] Gaussians -> [n,3,3] SU(3) links exp(i*eps*H)."""
    a = (g[:, 0::2] + 1j * g[:, 1::2]).reshape(-1, 3, 3)
    h = 0.5 * (a + np.conj(np.swapaxes(a, -1, -2)))
    tr = np.trace(h, axis1=-2, axis2=-1) / 3.0
    h = h - tr[:, None, None] * np.eye(3)
    w, v = np.linalg.eigh(h)
    u = np.einsum("nij,nj,nkj->nik", v, np.exp(1j * eps * w), np.conj(v))
    return su3_project(u)


def gauge_field(dims, eps: float, seed: int) -> np.ndarray:
    """Synthetic SU(3) gauge field, complex128 [T,Lz,Ly,Lx,4,3,3]."""
    lx, ly, lz, lt = (int(d) for d in dims)
    nlink = volume(dims) * 4
    out = np.empty((nlink, 3, 3), dtype=np.complex128)
    step = 1 << 18
    for a in range(0, nlink, step):
        b = min(nlink, a + step)
        g = gaussians(seed, GAUGE_STREAM, a * 18, (b - a) * 18).reshape(-1, 18)
        out[a:b] = _links_from_gaussians(g, eps)
    return out.reshape(lt, lz, ly, lx, 4, 3, 3)


def unit_gauge(dims) -> np.ndarray:
    lx, ly, lz, lt = (int(d) for d in dims)
    u = np.zeros((lt, lz, ly, lx, 4, 3, 3), dtype=np.complex128)
    u[..., 0, 0] = u[..., 1, 1] = u[..., 2, 2] = 1.0
    return u


def random_spinor(dims, seed: int, stream: int = 0x7370696E) -> np.ndarray:
    """Gaussian spinor field (re, im unit normal), complex128 [T,Lz,Ly,Lx,4,3]."""
    lx, ly, lz, lt = (int(d) for d in dims)
    n = volume(dims) * 12
    g = gaussians(seed, stream, 0, 2 * n)
    return (g[0::2] + 1j * g[1::2]).reshape(lt, lz, ly, lx, 4, 3)


def random_su3_field(dims, seed: int, eps: float = 1.0, stream: int = 0x67786630) -> np.ndarray:
    """One random SU(3) matrix g(x) per site, [T,Lz,Ly,Lx,3,3] (gauge transforms)."""
    lx, ly, lz, lt = (int(d) for d in dims)
    n = volume(dims)
    g = gaussians(seed, stream, 0, n * 18).reshape(-1, 18)
    return _links_from_gaussians(g, eps).reshape(lt, lz, ly, lx, 3, 3)


def momentum_list(p2max: int) -> np.ndarray:
    """Integer momenta (px,py,pz) with p^2 <= p2max, int32 [nmom,3].

    Order: nested loops pz, py, px ascending in [-m, m], keep p^2 <= p2max,
    stable sort by p^2 ("up to p^2 <= 9" -> 123 vectors)."""
    m = int(np.floor(np.sqrt(p2max)))
    rows = []
    for pz in range(-m, m + 1):
        for py in range(-m, m + 1):
            for px in range(-m, m + 1):
                if px * px + py * py + pz * pz <= p2max:
                    rows.append((px, py, pz))
    rows.sort(key=lambda p: p[0] ** 2 + p[1] ** 2 + p[2] ** 2)
    return np.array(rows, dtype=np.int32).reshape(-1, 3)


# BASELINE.json configs c1..c5 (dims = Lx,Ly,Lz,T)
CONFIGS = {
    "c1": dict(dims=(4, 4, 4, 8), eps=0.3, seed=1, kappa=0.156, mu=0.01, src_seed=2),
    "c2": dict(dims=(16, 16, 16, 32), eps=0.3, seed=3, kappa=0.1565, mu=0.004, src_seed=3),
    "c3": dict(dims=(24, 24, 24, 48), eps=0.25, seed=4, kappa=0.1563, mu=0.0055, src_seed=4,
               n_lp=100, n_hp=10, p2max=4),
    "c4": dict(dims=(32, 32, 32, 64), eps=0.2, seed=5, kappa=0.161231, mu=0.004, src_seed=5,
               n_lp=500, n_hp=20, p2max=9),
    "c5": dict(dims=(48, 48, 48, 96), eps=0.2, seed=6, kappa=0.1612, mu=0.003, src_seed=6),
}
