"""CPU ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front-end of ``oracle/tm_oracle.c`` (plain C, double precision, full
lattice; see that file's header for the passages it follows and its pins).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this package.  It imports nothing from
``paper_1401_6750_b200`` (the CUDA path) and the CUDA path never imports it.

All arrays are numpy complex128, C-contiguous, in the canonical shapes of
``paper_1401_6750_b200/inputs.py``:
  spinor [T,Lz,Ly,Lx,4,3], gauge [T,Lz,Ly,Lx,4,3,3]; dims = (Lx,Ly,Lz,T).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tm_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile tm_oracle.c -> liboracle.so with gcc (OpenMP over sites)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_true_residual.restype = ctypes.c_double
        _lib.orc_solve.restype = ctypes.c_int
    return _lib


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a, a.ctypes.data_as(ctypes.c_void_p)


def _dims(dims):
    return (ctypes.c_int * 4)(*[int(d) for d in dims])


def dims_of(field) -> tuple:
    lt, lz, ly, lx = field.shape[:4]
    return (lx, ly, lz, lt)


def gamma(mu: int) -> np.ndarray:
    """gamma_mu (mu = 0..3 = x,y,z,t; 4 = gamma5), 4x4 complex."""
    out = np.empty((4, 4), dtype=np.complex128)
    lib().orc_gamma(ctypes.c_int(mu), out.ctypes.data_as(ctypes.c_void_p))
    return out


def Gamma(n: int) -> np.ndarray:
    """Gamma_n = g_x^b0 g_y^b1 g_z^b2 g_t^b3, n = b0+2b1+4b2+8b3."""
    out = np.empty((4, 4), dtype=np.complex128)
    lib().orc_Gamma(ctypes.c_int(n), out.ctypes.data_as(ctypes.c_void_p))
    return out


def apply_M(psi, U, kappa, mu, tb=-1, dagger=False) -> np.ndarray:
    psi, p_psi = _c(psi)
    U, p_U = _c(U)
    out = np.empty_like(psi)
    lib().orc_apply_M(out.ctypes.data_as(ctypes.c_void_p), p_psi, p_U, _dims(dims_of(psi)),
                      ctypes.c_int(tb), ctypes.c_double(kappa), ctypes.c_double(mu),
                      ctypes.c_int(1 if dagger else 0))
    return out


def solve(eta, U, kappa, mu, rho, tb=-1, max_iter=10000):
    """Returns (s, iters, true_resid, status); status 0 = converged."""
    eta, p_eta = _c(eta)
    U, p_U = _c(U)
    s = np.empty_like(eta)
    it = ctypes.c_int(0)
    tr = ctypes.c_double(0)
    st = lib().orc_solve(s.ctypes.data_as(ctypes.c_void_p), p_eta, p_U, _dims(dims_of(eta)),
                         ctypes.c_int(tb), ctypes.c_double(kappa), ctypes.c_double(mu),
                         ctypes.c_double(rho), ctypes.c_int(max_iter),
                         ctypes.byref(it), ctypes.byref(tr))
    return s, it.value, tr.value, st


def true_residual(s, eta, U, kappa, mu, tb=-1) -> float:
    s, p_s = _c(s)
    eta, p_eta = _c(eta)
    U, p_U = _c(U)
    return lib().orc_true_residual(p_s, p_eta, p_U, _dims(dims_of(eta)), ctypes.c_int(tb),
                                   ctypes.c_double(kappa), ctypes.c_double(mu))


def cov_deriv(psi, U, m, tb=-1) -> np.ndarray:
    psi, p_psi = _c(psi)
    U, p_U = _c(U)
    out = np.empty_like(psi)
    lib().orc_cov_deriv(out.ctypes.data_as(ctypes.c_void_p), p_psi, p_U, _dims(dims_of(psi)),
                        ctypes.c_int(tb), ctypes.c_int(m))
    return out


def loops_sites(s, eta, U, kappa, mu, sites=None, tb=-1) -> np.ndarray:
    """Per-site 160 insertions, [nsites, 2, 80]; sites = flat lexicographic indices (None = all)."""
    s, p_s = _c(s)
    eta, p_eta = _c(eta)
    U, p_U = _c(U)
    V = int(np.prod(s.shape[:4]))
    if sites is None:
        sites = np.arange(V)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((len(sites), 2, 80), dtype=np.complex128)
    lib().orc_loops_sites(out.ctypes.data_as(ctypes.c_void_p), p_s, p_eta, p_U, _dims(dims_of(s)),
                          ctypes.c_int(tb), ctypes.c_double(kappa), ctypes.c_double(mu),
                          sites.ctypes.data_as(ctypes.c_void_p), ctypes.c_long(len(sites)))
    return out


def loops_project(s, eta, U, kappa, mu, momenta, tb=-1, t0=0, t1=None) -> np.ndarray:
    """Momentum-projected loops [2, 80, nmom, T] (timeslices outside [t0,t1) are zero)."""
    s, p_s = _c(s)
    eta, p_eta = _c(eta)
    U, p_U = _c(U)
    T = s.shape[0]
    if t1 is None:
        t1 = T
    mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
    out = np.zeros((2, 80, len(mom), T), dtype=np.complex128)
    lib().orc_loops_project(out.ctypes.data_as(ctypes.c_void_p), p_s, p_eta, p_U,
                            _dims(dims_of(s)), ctypes.c_int(tb), ctypes.c_double(kappa),
                            ctypes.c_double(mu), mom.ctypes.data_as(ctypes.c_void_p),
                            ctypes.c_int(len(mom)), ctypes.c_int(t0), ctypes.c_int(t1))
    return out


def tsm_combine(lp, hp) -> np.ndarray:
    """lp: [n_lp, ...], hp: [n_hp, ...] (HP sources = the first n_hp LP sources)."""
    lp, p_lp = _c(lp)
    hp, p_hp = _c(hp)
    n_lp, n_hp = lp.shape[0], hp.shape[0]
    out = np.empty(lp.shape[1:], dtype=np.complex128)
    ln = int(np.prod(lp.shape[1:]))
    lib().orc_tsm_combine(out.ctypes.data_as(ctypes.c_void_p), p_lp, ctypes.c_int(n_lp), p_hp,
                          ctypes.c_int(n_hp), ctypes.c_long(ln))
    return out


def binary_nfiles(n: int) -> int:
    """Number of files n sources touch: the smallest K with 2^K - 1 >= n."""
    k = 0
    while (1 << k) - 1 < n:
        k += 1
    return k


def binary_store(per_source):
    """sec 2.1.1 / Fig. 2: per_source [n, ...] -> (files [K, ...], counts [K]); file k sums sources 2^k-1 .. 2^(k+1)-2."""
    ps, p_ps = _c(per_source)
    n = ps.shape[0]
    ln = int(np.prod(ps.shape[1:]))
    K = binary_nfiles(n)
    files = np.empty((K,) + ps.shape[1:], dtype=np.complex128)
    counts = np.zeros(K, dtype=np.int32)
    lib().orc_binary_store(files.ctypes.data_as(ctypes.c_void_p), counts.ctypes.data_as(ctypes.c_void_p), p_ps,
                           ctypes.c_int(n), ctypes.c_long(ln))
    return files, counts


def binary_recover(files, counts, N: int):
    """Estimator from N sources = sum of the files named by the binary digits of N, / N (None if not recoverable)."""
    f, p_f = _c(files)
    counts = np.ascontiguousarray(counts, dtype=np.int32)
    out = np.empty(f.shape[1:], dtype=np.complex128)
    ln = int(np.prod(f.shape[1:]))
    lib().orc_binary_recover.restype = ctypes.c_int
    st = lib().orc_binary_recover(out.ctypes.data_as(ctypes.c_void_p), p_f, counts.ctypes.data_as(ctypes.c_void_p),
                                  ctypes.c_int(f.shape[0]), ctypes.c_int(N), ctypes.c_long(ln))
    return out if st == 0 else None


def loops_project_explicit(s, U, kappa, mu, momenta, tb=-1, t0=0, t1=None) -> np.ndarray:
    """Variant of reading 5: the generalised one-end trick with D_W applied explicitly,
    l[1] = s^dag g5 X g5 D_W s with g5 D_W s = g5 (M s) - 2 i kappa mu s, i.e. the loops of (s, eta := M s)."""
    return loops_project(s, apply_M(s, U, kappa, mu, tb), U, kappa, mu, momenta, tb, t0, t1)


def loops_project_sym(s, eta, U, kappa, mu, momenta, tb=-1, t0=0, t1=None) -> np.ndarray:
    """Variant of reading 4 (row f3): one-derivative insertions with the symmetrised derivative
    1/2 [s^dag g5 G (D psi) - (D s)^dag g5 G psi]; ultra-local entries as in loops_project."""
    s, p_s = _c(s)
    eta, p_eta = _c(eta)
    U, p_U = _c(U)
    T = s.shape[0]
    if t1 is None:
        t1 = T
    mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
    out = np.zeros((2, 80, len(mom), T), dtype=np.complex128)
    lib().orc_loops_project_sym(out.ctypes.data_as(ctypes.c_void_p), p_s, p_eta, p_U,
                                _dims(dims_of(s)), ctypes.c_int(tb), ctypes.c_double(kappa),
                                ctypes.c_double(mu), mom.ctypes.data_as(ctypes.c_void_p),
                                ctypes.c_int(len(mom)), ctypes.c_int(t0), ctypes.c_int(t1))
    return out


# ---------------------------------------------------------------------------- time dilution (row f4)
def time_dilute(eta, t0: int) -> np.ndarray:
    """eta^(t0): the noise vector restricted to timeslice t0 (reading 22)."""
    eta, p_eta = _c(eta)
    out = np.empty_like(eta)
    lib().orc_time_dilute(out.ctypes.data_as(ctypes.c_void_p), p_eta, _dims(dims_of(eta)), ctypes.c_int(t0))
    return out


def plain_loops_project(a, b, U, momenta, tb=-1, t0=0, t1=None) -> np.ndarray:
    """Plain bilinears sum_x e^{ipx} a^dag X_i b per timeslice, [80, nmom, T]; X_n = Gamma_n, X_{16+16m+n} = Gamma_n D_m
    (D_m on b); timeslices outside [t0, t1) are zero."""
    a, p_a = _c(a)
    b, p_b = _c(b)
    U, p_U = _c(U)
    T = a.shape[0]
    if t1 is None:
        t1 = T
    mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
    out = np.zeros((80, len(mom), T), dtype=np.complex128)
    lib().orc_plain_loops_project(out.ctypes.data_as(ctypes.c_void_p), p_a, p_b, p_U, _dims(dims_of(a)),
                                  ctypes.c_int(tb), mom.ctypes.data_as(ctypes.c_void_p), ctypes.c_int(len(mom)),
                                  ctypes.c_int(t0), ctypes.c_int(t1))
    return out


def loops_time_diluted(eta, U, kappa, mu, rho, momenta, tb=-1, max_iter=10000):
    """Time-diluted plain loops of ONE noise vector (reading 22), step by step: for every t0, restrict eta to the
    timeslice, solve M s = eta^(t0), contract that single timeslice.  Returns ([80, nmom, T], worst true residual)."""
    T = eta.shape[0]
    mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
    out = np.zeros((80, len(mom), T), dtype=np.complex128)
    worst = 0.0
    for t0 in range(T):
        e = time_dilute(eta, t0)
        s, _, tr, st = solve(e, U, kappa, mu, rho, tb, max_iter)
        if st != 0:
            raise RuntimeError("oracle solve did not converge")
        worst = max(worst, tr)
        out[:, :, t0] = plain_loops_project(e, s, U, mom, tb, t0, t0 + 1)[:, :, t0]
    return out, worst


# ---------------------------------------------------------------------------- hopping parameter expansion (row f4)
def apply_AinvH(v, U, kappa, mu, tb=-1) -> np.ndarray:
    """One factor of the expansion: A^-1 H v with A = 1 + 2 i kappa mu g5, H = A - M (reading 23)."""
    v, p_v = _c(v)
    U, p_U = _c(U)
    out = np.empty_like(v)
    lib().orc_apply_AinvH(out.ctypes.data_as(ctypes.c_void_p), p_v, p_U, _dims(dims_of(v)), ctypes.c_int(tb),
                          ctypes.c_double(kappa), ctypes.c_double(mu))
    return out


def hpe_exact(U, kappa, mu, momenta, tb=-1, order_local=4, order_deriv=2) -> np.ndarray:
    """Exact part sum_x e^{ipx} tr[X_i sum_{k<n_i} ((A^-1 H)^k A^-1)(x,x)] per timeslice, [80, nmom, T], by brute force
    over all 12 V unit vectors (small lattices only)."""
    U, p_U = _c(U)
    T, lz, ly, lx = U.shape[:4]
    mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
    out = np.zeros((80, len(mom), T), dtype=np.complex128)
    lib().orc_hpe_exact(out.ctypes.data_as(ctypes.c_void_p), p_U, _dims((lx, ly, lz, T)), ctypes.c_int(tb),
                        ctypes.c_double(kappa), ctypes.c_double(mu), ctypes.c_int(order_local), ctypes.c_int(order_deriv),
                        mom.ctypes.data_as(ctypes.c_void_p), ctypes.c_int(len(mom)))
    return out


def hpe_orders(order: int):
    """Reading 23: the ultra-local insertions are expanded to `order` (<= 4), the one-derivative ones to min(order, 2)
    (their order-3 term closes four-link loops and is not site-independent)."""
    if order < 0 or order > 4:
        raise ValueError("HPE order must be 0..4")
    return order, min(order, 2)


def loops_hpe(eta, s, U, kappa, mu, momenta, tb=-1, order=4, exact=None) -> np.ndarray:
    """HPE-improved plain loops of one (noise vector, solution) pair, step by step (reading 23):
    remainder eta^dag X_i (A^-1 H)^{n_i} s, projected per timeslice, plus the exact part.  [80, nmom, T].
    exact: the (source-independent) exact part if already computed."""
    n_loc, n_der = hpe_orders(order)
    mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
    v = {0: np.ascontiguousarray(s)}
    for k in range(1, max(n_loc, n_der) + 1):
        v[k] = apply_AinvH(v[k - 1], U, kappa, mu, tb)
    out = np.empty((80, len(mom), eta.shape[0]), dtype=np.complex128)
    out[:16] = plain_loops_project(eta, v[n_loc], U, mom, tb)[:16]
    out[16:] = plain_loops_project(eta, v[n_der], U, mom, tb)[16:]
    if exact is None:
        exact = hpe_exact(U, kappa, mu, mom, tb, n_loc, n_der)
    return out + exact
