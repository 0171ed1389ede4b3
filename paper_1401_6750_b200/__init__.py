"""paper_1401_6750_b200 -- thin Python binding of libtmloops.so (hand-written CUDA, sm_100a).

Argument marshalling only: every step of the hot path (Dslash, CG, contraction, projection,
TSM combination) runs inside the CUDA library behind the C ABI of ``include/tmloops.h``.
PyTorch is used for device memory and streams.  There is NO CPU fallback: importing works
without a GPU (so the symbol table can be checked), but every compute entry point needs a
CUDA device and raises ``TmError`` otherwise.  Nothing here imports ``oracle/``.

Names follow the C ABI: ``tm_dslash``, ``tm_cg_solve``, ``loop_contract_project``,
``tsm_estimate`` (methods of :class:`TmContext`).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import inputs  # noqa: F401  (seeded input generators; no method arithmetic)

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtmloops.so")

TM_OK, TM_EARG, TM_EDIM, TM_EPREC, TM_ECUDA, TM_ENOCONV, TM_EALLOC = range(7)
TM_F64, TM_F32, TM_F16, TM_BF16 = range(4)
TM_R18, TM_R12 = 18, 12
TM_OP_HOP, TM_OP_HOP_TWINV, TM_OP_XPAY, TM_OP_M_FULL, TM_OP_MHAT = range(5)
TM_OPT_GROUP, TM_OPT_CONTRACT_PATH, TM_OPT_POISON, TM_OPT_LANES = range(4)
PREC = {"f64": TM_F64, "f32": TM_F32, "f16": TM_F16, "bf16": TM_BF16}
PREC_BYTES = {TM_F64: 8, TM_F32: 4, TM_F16: 2, TM_BF16: 2}

EXPORTS = [
    "tm_create", "tm_destroy", "tm_last_error", "tm_load_gauge", "tm_field_bytes",
    "tm_field_import", "tm_field_export", "tm_dslash", "tm_dslash_multi", "tm_cg_solve", "loop_contract_project",
    "loop_contract_project_explicit", "loop_contract_project_sym", "loop_contract_project_timeslice",
    "loop_contract_project_fields", "loop_contract_project_fields_static", "loop_contract_static_scratch_bytes",
    "tsm_estimate", "tsm_estimate_host", "tsm_partial_sums_host", "tm_load_gauge_host",
    "loop_plain_project_timeslice", "tsm_estimate_time_diluted", "tm_launch_count", "tm_set_option", "tsm_partial_sums", "tsm_combine_sums",
    "tm_fma_peak",
    "loop_binary_nfiles", "loop_binary_accumulate", "loop_binary_recover", "tsm_estimate_binary",
    "loop_hpe_project", "tsm_estimate_hpe",
]


class TmError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"tmloops status {status}: {msg}")
        self.status = status


class tm_solve_params(ctypes.Structure):
    _fields_ = [("sloppy", ctypes.c_int), ("outer", ctypes.c_int), ("recon", ctypes.c_int),
                ("rho", ctypes.c_double), ("max_iter", ctypes.c_int), ("delta", ctypes.c_double)]


class tm_solve_info(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int), ("reliable_updates", ctypes.c_int),
                ("true_resid", ctypes.c_double), ("ms", ctypes.c_double)]


class tsm_params(ctypes.Structure):
    _fields_ = [("n_lp", ctypes.c_int), ("n_hp", ctypes.c_int),
                ("lp", tm_solve_params), ("hp", tm_solve_params),
                ("kappa", ctypes.c_double), ("mu", ctypes.c_double),
                ("h_momenta", ctypes.POINTER(ctypes.c_int)), ("nmom", ctypes.c_int),
                ("contract_acc_lp", ctypes.c_int), ("contract_acc_hp", ctypes.c_int),
                ("d_z4", ctypes.c_void_p), ("seed", ctypes.c_ulonglong),
                ("src_first", ctypes.c_int), ("src_stride", ctypes.c_int), ("d_solutions", ctypes.c_void_p)]


class tsm_info(ctypes.Structure):
    _fields_ = [("ms_total", ctypes.c_double), ("ms_lp_solve", ctypes.c_double),
                ("ms_hp_solve", ctypes.c_double), ("ms_contract", ctypes.c_double),
                ("iters_lp", ctypes.c_long), ("iters_hp", ctypes.c_long),
                ("worst_resid_lp", ctypes.c_double), ("worst_resid_hp", ctypes.c_double),
                ("launches", ctypes.c_int), ("lanes", ctypes.c_int)]


_lib = None


def load_library():
    """dlopen libtmloops.so (built in-tree by ``python -m paper_1401_6750_b200.build``).

    Fails loudly when the library is missing: there is no other implementation to fall back to."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise TmError(TM_ECUDA, f"{LIB_PATH} not built; run python -m paper_1401_6750_b200.build "
                                "(no CPU fallback exists)")
    L = ctypes.CDLL(LIB_PATH)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    L.tm_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(ci), ci, ci]
    L.tm_destroy.argtypes = [vp]
    L.tm_last_error.argtypes = [vp]
    L.tm_last_error.restype = ctypes.c_char_p
    L.tm_load_gauge.argtypes = [vp, vp, vp]
    L.tm_load_gauge_host.argtypes = [vp, vp, vp]
    L.tm_field_bytes.argtypes = [vp, ci, ci]
    L.tm_field_bytes.restype = ctypes.c_size_t
    L.tm_field_import.argtypes = [vp, vp, vp, ci, vp]
    L.tm_field_export.argtypes = [vp, vp, vp, ci, vp]
    L.tm_dslash.argtypes = [vp, vp, vp, vp, ci, ci, ci, cd, cd, ci, ci, vp]
    L.tm_dslash_multi.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, cd, cd, ci, vp]
    L.tm_cg_solve.argtypes = [vp, vp, vp, cd, cd, ctypes.POINTER(tm_solve_params),
                              ctypes.POINTER(tm_solve_info), vp]
    L.loop_contract_project.argtypes = [vp, vp, vp, vp, cd, cd, ctypes.POINTER(ci), ci, ci, vp]
    L.loop_contract_project_fields.argtypes = [vp, vp, vp, vp, cd, cd, ctypes.POINTER(ci), ci, ci, vp]
    L.loop_contract_project_fields_static.argtypes = [vp, vp, vp, vp, cd, cd, ctypes.POINTER(ci), ci, ci, vp]
    L.loop_contract_static_scratch_bytes.restype = ctypes.c_size_t
    L.loop_contract_static_scratch_bytes.argtypes = []
    L.loop_contract_project_timeslice.argtypes = [vp, vp, vp, vp, cd, cd, ctypes.POINTER(ci), ci, ci, ci, vp]
    L.loop_contract_project_sym.argtypes = [vp, vp, vp, vp, cd, cd, ctypes.POINTER(ci), ci, ci, vp]
    L.loop_contract_project_explicit.argtypes = [vp, vp, vp, cd, cd, ctypes.POINTER(ci), ci, ci, vp]
    L.tsm_estimate.argtypes = [vp, vp, vp, ctypes.POINTER(tsm_params), ctypes.POINTER(tsm_info), vp]
    L.tsm_estimate_host.argtypes = [vp, vp, vp, ctypes.POINTER(tsm_params), ctypes.POINTER(tsm_info), vp]
    L.loop_plain_project_timeslice.argtypes = [vp, vp, vp, vp, ctypes.POINTER(ci), ci, ci, ci, vp]
    L.tsm_estimate_time_diluted.argtypes = [vp, vp, vp, ctypes.POINTER(tsm_params), ctypes.POINTER(tsm_info), vp]
    L.loop_hpe_project.argtypes = [vp, vp, vp, vp, cd, cd, ctypes.POINTER(ci), ci, ci, ci, vp]
    L.tsm_estimate_hpe.argtypes = [vp, vp, vp, ctypes.POINTER(tsm_params), ci, ctypes.POINTER(tsm_info), vp]
    L.tsm_partial_sums_host.argtypes = [vp, vp, vp, ctypes.POINTER(tsm_params), ctypes.POINTER(tsm_info), vp]
    L.loop_binary_nfiles.argtypes = [ci]
    L.loop_binary_nfiles.restype = ci
    L.loop_binary_accumulate.argtypes = [vp, vp, vp, ci, ctypes.c_size_t, vp]
    L.loop_binary_recover.argtypes = [vp, vp, vp, ci, ci, ctypes.c_size_t, vp]
    L.tsm_estimate_binary.argtypes = [vp, vp, vp, vp, ctypes.POINTER(tsm_params), ctypes.POINTER(tsm_info), vp]
    L.tm_launch_count.argtypes = [vp]
    L.tm_set_option.argtypes = [vp, ci, ci]
    L.tsm_partial_sums.argtypes = [vp, vp, vp, ctypes.POINTER(tsm_params), ctypes.POINTER(tsm_info), vp]
    L.tsm_combine_sums.argtypes = [vp, vp, vp, ci, ci, ci, vp]
    L.tm_fma_peak.argtypes = [vp, ci, ci, ctypes.POINTER(cd), vp]
    L.tm_launch_count.restype = ctypes.c_long
    _lib = L
    return L


def _torch():
    import torch
    return torch


def _stream():
    return ctypes.c_void_p(_torch().cuda.current_stream().cuda_stream)


def _solve_params(sloppy, outer, recon, rho, max_iter, delta):
    p = tm_solve_params()
    p.sloppy = PREC[sloppy] if isinstance(sloppy, str) else int(sloppy)
    p.outer = PREC[outer] if isinstance(outer, str) else int(outer)
    p.recon = int(recon)
    p.rho = float(rho)
    p.max_iter = int(max_iter)
    p.delta = float(delta)
    return p


class TmContext:
    """Owns one ``tm_ctx`` (lattice geometry + private gauge copies + workspaces) on one GPU."""

    def __init__(self, dims, t_boundary: int = -1, device: int = 0):
        self.lib = load_library()
        self.dims = tuple(int(d) for d in dims)
        self.device = int(device)
        self.V = int(np.prod(self.dims))
        self.T = self.dims[3]
        h = ctypes.c_void_p()
        st = self.lib.tm_create(ctypes.byref(h), (ctypes.c_int * 4)(*self.dims), int(t_boundary),
                                self.device)
        if st != TM_OK:
            raise TmError(st, self.lib.tm_last_error(None).decode())
        self.h = h
        self.tdev = _torch().device("cuda", self.device)

    def close(self):
        if getattr(self, "h", None):
            self.lib.tm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def _check(self, st, allow=()):
        if st != TM_OK and st not in allow:
            raise TmError(st, self.lib.tm_last_error(self.h).decode())
        return st

    def _dev(self, a, dtype=None):
        """numpy / torch -> contiguous torch tensor on this context's device."""
        torch = _torch()
        if isinstance(a, np.ndarray):
            a = torch.from_numpy(np.ascontiguousarray(a))
        a = a.to(self.tdev)
        if dtype is not None and a.dtype != dtype:
            a = a.to(dtype)
        return a.contiguous()

    # ------------------------------------------------------------------ fields
    def launch_count(self) -> int:
        return int(self.lib.tm_launch_count(self.h))

    def tm_set_option(self, opt: int, value: int):
        """TM_OPT_GROUP (0 = automatic | 1 | 2 | 4 | 8), TM_OPT_CONTRACT_PATH (0 = automatic | 1 .. 4), TM_OPT_POISON (0 | 1) or TM_OPT_LANES (0 = automatic | 1 | 2); see tmloops.h."""
        self._check(self.lib.tm_set_option(self.h, int(opt), int(value)))

    def tm_fma_peak(self, mode: int = 1, iters: int = 4096) -> float:
        """Measured fp32 FMA peak in TFLOP/s (mode 0: FFMA, 1: FFMA2)."""
        v = ctypes.c_double(0.0)
        self._check(self.lib.tm_fma_peak(self.h, int(mode), int(iters), ctypes.byref(v), _stream()))
        return float(v.value)

    def tm_load_gauge(self, U):
        """U: complex128 [T,Lz,Ly,Lx,4,3,3] (numpy or torch)."""
        torch = _torch()
        U = self._dev(U, torch.complex128)
        assert U.numel() == self.V * 36
        self._check(self.lib.tm_load_gauge(self.h, U.data_ptr(), _stream()))     # stream-ordered, like U's own lifetime

    def tm_load_gauge_host(self, U_host):
        """U_host: CPU complex128 tensor [T,Lz,Ly,Lx,4,3,3] (pinned: asynchronous upload straight into the context's master).
        The caller keeps it alive and unchanged until the stream has passed the copy."""
        torch = _torch()
        assert U_host.device.type == "cpu" and U_host.dtype == torch.complex128 and U_host.is_contiguous()
        assert U_host.numel() == self.V * 36
        self._check(self.lib.tm_load_gauge_host(self.h, U_host.data_ptr(), _stream()))

    def tm_field_bytes(self, prec, full_lattice=True) -> int:
        return int(self.lib.tm_field_bytes(self.h, int(prec), 1 if full_lattice else 0))

    def empty_field(self, prec, full_lattice=True):
        return _torch().empty(self.tm_field_bytes(prec, full_lattice), dtype=_torch().uint8,
                              device=self.tdev)

    def tm_field_import(self, canon, prec):
        """canonical complex128 [T,Lz,Ly,Lx,4,3] -> internal full-lattice field (uint8 tensor)."""
        torch = _torch()
        canon = self._dev(canon, torch.complex128)
        assert canon.numel() == self.V * 12
        out = self.empty_field(prec, True)
        self._check(self.lib.tm_field_import(self.h, out.data_ptr(), canon.data_ptr(), int(prec), _stream()))
        return out

    def tm_field_export(self, internal, prec):
        torch = _torch()
        lx, ly, lz, lt = self.dims
        out = torch.empty((lt, lz, ly, lx, 4, 3), dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.tm_field_export(self.h, out.data_ptr(), internal.data_ptr(), int(prec), _stream()))
        return out

    def parity_views(self, internal):
        """(even, odd) halves of a full-lattice internal field."""
        n = internal.numel() // 2
        return internal[:n], internal[n:]

    # ------------------------------------------------------------------ operator
    def tm_dslash(self, out, inp, x, op, out_parity, dagger, kappa, mu, prec, recon):
        """One operator application on INTERNAL fields (uint8 tensors); see tmloops.h."""
        self._check(self.lib.tm_dslash(self.h, out.data_ptr(), inp.data_ptr(),
                                       x.data_ptr() if x is not None else None, int(op),
                                       int(out_parity), int(bool(dagger)), float(kappa), float(mu),
                                       int(prec), int(recon), _stream()))
        return out

    def tm_dslash_multi(self, out, inp, x, nb, op, out_parity, dagger, kappa, mu, prec):
        """nb (1, 2, 4, 8) stacked internal parity fields (source b at b parity fields behind source 0) in one launch."""
        self._check(self.lib.tm_dslash_multi(self.h, out.data_ptr(), inp.data_ptr(),
                                             x.data_ptr() if x is not None else None, int(nb), int(op), int(out_parity),
                                             int(bool(dagger)), float(kappa), float(mu), int(prec), _stream()))
        return out

    def apply_M(self, psi, kappa, mu, prec=TM_F64, recon=TM_R18, dagger=False):
        """Convenience for tests: canonical in -> canonical out through TM_OP_M_FULL."""
        fin = self.tm_field_import(psi, prec)
        fout = self.empty_field(prec, True)
        self.tm_dslash(fout, fin, None, TM_OP_M_FULL, 0, dagger, kappa, mu, prec, recon)
        return self.tm_field_export(fout, prec)

    # ------------------------------------------------------------------ solver
    def tm_cg_solve(self, eta, kappa, mu, sloppy="f64", outer="f64", recon=TM_R18, rho=1e-10,
                    max_iter=5000, delta=0.1, raise_on_noconv=True):
        """eq. 2.1: returns (s canonical complex128 cuda tensor, info dict)."""
        torch = _torch()
        eta = self._dev(eta, torch.complex128)
        s = torch.empty_like(eta)
        p = _solve_params(sloppy, outer, recon, rho, max_iter, delta)
        info = tm_solve_info()
        st = self.lib.tm_cg_solve(self.h, s.data_ptr(), eta.data_ptr(), float(kappa), float(mu),
                                  ctypes.byref(p), ctypes.byref(info), _stream())
        self._check(st, allow=() if raise_on_noconv else (TM_ENOCONV,))
        return s, dict(iters=info.iters, reliable_updates=info.reliable_updates,
                       true_resid=info.true_resid, ms=info.ms, status=st)

    # ------------------------------------------------------------------ contraction
    def loop_contract_project(self, s, eta, kappa, mu, momenta, acc=TM_F64):
        """sec 2.1.1/2.2: complex128 [2,80,nmom,T] cuda tensor of the 160 projected insertions."""
        torch = _torch()
        s = self._dev(s, torch.complex128)
        eta = self._dev(eta, torch.complex128)
        mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
        out = torch.empty((2, 80, len(mom), self.T), dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.loop_contract_project(
            self.h, out.data_ptr(), s.data_ptr(), eta.data_ptr(), float(kappa), float(mu),
            mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), len(mom), int(acc), _stream()))
        return out

    def loop_contract_project_fields(self, s_int, eta_int, kappa, mu, momenta, acc=TM_F32, out=None):
        """loop_contract_project on internal-layout fields (tm_field_import(.., acc)): no layout conversion inside."""
        torch = _torch()
        mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
        if out is None:
            out = torch.empty((2, 80, len(mom), self.T), dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.loop_contract_project_fields(
            self.h, out.data_ptr(), s_int.data_ptr(), eta_int.data_ptr(), float(kappa), float(mu),
            mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), len(mom), int(acc), _stream()))
        return out

    def loop_contract_project_fields_static(self, s_int, eta_int, kappa, mu, momenta, acc=TM_F32, out=None):
        """loop_contract_project_fields without any allocation inside the call: scratch in the library's static device
        array (loop_contract_static_scratch_bytes(); small lattices only; calls on one device must not overlap).  `out`
        should be passed by callers that must not allocate (the default allocates it with torch)."""
        torch = _torch()
        mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
        if out is None:
            out = torch.empty((2, 80, len(mom), self.T), dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.loop_contract_project_fields_static(
            self.h, out.data_ptr(), s_int.data_ptr(), eta_int.data_ptr(), float(kappa), float(mu),
            mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), len(mom), int(acc), _stream()))
        return out

    def loop_contract_static_scratch_bytes(self):
        return int(self.lib.loop_contract_static_scratch_bytes())

    def loop_contract_project_timeslice(self, s, eta, kappa, mu, momenta, t0, acc=TM_F64):
        """Single-timeslice contraction: column t0 of the [2,80,nmom,T] output, zeros elsewhere."""
        torch = _torch()
        s = self._dev(s, torch.complex128)
        eta = self._dev(eta, torch.complex128)
        mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
        out = torch.empty((2, 80, len(mom), self.T), dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.loop_contract_project_timeslice(
            self.h, out.data_ptr(), s.data_ptr(), eta.data_ptr(), float(kappa), float(mu),
            mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), len(mom), int(t0), int(acc), _stream()))
        return out

    def loop_contract_project_sym(self, s, eta, kappa, mu, momenta, acc=TM_F64):
        """Row f3 variant: one-derivative insertions with the symmetrised derivative (momenta closed under p -> -p)."""
        torch = _torch()
        s = self._dev(s, torch.complex128)
        eta = self._dev(eta, torch.complex128)
        mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
        out = torch.empty((2, 80, len(mom), self.T), dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.loop_contract_project_sym(
            self.h, out.data_ptr(), s.data_ptr(), eta.data_ptr(), float(kappa), float(mu),
            mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), len(mom), int(acc), _stream()))
        return out

    def loop_contract_project_explicit(self, s, kappa, mu, momenta, acc=TM_F64):
        """Row f3 variant: the loops of (s, eta := M s), i.e. D_W applied explicitly in the f = 1 insertions."""
        torch = _torch()
        s = self._dev(s, torch.complex128)
        mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
        out = torch.empty((2, 80, len(mom), self.T), dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.loop_contract_project_explicit(
            self.h, out.data_ptr(), s.data_ptr(), float(kappa), float(mu),
            mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), len(mom), int(acc), _stream()))
        return out

    # ------------------------------------------------------------------ TSM
    def _tsm_params(self, n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp, acc_hp, d_z4, seed,
                    src_first=0, src_stride=1, d_solutions=None):
        mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
        P = tsm_params()
        P.n_lp, P.n_hp = int(n_lp), int(n_hp)
        P.lp = _solve_params(**lp)
        P.hp = _solve_params(**hp)
        P.kappa, P.mu = float(kappa), float(mu)
        P.h_momenta = mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int))
        P.nmom = len(mom)
        P.contract_acc_lp, P.contract_acc_hp = int(acc_lp), int(acc_hp)
        P.d_z4 = d_z4
        P.seed = int(seed)
        P.src_first, P.src_stride = int(src_first), int(src_stride)
        P.d_solutions = d_solutions
        return P, mom

    @staticmethod
    def _tsm_info(info, st):
        return dict(ms_total=info.ms_total, ms_lp_solve=info.ms_lp_solve, ms_hp_solve=info.ms_hp_solve,
                    ms_contract=info.ms_contract, iters_lp=info.iters_lp, iters_hp=info.iters_hp, lanes=info.lanes,
                    worst_resid_lp=info.worst_resid_lp, worst_resid_hp=info.worst_resid_hp,
                    launches=info.launches, status=st)

    def tsm_estimate(self, n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp=TM_F32, acc_hp=TM_F64,
                     z4=None, seed=0, per_source=False, raise_on_noconv=True, solutions=False,
                     src_first=0, src_stride=1, partial_sums=False):
        """sec 2.1: TSM estimate, complex128 [2,80,nmom,T] (device-resident inputs).

        z4: optional uint8 cuda tensor [n_lp, 3V] of packed Z4 exponents (None: generated on the
        device from ``seed``).  lp / hp: dicts(sloppy, outer, recon, rho, max_iter, delta).
        solutions=True: info["solutions"] = complex128 [n_lp + n_hp, T,Lz,Ly,Lx,4,3], the run's own solutions.
        src_first / src_stride: local source j is global source src_first + j * src_stride (sharding by source).
        partial_sums=True: the first return value is the raw accumulators [3,2,80,nmom,T] (tsm_partial_sums)."""
        torch = _torch()
        d_z4 = None
        if z4 is not None:
            z4 = self._dev(z4, torch.uint8)
            assert z4.numel() == n_lp * 3 * self.V
            d_z4 = z4.data_ptr()
        sol = None
        if solutions:
            lx, ly, lz, lt = self.dims
            sol = torch.empty((n_lp + n_hp, lt, lz, ly, lx, 4, 3), dtype=torch.complex128, device=self.tdev)
        P, mom = self._tsm_params(n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp, acc_hp, d_z4, seed,
                                  src_first, src_stride, sol.data_ptr() if sol is not None else None)
        shape = (2, 80, len(mom), self.T)
        out = torch.empty(((3,) + shape) if partial_sums else shape, dtype=torch.complex128, device=self.tdev)
        ps = None
        if per_source:
            ps = torch.empty((n_lp + n_hp,) + shape, dtype=torch.complex128, device=self.tdev)
        info = tsm_info()
        fn = self.lib.tsm_partial_sums if partial_sums else self.lib.tsm_estimate
        st = fn(self.h, out.data_ptr(), ps.data_ptr() if ps is not None else None,
                ctypes.byref(P), ctypes.byref(info), _stream())
        self._check(st, allow=() if raise_on_noconv else (TM_ENOCONV,))
        d = self._tsm_info(info, st)
        if sol is not None:
            d["solutions"] = sol
        return out, ps, d

    # ------------------------------------------------------------------ time dilution (row f4)
    def loop_plain_project_timeslice(self, a, b, momenta, t0=-1, acc=TM_F64):
        """Plain bilinears a^dag X_i b on timeslice t0 (-1: every timeslice), complex128 [80, nmom, T]."""
        torch = _torch()
        a = self._dev(a, torch.complex128)
        b = self._dev(b, torch.complex128)
        mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
        out = torch.empty((80, len(mom), self.T), dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.loop_plain_project_timeslice(
            self.h, out.data_ptr(), a.data_ptr(), b.data_ptr(),
            mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), len(mom), int(t0), int(acc), _stream()))
        return out

    def tsm_estimate_time_diluted(self, n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp=TM_F32, acc_hp=TM_F64,
                                  z4=None, seed=0, per_source=False, raise_on_noconv=True, src_first=0, src_stride=1):
        """TSM estimate of the time-diluted plain loops: (out [80,nmom,T], per_source | None, info)."""
        torch = _torch()
        d_z4 = None
        if z4 is not None:
            z4 = self._dev(z4, torch.uint8)
            assert z4.numel() == n_lp * 3 * self.V
            d_z4 = z4.data_ptr()
        P, mom = self._tsm_params(n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp, acc_hp, d_z4, seed, src_first, src_stride)
        shape = (80, len(mom), self.T)
        out = torch.empty(shape, dtype=torch.complex128, device=self.tdev)
        ps = torch.empty((n_lp + n_hp,) + shape, dtype=torch.complex128, device=self.tdev) if per_source else None
        info = tsm_info()
        st = self.lib.tsm_estimate_time_diluted(self.h, out.data_ptr(), ps.data_ptr() if ps is not None else None,
                                                ctypes.byref(P), ctypes.byref(info), _stream())
        self._check(st, allow=() if raise_on_noconv else (TM_ENOCONV,))
        return out, ps, self._tsm_info(info, st)

    # ------------------------------------------------------------------ hopping parameter expansion (row f4)
    def loop_hpe_project(self, eta, s, kappa, mu, momenta, order=4, acc=TM_F64):
        """HPE-improved plain loops of one (eta, s) pair (reading 23), complex128 [80, nmom, T]."""
        torch = _torch()
        eta = self._dev(eta, torch.complex128)
        s = self._dev(s, torch.complex128)
        mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
        out = torch.empty((80, len(mom), self.T), dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.loop_hpe_project(
            self.h, out.data_ptr(), eta.data_ptr(), s.data_ptr(), float(kappa), float(mu),
            mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), len(mom), int(order), int(acc), _stream()))
        return out

    def tsm_estimate_hpe(self, n_lp, n_hp, kappa, mu, momenta, lp, hp, order=4, acc_lp=TM_F32, acc_hp=TM_F64,
                         z4=None, seed=0, per_source=False, raise_on_noconv=True, src_first=0, src_stride=1):
        """TSM estimate of the HPE-improved plain loops: (out [80,nmom,T], per_source | None, info)."""
        torch = _torch()
        d_z4 = None
        if z4 is not None:
            z4 = self._dev(z4, torch.uint8)
            assert z4.numel() == n_lp * 3 * self.V
            d_z4 = z4.data_ptr()
        P, mom = self._tsm_params(n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp, acc_hp, d_z4, seed, src_first, src_stride)
        shape = (80, len(mom), self.T)
        out = torch.empty(shape, dtype=torch.complex128, device=self.tdev)
        ps = torch.empty((n_lp + n_hp,) + shape, dtype=torch.complex128, device=self.tdev) if per_source else None
        info = tsm_info()
        st = self.lib.tsm_estimate_hpe(self.h, out.data_ptr(), ps.data_ptr() if ps is not None else None,
                                       ctypes.byref(P), int(order), ctypes.byref(info), _stream())
        self._check(st, allow=() if raise_on_noconv else (TM_ENOCONV,))
        return out, ps, self._tsm_info(info, st)

    def tsm_combine_sums(self, sums, n_lp_total, n_hp_total):
        """out = S_LP / n_lp_total + (S_HP - S_LPc) / n_hp_total from the (all-reduced) raw accumulators [3,2,80,nmom,T]."""
        torch = _torch()
        assert sums.dtype == torch.complex128 and sums.is_contiguous() and sums.shape[0] == 3
        out = torch.empty(tuple(sums.shape[1:]), dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.tsm_combine_sums(self.h, out.data_ptr(), sums.data_ptr(), int(n_lp_total), int(n_hp_total),
                                              int(sums.shape[3]), _stream()))
        return out

    # ------------------------------------------------------------------ binary storage (sec 2.1.1, Fig. 2)
    def loop_binary_nfiles(self, n_sources: int) -> int:
        return int(self.lib.loop_binary_nfiles(int(n_sources)))

    def loop_binary_accumulate(self, files, loop, r: int):
        """files: complex128 cuda tensor [nfiles, ...] (zeroed by the caller); loop: one per-source array."""
        self._check(self.lib.loop_binary_accumulate(self.h, files.data_ptr(), loop.data_ptr(), int(r),
                                                    loop.numel(), _stream()))

    def loop_binary_recover(self, files, n_stored: int, N: int):
        torch = _torch()
        out = torch.empty(files.shape[1:], dtype=torch.complex128, device=self.tdev)
        self._check(self.lib.loop_binary_recover(self.h, out.data_ptr(), files.data_ptr(), int(n_stored), int(N),
                                                 out.numel(), _stream()))
        return out

    def tsm_estimate_binary(self, n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp=TM_F32, acc_hp=TM_F64,
                            z4=None, seed=0, raise_on_noconv=True):
        """tsm_estimate that also returns the binary-storage files: (out, files_lp, files_corr, info)."""
        torch = _torch()
        d_z4 = None
        if z4 is not None:
            z4 = self._dev(z4, torch.uint8)
            assert z4.numel() == n_lp * 3 * self.V
            d_z4 = z4.data_ptr()
        P, mom = self._tsm_params(n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp, acc_hp, d_z4, seed)
        shape = (2, 80, len(mom), self.T)
        out = torch.empty(shape, dtype=torch.complex128, device=self.tdev)
        f_lp = torch.empty((self.loop_binary_nfiles(n_lp),) + shape, dtype=torch.complex128, device=self.tdev)
        f_co = torch.empty((max(1, self.loop_binary_nfiles(n_hp)),) + shape, dtype=torch.complex128, device=self.tdev)
        info = tsm_info()
        st = self.lib.tsm_estimate_binary(self.h, out.data_ptr(), f_lp.data_ptr(), f_co.data_ptr() if n_hp else None,
                                          ctypes.byref(P), ctypes.byref(info), _stream())
        self._check(st, allow=() if raise_on_noconv else (TM_ENOCONV,))
        return out, f_lp, (f_co if n_hp else None), self._tsm_info(info, st)

    def tsm_estimate_host(self, n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp=TM_F32, acc_hp=TM_F64,
                          z4_host=None, seed=0, out_host=None, raise_on_noconv=True,
                          src_first=0, src_stride=1, partial_sums=False):
        """Same through HOST buffers: z4_host (numpy/torch CPU uint8 [n_lp,3V], pinned or not) is uploaded by a copy
        stream running ahead of the solves and the result (partial_sums: the raw accumulators [3,2,80,nmom,T]) is
        copied back inside the call."""
        torch = _torch()
        h_z4 = None
        if z4_host is not None:
            if isinstance(z4_host, np.ndarray):
                z4_host = torch.from_numpy(z4_host)
            assert z4_host.device.type == "cpu" and z4_host.dtype == torch.uint8 and z4_host.is_contiguous()
            assert z4_host.numel() == n_lp * 3 * self.V
            h_z4 = z4_host.data_ptr()
        P, mom = self._tsm_params(n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp, acc_hp, None, seed, src_first, src_stride)
        shape = (2, 80, len(mom), self.T)
        if partial_sums:
            shape = (3,) + shape
        if out_host is None:
            out_host = torch.empty(shape, dtype=torch.complex128).pin_memory()
        assert out_host.device.type == "cpu" and out_host.dtype == torch.complex128 and tuple(out_host.shape) == shape
        info = tsm_info()
        fn = self.lib.tsm_partial_sums_host if partial_sums else self.lib.tsm_estimate_host
        st = fn(self.h, out_host.data_ptr(), h_z4, ctypes.byref(P), ctypes.byref(info), _stream())
        self._check(st, allow=() if raise_on_noconv else (TM_ENOCONV,))
        return out_host, self._tsm_info(info, st)
