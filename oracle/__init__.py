"""CPU oracle for the TDSLDA/BdG step (TEST INFRASTRUCTURE ONLY).

ctypes front end of ``wslda_oracle.c``.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the CUDA library never does.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libwslda_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C99 + OpenMP)."""
    src = os.path.join(_HERE, "wslda_oracle.c")
    hdr = os.path.join(_HERE, "wslda_oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _SO, src, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


class Params(C.Structure):
    _fields_ = [("mode", C.c_int), ("dims", C.c_int * 3), ("dx", C.c_double * 3), ("n_wf", C.c_int64),
                ("func_id", C.c_int), ("force_a1", C.c_int), ("spin_symmetric", C.c_int), ("kin_form", C.c_int),
                ("ab_order", C.c_int), ("am_order", C.c_int), ("subtract_mean_energy", C.c_int),
                ("normalize", C.c_int), ("four_pi_as", C.c_double), ("C", C.c_double), ("E_cut", C.c_double),
                ("lambda_mode", C.c_int), ("rho_floor", C.c_double), ("current_terms", C.c_int),
                ("quantum_friction", C.c_int), ("qf_alpha", C.c_double), ("qf_beta", C.c_double), ("qf_gamma", C.c_double),
                ("qf_rho0", C.c_double), ("qf_nreq", C.c_double)]


FIELD = dict(rho_a=0, rho_b=1, tau_a=2, tau_b=3, nu=4, ja_x=5, ja_y=6, ja_z=7, jb_x=8, jb_y=9, jb_z=10,
             alpha_a=16, alpha_b=17, U_a=18, U_b=19, delta=20, lap_alpha_a=21, lap_alpha_b=22, lambda_c=23,
             g_eff=24, V_a=25, V_b=26, Aa_x=27, Aa_y=28, Aa_z=29, Ab_x=30, Ab_y=31, Ab_z=32, bp=33)
_COMPLEX = {4, 20, 33}

_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def fft1d(x, sign=-1):
    a = _c128(x).copy()
    rc = lib().orc_fft1d(_p(a), C.c_int(a.size), C.c_int(sign))
    if rc:
        raise ValueError("orc_fft1d: n must be a power of two")
    return a


def dft1d_naive(x, sign=-1):
    a = _c128(x)
    out = np.empty_like(a)
    lib().orc_dft1d_naive(_p(a), _p(out), C.c_int(a.size), C.c_int(sign))
    return out


def derivatives(field, dx):
    """Laplacian and gradient of a complex field on its (1-3)-D periodic lattice (Eqs. 25-26)."""
    a = _c128(field)
    nd = a.ndim
    dims = (C.c_int * 3)(*(list(a.shape) + [1] * (3 - nd)))
    dxs = (C.c_double * 3)(*(list(dx) + [1.0] * (3 - len(dx))))
    lap = np.empty_like(a)
    grad = np.empty((nd,) + a.shape, dtype=np.complex128)
    rc = lib().orc_derivatives(C.c_int(nd), dims, dxs, _p(a), _p(lap), _p(grad))
    if rc:
        raise ValueError("orc_derivatives failed")
    return lap, grad


class Oracle:
    """One oracle context.  Spinor buffers are numpy complex128 arrays of shape [n_wf, 2, *held_dims]."""

    def __init__(self, mode, dims, dx, n_wf, func_id=0, force_a1=0, spin_symmetric=0, kin_form=0, ab_order=4,
                 am_order=5, subtract_mean_energy=1, normalize=1, four_pi_as=-1.0, C_=-11.11, E_cut=None,
                 lambda_mode=0, rho_floor=1e-14, current_terms=0, quantum_friction=0, qf_alpha=0.0, qf_beta=0.0,
                 qf_gamma=0.0, qf_rho0=1.0, qf_nreq=1.0):
        dims = list(dims) + [1] * (3 - len(dims))
        dx = list(dx) + [1.0] * (3 - len(dx))
        if E_cut is None:
            E_cut = np.pi ** 2 / (2 * dx[0] ** 2)          # Eq. 22
        self.p = Params(mode, (C.c_int * 3)(*dims), (C.c_double * 3)(*dx), n_wf, func_id, force_a1,
                        spin_symmetric, kin_form, ab_order, am_order, subtract_mean_energy, normalize,
                        four_pi_as, C_, E_cut, lambda_mode, rho_floor, current_terms, quantum_friction, qf_alpha, qf_beta,
                        qf_gamma, qf_rho0, qf_nreq)
        self.mode, self.dims, self.dx, self.n_wf = mode, dims, dx, n_wf
        self.shape = tuple(dims[:mode])
        self.M = int(np.prod(self.shape))
        self.dV = float(np.prod(dx[:mode]))
        self.ctx = C.c_void_p()
        rc = lib().orc_create(C.byref(self.ctx), C.byref(self.p))
        if rc:
            raise ValueError("orc_create rejected the parameters")
        self.m = lib().orc_history_length(self.ctx)

    def __del__(self):
        if getattr(self, "ctx", None):
            lib().orc_destroy(self.ctx)
            self.ctx = None

    def _chk(self, rc, what):
        if rc:
            raise RuntimeError(f"oracle {what} failed ({rc})")

    def set_modes(self, kperp, mult, first):
        kperp, mult = _f64(kperp), _f64(mult)
        first = np.ascontiguousarray(first, dtype=np.int64)
        self._chk(lib().orc_set_modes(self.ctx, C.c_int(len(mult)), _p(kperp), _p(mult), _p(first)), "set_modes")

    def set_weights(self, w_a, w_b):
        self._chk(lib().orc_set_weights(self.ctx, _p(_f64(w_a)), _p(_f64(w_b))), "set_weights")

    def set_mu(self, mu_a, mu_b):
        self._chk(lib().orc_set_mu(self.ctx, C.c_double(mu_a), C.c_double(mu_b)), "set_mu")

    def set_external(self, vext_a=None, vext_b=None, delta_ext=None):
        a = _f64(vext_a) if vext_a is not None else None
        b = _f64(vext_b) if vext_b is not None else None
        d = _c128(delta_ext) if delta_ext is not None else None
        self._chk(lib().orc_set_external(self.ctx, _p(a), _p(b), _p(d)), "set_external")

    def set_potentials(self, alpha_a, alpha_b, U_a, U_b, delta):
        self._chk(lib().orc_set_potentials(self.ctx, _p(_f64(alpha_a)), _p(_f64(alpha_b)), _p(_f64(U_a)),
                                           _p(_f64(U_b)), _p(_c128(delta))), "set_potentials")

    def get_field(self, name):
        fid = FIELD[name]
        out = np.empty(self.shape, dtype=np.complex128 if fid in _COMPLEX else np.float64)
        self._chk(lib().orc_get_field(self.ctx, C.c_int(fid), _p(out)), "get_field")
        return out

    def set_field(self, name, value):
        fid = FIELD[name]
        v = _c128(value) if fid in _COMPLEX else _f64(value)
        self._chk(lib().orc_set_field(self.ctx, C.c_int(fid), _p(v)), "set_field")

    def apply_h(self, psi, n_first=0, n_count=None):
        psi = _c128(psi)
        n_count = self.n_wf - n_first if n_count is None else n_count
        hpsi = np.zeros_like(psi)
        eps = np.zeros(self.n_wf)
        self._chk(lib().orc_apply_h(self.ctx, _p(psi), _p(hpsi), _p(eps), C.c_int64(n_first), C.c_int64(n_count)),
                  "apply_h")
        return hpsi, eps

    def densities(self, psi, n_first=0, n_count=None, accumulate=0):
        psi = _c128(psi)
        n_count = self.n_wf - n_first if n_count is None else n_count
        self._chk(lib().orc_densities(self.ctx, _p(psi), C.c_int64(n_first), C.c_int64(n_count),
                                      C.c_int(accumulate)), "densities")

    def update_potentials(self):
        self._chk(lib().orc_update_potentials(self.ctx), "update_potentials")

    def functional_point(self, rho_a, rho_b, tau_a, tau_b, nu, vext_a=0.0, vext_b=0.0, lambda_in=None, j_a=None, j_b=None):
        vin = (C.c_double * 9)(rho_a, rho_b, tau_a, tau_b, complex(nu).real, complex(nu).imag, vext_a, vext_b,
                               0.0 if lambda_in is None else lambda_in)
        out = (C.c_double * 10)()
        ja = (C.c_double * 3)(*(j_a if j_a is not None else (0.0, 0.0, 0.0)))
        jb = (C.c_double * 3)(*(j_b if j_b is not None else (0.0, 0.0, 0.0)))
        A = (C.c_double * 6)()
        self._chk(lib().orc_functional_point_j(self.ctx, vin, ja, jb, C.c_int(lambda_in is not None), out, A), "functional")
        return dict(alpha_a=out[0], alpha_b=out[1], V_a=out[2], V_b=out[3], delta=complex(out[4], out[5]),
                    lambda_c=out[6], g_eff=out[7], edens=out[8], A_a=np.array(A[0:3]), A_b=np.array(A[3:6]))

    def set_velocity(self, vel_a=None, vel_b=None):
        """External velocity fields v_ext_sigma, arrays [3, *held_dims] (components along non-held axes are ignored)."""
        def prep(v):
            if v is None:
                return None
            a = np.zeros((3, self.M))
            v = np.asarray(v, dtype=np.float64).reshape(len(v), self.M)
            a[: len(v)] = v
            return a
        va, vb = prep(vel_a), prep(vel_b)
        self._chk(lib().orc_set_velocity(self.ctx, _p(va), _p(vb)), "set_velocity")

    def _hist_ptrs(self, f_hist):
        assert len(f_hist) == self.m
        return (C.c_void_p * self.m)(*[a.ctypes.data for a in f_hist])

    @staticmethod
    def _reorder(f_hist, ptrs):
        by_addr = {a.ctypes.data: a for a in f_hist}
        return [by_addr[p] for p in ptrs]

    def abm_init(self, phi, f_hist, dt, selfstart=1):
        """phi (in/out, complex128 contiguous) and the list of m history buffers; returns the reordered list."""
        ptrs = self._hist_ptrs(f_hist)
        self._chk(lib().orc_abm_init(self.ctx, _p(phi), ptrs, C.c_double(dt), C.c_int(selfstart)), "abm_init")
        return self._reorder(f_hist, list(ptrs))

    def abm_step(self, phi, f_hist, dt):
        ptrs = self._hist_ptrs(f_hist)
        self._chk(lib().orc_abm_step(self.ctx, _p(phi), ptrs, C.c_double(dt)), "abm_step")
        return self._reorder(f_hist, list(ptrs))

    def energy(self):
        out = (C.c_double * 10)()
        self._chk(lib().orc_energy(self.ctx, out), "energy")
        return dict(zip(["N_a", "N_b", "E_kin", "E_pot", "E_pair", "E_pot_ext", "E_pair_ext", "E_total", "E_curr",
                         "E_vel_ext"], out))


def num_threads():
    return lib().orc_num_threads()
