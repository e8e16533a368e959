"""Thin ctypes binding of libwslda (include/wslda.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of ``csrc/``; PyTorch is used for device memory and streams.
There is no CPU fallback: without the built library or without a CUDA device the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libwslda.so")
_SRC_DIR = os.path.join(_HERE, "csrc")
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-shared",
              "-Xcompiler", "-fPIC"]


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/wslda.cu for sm_100a into libwslda.so (in-tree)."""
    srcs = [os.path.join(_SRC_DIR, f) for f in os.listdir(_SRC_DIR)]
    srcs.append(os.path.join(os.path.dirname(_HERE), "include", "wslda.h"))
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= max(os.path.getmtime(s) for s in srcs):
        return _SO
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [os.path.join(_SRC_DIR, "wslda.cu"), "-o", _SO]
    subprocess.run(cmd, check=True)
    return _SO


class Functional(C.Structure):
    _fields_ = [("func_id", C.c_int), ("force_a1", C.c_int), ("spin_symmetric", C.c_int), ("kin_form", C.c_int),
                ("ab_order", C.c_int), ("am_order", C.c_int), ("subtract_mean_energy", C.c_int), ("normalize", C.c_int),
                ("four_pi_as", C.c_double), ("C", C.c_double), ("E_cut", C.c_double), ("lambda_mode", C.c_int),
                ("rho_floor", C.c_double), ("current_terms", C.c_int), ("quantum_friction", C.c_int),
                ("qf_alpha", C.c_double), ("qf_beta", C.c_double), ("qf_gamma", C.c_double), ("qf_rho0", C.c_double),
                ("qf_nreq", C.c_double)]


class Tuning(C.Structure):
    _fields_ = [("disable_fused3d", C.c_int), ("disable_persistent", C.c_int), ("disable_axis_split", C.c_int),
                ("enable_tma_stage", C.c_int), ("disable_mega64", C.c_int), ("disable_onchip", C.c_int),
                ("fused_chunk", C.c_int), ("fused_streams", C.c_int), ("group", C.c_int), ("p_planes", C.c_int),
                ("x_rows", C.c_int), ("persistent_ctas", C.c_int), ("onchip_ctas", C.c_int), ("chunk_mb", C.c_double),
                ("fft_radix", C.c_int), ("spin_limit", C.c_int), ("tma_group", C.c_int), ("tma_block", C.c_int),
                ("tma_ring", C.c_int), ("tma_lag", C.c_int), ("dmma_stage", C.c_int), ("dmma_ctas", C.c_int)]


def fp64_probe():
    """Measured FP64 FMA rate of the current device in flop/s (wslda_fp64_probe) and its SM count."""
    f, n = C.c_double(), C.c_double()
    rc = lib().wslda_fp64_probe(C.byref(f), C.byref(n))
    if rc:
        raise WsldaError(f"fp64_probe failed ({rc}): {lib().wslda_last_error(None).decode()}")
    return f.value, int(n.value)


STATIC_MAX_SIDE, STATIC_MAX_SPINORS = 64, 65536


def gradient_densities_static(psi, cw_a, cw_b, dx, tau, j):
    """wslda_gradient_densities_static: tau [2][M] and j [2][3][M] of the spinors psi [n][2][N][N][N] (N = 32 | 64) on
    the current torch stream, with the kernel's scratch in the library's static device array: the call allocates nothing
    (the caller passes the outputs).  Calls that overlap on the GPU race on that array."""
    import torch
    for t, dt, name in ((psi, torch.complex128, "psi"), (cw_a, torch.float64, "cw_a"), (cw_b, torch.float64, "cw_b"),
                        (tau, torch.float64, "tau"), (j, torch.float64, "j")):
        if t is None and name in ("tau", "j"):
            continue
        if not (t.is_cuda and t.is_contiguous() and t.dtype == dt):
            raise WsldaError(f"gradient_densities_static: {name} must be a contiguous CUDA tensor of {dt}")
    if psi.dim() != 5 or psi.shape[1] != 2 or not (psi.shape[2] == psi.shape[3] == psi.shape[4]):
        raise WsldaError("gradient_densities_static: psi must be [n][2][N][N][N]")
    n, N = int(psi.shape[0]), int(psi.shape[2])
    M = N ** 3
    if cw_a.numel() < n or cw_b.numel() < n or (tau is not None and tau.numel() < 2 * M) or (j is not None and j.numel() < 6 * M):
        raise WsldaError("gradient_densities_static: a weight or output tensor is too small")
    d3 = (C.c_double * 3)(*[float(v) for v in dx])
    rc = lib().wslda_gradient_densities_static(psi.data_ptr(), cw_a.data_ptr(), cw_b.data_ptr(), n, N, d3,
                                               tau.data_ptr() if tau is not None else None,
                                               j.data_ptr() if j is not None else None,
                                               C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc:
        raise WsldaError(f"gradient_densities_static failed ({rc}): {lib().wslda_last_error(None).decode()}")


def set_tuning(**kw):
    """Process-wide kernel selection / tile sizes for contexts created afterwards (wslda_set_tuning); no arguments
    restores the defaults."""
    if not kw:
        lib().wslda_set_tuning(None)
        return
    t = Tuning()
    for k, v in kw.items():
        if not hasattr(t, k):
            raise TypeError(f"unknown tuning field {k}")
        setattr(t, k, v)
    lib().wslda_set_tuning(C.byref(t))


FIELD = dict(rho_a=0, rho_b=1, tau_a=2, tau_b=3, nu=4, ja_x=5, ja_y=6, ja_z=7, jb_x=8, jb_y=9, jb_z=10,
             alpha_a=16, alpha_b=17, U_a=18, U_b=19, delta=20, lap_alpha_a=21, lap_alpha_b=22, lambda_c=23,
             g_eff=24, V_a=25, V_b=26, Aa_x=27, Aa_y=28, Aa_z=29, Ab_x=30, Ab_y=31, Ab_z=32, bp=33)
_COMPLEX = {4, 20, 33}
D_RHO, D_NU, D_TAU, D_J, D_ALL, D_BP = 1, 2, 4, 8, 15, 16
SYMBOLS = ["wslda_workspace_bytes", "wslda_ctx_create", "wslda_ctx_destroy", "wslda_set_modes", "wslda_set_weights",
           "wslda_set_mu", "wslda_set_external", "wslda_set_potentials", "wslda_get_field", "wslda_set_field",
           "wslda_apply_h", "wslda_densities", "wslda_update_potentials", "wslda_history_length", "wslda_abm_init",
           "wslda_abm_step", "wslda_abm_step_host", "wslda_launch_count", "wslda_last_error", "wslda_profile",
           "wslda_profile_report", "wslda_set_reduce_hook", "wslda_set_tuning", "wslda_set_external_velocity",
           "wslda_energy", "wslda_watchdog", "wslda_fp64_probe", "wslda_static_scratch_bytes",
           "wslda_gradient_densities_static"]
OBS = ["N_a", "N_b", "E_kin", "E_pot", "E_pair", "E_pot_ext", "E_pair_ext", "E_total", "E_curr", "E_vel_ext"]
REDUCE_HOOK = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p)

_lib = None


def lib():
    """Load libwslda.so (building it if the sources are newer); raises if that fails."""
    global _lib
    if _lib is None:
        build()                                   # no-op when libwslda.so is newer than every source
        L = C.CDLL(_SO)
        L.wslda_workspace_bytes.restype = C.c_size_t
        L.wslda_workspace_bytes.argtypes = [C.POINTER(C.c_int), C.c_int, C.c_int64, C.POINTER(Functional)]
        L.wslda_ctx_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(C.c_int), C.POINTER(C.c_double), C.c_int,
                                       C.c_int64, C.POINTER(Functional), C.c_void_p, C.c_size_t]
        L.wslda_ctx_destroy.argtypes = [C.c_void_p]
        L.wslda_set_modes.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.wslda_set_weights.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.wslda_set_mu.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.wslda_set_external.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.wslda_set_potentials.argtypes = [C.c_void_p] + [C.c_void_p] * 6
        L.wslda_get_field.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.wslda_set_field.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.wslda_apply_h.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p]
        L.wslda_densities.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_uint, C.c_int, C.c_void_p]
        L.wslda_update_potentials.argtypes = [C.c_void_p, C.c_void_p]
        L.wslda_history_length.argtypes = [C.c_void_p]
        L.wslda_abm_init.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p), C.c_double, C.c_int, C.c_void_p]
        L.wslda_abm_step.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p), C.c_double, C.c_void_p]
        L.wslda_abm_step_host.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p), C.c_void_p,
                                          C.POINTER(C.c_void_p), C.c_double, C.c_void_p]
        L.wslda_set_reduce_hook.argtypes = [C.c_void_p, REDUCE_HOOK, C.c_void_p]
        L.wslda_set_tuning.argtypes = [C.c_void_p]
        L.wslda_set_external_velocity.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.wslda_fp64_probe.argtypes = [C.c_void_p, C.c_void_p]
        L.wslda_static_scratch_bytes.restype = C.c_size_t
        L.wslda_static_scratch_bytes.argtypes = []
        L.wslda_gradient_densities_static.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int,
                                                      C.POINTER(C.c_double), C.c_void_p, C.c_void_p, C.c_void_p]
        L.wslda_energy.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.wslda_watchdog.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        L.wslda_profile.argtypes = [C.c_void_p, C.c_int]
        L.wslda_profile_report.argtypes = [C.c_void_p, C.c_char_p, C.c_size_t]
        L.wslda_launch_count.restype = C.c_int64
        L.wslda_launch_count.argtypes = [C.c_void_p]
        L.wslda_last_error.restype = C.c_char_p
        L.wslda_last_error.argtypes = [C.c_void_p]
        _lib = L
    return _lib


class WsldaError(RuntimeError):
    pass


def make_functional(func_id=0, force_a1=0, spin_symmetric=0, kin_form=0, ab_order=4, am_order=5,
                    subtract_mean_energy=1, normalize=1, four_pi_as=-1.0, C_=-11.11, E_cut=None, lambda_mode=0,
                    rho_floor=1e-14, dx0=1.0, current_terms=0, quantum_friction=0, qf_alpha=0.0, qf_beta=0.0, qf_gamma=0.0,
                    qf_rho0=1.0, qf_nreq=1.0):
    if E_cut is None:
        E_cut = 3.141592653589793 ** 2 / (2 * dx0 ** 2)      # Eq. 22
    return Functional(func_id, force_a1, spin_symmetric, kin_form, ab_order, am_order, subtract_mean_energy, normalize,
                      four_pi_as, C_, E_cut, lambda_mode, rho_floor, current_terms, quantum_friction, qf_alpha, qf_beta,
                      qf_gamma, qf_rho0, qf_nreq)


def workspace_bytes(dims, mode, n_wf, functional) -> int:
    d = (C.c_int * 3)(*(list(dims) + [1] * (3 - len(dims))))
    return int(lib().wslda_workspace_bytes(d, int(mode), int(n_wf), C.byref(functional)))


class Context:
    """One wslda context on the current CUDA device.  Spinor buffers are torch complex128 CUDA tensors of shape
    [n_wf, 2, *held_dims]; fields are float64 / complex128 CUDA tensors of shape held_dims."""

    def __init__(self, mode, dims, dx, n_wf, **fkw):
        import torch
        if not torch.cuda.is_available():
            raise WsldaError("wslda needs a CUDA device (there is no CPU fallback)")
        self.torch = torch
        dims = list(dims) + [1] * (3 - len(dims))
        dx = list(dx) + [1.0] * (3 - len(dx))
        self.f = make_functional(dx0=dx[0], **fkw)
        self.mode, self.dims, self.dx, self.n_wf = int(mode), dims, dx, int(n_wf)
        self.shape = tuple(dims[:mode])
        self.M = 1
        for s in self.shape:
            self.M *= s
        nbytes = workspace_bytes(dims, mode, n_wf, self.f)
        if nbytes == 0:
            raise WsldaError("wslda_workspace_bytes rejected the problem (dims must be powers of two >= 2)")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        self.ctx = C.c_void_p()
        d = (C.c_int * 3)(*dims)
        x = (C.c_double * 3)(*dx)
        rc = lib().wslda_ctx_create(C.byref(self.ctx), d, x, self.mode, self.n_wf, C.byref(self.f),
                                    self.workspace.data_ptr(), nbytes)
        if rc:
            raise WsldaError(f"wslda_ctx_create failed ({rc}): {lib().wslda_last_error(None).decode()}")
        self.m = lib().wslda_history_length(self.ctx)

    def __del__(self):
        if getattr(self, "ctx", None) and _lib is not None:      # at interpreter exit the module may already be torn down
            _lib.wslda_ctx_destroy(self.ctx)
            self.ctx = None

    # -- helpers
    def _chk(self, rc, what):
        if rc:
            raise WsldaError(f"{what} failed ({rc}): {lib().wslda_last_error(self.ctx).decode()}")

    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream().cuda_stream)

    def _dev(self, a, dtype, numel=None):
        t = self.torch
        if a is None:
            return None
        if not isinstance(a, t.Tensor):
            a = t.as_tensor(a)
        a = a.to(device="cuda", dtype=dtype).contiguous()
        if numel is not None and a.numel() != numel:
            raise WsldaError(f"expected {numel} elements, got {a.numel()}")
        return a

    def _spinors(self, x, what):
        """The library reads raw pointers: refuse anything that is not a contiguous complex128 CUDA tensor of the
        whole-batch shape [n_wf, 2, *held_dims] (a slice, a float32 or a host tensor would be read out of bounds)."""
        t = self.torch
        want = (self.n_wf, 2) + self.shape
        if not (isinstance(x, t.Tensor) and x.is_cuda and x.dtype == t.complex128 and x.is_contiguous() and tuple(x.shape) == want):
            raise WsldaError(f"{what}: need a contiguous complex128 CUDA tensor of shape {want}")
        return x

    @staticmethod
    def _ptr(t):
        return None if t is None else C.c_void_p(t.data_ptr())

    # -- setters
    def set_modes(self, kperp, mult, first):
        import numpy as np
        kperp = np.ascontiguousarray(kperp, dtype=np.float64)
        mult = np.ascontiguousarray(mult, dtype=np.float64)
        first = np.ascontiguousarray(first, dtype=np.int64)
        if kperp.size != 2 * len(mult) or len(first) != len(mult) + 1:
            raise WsldaError("set_modes: need kperp[n_modes][2], mult[n_modes], first[n_modes + 1]")
        self._chk(lib().wslda_set_modes(self.ctx, len(mult), kperp.ctypes.data, mult.ctypes.data, first.ctypes.data,
                                        self._stream()), "set_modes")

    def set_weights(self, w_a, w_b):
        t = self.torch
        a, b = self._dev(w_a, t.float64, self.n_wf), self._dev(w_b, t.float64, self.n_wf)
        self._chk(lib().wslda_set_weights(self.ctx, self._ptr(a), self._ptr(b), self._stream()), "set_weights")
        t.cuda.current_stream().synchronize()            # a, b are temporaries: keep them alive until the copy is done

    def set_mu(self, mu_a, mu_b):
        self._chk(lib().wslda_set_mu(self.ctx, float(mu_a), float(mu_b)), "set_mu")

    def set_external(self, vext_a=None, vext_b=None, delta_ext=None):
        t = self.torch
        a, b, d = self._dev(vext_a, t.float64, self.M), self._dev(vext_b, t.float64, self.M), self._dev(delta_ext, t.complex128, self.M)
        self._chk(lib().wslda_set_external(self.ctx, self._ptr(a), self._ptr(b), self._ptr(d), self._stream()), "set_external")
        t.cuda.current_stream().synchronize()

    def set_velocity(self, vel_a=None, vel_b=None):
        """External velocity fields v_ext_sigma, arrays [<=3, *held_dims]; needs current_terms=1."""
        t = self.torch

        def prep(v):
            if v is None:
                return None
            v = self._dev(v, t.float64)
            out = t.zeros((3, self.M), dtype=t.float64, device="cuda")
            out[: v.shape[0]] = v.reshape(v.shape[0], self.M)
            return out
        a, b = prep(vel_a), prep(vel_b)
        self._chk(lib().wslda_set_external_velocity(self.ctx, self._ptr(a), self._ptr(b), self._stream()), "set_external_velocity")
        t.cuda.current_stream().synchronize()

    def set_potentials(self, alpha_a, alpha_b, U_a, U_b, delta):
        t = self.torch
        args = [self._dev(x, t.float64, self.M) for x in (alpha_a, alpha_b, U_a, U_b)] + [self._dev(delta, t.complex128, self.M)]
        self._chk(lib().wslda_set_potentials(self.ctx, *[self._ptr(x) for x in args], self._stream()), "set_potentials")
        t.cuda.current_stream().synchronize()

    def get_field(self, name):
        t = self.torch
        fid = FIELD[name]
        out = t.empty(self.shape, dtype=t.complex128 if fid in _COMPLEX else t.float64, device="cuda")
        self._chk(lib().wslda_get_field(self.ctx, fid, self._ptr(out), self._stream()), "get_field")
        return out

    def set_field(self, name, value):
        t = self.torch
        fid = FIELD[name]
        v = self._dev(value, t.complex128 if fid in _COMPLEX else t.float64)
        self._chk(lib().wslda_set_field(self.ctx, fid, self._ptr(v), self._stream()), "set_field")
        t.cuda.current_stream().synchronize()

    # -- the path
    def apply_h(self, psi, hpsi=None, eps=None, n_first=0, n_count=None):
        t = self.torch
        n_count = self.n_wf - n_first if n_count is None else n_count
        self._spinors(psi, "apply_h psi")
        if hpsi is None:
            hpsi = t.zeros_like(psi)
        if eps is None:
            eps = t.zeros(self.n_wf, dtype=t.float64, device="cuda")
        self._spinors(hpsi, "apply_h hpsi")
        if not (eps.is_cuda and eps.dtype == t.float64 and eps.is_contiguous() and eps.numel() == self.n_wf):
            raise WsldaError("apply_h eps: need a contiguous float64 CUDA tensor of n_wf elements")
        self._chk(lib().wslda_apply_h(self.ctx, self._ptr(psi), self._ptr(hpsi), self._ptr(eps), n_first, n_count,
                                      self._stream()), "apply_h")
        return hpsi, eps

    def densities(self, psi, n_first=0, n_count=None, which=D_ALL, accumulate=0):
        n_count = self.n_wf - n_first if n_count is None else n_count
        self._spinors(psi, "densities psi")
        self._chk(lib().wslda_densities(self.ctx, self._ptr(psi), n_first, n_count, which, accumulate, self._stream()),
                  "densities")

    def energy(self, out=None):
        """Observables of Eqs. 33a-g as a float64 CUDA tensor of 10 (order: OBS); no host synchronisation."""
        t = self.torch
        if out is None:
            out = t.empty(len(OBS), dtype=t.float64, device="cuda")
        self._chk(lib().wslda_energy(self.ctx, self._ptr(out), self._stream()), "energy")
        return out

    def watchdog(self, ref, tol_number, tol_energy, out=None):
        """Device-side conservation check against `ref` (a tensor from energy()); a violation poisons the context."""
        t = self.torch
        if out is None:
            out = t.empty(len(OBS), dtype=t.float64, device="cuda")
        self._chk(lib().wslda_watchdog(self.ctx, self._ptr(ref), float(tol_number), float(tol_energy), self._ptr(out),
                                       self._stream()), "watchdog")
        return out

    def update_potentials(self):
        self._chk(lib().wslda_update_potentials(self.ctx, self._stream()), "update_potentials")

    def _hist(self, f_hist):
        if len(f_hist) != self.m:
            raise WsldaError(f"need {self.m} history buffers")
        for x in f_hist:
            self._spinors(x, "history buffer")
        return (C.c_void_p * self.m)(*[x.data_ptr() for x in f_hist])

    @staticmethod
    def _reorder(f_hist, ptrs):
        by = {x.data_ptr(): x for x in f_hist}
        return [by[p] for p in ptrs]

    def abm_init(self, phi, f_hist, dt, selfstart=1):
        self._spinors(phi, "abm_init phi")
        ptrs = self._hist(f_hist)
        self._chk(lib().wslda_abm_init(self.ctx, self._ptr(phi), ptrs, float(dt), int(selfstart), self._stream()), "abm_init")
        return self._reorder(f_hist, list(ptrs))

    def abm_step(self, phi, f_hist, dt):
        self._spinors(phi, "abm_step phi")
        ptrs = self._hist(f_hist)
        self._chk(lib().wslda_abm_step(self.ctx, self._ptr(phi), ptrs, float(dt), self._stream()), "abm_step")
        return self._reorder(f_hist, list(ptrs))

    def abm_step_host(self, phi_host, f_hist_host, phi, f_hist, dt):
        """End-to-end step from (pinned) host tensors; returns the permuted (host, device) history lists."""
        t = self.torch
        want = (self.n_wf, 2) + self.shape
        for x in [phi_host] + list(f_hist_host):
            if x.is_cuda or x.dtype != t.complex128 or not x.is_contiguous() or tuple(x.shape) != want:
                raise WsldaError(f"abm_step_host: host buffers must be contiguous complex128 CPU tensors of shape {want}")
        self._spinors(phi, "abm_step_host phi")
        hp = (C.c_void_p * self.m)(*[x.data_ptr() for x in f_hist_host])
        dp = self._hist(f_hist)
        self._chk(lib().wslda_abm_step_host(self.ctx, C.c_void_p(phi_host.data_ptr()), hp, self._ptr(phi), dp, float(dt),
                                            self._stream()), "abm_step_host")
        byh = {x.data_ptr(): x for x in f_hist_host}
        return [byh[p] for p in hp], self._reorder(f_hist, list(dp))

    # -- sharding over the spinor index (include/wslda.h: wslda_set_reduce_hook)
    def set_reduce_hook(self, fn):
        """fn(block, stream_ptr): sum the float64 CUDA tensor `block` (a view of this context's density block) in
        place over the ranks, enqueued on the CUDA stream `stream_ptr`.  None removes the hook."""
        if fn is None:
            self._hook = None
            self._chk(lib().wslda_set_reduce_hook(self.ctx, C.cast(None, REDUCE_HOOK), None), "set_reduce_hook")
            return
        t, base = self.torch, self.workspace.data_ptr()

        def _cb(_user, block, count, stream):
            off = int(block) - base
            fn(self.workspace[off:off + 8 * int(count)].view(t.float64), int(stream or 0))

        self._hook = REDUCE_HOOK(_cb)                       # keep the trampoline alive as long as the context
        self._chk(lib().wslda_set_reduce_hook(self.ctx, self._hook, None), "set_reduce_hook")

    def set_density_allreduce(self, group=None):
        """Shard the spinors over the ranks of a torch.distributed group (NCCL over NVLink/NVSwitch): every density
        build is summed over the ranks with one all-reduce on the stream the step runs on."""
        import torch.distributed as dist
        t = self.torch

        def _allreduce(block, stream):
            cur = t.cuda.current_stream()
            if stream and stream != cur.cuda_stream:
                with t.cuda.stream(t.cuda.ExternalStream(stream)):
                    dist.all_reduce(block, op=dist.ReduceOp.SUM, group=group)
            else:
                dist.all_reduce(block, op=dist.ReduceOp.SUM, group=group)

        self.set_reduce_hook(_allreduce)

    def profile(self, enable=True):
        self._chk(lib().wslda_profile(self.ctx, int(bool(enable))), "profile")

    def profile_report(self):
        """{kernel name: (launches, total_ms, algorithmic bytes, algorithmic flops, attributed_ms)} recorded since
        profile(True); synchronises the device.  attributed_ms shares overlapped time among concurrent launches."""
        buf = C.create_string_buffer(1 << 16)
        lib().wslda_profile_report(self.ctx, buf, len(buf))
        out = {}
        for line in buf.value.decode().splitlines():
            name, cnt, ms, nbytes, flops, share = line.split()
            out[name] = (int(cnt), float(ms), float(nbytes), float(flops), float(share))
        return out

    def launch_count(self):
        return int(lib().wslda_launch_count(self.ctx))
