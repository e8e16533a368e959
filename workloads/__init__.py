"""Seeded synthetic inputs for the TDSLDA/BdG step (shared by the oracle tests, the GPU tests and bench.py).

This module holds NONE of the method's arithmetic (no H, no densities, no functional, no integrator): it only
produces input arrays -- initial spinors, external fields, fixed potentials, weights, transverse-mode tables --
as pure functions of (seed, index), so that the CPU oracle and the CUDA library see identical bits.  The recipes
restate SURVEY.md section 8(d) / DESIGN.md section 5; they stand in for the paper's physical set-ups (uniform
gas, harmonic traps, vortices), whose actual wave-function files are not available.

Random numbers: counter-based SplitMix64 -> uniform (0,1) -> Box-Muller normal.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

_GOLD = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, start: int, count: int) -> np.ndarray:
    """Outputs number start..start+count-1 of the SplitMix64 stream of `seed` (counter-based)."""
    with np.errstate(over="ignore"):
        idx = np.arange(start + 1, start + count + 1, dtype=np.uint64)
        z = np.uint64(seed) + idx * _GOLD
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        return z ^ (z >> np.uint64(31))


def uniform01(seed: int, start: int, count: int) -> np.ndarray:
    """Uniform on (0,1): top 53 bits, shifted by half an ulp so that 0 never occurs."""
    return ((splitmix64(seed, start, count) >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed: int, start: int, count: int) -> np.ndarray:
    """Standard normals number start..start+count-1 of stream `seed` (Box-Muller on pairs of uniforms)."""
    first = start // 2
    npair = (start + count + 1) // 2 - first
    u = uniform01(seed, 2 * first, 2 * npair)
    r = np.sqrt(-2.0 * np.log(u[0::2]))
    t = 2.0 * np.pi * u[1::2]
    z = np.empty(2 * npair)
    z[0::2] = r * np.cos(t)
    z[1::2] = r * np.sin(t)
    off = start - 2 * first
    return z[off:off + count]


def kgrid(n: int, dx: float) -> np.ndarray:
    """Wave numbers of an n-point periodic axis (Eq. 25)."""
    l = np.arange(n)
    return 2.0 * np.pi * np.where(l < n // 2, l, l - n) / (n * dx)


@dataclass
class Workload:
    name: str
    mode: int
    dims: tuple            # (Nx, Ny, Nz) -- all three
    dx: tuple
    n_wf: int
    func_id: int           # 0 fixed, 1 BdG, 2 ASLDA
    force_a1: int
    spin_symmetric: int
    kin_form: int
    ab_order: int
    am_order: int
    dt: float
    n_steps: int
    mu: tuple
    subtract_mean_energy: int = 1
    normalize: int = 1
    four_pi_as: float = -1.0
    E_cut: float | None = None
    lambda_mode: int = 0
    # plane-wave table of the initial spinors: k-index tuple on the held axes, branch (+1/-1), mode id
    kidx: np.ndarray = None
    branch: np.ndarray = None
    mode_of: np.ndarray = None
    kperp: np.ndarray = None      # [n_modes, 2]
    mult: np.ndarray = None       # [n_modes]
    first: np.ndarray = None      # [n_modes+1]
    mu_eff: float = 0.5           # parameters of the closed-form uniform spinors
    delta0: float = 0.2
    alpha0: float = 1.0
    noise: float = 0.0
    noise_seed: int = 0
    w_a: np.ndarray = None
    w_b: np.ndarray = None
    E: np.ndarray = None
    vext_a: np.ndarray = None
    vext_b: np.ndarray = None
    delta_ext: np.ndarray = None
    fixed: dict = field(default_factory=dict)   # alpha_a, alpha_b, U_a, U_b, delta for func_id == 0
    n_base: int = 0               # global index of spinor 0 (non-zero for one rank's shard, see shard())

    @property
    def shape(self):
        return tuple(self.dims[:self.mode])

    @property
    def M(self):
        return int(np.prod(self.shape))

    @property
    def dV(self):
        return float(np.prod(self.dx[:self.mode]))

    @property
    def history(self):
        return max(self.ab_order, self.am_order - 1)

    def spinors(self, n0: int = 0, n1: int | None = None) -> np.ndarray:
        """Initial spinors n0..n1-1 as complex128 [n, 2, *shape]: closed-form uniform-Delta BdG plane waves
        (u_k, v_k) e^{ik.r}/sqrt(V) (+ branch) or (-v_k, u_k) e^{ik.r}/sqrt(V) (- branch), plus optional seeded
        noise, then normalised to dV * sum(|u|^2+|v|^2) = 1."""
        n1 = self.n_wf if n1 is None else n1
        shape, nd = self.shape, self.mode
        ks = [kgrid(shape[d], self.dx[d]) for d in range(nd)]
        pos = [np.arange(shape[d]) * self.dx[d] for d in range(nd)]
        vol = self.M * self.dV
        out = np.empty((n1 - n0, 2) + shape, dtype=np.complex128)
        for i, n in enumerate(range(n0, n1)):
            kk = [ks[d][self.kidx[n, d]] for d in range(nd)]
            kp2 = 0.0 if self.kperp is None else float(np.sum(self.kperp[self.mode_of[n]] ** 2))
            eps = self.alpha0 * (sum(k * k for k in kk) + kp2) / 2.0 - self.mu_eff
            En = np.sqrt(eps * eps + self.delta0 ** 2)
            u, v = np.sqrt(0.5 * (1 + eps / En)), np.sqrt(0.5 * (1 - eps / En))
            if self.branch[n] < 0:
                u, v = -v, u
            pw = np.exp(1j * kk[0] * pos[0])
            for d in range(1, nd):
                pw = np.multiply.outer(pw, np.exp(1j * kk[d] * pos[d]))
            pw = pw / np.sqrt(vol)
            out[i, 0] = u * pw
            out[i, 1] = v * pw
        if self.noise > 0:
            cnt = (n1 - n0) * 4 * self.M
            z = normal(self.noise_seed, (self.n_base + n0) * 4 * self.M, cnt).reshape((n1 - n0, 2) + shape + (2,))
            out += self.noise * (z[..., 0] + 1j * z[..., 1]) / np.sqrt(vol)
            nrm = np.sqrt(np.sum(np.abs(out) ** 2, axis=tuple(range(1, nd + 2)), keepdims=True) * self.dV)
            out /= nrm
        return out


def spinors_device(w: "Workload", n0: int, n1: int, out):
    """Fill the torch CUDA tensor `out` ([n1-n0, 2, *shape] complex128) with spinors n0..n1-1 of the recipe of
    Workload.spinors, generated on the device (bench-sized batches; the noise comes from torch's seeded
    generator instead of SplitMix64, so the bits differ from the numpy path but the distribution is the same)."""
    import torch
    dev = out.device
    shape, nd = w.shape, w.mode
    vol = w.M * w.dV
    g = torch.Generator(device=dev)
    step = max(1, (1 << 24) // w.M)
    for a in range(n0, n1, step):
        b = min(n1, a + step)
        kidx = np.asarray(w.kidx[a:b])
        kk = [kgrid(shape[d], w.dx[d])[kidx[:, d]] for d in range(nd)]
        kp2 = np.zeros(b - a) if w.kperp is None else np.sum(np.asarray(w.kperp)[w.mode_of[a:b]] ** 2, axis=1)
        eps = w.alpha0 * (sum(k * k for k in kk) + kp2) / 2.0 - w.mu_eff
        En = np.sqrt(eps * eps + w.delta0 ** 2)
        u, v = np.sqrt(0.5 * (1 + eps / En)), np.sqrt(0.5 * (1 - eps / En))
        neg = np.asarray(w.branch[a:b]) < 0
        u, v = np.where(neg, -v, u), np.where(neg, u, v)
        phase = torch.zeros((b - a,) + shape, dtype=torch.float64, device=dev)
        for d in range(nd):
            pos = torch.arange(shape[d], dtype=torch.float64, device=dev) * w.dx[d]
            view = [1] * (nd + 1); view[d + 1] = shape[d]
            kd = torch.as_tensor(kk[d], device=dev).view([-1] + [1] * nd)
            phase = phase + kd * pos.view(view)
        pw = torch.polar(torch.full_like(phase, 1.0 / np.sqrt(vol)), phase)
        o = out[a - n0:b - n0]
        o[:, 0] = torch.as_tensor(u, device=dev).view([-1] + [1] * nd) * pw
        o[:, 1] = torch.as_tensor(v, device=dev).view([-1] + [1] * nd) * pw
        if w.noise > 0:
            g.manual_seed(w.noise_seed * 1000003 + a)
            z = torch.randn((b - a, 2) + shape + (2,), dtype=torch.float64, device=dev, generator=g)
            o += (w.noise / np.sqrt(vol)) * torch.view_as_complex(z)
            nrm = torch.sqrt(torch.sum(o.real ** 2 + o.imag ** 2, dim=tuple(range(1, nd + 2)), keepdim=True) * w.dV)
            o /= nrm
    return out


def shard_range(n_wf: int, rank: int, world: int):
    """Contiguous near-equal share [n0, n1) of the spinor index for `rank` of `world` (nwf/np each)."""
    return n_wf * rank // world, n_wf * (rank + 1) // world


def shard(w: "Workload", n0: int, n1: int) -> "Workload":
    """The workload restricted to spinors n0..n1-1 -- one rank's share when the spinor index is sharded over GPUs:
    weights and plane-wave table sliced, transverse-mode table shifted and clipped (modes outside the range become
    empty), lattice, functional and external fields unchanged.  v.spinors() returns the same spinors as
    w.spinors(n0, n1)."""
    import copy
    v = copy.copy(w)
    v.n_wf = n1 - n0
    v.n_base = w.n_base + n0
    for k in ("kidx", "branch", "mode_of", "w_a", "w_b", "E"):
        a = getattr(w, k)
        if a is not None:
            setattr(v, k, a[n0:n1])
    if w.first is not None:
        v.first = np.clip(np.asarray(w.first) - n0, 0, n1 - n0)
    return v


def _coords_centered(shape, dx):
    ax = [dx[d] * (np.arange(shape[d]) - shape[d] // 2) for d in range(len(shape))]
    return np.meshgrid(*ax, indexing="ij")


def _plane_wave_table(shape, dx, mu_eff, delta0, alpha0=1.0, kp2=0.0):
    """All lattice momenta on the held axes in index order with their uniform quasi-energies."""
    ks = [kgrid(shape[d], dx[d]) for d in range(len(shape))]
    grids = np.meshgrid(*[np.arange(s) for s in shape], indexing="ij")
    kidx = np.stack([g.ravel() for g in grids], axis=1)
    k2 = sum(ks[d][kidx[:, d]] ** 2 for d in range(len(shape)))
    eps = alpha0 * (k2 + kp2) / 2.0 - mu_eff
    return kidx, np.sqrt(eps ** 2 + delta0 ** 2)


def _smooth_field(seed, shape, dx, ell=4.0, amp=0.1):
    """White noise -> spectral Gaussian filter exp(-k^2 ell^2 / 2) -> scaled to max-abs amp (input recipe only)."""
    M = int(np.prod(shape))
    w = normal(seed, 0, M).reshape(shape)
    ks = np.meshgrid(*[kgrid(shape[d], dx[d]) for d in range(len(shape))], indexing="ij")
    k2 = sum(k * k for k in ks)
    f = np.fft.ifftn(np.fft.fftn(w) * np.exp(-0.5 * k2 * ell * ell)).real
    return amp * f / np.max(np.abs(f))


def cfg1(n_wf=None):
    """configs[0]: 3D BdG 8^3, fixed noisy potentials, full basis of 1024 closed-form spinors, AB4AM4."""
    shape, dx = (8, 8, 8), (1.0, 1.0, 1.0)
    M = 512
    kidx, E = _plane_wave_table(shape, dx, 0.5, 0.2)
    kidx = np.repeat(kidx, 2, axis=0)
    branch = np.tile(np.array([1, -1]), M)
    n_wf = 2 * M if n_wf is None else n_wf
    En = np.repeat(E, 2) * branch
    delta = 0.2 + 0.02 * (normal(101, 0, 2 * M)[0::2] + 1j * normal(101, 0, 2 * M)[1::2])
    U = 0.05 * normal(102, 0, M)
    one = np.ones(shape)
    return Workload("cfg1_bdg_8x8x8", 3, shape, dx, n_wf, 0, 1, 0, 0, 4, 4, 0.005, 100, (0.5, 0.5),
                    kidx=kidx[:n_wf], branch=branch[:n_wf], mode_of=np.zeros(n_wf, dtype=np.int64), mu_eff=0.5,
                    delta0=0.2, E=En[:n_wf], w_a=(En[:n_wf] < 0).astype(float), w_b=(En[:n_wf] > 0).astype(float),
                    fixed=dict(alpha_a=one, alpha_b=one, U_a=U.reshape(shape), U_b=U.reshape(shape),
                               delta=delta.reshape(shape)))


def cfg2(n_modes_side=32, nx=128, n_steps=200):
    """configs[1]: quasi-1D SLDA (FORCE_A1), Nx=128, 32x32 transverse modes, 256 spinors per mode, self-consistent."""
    dx = (1.0, 1.0, 1.0)
    ny = nz = n_modes_side
    ky, kz = kgrid(ny, dx[1]), kgrid(nz, dx[2])
    kperp = np.stack([np.repeat(ky, nz), np.tile(kz, ny)], axis=1)
    n_modes = ny * nz
    per = 2 * nx
    n_wf = n_modes * per
    kidx = np.tile(np.repeat(np.arange(nx), 2), n_modes)[:, None]
    branch = np.tile(np.array([1, -1]), n_wf // 2)
    mode_of = np.repeat(np.arange(n_modes), per)
    mu_eff, delta0, eF = 0.45, 0.25, 0.5
    kx = kgrid(nx, dx[0])
    eps = (kx[kidx[:, 0]] ** 2 + np.sum(kperp[mode_of] ** 2, axis=1)) / 2 - mu_eff
    E = np.sqrt(eps ** 2 + delta0 ** 2) * branch
    E_c = np.pi ** 2 / 2
    inside = (np.abs(E) < E_c).astype(float)
    u = uniform01(201, 0, 2)
    q = 1 + int(u[0] * 3)
    phase = 2 * np.pi * u[1]
    x = np.arange(nx) * dx[0]
    vext = 0.1 * eF * np.cos(2 * np.pi * q * x / (nx * dx[0]) + phase)
    return Workload(f"cfg2_q1d_{nx}x{ny}x{nz}", 1, (nx, ny, nz), dx, n_wf, 2, 1, 0, 0, 4, 5, 0.01, n_steps, (0.2, 0.2),
                    kidx=kidx, branch=branch, mode_of=mode_of, kperp=kperp, mult=np.ones(n_modes),
                    first=np.arange(n_modes + 1, dtype=np.int64) * per, mu_eff=mu_eff, delta0=delta0, E=E,
                    w_a=(E < 0) * inside, w_b=(E > 0) * inside, vext_a=vext, vext_b=vext, E_cut=E_c)


def cfg3(n_side=64, n_kz=16, nz=32, n_steps=100):
    """configs[2]: quasi-2D SLDA vortex, 64^2, 16 kz values, 4096 positive-energy spinors per kz."""
    dx = (1.0, 1.0, 1.0)
    shape = (n_side, n_side)
    M = n_side * n_side
    kz = 2 * np.pi * np.arange(n_kz) / (nz * dx[2])
    kperp = np.stack([kz, np.zeros(n_kz)], axis=1)
    mult = np.where(np.arange(n_kz) == 0, 1.0, 2.0)
    mu_eff, delta0 = 0.45, 0.25
    kidx0, _ = _plane_wave_table(shape, dx, mu_eff, delta0)
    kidx = np.tile(kidx0, (n_kz, 1))
    mode_of = np.repeat(np.arange(n_kz), M)
    n_wf = n_kz * M
    kxy = [kgrid(n_side, 1.0)[kidx[:, d]] for d in range(2)]
    eps = (kxy[0] ** 2 + kxy[1] ** 2 + kz[mode_of] ** 2) / 2 - mu_eff
    E = np.sqrt(eps ** 2 + delta0 ** 2)
    E_c = np.pi ** 2 / 2
    X, Y = _coords_centered(shape, dx)
    r = np.sqrt(X ** 2 + Y ** 2)
    theta = np.arctan2(Y, X)
    z = normal(301, 0, 2 * M)
    dext = 0.3 * np.tanh(r / 2) * np.exp(1j * theta) + 0.01 * (z[0::2] + 1j * z[1::2]).reshape(shape)
    vext = 0.5 * 0.05 ** 2 * r ** 2
    return Workload(f"cfg3_q2d_{n_side}x{n_side}x{n_kz}kz", 2, (n_side, n_side, nz), dx, n_wf, 2, 1, 1, 0, 4, 5, 0.01,
                    n_steps, (0.2, 0.2), kidx=kidx, branch=np.ones(n_wf, dtype=np.int64), mode_of=mode_of,
                    kperp=kperp, mult=mult, first=np.arange(n_kz + 1, dtype=np.int64) * M, mu_eff=mu_eff,
                    delta0=delta0, E=E, w_a=np.zeros(n_wf), w_b=(E < E_c).astype(float), vext_a=vext, vext_b=vext,
                    delta_ext=dext, E_cut=E_c)


def cfg4(n_side=32, n_wf=None, kin_form=1, n_steps=50):
    """configs[3]: 3D SLDA (ASLDA formulas, general-alpha path) in a harmonic trap, 32^3, 16384 spinors."""
    dx = (1.0, 1.0, 1.0)
    shape = (n_side,) * 3
    M = n_side ** 3
    n_wf = M // 2 if n_wf is None else n_wf
    mu_eff, delta0, alpha0 = 0.45, 0.25, 1.094
    kidx, E = _plane_wave_table(shape, dx, mu_eff, delta0, alpha0)
    order = np.argsort(E, kind="stable")[:n_wf]
    X, Y, Z = _coords_centered(shape, dx)
    vext = 0.5 * 0.1 ** 2 * (X ** 2 + Y ** 2 + Z ** 2)
    E_c = np.pi ** 2 / 2
    return Workload(f"cfg4_3d_{n_side}^3_kin{kin_form}", 3, shape, dx, n_wf, 2, 0, 1, kin_form, 4, 5, 0.005, n_steps,
                    (0.2, 0.2), kidx=kidx[order], branch=np.ones(n_wf, dtype=np.int64),
                    mode_of=np.zeros(n_wf, dtype=np.int64), mu_eff=mu_eff, delta0=delta0, alpha0=alpha0, noise=0.01,
                    noise_seed=401, E=E[order], w_a=np.zeros(n_wf), w_b=(E[order] < E_c).astype(float), vext_a=vext,
                    vext_b=vext, E_cut=E_c)


def cfg5(n_side=64, n_wf=512, kin_form=1, n_steps=4):
    """configs[4]: 3D ASLDA-like spin-imbalanced throughput case: fixed smooth alpha_sigma, U_sigma, Delta."""
    dx = (1.0, 1.0, 1.0)
    shape = (n_side,) * 3
    f = [_smooth_field(500 + i, shape, dx) for i in range(1, 7)]
    fixed = dict(alpha_a=1.10 + f[0], alpha_b=1.05 + f[1], U_a=f[2], U_b=f[3], delta=0.25 + (f[4] + 1j * f[5]))
    mu_eff, delta0 = 0.5, 0.25
    kidx, E = _plane_wave_table(shape, dx, mu_eff, delta0)
    return Workload(f"cfg5_3d_{n_side}^3_fixed_kin{kin_form}", 3, shape, dx, n_wf, 0, 0, 0, kin_form, 4, 5, 0.005,
                    n_steps, (0.6, 0.4), kidx=kidx[:n_wf], branch=np.ones(n_wf, dtype=np.int64),
                    mode_of=np.zeros(n_wf, dtype=np.int64), mu_eff=mu_eff, delta0=delta0, noise=0.01, noise_seed=506,
                    E=E[:n_wf], w_a=np.zeros(n_wf), w_b=np.ones(n_wf), fixed=fixed)


def random_spinors(seed, n_wf, shape, dV=1.0):
    """Seeded random normalised spinors [n_wf, 2, *shape] (for property tests)."""
    M = int(np.prod(shape))
    z = normal(seed, 0, n_wf * 4 * M).reshape((n_wf, 2) + tuple(shape) + (2,))
    psi = z[..., 0] + 1j * z[..., 1]
    nrm = np.sqrt(np.sum(np.abs(psi) ** 2, axis=tuple(range(1, psi.ndim)), keepdims=True) * dV)
    return psi / nrm


# ---- context plumbing: hand a Workload's inputs to a context object (the oracle's or the CUDA library's; both expose the
# same setters).  Argument marshalling only -- used by tests/harness.py, bench.py and __graft_entry__.smoke().
def context_kwargs(w: "Workload", over=None) -> dict:
    kw = dict(func_id=w.func_id, force_a1=w.force_a1, spin_symmetric=w.spin_symmetric, kin_form=w.kin_form,
              ab_order=w.ab_order, am_order=w.am_order, subtract_mean_energy=w.subtract_mean_energy,
              normalize=w.normalize, four_pi_as=w.four_pi_as, E_cut=w.E_cut, lambda_mode=w.lambda_mode)
    if getattr(w, "current_terms", 0):
        kw["current_terms"] = 1
    if getattr(w, "friction", None):                      # dict(qf_alpha=..., qf_beta=..., qf_gamma=..., qf_rho0=..., qf_nreq=...)
        kw["quantum_friction"] = 1
        kw.update(w.friction)
    kw.update(over or {})
    return kw


def configure(c, w: "Workload", n_wf: int | None = None):
    """Set chemical potentials, the mode table (clipped to the first n_wf spinors), weights, external and fixed fields."""
    n_wf = w.n_wf if n_wf is None else n_wf
    c.set_mu(*w.mu)
    if w.kperp is not None:
        c.set_modes(w.kperp, w.mult, np.minimum(np.asarray(w.first), n_wf))
    c.set_weights(np.asarray(w.w_a[:n_wf]), np.asarray(w.w_b[:n_wf]))
    if w.vext_a is not None or w.delta_ext is not None:
        shp = w.shape
        va = None if w.vext_a is None else np.broadcast_to(w.vext_a.reshape(shp), shp).copy()
        vb = None if w.vext_b is None else np.broadcast_to(w.vext_b.reshape(shp), shp).copy()
        c.set_external(va, vb, w.delta_ext)
    if w.fixed:
        c.set_potentials(**w.fixed)
    if getattr(w, "vel", None) is not None:               # external velocity fields (v_a, v_b), only with current_terms
        c.set_velocity(*w.vel)
    return c
