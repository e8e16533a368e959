"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Every check compares the oracle with something that is NOT the oracle: closed forms typed out here, dense
matrices built with numpy from Eqs. 28a/b, numpy's eigh / FFT as independent third parties, conservation laws.
"""
import os

import numpy as np
import pytest

import oracle as orc
import workloads as wl

TWO_PI = 2 * np.pi


def relerr(x, ref):
    return np.max(np.abs(np.asarray(x) - np.asarray(ref))) / np.max(np.abs(ref))


# ---------------------------------------------------------------------------------------------- P1: transforms
@pytest.mark.parametrize("n", [2, 4, 8, 16, 32, 64, 128, 256])
def test_p1_fft_vs_naive_dft_and_numpy(n):
    x = wl.normal(7, 0, 2 * n).view(np.complex128)
    f = orc.fft1d(x, -1)
    assert relerr(f, orc.dft1d_naive(x, -1)) < 1e-13
    assert relerr(f, np.fft.fft(x)) < 1e-13                       # library routine, same sign convention
    assert relerr(orc.fft1d(f, +1) / n, x) < 1e-13                # inverse(forward(x)) = x
    # definition typed out once more for a single output bin (guards the sign of the exponent)
    l = 3 % n
    assert abs(f[l] - np.sum(x * np.exp(-1j * TWO_PI * l * np.arange(n) / n))) < 1e-11


def test_p1_fft_rejects_non_power_of_two():
    with pytest.raises(ValueError):
        orc.fft1d(np.zeros(12, dtype=complex))


# ------------------------------------------------------------------- P2: Eq. 28a/b derivative matrices
def d1_matrix(n, dx):
    L = n * dx
    l = np.arange(n)
    d = l[:, None] - l[None, :]
    with np.errstate(divide="ignore", invalid="ignore"):
        m = np.pi / L * (-1.0) ** d / np.tan(np.pi * d / n)
    m[d == 0] = 0.0
    return m


def d2_matrix(n, dx):
    L = n * dx
    l = np.arange(n)
    d = l[:, None] - l[None, :]
    with np.errstate(divide="ignore", invalid="ignore"):
        m = 2 * np.pi ** 2 / L ** 2 * (-1.0) ** (d - 1) / np.sin(np.pi * d / n) ** 2
    m[d == 0] = -np.pi ** 2 / (3 * dx ** 2) * (1 + 2.0 / n ** 2)
    return m


@pytest.mark.parametrize("n,dx", [(8, 1.0), (16, 0.7), (32, 1.3)])
def test_p2_derivative_matrices_1d(n, dx):
    f = wl.normal(11, 0, 2 * n).view(np.complex128)
    lap, grad = orc.derivatives(f, [dx])
    assert relerr(grad[0], d1_matrix(n, dx) @ f) < 1e-13
    assert relerr(lap, d2_matrix(n, dx) @ f) < 1e-13


def test_p2_derivative_matrices_3d_axes():
    shape, dx = (4, 8, 16), (1.0, 0.5, 2.0)
    f = wl.normal(12, 0, 2 * int(np.prod(shape))).view(np.complex128).reshape(shape)
    lap, grad = orc.derivatives(f, dx)
    D1 = [d1_matrix(shape[a], dx[a]) for a in range(3)]
    D2 = [d2_matrix(shape[a], dx[a]) for a in range(3)]
    assert relerr(grad[0], np.einsum("ij,jkl->ikl", D1[0], f)) < 1e-13
    assert relerr(grad[1], np.einsum("ij,kjl->kil", D1[1], f)) < 1e-13
    assert relerr(grad[2], np.einsum("ij,klj->kli", D1[2], f)) < 1e-13
    ref = (np.einsum("ij,jkl->ikl", D2[0], f) + np.einsum("ij,kjl->kil", D2[1], f) + np.einsum("ij,klj->kli", D2[2], f))
    assert relerr(lap, ref) < 1e-13


def test_p2_real_field_has_real_odd_derivative():
    """Footnote 6: zeroing the Nyquist mode keeps the first derivative of a real field real."""
    f = wl.normal(13, 0, 16).astype(np.complex128)
    _, grad = orc.derivatives(f, [1.0])
    assert np.max(np.abs(grad[0].imag)) < 1e-14


# --------------------------------------------------------------------------------------------- helpers for H
def dense_h(shape, dx, alpha_a, alpha_b, U_a, U_b, delta, mu, kin_form, kp2=0.0):
    """Dense 2M x 2M BdG matrix of Eq. 5 from Eqs. 28a/b, 39a-c, 40 (numpy only)."""
    nd = len(shape)
    M = int(np.prod(shape))

    def axis_op(mat, a):
        ops = [np.eye(s) for s in shape]
        ops[a] = mat
        out = ops[0]
        for o in ops[1:]:
            out = np.kron(out, o)
        return out

    D1 = [axis_op(d1_matrix(shape[a], dx[a]), a) for a in range(nd)]
    lap = sum(axis_op(d2_matrix(shape[a], dx[a]), a) for a in range(nd))

    def kin(alpha):
        A = np.diag(alpha.ravel())
        if kin_form == 0:
            return -0.5 * lap + 0.5 * kp2 * np.eye(M)
        if kin_form == 1:
            lap_alpha = np.diag(lap @ alpha.ravel())
            return -0.25 * (lap @ A + A @ lap - lap_alpha) + 0.5 * kp2 * A
        return -0.5 * sum(D1[a] @ A @ D1[a] for a in range(nd)) + 0.5 * kp2 * A

    ha = kin(alpha_a) + np.diag(U_a.ravel() - mu[0])
    hb = kin(alpha_b) + np.diag(U_b.ravel() - mu[1])
    D = np.diag(delta.ravel())
    return np.block([[ha, D], [D.conj(), -hb]])


def random_fields(seed, shape):
    M = int(np.prod(shape))
    z = wl.normal(seed, 0, 6 * M).reshape(6, *shape)
    return dict(alpha_a=1.1 + 0.2 * np.tanh(z[0]), alpha_b=0.9 + 0.2 * np.tanh(z[1]), U_a=0.3 * z[2], U_b=0.3 * z[3],
                delta=0.2 + 0.1 * (z[4] + 1j * z[5]))


def make_fixed(shape, dx, n_wf, kin_form, fields, mu=(0.4, 0.3), mode=None, full_dims=None, **kw):
    mode = len(shape) if mode is None else mode
    dims = list(shape) if full_dims is None else full_dims
    o = orc.Oracle(mode, dims, dx, n_wf, func_id=0, kin_form=kin_form, **kw)
    o.set_mu(*mu)
    o.set_potentials(**fields)
    return o


# ----------------------------------------------------------------------------- P3: closed-form uniform eigenstates
@pytest.mark.parametrize("kin_form,alpha0", [(0, 1.0), (1, 1.0), (1, 1.3), (2, 1.3)])
def test_p3_uniform_plane_wave_eigenstates(kin_form, alpha0):
    shape, dx, mu, d0 = (8, 4, 4), (1.0, 1.2, 0.8), 0.5, 0.2 + 0.1j
    M = int(np.prod(shape))
    one = np.ones(shape)
    o = make_fixed(shape, dx, 2, kin_form, dict(alpha_a=alpha0 * one, alpha_b=alpha0 * one, U_a=0 * one, U_b=0 * one,
                                                 delta=d0 * one), mu=(mu, mu))
    ks = [wl.kgrid(shape[a], dx[a]) for a in range(3)]
    pos = np.meshgrid(*[np.arange(shape[a]) * dx[a] for a in range(3)], indexing="ij")
    # one generic k and (for the second-derivative forms, which keep the Nyquist mode) one Nyquist k
    for kidx in [(3, 1, 3), (4, 2, 1)] if kin_form != 2 else [(3, 1, 3)]:
        k = [ks[a][kidx[a]] for a in range(3)]
        eps = alpha0 * sum(x * x for x in k) / 2 - mu
        E = np.sqrt(eps ** 2 + abs(d0) ** 2)
        u, v = np.sqrt((1 + eps / E) / 2), np.sqrt((1 - eps / E) / 2) * np.conj(d0) / abs(d0)
        pw = np.exp(1j * sum(k[a] * pos[a] for a in range(3))) / np.sqrt(M * np.prod(dx))
        psi = np.stack([np.stack([u * pw, v * pw]), np.stack([-np.conj(v) * pw, u * pw])])
        h, eps_n = o.apply_h(psi)
        assert relerr(h[0], E * psi[0]) < 1e-13               # E = +sqrt((k^2/2 - mu)^2 + |Delta|^2)
        assert relerr(h[1], -E * psi[1]) < 1e-13              # partner branch, E = -sqrt(...)
        assert abs(eps_n[0] - E) < 1e-13 and abs(eps_n[1] + E) < 1e-13


# ------------------------------------------------------------------------------------------- P4: Hermiticity
@pytest.mark.parametrize("kin_form", [0, 1, 2])
@pytest.mark.parametrize("shape,dx", [((8, 4, 8), (1.0, 0.9, 1.1)), ((16, 8), (1.0, 1.0)), ((32,), (0.8,))])
def test_p4_hermiticity(kin_form, shape, dx):
    f = random_fields(21, shape)
    o = make_fixed(shape, dx, 2, kin_form, f)
    if len(shape) < 3:
        o.set_modes([[0.3, -0.2]], [1.0], [0, 2])
    psi = wl.random_spinors(22, 2, shape)
    h, _ = o.apply_h(psi)
    lhs = np.vdot(psi[0], h[1])                    # <phi|H psi>
    rhs = np.conj(np.vdot(psi[1], h[0]))           # <H phi|psi> = <psi|H phi>^*
    assert abs(lhs - rhs) < 1e-13 * max(1.0, abs(lhs))


# ---------------------------------------------------------------------- P5: dense H from Eqs. 28/39/40 (numpy)
@pytest.mark.parametrize("kin_form", [0, 1, 2])
def test_p5_dense_matvec_3d(kin_form):
    shape, dx, mu = (4, 4, 8), (1.0, 1.1, 0.9), (0.4, 0.3)
    f = random_fields(31, shape)
    o = make_fixed(shape, dx, 3, kin_form, f, mu=mu)
    H = dense_h(shape, dx, f["alpha_a"], f["alpha_b"], f["U_a"], f["U_b"], f["delta"], mu, kin_form)
    assert np.max(np.abs(H - H.conj().T)) < 1e-12
    psi = wl.random_spinors(32, 3, shape)
    h, eps = o.apply_h(psi)
    for n in range(3):
        ref = H @ psi[n].ravel()
        assert relerr(h[n].ravel(), ref) < 1e-12
        assert abs(eps[n] - np.real(np.vdot(psi[n].ravel(), ref)) * np.prod(dx)) < 1e-12


@pytest.mark.parametrize("kin_form", [0, 1])
def test_p5_dense_matvec_transverse_mode(kin_form):
    """quasi-2D substitution mu -> mu - alpha kz^2 / 2."""
    shape, dx, mu, kz = (8, 8), (1.0, 1.0), (0.4, 0.3), 0.7
    f = random_fields(33, shape)
    o = make_fixed(shape, dx, 1, kin_form, f, mu=mu, full_dims=[8, 8, 16])
    o.set_modes([[kz, 0.0]], [2.0], [0, 1])
    H = dense_h(shape, dx, f["alpha_a"], f["alpha_b"], f["U_a"], f["U_b"], f["delta"], mu, kin_form, kp2=kz * kz)
    psi = wl.random_spinors(34, 1, shape)
    h, _ = o.apply_h(psi)
    assert relerr(h[0].ravel(), H @ psi[0].ravel()) < 1e-12


def test_p5_spectrum_symmetric_for_spin_symmetric_h():
    """h_a - mu_a = h_b - mu_b  =>  eigenvalues come in +-E pairs."""
    shape, dx = (4, 4, 4), (1.0, 1.0, 1.0)
    f = random_fields(35, shape)
    f["alpha_b"], f["U_b"] = f["alpha_a"], f["U_a"]
    H = dense_h(shape, dx, f["alpha_a"], f["alpha_b"], f["U_a"], f["U_b"], f["delta"], (0.4, 0.4), 1)
    E = np.linalg.eigvalsh(H)
    assert np.max(np.abs(E + E[::-1])) < 1e-12


# ------------------------------------------------------------------ P6/P7: integrator order against exact exp(-iHt)
def evolve_oracle(o, psi0, dt, n_steps, selfstart=1):
    phi = np.ascontiguousarray(psi0.copy())
    hist = [np.zeros_like(phi) for _ in range(o.m)]
    hist = o.abm_init(phi, hist, dt, selfstart)
    for _ in range(n_steps - (o.m - 1 if selfstart else 0)):
        hist = o.abm_step(phi, hist, dt)
    return phi


@pytest.mark.parametrize("ab,am,order", [(3, 4, 4), (4, 4, 4), (4, 5, 5), (5, 5, 5)])
def test_p6_order_of_convergence_against_exact_propagator(ab, am, order):
    shape, dx, mu = (16,), (1.0,), (0.4, 0.3)
    f = random_fields(41, shape)
    H = dense_h(shape, dx, f["alpha_a"], f["alpha_b"], f["U_a"], f["U_b"], f["delta"], mu, 1)
    lam, V = np.linalg.eigh(H)
    psi0 = wl.random_spinors(42, 2, shape)
    T = 0.32
    errs = []
    for nst in (32, 64):
        o = make_fixed(shape, dx, 2, 1, f, mu=mu, ab_order=ab, am_order=am, subtract_mean_energy=0, normalize=0)
        phi = evolve_oracle(o, psi0, T / nst, nst)
        exact = np.stack([(V @ (np.exp(-1j * lam * T) * (V.conj().T @ psi0[n].ravel()))).reshape(2, *shape)
                          for n in range(2)])
        errs.append(relerr(phi, exact))
    slope = np.log2(errs[0] / errs[1])
    assert errs[1] < 1e-5
    assert order - 0.6 < slope < order + 1.2, (errs, slope)


def test_p6_energy_shift_changes_only_a_phase():
    """Eqs. 41 vs 44a differ by exp(-i int <H>_n dt): compare |<exact|phi>| = 1."""
    shape, dx, mu = (16,), (1.0,), (0.4, 0.3)
    f = random_fields(43, shape)
    H = dense_h(shape, dx, f["alpha_a"], f["alpha_b"], f["U_a"], f["U_b"], f["delta"], mu, 1)
    lam, V = np.linalg.eigh(H)
    psi0 = wl.random_spinors(44, 1, shape)
    o = make_fixed(shape, dx, 1, 1, f, mu=mu, subtract_mean_energy=1, normalize=1)
    T, nst = 0.2, 40
    phi = evolve_oracle(o, psi0, T / nst, nst)
    exact = V @ (np.exp(-1j * lam * T) * (V.conj().T @ psi0[0].ravel()))
    ov = np.vdot(exact, phi[0].ravel())
    assert abs(abs(ov) - 1.0) < 1e-9
    # the phase is the time integral of the conserved <H>
    e0 = np.real(np.vdot(psi0[0].ravel(), H @ psi0[0].ravel()))
    assert abs(np.angle(ov * np.exp(-1j * e0 * T))) < 1e-8


def test_p7_abm_tables_on_scalar_ode():
    """On a 2-point lattice with uniform fields the k=0 spinor obeys y' = -i w y: compare with exp(-i w t);
    also exactness conditions of the printed coefficient tables (Eqs. 46-50)."""
    from fractions import Fraction as F
    tabs = {"AB3": [F(23, 12), F(-16, 12), F(5, 12)], "AB4": [F(55, 24), F(-59, 24), F(37, 24), F(-9, 24)],
            "AB5": [F(1901, 720), F(-2774, 720), F(2616, 720), F(-1274, 720), F(251, 720)]}
    for name, b in tabs.items():                     # AB_s integrates t^q exactly for q < s from history at t=-1,-2,..
        for q in range(len(b)):
            assert sum(bi * F(-(i), 1) ** q for i, bi in enumerate(b)) == F(1, q + 1), name
    am = {"AM4": [F(9, 24), F(19, 24), F(-5, 24), F(1, 24)], "AM5": [F(251, 720), F(646, 720), F(-264, 720), F(106, 720), F(-19, 720)]}
    for name, c in am.items():                       # nodes t = 1, 0, -1, ...; integral of t^q over [0,1]
        for q in range(len(c)):
            assert sum(ci * F(1 - i, 1) ** q for i, ci in enumerate(c)) == F(1, q + 1), name
    one = np.ones(2)
    w = 0.37
    o = make_fixed((2,), (1.0,), 1, 0, dict(alpha_a=one, alpha_b=one, U_a=w * one, U_b=0 * one, delta=0j * one),
                   mu=(0.0, 0.0), ab_order=4, am_order=5, subtract_mean_energy=0, normalize=0)
    psi0 = np.zeros((1, 2, 2), dtype=complex)
    psi0[0, 0] = 1 / np.sqrt(2)
    e = []
    for nst in (20, 40):
        phi = evolve_oracle(o, psi0, 2.0 / nst, nst)
        e.append(abs(phi[0, 0, 0] - np.exp(-1j * w * 2.0) / np.sqrt(2)))
    assert 4.4 < np.log2(e[0] / e[1]) < 6.2


# ---------------------------------------------------------------- P8: stationary state does not move (Eqs. 43-44)
def test_p8_stationary_state_with_shift_stays_put():
    w = wl.cfg1(n_wf=64)
    one = np.ones(w.shape)
    o = make_fixed(w.shape, w.dx, w.n_wf, 0, dict(alpha_a=one, alpha_b=one, U_a=0 * one, U_b=0 * one, delta=0.2 * one),
                   mu=(0.5, 0.5), ab_order=4, am_order=4)
    psi0 = w.spinors()
    h, eps = o.apply_h(psi0)
    assert relerr(eps, w.E) < 1e-13
    phi = evolve_oracle(o, psi0, 0.005, 100, selfstart=1)
    assert relerr(phi, psi0) < 1e-12
    phi = evolve_oracle(o, psi0, 0.005, 100, selfstart=0)      # f_k = 0 start
    assert relerr(phi, psi0) < 1e-12


# --------------------------------------------------------------------- P9/P10/P17: densities of the uniform system
def uniform_oracle(w, **kw):
    o = orc.Oracle(w.mode, w.dims, w.dx, w.n_wf, func_id=0, **kw)
    o.set_weights(w.w_a, w.w_b)
    return o


def test_p9_completeness_full_basis():
    w = wl.cfg1()
    o = uniform_oracle(w)
    o.set_weights(np.ones(w.n_wf), np.ones(w.n_wf))
    psi = w.spinors()
    o.densities(psi)
    assert relerr(o.get_field("rho_a"), np.full(w.shape, 1 / w.dV)) < 1e-12    # sum_n |u_n(r)|^2 = 1/dV
    assert relerr(o.get_field("rho_b"), np.full(w.shape, 1 / w.dV)) < 1e-12
    o.set_weights(np.zeros(w.n_wf), 2 * np.ones(w.n_wf))                       # nu = sum_n u_n v_n^* = 0
    o.densities(psi)
    assert np.max(np.abs(o.get_field("nu"))) < 1e-13


def test_p10_uniform_density_closed_forms():
    w = wl.cfg1()
    o = uniform_oracle(w)
    psi = w.spinors()
    o.densities(psi)
    ks = [wl.kgrid(8, 1.0)] * 3
    K = np.meshgrid(*ks, indexing="ij")
    kt = [np.where(np.arange(8) == 4, 0.0, k) for k in ks]       # Nyquist-zeroed for first derivatives
    KT = np.meshgrid(*kt, indexing="ij")
    eps = sum(k * k for k in K) / 2 - 0.5
    E = np.sqrt(eps ** 2 + 0.04)
    vol = 512.0
    v2, u2 = 0.5 * (1 - eps / E), 0.5 * (1 + eps / E)
    # general Eq. 7 weights at T=0: (+) states carry w_b=1, (-) states (u,v)=(-v_k,u_k) carry w_a=1
    assert relerr(o.get_field("rho_b"), np.full(w.shape, np.sum(v2) / vol)) < 1e-13
    assert relerr(o.get_field("rho_a"), np.full(w.shape, np.sum(v2) / vol)) < 1e-13
    kt2 = sum(k * k for k in KT)
    assert relerr(o.get_field("tau_b"), np.full(w.shape, np.sum(kt2 * v2) / vol)) < 1e-13
    # nu = 1/2 sum (w_b - w_a) u v^*: (+) gives +u_k v_k/2, (-) gives -(-v_k u_k)/2  =>  sum_k Delta/(2E)/V
    assert relerr(o.get_field("nu"), np.full(w.shape, np.sum(0.2 / (2 * E)) / vol)) < 1e-13
    for f in ("ja_x", "ja_y", "ja_z", "jb_x", "jb_y", "jb_z"):
        assert np.max(np.abs(o.get_field(f))) < 1e-14


def test_p10_single_plane_wave_current_sign():
    """One spinor (0, e^{ikr}/sqrt V) with w_b=1: j_b = Im[v grad v^*] = -k |v|^2; (e^{ikr},0) with w_a=1: j_a = +k|u|^2."""
    shape, dx = (8, 8, 4), (1.0, 0.5, 2.0)
    vol = np.prod(shape) * np.prod(dx)
    o = orc.Oracle(3, shape, dx, 2)
    o.set_weights([1.0, 0.0], [0.0, 1.0])
    ks = [wl.kgrid(shape[a], dx[a]) for a in range(3)]
    kidx = (2, 7, 1)
    k = np.array([ks[a][kidx[a]] for a in range(3)])
    pos = np.meshgrid(*[np.arange(shape[a]) * dx[a] for a in range(3)], indexing="ij")
    pw = np.exp(1j * sum(k[a] * pos[a] for a in range(3))) / np.sqrt(vol)
    psi = np.zeros((2, 2) + shape, dtype=complex)
    psi[0, 0] = pw
    psi[1, 1] = pw
    o.densities(psi)
    for a, nm in enumerate("xyz"):
        assert relerr(o.get_field("ja_" + nm), np.full(shape, k[a] / vol)) < 1e-13
        assert relerr(o.get_field("jb_" + nm), np.full(shape, -k[a] / vol)) < 1e-13
    assert relerr(o.get_field("tau_a"), np.full(shape, np.sum(k * k) / vol)) < 1e-13


def test_p17_general_vs_spin_symmetric_densities():
    """Eq. 8 (E>0 only, folded) = Eq. 7 over both branches with partner states [v^*, -u^*]."""
    shape, dx, n = (4, 8, 4), (1.0, 1.0, 1.0), 5
    psi = wl.random_spinors(51, n, shape)
    fb = wl.uniform01(52, 0, n)                          # f_beta(-E_n) in (0,1), f_beta(E_n) = 1 - that
    o_sym = orc.Oracle(3, shape, dx, n, spin_symmetric=1)
    o_sym.set_weights(1 - fb, fb)
    o_sym.densities(psi)
    partner = np.stack([np.conj(psi[:, 1]), -np.conj(psi[:, 0])], axis=1)
    both = np.concatenate([psi, partner])
    o_gen = orc.Oracle(3, shape, dx, 2 * n, spin_symmetric=0)
    o_gen.set_weights(np.concatenate([1 - fb, fb]), np.concatenate([fb, 1 - fb]))   # partner has energy -E_n
    o_gen.densities(both)
    for f in ("rho_a", "rho_b", "tau_a", "tau_b", "nu", "ja_x", "ja_y", "ja_z", "jb_x", "jb_y", "jb_z"):
        assert relerr(o_sym.get_field(f), o_gen.get_field(f)) < 1e-13, f


def test_p10_density_accumulate_over_batches():
    shape, n = (8, 8), 7
    psi = wl.random_spinors(53, n, shape)
    o = orc.Oracle(2, list(shape) + [4], (1.0, 1.0, 1.0), n)
    o.set_modes([[0.1, 0], [0.4, 0]], [1.0, 2.0], [0, 3, 7])
    o.densities(psi)
    full = {f: o.get_field(f) for f in ("rho_b", "tau_b", "nu", "jb_x")}
    o.densities(psi, 0, 4, accumulate=0)
    o.densities(psi, 4, 3, accumulate=1)
    for f, v in full.items():
        assert relerr(o.get_field(f), v) < 1e-14


# ----------------------------------------------------------------- P16: 3D vs quasi-2D / quasi-1D
@pytest.mark.parametrize("mode", [2, 1])
def test_p16_reduced_modes_match_3d(mode):
    dims, dx = (8, 4, 4), (1.0, 1.1, 0.9)
    held = dims[:mode]
    f = random_fields(61, held)                                   # fields independent of the transverse axes
    mu = (0.4, 0.3)
    kt = [wl.kgrid(dims[a], dx[a]) for a in range(mode, 3)]
    # transverse modes without their Nyquist members (R17): the 3D gradient zeroes those, Eqs. 29c/30c keep them
    tm = [[(i, k) for i, k in enumerate(kk) if i != len(kk) // 2] for kk in kt]
    modes = [(a,) for a in tm[0]] if mode == 2 else [(a, b) for a in tm[0] for b in tm[1]]
    per = 2
    nq = len(modes) * per
    psi_q = wl.random_spinors(62, nq, held, dV=np.prod(dx[:mode]))
    Lp = np.prod([dims[a] * dx[a] for a in range(mode, 3)])
    kperp = np.array([[m[0][1], m[1][1] if mode == 1 else 0.0] for m in modes])
    oq = make_fixed(held, dx, nq, 1, f, mu=mu, mode=mode, full_dims=list(dims))
    oq.set_modes(kperp, np.ones(len(modes)), np.arange(len(modes) + 1) * per)
    wa, wb = wl.uniform01(63, 0, nq), wl.uniform01(64, 0, nq)
    oq.set_weights(wa, wb)
    # the same states on the full 3D lattice: phi(x,y) e^{i kz z}/sqrt(Lz) (Eq. 29a / 30a)
    tpos = [np.arange(dims[a]) * dx[a] for a in range(mode, 3)]
    psi3 = np.zeros((nq, 2) + dims, dtype=complex)
    for n in range(nq):
        m = modes[n // per]
        ph = np.exp(1j * m[0][1] * tpos[0])
        if mode == 1:
            ph = np.multiply.outer(ph, np.exp(1j * m[1][1] * tpos[1]))
        psi3[n] = np.multiply.outer(psi_q[n], ph) / np.sqrt(Lp)
    f3 = {k: np.broadcast_to(v.reshape(v.shape + (1,) * (3 - mode)), dims).copy() for k, v in f.items()}
    o3 = make_fixed(dims, dx, nq, 1, f3, mu=mu)
    o3.set_weights(wa, wb)
    hq, eq = oq.apply_h(psi_q)
    h3, e3 = o3.apply_h(psi3)
    assert relerr(eq, e3) < 1e-12
    sl = (slice(None),) * (2 + mode) + (0,) * (3 - mode)
    assert relerr(hq, h3[sl] * np.sqrt(Lp)) < 1e-12          # transverse phase is 1 at the origin of those axes
    oq.densities(psi_q)
    o3.densities(psi3)
    for fld in ["rho_a", "rho_b", "tau_a", "tau_b", "nu", "ja_x", "jb_x"] + (["ja_y", "jb_y"] if mode == 2 else []):
        assert relerr(oq.get_field(fld), o3.get_field(fld)[sl[2:]]) < 1e-12, fld


# ------------------------------------------------------------------------------- P12/P14/P15: pointwise functional
def slda(force_a1=0, **kw):
    o = orc.Oracle(3, (4, 4, 4), (1.0, 1.0, 1.0), 1, func_id=2, force_a1=force_a1, kin_form=1, **kw)
    o.set_mu(0.35, 0.25)
    return o


def test_p12_lambda_c_against_principal_value_integral():
    """Lambda_c (Eq. 20) = PV int_0^kc d^3k/(2pi)^3 1/(alpha (k^2 - k0^2)) ... the regulator of the uniform gas:
    closed form vs numerical quadrature, both signs of k0^2, and continuity at k0 = 0."""
    from scipy.integrate import quad
    o = slda(force_a1=1, E_cut=4.0)
    for vext in (-0.4, 0.1, 0.29, 0.31, 0.8, 2.0):           # moves k0^2 = 2(mu+ - V+)/alpha through zero
        r = o.functional_point(0.01, 0.01, 0.0, 0.0, 0.0, vext, vext)
        V0 = r["V_a"]                                        # nu = 0 -> no pairing part
        k02 = 2 * (0.30 - V0 - vext)
        kc2 = 2 * (4.0 + 0.30 - V0 - vext)
        kc = np.sqrt(kc2)
        if k02 > 0:
            k0 = np.sqrt(k02)
            # PV int_0^kc k^2/(k^2-k0^2) dk = kc + k0^2 PV int dk/(k^2-k0^2); use cauchy weight 1/(k-k0)
            pv = quad(lambda k: 1.0 / (k + k0), 0, kc, weight="cauchy", wvar=k0)[0]
            integral = kc + k02 * pv
        else:
            integral = quad(lambda k: k * k / (k * k - k02), 0, kc)[0]
        assert abs(r["lambda_c"] - integral / (2 * np.pi ** 2)) < 1e-10
    V0 = o.functional_point(0.01, 0.01, 0, 0, 0)["V_a"]
    a = o.functional_point(0.01, 0.01, 0, 0, 0, 0.3 - V0 - 1e-10, 0.3 - V0 - 1e-10)      # k0^2 -> 0+
    b = o.functional_point(0.01, 0.01, 0, 0, 0, 0.3 - V0 + 1e-10, 0.3 - V0 + 1e-10)      # k0^2 -> 0-
    assert abs(a["lambda_c"] - b["lambda_c"]) < 1e-4 * a["lambda_c"]


@pytest.mark.parametrize("force_a1", [0, 1])
def test_p14_potentials_are_derivatives_of_energy_density(force_a1):
    o = slda(force_a1=force_a1)
    ra, rb, ta, tb, nu = 0.021, 0.013, 0.05, 0.02, 0.004 - 0.003j
    base = o.functional_point(ra, rb, ta, tb, nu)
    lam = base["lambda_c"]

    def e(ra_, rb_, ta_=ta, tb_=tb, nu_=nu):
        return o.functional_point(ra_, rb_, ta_, tb_, nu_, lambda_in=lam)["edens"]

    h = 1e-6
    assert abs((e(ra + h, rb) - e(ra - h, rb)) / (2 * h) - base["V_a"]) < 1e-7       # V_a = dE/d rho_a
    assert abs((e(ra, rb + h) - e(ra, rb - h)) / (2 * h) - base["V_b"]) < 1e-7
    assert abs(2 * (e(ra, rb, ta + h) - e(ra, rb, ta - h)) / (2 * h) - base["alpha_a"]) < 1e-8   # alpha = 2 dE/d tau
    assert abs(2 * (e(ra, rb, ta, tb + h) - e(ra, rb, ta, tb - h)) / (2 * h) - base["alpha_b"]) < 1e-8
    # Delta = -dE/d nu^* : for E = g |nu|^2, dE/d nu^* = g nu  (Wirtinger) = [dE/dRe + i dE/dIm]/2
    dre = (e(ra, rb, nu_=nu + h) - e(ra, rb, nu_=nu - h)) / (2 * h)
    dim = (e(ra, rb, nu_=nu + 1j * h) - e(ra, rb, nu_=nu - 1j * h)) / (2 * h)
    assert abs(-(dre + 1j * dim) / 2 - base["delta"]) < 1e-8
    if force_a1:
        assert base["alpha_a"] == 1.0 and base["alpha_b"] == 1.0


def test_p14_aslda_constants_at_p0_and_p1():
    o = slda()
    r = o.functional_point(0.01, 0.01, 0, 0, 0)
    assert abs(r["alpha_a"] - 1.094) < 1e-15 and abs(r["alpha_b"] - 1.094) < 1e-15       # Eq. 12a at p = 0
    r = o.functional_point(0.02, 0.0, 0, 0, 0)
    assert abs(r["alpha_a"] - (1.094 + 0.156 * 8 / 15 - 0.532 / 3)) < 1e-14             # p = 1
    assert abs(r["alpha_b"] - (1.094 - 0.156 * 8 / 15 - 0.532 / 3)) < 1e-14             # A_b(p) = A_a(-p)


def test_p15_bdg_limit():
    """A=1, B=0, C/rho^(1/3) = 4 pi a_s: V=0, alpha=1, Delta = -g nu with 1/g = 1/(4 pi a_s) - Lambda_c (Eq. 11)."""
    o = orc.Oracle(3, (4, 4, 4), (1.0, 1.0, 1.0), 1, func_id=1, four_pi_as=-4.0)
    o.set_mu(0.5, 0.5)
    nu = 0.01 + 0.02j
    r = o.functional_point(0.02, 0.02, 0.03, 0.03, nu, 0.1, 0.1)
    assert r["V_a"] == 0.0 and r["V_b"] == 0.0 and r["alpha_a"] == 1.0 and r["alpha_b"] == 1.0
    k0, kc = np.sqrt(2 * 0.4), np.sqrt(2 * (np.pi ** 2 / 2 + 0.4))
    lam = kc / (2 * np.pi ** 2) * (1 - k0 / (2 * kc) * np.log((kc + k0) / (kc - k0)))
    assert abs(r["lambda_c"] - lam) < 1e-15
    assert abs(r["delta"] + nu / (1 / -4.0 - lam)) < 1e-15


def test_p13_uniform_unitary_gas_values():
    """SLDA at p=0 in the continuum with a large cutoff reproduces the paper's printed Delta/eF = 0.51(1),
    E/E_FG = 0.39(1) (Eq. 12d) -- pins the sign reading of Eq. 19 (R1) and V_sigma (R2)."""
    from scipy.integrate import quad
    from scipy.optimize import fsolve
    kF = 1.0
    rho = kF ** 3 / (3 * np.pi ** 2)
    eF = 0.5
    Ec = 0.5 * (25.0 * kF) ** 2
    alpha = 1.094

    def moments(mu_eff, D):
        kmax = np.sqrt(2 * (np.sqrt(max(Ec * Ec - D * D, 0.0)) + mu_eff) / alpha)   # E_k < E_c
        ek = lambda k: alpha * k * k / 2 - mu_eff
        Ek = lambda k: np.sqrt(ek(k) ** 2 + D * D)
        pts = [np.sqrt(2 * max(mu_eff, 0.01) / alpha)]
        n = quad(lambda k: k * k * 0.5 * (1 - ek(k) / Ek(k)), 0, kmax, points=pts, limit=400)[0] / (2 * np.pi ** 2)
        t = quad(lambda k: k ** 4 * 0.5 * (1 - ek(k) / Ek(k)), 0, kmax, points=pts, limit=400)[0] / (2 * np.pi ** 2)
        a = quad(lambda k: k * k * D / (2 * Ek(k)), 0, kmax, points=pts, limit=400)[0] / (2 * np.pi ** 2)
        return n, t, a

    def resid(x):
        mu, D, U = x
        o = orc.Oracle(3, (4, 4, 4), (1.0, 1.0, 1.0), 1, func_id=2, kin_form=1, E_cut=Ec)
        o.set_mu(mu, mu)
        n, t, a = moments(mu - U, D)
        r = o.functional_point(n, n, t, t, a)
        return [2 * n - rho, r["delta"].real - D, r["V_a"] - U]

    mu, D, U = fsolve(resid, [0.4 * eF, 0.5 * eF, -0.25], xtol=1e-12)
    o = orc.Oracle(3, (4, 4, 4), (1.0, 1.0, 1.0), 1, func_id=2, kin_form=1, E_cut=Ec)
    o.set_mu(mu, mu)
    n, t, a = moments(mu - U, D)
    r = o.functional_point(n, n, t, t, a)
    assert abs(2 * n - rho) < 1e-9
    gold = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "eq12d_unitary_gas.txt")):
        if line.strip() and not line.startswith("#"):
            name, val, unc = line.split()
            gold[name] = (float(val), float(unc))
    assert alpha == gold["A_at_p0"][0]
    # the paper's printed values with their printed uncertainty (+ the finite-cutoff shift of the gap, < 0.01)
    assert abs(D / eF - gold["Delta_over_eF"][0]) <= gold["Delta_over_eF"][1] + 0.01, D / eF
    assert abs(r["edens"] / (0.6 * rho * eF) - gold["E_over_EFG"][0]) <= gold["E_over_EFG"][1] + 0.01
    assert 0.49 <= D / eF <= 0.52, D / eF
    assert 0.38 <= r["edens"] / (0.6 * rho * eF) <= 0.41, r["edens"] / (0.6 * rho * eF)
    assert abs(mu / eF - r["edens"] / (0.6 * rho * eF)) < 0.02      # mu = xi eF at unitarity (thermodynamics)


# ------------------------------------------------------------- P11: conservation laws of the self-consistent evolution
def test_p11_conservation_selfconsistent_bdg_full_basis():
    """Full basis (all 2M states of the BdG matrix), BdG functional (Lambda_c static since V+ = V_ext, alpha = 1):
    norm, orthonormality (Eq. 16), particle number and total energy are conserved up to the integrator error."""
    shape, dx = (4, 4, 2), (1.0, 1.0, 1.0)
    M = int(np.prod(shape))
    mu = (0.6, 0.6)
    z = wl.normal(71, 0, M).reshape(shape)
    vext = 0.2 * z
    delta0 = 0.3 + 0.05 * wl.normal(72, 0, M).reshape(shape)
    one = np.ones(shape)
    H = dense_h(shape, dx, one, one, vext, vext, delta0.astype(complex), mu, 0)
    lam, V = np.linalg.eigh(H)
    psi0 = np.ascontiguousarray(V.T.reshape(2 * M, 2, *shape))    # dV = 1: eigenvectors are already normalised
    o = orc.Oracle(3, shape, dx, 2 * M, func_id=1, kin_form=0, four_pi_as=-6.0, ab_order=4, am_order=5,
                   subtract_mean_energy=1, normalize=0)
    o.set_mu(*mu)
    o.set_external(vext, vext)
    o.set_weights((lam < 0).astype(float), (lam > 0).astype(float))
    lap = -2.0 * dense_h(shape, dx, one, one, 0 * one, 0 * one, 0j * one, (0.0, 0.0), 0)[:M, :M]   # sum_d D2_d (Eq. 28b)

    def conserved_energy(phi):
        """E_kin + E_pair + E_pot.ext (Eqs. 33a, c, e).  E_kin is written as sum_n w <psi|-lap/2|psi>, the form H itself
        uses: Eq. 33a's tau comes from first derivatives with the Nyquist mode dropped and equals it only
        for states without Nyquist content, which a full basis on a 4x4x2 lattice certainly has."""
        o.densities(phi)
        o.update_potentials()
        e = o.energy()
        u, v = phi[:, 0].reshape(2 * M, M), phi[:, 1].reshape(2 * M, M)
        wa, wb = (lam < 0).astype(float), (lam > 0).astype(float)
        ekin = -0.5 * np.real(np.sum(wa * np.einsum("ni,ij,nj->n", u.conj(), lap, u))
                              + np.sum(wb * np.einsum("ni,ij,nj->n", v.conj(), lap, v)))
        return ekin + e["E_pair"] + e["E_pot_ext"], e

    drift = []
    for dt, nst in ((0.004, 40), (0.002, 80)):
        phi = psi0.copy()
        hist = [np.zeros_like(phi) for _ in range(o.m)]
        hist = o.abm_init(phi, hist, dt, 1)
        E0, e0 = conserved_energy(phi)
        for _ in range(nst):
            hist = o.abm_step(phi, hist, dt)
        E1, e1 = conserved_energy(phi)
        flat = phi.reshape(2 * M, -1)
        gram = flat.conj() @ flat.T
        assert np.max(np.abs(gram - np.eye(2 * M))) < 1e-8
        assert abs(e1["N_a"] - e0["N_a"]) < 1e-9 * max(1, e0["N_a"]) and abs(e1["N_b"] - e0["N_b"]) < 1e-9 * max(1, e0["N_b"])
        assert abs(e1["E_pair"] - e0["E_pair"]) > 1e-5        # energy really flows between the terms
        assert relerr(phi, psi0) > 1e-4                       # the state really moved (initial Delta not self-consistent)
        drift.append(abs(E1 - E0) / abs(E0))
    assert drift[0] < 1e-6 and drift[1] < drift[0] / 8, drift   # integrator-level drift, shrinking like dt^p


# ------------------------------------------------ P16b: the mode multiplicity (Eqs. 29b-e; k_z list PAPER.md:889)
def test_p16_mode_multiplicity_folds_plus_minus_kz():
    """configs[2] keeps k_z >= 0 only and gives every k_z > 0 mode multiplicity 2 (R16).  A quasi-2D run with modes
    k_z = 0, k_1, k_2, k_3 of multiplicity 1, 2, 2, 2 must give the densities of the FULL 3-D lattice that holds the same
    in-plane spinors with e^{+i k_z z} AND e^{-i k_z z}: rho, tau, nu are even in k_z and j_x, j_y do not depend on it.
    A multiplicity that is dropped, squared or applied to the wrong mode fails this."""
    dims, dx = (8, 4, 8), (1.0, 1.1, 0.9)
    held = dims[:2]
    kz = wl.kgrid(dims[2], dx[2])[: dims[2] // 2]                 # 0, k_1, k_2, k_3 (no Nyquist member, R16/R17)
    mult = np.array([1.0] + [2.0] * (len(kz) - 1))
    per = 3
    nq = len(kz) * per
    psi_q = wl.random_spinors(161, nq, held, dV=np.prod(dx[:2]))
    wa, wb = wl.uniform01(162, 0, nq), wl.uniform01(163, 0, nq)
    f = random_fields(164, held)
    oq = make_fixed(held, dx, nq, 1, f, mode=2, full_dims=list(dims))
    oq.set_modes(np.stack([kz, 0 * kz], 1), mult, np.arange(len(kz) + 1) * per)
    oq.set_weights(wa, wb)
    oq.densities(psi_q)
    Lz = dims[2] * dx[2]
    z = np.arange(dims[2]) * dx[2]
    states, w3a, w3b = [], [], []
    for n in range(nq):
        k = kz[n // per]
        for sgn in ((1.0,) if k == 0 else (1.0, -1.0)):
            states.append(np.multiply.outer(psi_q[n], np.exp(1j * sgn * k * z)) / np.sqrt(Lz))
            w3a.append(wa[n]); w3b.append(wb[n])
    psi3 = np.ascontiguousarray(np.array(states))
    assert len(states) == per * (1 + 2 * (len(kz) - 1))
    f3 = {k: np.broadcast_to(v[..., None], dims).copy() for k, v in f.items()}
    o3 = make_fixed(dims, dx, len(states), 1, f3)
    o3.set_weights(np.array(w3a), np.array(w3b))
    o3.densities(psi3)
    for fld in ("rho_a", "rho_b", "tau_a", "tau_b", "nu", "ja_x", "ja_y", "jb_x", "jb_y"):
        assert relerr(oq.get_field(fld), o3.get_field(fld)[..., 0]) < 1e-12, fld
    assert np.abs(o3.get_field("ja_z")).max() < 1e-13 * np.abs(o3.get_field("ja_x")).max() + 1e-15    # +k_z and -k_z cancel


# ------------------------------------------------------------------- O8: the energy terms (Eqs. 33a, b, f PAPER.md:479-512)
def test_o8_kinetic_energy_is_the_expectation_value_of_the_kinetic_operator():
    """Eq. 33a (in-scope form, no current term): E_kin = int sum_sigma alpha_sigma tau_sigma / 2.  With first derivatives
    taken as in Eq. 26 (Nyquist dropped) summation by parts is exact, so for H = -1/2 sum_j d_j alpha d_j (DIVGRAD, U = mu =
    Delta = 0) E_kin = sum_n c_n [w^a_n <u|H_uu|u> + w^b_n <v|(-H_vv)|v>] -- evaluated through orc_apply_h, which the dense
    matrices of P5 pin, not through the density routine."""
    shape, dx = (8, 4, 8), (1.0, 0.9, 1.1)
    n = 7
    f = random_fields(171, shape)
    zero = np.zeros(shape)
    fields = dict(alpha_a=f["alpha_a"], alpha_b=f["alpha_b"], U_a=zero, U_b=zero, delta=zero.astype(complex))
    o = make_fixed(shape, dx, n, 2, fields, mu=(0.0, 0.0))
    wa, wb = wl.uniform01(172, 0, n), wl.uniform01(173, 0, n)
    o.set_weights(wa, wb)
    dV = float(np.prod(dx))
    psi = wl.random_spinors(174, n, shape, dV=dV)
    h, _ = o.apply_h(psi)
    eu = np.real(np.sum(psi[:, 0].conj() * h[:, 0], axis=(1, 2, 3))) * dV
    ev = np.real(np.sum(psi[:, 1].conj() * h[:, 1], axis=(1, 2, 3))) * dV
    o.densities(psi)
    e = o.energy()
    assert abs(e["E_kin"] - np.sum(wa * eu - wb * ev)) < 1e-12 * abs(e["E_kin"])
    assert e["E_kin"] > 0 and abs(e["E_pot"]) == 0 and abs(e["E_pair"]) < 1e-15


def test_o8_potential_energy_restores_the_normal_state_energy_of_eq_12b():
    """Eq. 12b is built so that a free Fermi sea (nu = 0, tau_sigma = (3/5)(6 pi^2 rho_sigma)^{2/3} rho_sigma) has the
    energy (3/5) rho eps_F 2^{2/3} (0.357 + 0.642 p^2): the alpha-dependent terms of E_kin (33a) and E_pot (33b)
    cancel.  That closed form pins E_pot once E_kin is pinned, at p = 0 and at finite polarisation."""
    shape, dx = (4, 4, 4), (1.0, 1.0, 1.0)
    V = float(np.prod(shape))
    for ra, rb in ((0.02, 0.02), (0.03, 0.01), (0.011, 0.027)):
        o = orc.Oracle(3, shape, dx, 1, func_id=2, kin_form=1)
        one = np.ones(shape)
        ta = 0.6 * (6 * np.pi ** 2 * ra) ** (2 / 3) * ra
        tb = 0.6 * (6 * np.pi ** 2 * rb) ** (2 / 3) * rb
        for name, v in (("rho_a", ra), ("rho_b", rb), ("tau_a", ta), ("tau_b", tb)):
            o.set_field(name, v * one)
        o.set_field("nu", 0j * one)
        o.update_potentials()
        e = o.energy()
        rho, p = ra + rb, (ra - rb) / (ra + rb)
        eF = 0.5 * (3 * np.pi ** 2 * rho) ** (2 / 3)
        want = 0.6 * rho * eF * 2 ** (2 / 3) * (0.357 + 0.642 * p * p) * V
        assert abs(e["E_kin"] + e["E_pot"] - want) < 1e-12 * want, (ra, rb)
        assert e["E_pot"] < 0 < e["E_kin"]


def test_o8_external_pairing_energy_is_the_response_of_eps_n_to_delta_ext():
    """Eq. 33f: E_pair.ext = -int (Delta_ext nu^* + h.c.).  Switching Delta_ext on changes <psi_n|H|psi_n> by
    2 Re int u_n^* Delta_ext v_n (Eq. 5), and nu = 1/2 sum (w^b - w^a) c_n u_n v_n^* (Eq. 7e), so
    E_pair.ext = -1/2 sum_n c_n (w^b_n - w^a_n) [eps_n(Delta_ext) - eps_n(0)] -- through orc_apply_h's eps_n."""
    shape, dx = (8, 4, 4), (1.0, 1.0, 1.2)
    n = 6
    M = int(np.prod(shape))
    dV = float(np.prod(dx))
    f = random_fields(181, shape)
    psi = wl.random_spinors(182, n, shape, dV=dV)
    wa, wb = wl.uniform01(183, 0, n), wl.uniform01(184, 0, n)
    dext = 0.3 * (wl.normal(185, 0, M) + 1j * wl.normal(186, 0, M)).reshape(shape)
    o = make_fixed(shape, dx, n, 1, f)
    o.set_weights(wa, wb)
    _, e0 = o.apply_h(psi)
    o.set_external(None, None, dext)
    _, e1 = o.apply_h(psi)
    o.densities(psi)
    e = o.energy()
    want = -0.5 * np.sum((wb - wa) * (e1 - e0))
    assert abs(e["E_pair_ext"] - want) < 1e-11 * abs(want) and abs(want) > 1e-5


# ------------------------------------------------------- O7: the midpoint rebuild of the starter (Eq. 53)
def test_o7_starter_rebuilds_the_potentials_at_the_midpoint():
    """Self-consistent BdG on 4x4x2 (Lambda_c static, so Delta(t) = -g_eff(r) nu(t) is the whole nonlinearity).  The
    starter's single step is exp(-i dt H[phi^(p)]) phi with H rebuilt from the half-step predictor phi^(p) (Eq. 53): a
    midpoint rule, local error O(dt^3).  Without that rebuild H would be the one of time t and the local error O(dt^2).
    Reference: the same nonlinear ODE written with the dense matrices of Eq. 28b and integrated by scipy's DOP853."""
    from scipy.integrate import solve_ivp
    shape, dx = (4, 4, 2), (1.0, 1.0, 1.0)
    M = int(np.prod(shape))
    mu = (0.6, 0.6)
    vext = 0.2 * wl.normal(191, 0, M).reshape(shape)
    delta0 = 0.3 + 0.05 * wl.normal(192, 0, M).reshape(shape)
    one = np.ones(shape)
    H0 = dense_h(shape, dx, one, one, vext, vext, delta0.astype(complex), mu, 0)
    lam, Vv = np.linalg.eigh(H0)
    psi0 = np.ascontiguousarray(Vv.T.reshape(2 * M, 2, *shape))
    wa, wb = (lam < 0).astype(float), (lam > 0).astype(float)

    def oracle(am):
        o = orc.Oracle(3, shape, dx, 2 * M, func_id=1, kin_form=0, four_pi_as=-6.0, ab_order=4, am_order=am,
                       subtract_mean_energy=0, normalize=0)
        o.set_mu(*mu); o.set_external(vext, vext); o.set_weights(wa, wb)
        return o

    o = oracle(5)
    o.densities(psi0); o.update_potentials()
    geff = o.get_field("g_eff").ravel()
    assert relerr(o.get_field("delta").ravel(), -geff * o.get_field("nu").ravel()) < 1e-13      # Eq. 10
    Hkin = dense_h(shape, dx, one, one, vext, vext, 0j * one, mu, 0)                              # everything but Delta

    def rhs(t, y):
        phi = y.reshape(2 * M, 2, M)
        u, v = phi[:, 0], phi[:, 1]
        nu = 0.5 * np.sum((wb - wa)[:, None] * u * v.conj(), axis=0)                              # Eq. 7e, dV = L_perp = 1
        d = -geff * nu
        hu = u @ Hkin[:M, :M].T + d[None] * v
        hv = d.conj()[None] * u + v @ Hkin[M:, M:].T
        return (-1j * np.stack([hu, hv], 1)).ravel()

    def starter_error(dt):
        oo = oracle(5)
        phi = psi0.copy()
        hist = [np.zeros_like(phi) for _ in range(oo.m)]
        oo.abm_init(phi, hist, dt, 1)                                                            # m - 1 = 3 starter steps
        ref = solve_ivp(rhs, (0.0, 3 * dt), psi0.ravel().astype(complex), method="DOP853", rtol=1e-12, atol=1e-14).y[:, -1]
        return np.max(np.abs(phi.ravel() - ref))

    e1, e2 = starter_error(0.02), starter_error(0.01)
    assert e1 > 1e-9                                             # far above rounding: the ratio below means something
    assert 6.0 < e1 / e2 < 10.0, (e1, e2)                        # dt^3 (8); a starter with H frozen at time t gives dt^2 (4)
