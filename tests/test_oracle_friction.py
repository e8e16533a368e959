"""Pins of the oracle's quantum-friction terms: V^(d) = -(alpha_qf / rho_0) div j (Eq. 66),
Delta^(d) = Delta [beta_qf sin(theta_nu - theta_B') + i gamma_qf (N - N_req) / N_req] (Eqs. 67-70).
CPU only; the independent routes go through orc_apply_h (pinned by dense matrices) and through physics."""
import numpy as np

import oracle as orc
import workloads as wl
from test_oracle_pins import relerr


def _band_limited(seed, n, shape, kmax=1):
    """Spinors with Fourier content |index| <= kmax on every axis: products of two of them stay below Nyquist."""
    k = [np.fft.fftfreq(s) * s for s in shape]
    mask = np.ones(shape, dtype=bool)
    for a, kk in enumerate(k):
        sh = [1] * len(shape); sh[a] = -1
        mask &= (np.abs(kk) <= kmax).reshape(sh)
    z = (wl.normal(seed, 0, 2 * n * 2 * int(np.prod(shape))).reshape(2, n, 2, *shape))
    f = (z[0] + 1j * z[1]) * mask
    psi = np.fft.ifftn(f, axes=tuple(range(2, 2 + len(shape))))
    psi /= np.sqrt(np.sum(np.abs(psi) ** 2, axis=tuple(range(1, 2 + len(shape))), keepdims=True))
    return np.ascontiguousarray(psi)


def _bdg(shape, n, **kw):
    o = orc.Oracle(3, shape, (1.0, 1.0, 1.0), n, func_id=1, kin_form=0, four_pi_as=-4.0, **kw)
    o.set_mu(0.5, 0.5)
    return o


def test_q1_dissipative_mean_field_is_minus_the_density_rate():
    """Continuity: with a real local potential and no pairing, d rho_sigma / dt = -div j_sigma, and d|u|^2/dt =
    2 Im(u^* (H psi)_u), d|v|^2/dt = 2 Im(v^* (H psi)_v) (Eq. 15).  So div j_a = -sum_n c w^a 2 Im(u^* Hu) and
    div j_b = -sum_n c w^b 2 Im(v^* Hv), from orc_apply_h on band-limited spinors (exact on the lattice) -- which
    fixes the divergence, its sign and the prefactor -alpha_qf / rho_0 of Eq. 66."""
    shape = (8, 8, 8)
    n = 5
    psi = _band_limited(301, n, shape)
    wa, wb = wl.uniform01(302, 0, n), wl.uniform01(303, 0, n)
    fixed = orc.Oracle(3, shape, (1.0, 1.0, 1.0), n, func_id=0, kin_form=0)
    one = np.ones(shape)
    fixed.set_potentials(one, one, 0 * one, 0 * one, 0j * one)          # H = diag(-lap/2, +lap/2)
    h, _ = fixed.apply_h(psi)
    rate_a = np.sum(wa[:, None, None, None] * 2 * np.imag(psi[:, 0].conj() * h[:, 0]), axis=0)
    rate_b = np.sum(wb[:, None, None, None] * 2 * np.imag(psi[:, 1].conj() * h[:, 1]), axis=0)
    aq, r0 = 7.0, 0.013
    res = []
    for qf in (0, 1):
        o = _bdg(shape, n, quantum_friction=qf, qf_alpha=aq, qf_rho0=r0, qf_nreq=1.0)
        o.set_weights(wa, wb)
        o.densities(psi)
        o.update_potentials()
        res.append((o.get_field("V_a"), o.get_field("V_b"), o.get_field("U_a")))
    dVa, dVb = res[1][0] - res[0][0], res[1][1] - res[0][1]
    assert relerr(dVa, (aq / r0) * rate_a) < 1e-11 and relerr(dVb, (aq / r0) * rate_b) < 1e-11
    assert relerr(res[1][2] - res[0][2], dVa) < 1e-13 and np.abs(dVa).max() > 1e-6


def test_q2_kinetic_anomalous_density_through_apply_h():
    """Eq. 68: B' = -1/2 sum_n [u lap v^* + v^* lap u] with the weights of nu (R29).  With H = diag(-lap/2, +lap/2):
    lap u = -2 (H psi)_u and lap v = +2 (H psi)_v, hence B' = sum_n wn [v^* (H psi)_u - u conj((H psi)_v)]."""
    shape = (8, 4, 8)
    n = 6
    psi = wl.random_spinors(311, n, shape)
    wa, wb = wl.uniform01(312, 0, n), wl.uniform01(313, 0, n)
    fixed = orc.Oracle(3, shape, (1.0, 1.0, 1.0), n, func_id=0, kin_form=0)
    one = np.ones(shape)
    fixed.set_potentials(one, one, 0 * one, 0 * one, 0j * one)
    h, _ = fixed.apply_h(psi)
    wn = (0.5 * (wb - wa))[:, None, None, None]
    want = np.sum(wn * (psi[:, 1].conj() * h[:, 0] - psi[:, 0] * h[:, 1].conj()), axis=0)
    fixed.set_weights(wa, wb)
    fixed.densities(psi)
    assert relerr(fixed.get_field("bp"), want) < 1e-12
    fixed.densities(psi[:3], 0, 3); fixed.densities(psi, 3, 3, accumulate=1)      # accumulates like every density
    assert relerr(fixed.get_field("bp"), want) < 1e-12


def _uniform_state(shape, mu, delta0):
    """Plane-wave BCS spinors of the uniform solution (positive branch), real positive u, v (times e^{ik.r})."""
    k = [wl.kgrid(s, 1.0) for s in shape]
    K = np.stack(np.meshgrid(*k, indexing="ij"), 0).reshape(3, -1)
    eps = 0.5 * np.sum(K ** 2, 0) - mu
    E = np.sqrt(eps ** 2 + delta0 ** 2)
    r = np.stack(np.meshgrid(*[np.arange(s) for s in shape], indexing="ij"), 0).reshape(3, -1)
    ph = np.exp(1j * K.T @ r) / np.sqrt(r.shape[1])
    u = np.sqrt(0.5 * (1 + eps / E))[:, None] * ph
    v = np.sqrt(0.5 * (1 - eps / E))[:, None] * ph
    return np.ascontiguousarray(np.stack([u, v], 1).reshape(-1, 2, *shape)), E


def test_q3_equilibrium_feels_no_friction():
    """In the uniform paired state j = 0 and nu, B' have the same phase (both sum_k k-even positive weights times u v),
    so with N_req = N every dissipative term vanishes: the potentials are those of the friction-free functional."""
    shape = (4, 4, 4)
    psi, E = _uniform_state(shape, 0.5, 0.3)
    n = psi.shape[0]
    res = []
    for qf in (0, 1):
        o = _bdg(shape, n, quantum_friction=qf, qf_alpha=8.0, qf_beta=5.0, qf_gamma=0.1, qf_rho0=0.05, qf_nreq=1.0,
                 spin_symmetric=1)
        o.set_weights(np.zeros(n), np.ones(n))
        o.densities(psi)
        if qf:
            o2 = _bdg(shape, n, quantum_friction=1, qf_alpha=8.0, qf_beta=5.0, qf_gamma=0.1, qf_rho0=0.05,
                      qf_nreq=res[0][2], spin_symmetric=1)
            o2.set_weights(np.zeros(n), np.ones(n)); o2.densities(psi); o = o2
        o.update_potentials()
        e = o.energy()
        res.append((o.get_field("delta"), o.get_field("V_a"), e["N_a"] + e["N_b"], o.get_field("bp"), o.get_field("nu")))
    assert relerr(res[1][0], res[0][0]) < 1e-12 and np.abs(res[1][1] - res[0][1]).max() < 1e-12
    bp, nu = res[1][3], res[1][4]
    assert np.all(bp.real > 0) and np.all(nu.real > 0) and np.abs(bp.imag).max() < 1e-14 and np.abs(nu.imag).max() < 1e-14


def test_q4_particle_number_term_of_eq_70():
    """beta_qf = 0: Delta^(d) / Delta = i gamma_qf (N - N_req) / N_req at every point, N = int (rho_a + rho_b)."""
    shape = (4, 4, 4)
    n = 5
    psi = wl.random_spinors(331, n, shape)
    wa, wb = wl.uniform01(332, 0, n), wl.uniform01(333, 0, n)
    N = float(np.sum(wa[:, None, None, None] * np.abs(psi[:, 0]) ** 2 + wb[:, None, None, None] * np.abs(psi[:, 1]) ** 2))
    d = []
    for qf in (0, 1):
        o = _bdg(shape, n, quantum_friction=qf, qf_gamma=0.1, qf_nreq=0.8 * N, qf_rho0=1.0)
        o.set_weights(wa, wb); o.densities(psi); o.update_potentials()
        d.append(o.get_field("delta"))
    ratio = (d[1] - d[0]) / d[0]
    assert np.abs(ratio - 1j * 0.1 * (N - 0.8 * N) / (0.8 * N)).max() < 1e-12


def test_q5_friction_lowers_the_energy_of_a_sloshing_cloud():
    """The point of Eq. 66: with currents present the total energy decreases, while the same run
    without friction conserves it.  Self-consistent BdG, full basis, a state kicked into motion."""
    from test_oracle_pins import dense_h
    shape, dx = (4, 4, 2), (1.0, 1.0, 1.0)
    M = int(np.prod(shape))
    mu = (0.6, 0.6)
    vext = 0.3 * np.cos(2 * np.pi * np.arange(4) / 4)[:, None, None] * np.ones(shape)
    one = np.ones(shape)
    H = dense_h(shape, dx, one, one, vext, vext, (0.3 * one).astype(complex), mu, 0)
    lam, V = np.linalg.eigh(H)
    psi0 = np.ascontiguousarray(V.T.reshape(2 * M, 2, *shape))
    kick = np.exp(1j * 2 * np.pi * np.arange(4) / 4)[:, None, None] * np.ones(shape)     # a boost along x
    psi0[:, 0] *= kick; psi0[:, 1] *= kick.conj()
    lap = -2.0 * dense_h(shape, dx, one, one, 0 * one, 0 * one, 0j * one, (0.0, 0.0), 0)[:M, :M]
    wa, wb = (lam < 0).astype(float), (lam > 0).astype(float)

    def energy(o, phi):
        o.densities(phi); o.update_potentials()
        e = o.energy()
        u, v = phi[:, 0].reshape(2 * M, M), phi[:, 1].reshape(2 * M, M)
        ekin = -0.5 * np.real(np.sum(wa * np.einsum("ni,ij,nj->n", u.conj(), lap, u)) + np.sum(wb * np.einsum("ni,ij,nj->n", v.conj(), lap, v)))
        return ekin + e["E_pair"] + e["E_pot_ext"], e["N_a"] + e["N_b"]

    out = []
    for qf in (0, 1):
        o = orc.Oracle(3, shape, dx, 2 * M, func_id=1, kin_form=0, four_pi_as=-6.0, ab_order=4, am_order=5, normalize=0,
                       quantum_friction=qf, qf_alpha=6.0, qf_rho0=1.0, qf_nreq=1.0)
        o.set_mu(*mu); o.set_external(vext, vext); o.set_weights(wa, wb)
        phi = psi0.copy()
        hist = [np.zeros_like(phi) for _ in range(o.m)]
        hist = o.abm_init(phi, hist, 0.004, 1)
        probe = orc.Oracle(3, shape, dx, 2 * M, func_id=1, kin_form=0, four_pi_as=-6.0)      # friction-free energy meter
        probe.set_mu(*mu); probe.set_external(vext, vext); probe.set_weights(wa, wb)
        E0, N0 = energy(probe, phi)
        for _ in range(60):
            hist = o.abm_step(phi, hist, 0.004)
        E1, N1 = energy(probe, phi)
        out.append((E0, E1, N0, N1))
    (a0, a1, _, _), (b0, b1, n0, n1) = out
    assert abs(a1 - a0) < 1e-6 * abs(a0)                        # conservative run: energy stays
    assert b1 < b0 - 1e-4 * abs(b0)                             # dissipative run: energy goes down, visibly
    assert abs(n1 - n0) < 1e-8 * n0                             # a real potential cannot change the particle number
