"""Pins of the oracle's current / velocity coupling: the term -(i/2){A_sigma - v_ext_sigma, grad} of
Eq. 4c, the current potential A_sigma = dE/dj_sigma and the j-terms of Eqs. 9b-c
 and of the energies 33a, d, g.  CPU only; numpy is the independent party."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl
from test_oracle_pins import d1_matrix, dense_h, random_fields, relerr


def _vel(seed, shape, amp=0.3):
    M = int(np.prod(shape))
    return amp * wl.normal(seed, 0, 3 * M).reshape(3, *shape)


def _fixed(shape, dx, n, kin_form, f, mu=(0.4, 0.3)):
    o = orc.Oracle(len(shape), shape, dx, n, func_id=0, kin_form=kin_form, current_terms=1)
    o.set_mu(*mu)
    o.set_potentials(**f)
    return o


@pytest.mark.parametrize("kin_form", [0, 1, 2])
@pytest.mark.parametrize("shape,dx", [((8, 4, 8), (1.0, 0.9, 1.1)), ((16, 8), (1.0, 1.2))])
def test_c1_current_term_keeps_h_hermitian(kin_form, shape, dx):
    """With a random (rough) real velocity field the discrete -(i/2)(W.D + D.W) is exactly Hermitian, because the
    first-derivative matrix of Eq. 28a is anti-Hermitian: <phi|H psi> = <H phi|psi> to rounding (DESIGN R27)."""
    f = random_fields(201, shape)
    o = _fixed(shape, dx, 2, kin_form, f)
    nd = len(shape)
    o.set_velocity(_vel(202, shape)[:nd], _vel(203, shape)[:nd])
    psi = wl.random_spinors(204, 2, shape, dV=float(np.prod(dx)))
    h, _ = o.apply_h(psi)
    a = np.vdot(psi[0], h[1])
    b = np.vdot(h[0], psi[1])
    assert abs(a - b) < 1e-12 * max(abs(a), 1.0)
    o0 = _fixed(shape, dx, 2, kin_form, f)                      # and the term is really there
    h0, _ = o0.apply_h(psi)
    assert relerr(h, h0) > 1e-2


def _axis_op(mat, a, shape):
    ops = [np.eye(s) for s in shape]
    ops[a] = mat
    out = ops[0]
    for q in ops[1:]:
        out = np.kron(out, q)
    return out


@pytest.mark.parametrize("kin_form", [0, 1, 2])
def test_c2_dense_matvec_with_velocity_field(kin_form):
    """Eq. 4b with h of Eq. 4c: block (u,u) gets C_a = -(i/2) sum_j (W_a,j D_j + D_j W_a,j), block (v,v) is -h_b^* and so
    gets -conj(C_b) = -(i/2) sum_j (W_b,j D_j + D_j W_b,j) as well; D_j from Eq. 28a, W = A - v_ext = -v_ext here."""
    shape, dx = (4, 8, 4), (1.0, 0.8, 1.1)
    M = int(np.prod(shape))
    f = random_fields(211, shape)
    mu = (0.4, 0.3)
    va, vb = _vel(212, shape), _vel(213, shape)
    H = dense_h(shape, dx, f["alpha_a"], f["alpha_b"], f["U_a"], f["U_b"], f["delta"], mu, kin_form).astype(complex)
    for blk, v in ((0, va), (1, vb)):
        C = np.zeros((M, M), dtype=complex)
        for a in range(3):
            D = _axis_op(d1_matrix(shape[a], dx[a]), a, shape)
            W = np.diag(-v[a].ravel())
            C += -0.5j * (W @ D + D @ W)
        H[blk * M:(blk + 1) * M, blk * M:(blk + 1) * M] += C
    assert np.max(np.abs(H - H.conj().T)) < 1e-12
    o = _fixed(shape, dx, 3, kin_form, f, mu)
    o.set_velocity(va, vb)
    psi = wl.random_spinors(214, 3, shape, dV=float(np.prod(dx)))
    h, e = o.apply_h(psi)
    ref = (H @ psi.reshape(3, 2 * M).T).T.reshape(psi.shape)
    assert relerr(h, ref) < 1e-12
    assert relerr(e, np.real(np.einsum("ni,ni->n", psi.reshape(3, -1).conj(), ref.reshape(3, -1))) * np.prod(dx)) < 1e-12


def _aslda(shape, dx, n, **kw):
    o = orc.Oracle(3, shape, dx, n, func_id=2, kin_form=1, current_terms=1, **kw)
    o.set_mu(0.5, 0.4)
    return o


def test_c3_galilean_boost_of_the_energy():
    """Eqs. 9b + 9c are Galilean covariant: boosting every u_n by e^{iq.r} and every v_n by e^{-iq.r} leaves rho, p and
    alpha alone, turns j_sigma into j_sigma + q rho_sigma, tau_sigma into tau_sigma + 2 q.j_sigma + q^2 rho_sigma, and
    must change the energy by q.J + q^2 N / 2 exactly -- only if the (1 - alpha) j^2 / 2 rho terms are there with the
    right sign and weight (alpha != 1: a polarised ASLDA state).  Band-limited spinors keep every product alias-free."""
    shape, dx = (16, 8, 8), (1.0, 1.0, 1.0)
    n = 6
    dV, V = 1.0, float(np.prod(shape))
    rng_u = wl.normal(221, 0, 2 * n * 2 * 27).reshape(n, 2, 3, 3, 3, 2)
    k = [wl.kgrid(s, 1.0) for s in shape]
    x = [np.arange(s) * 1.0 for s in shape]
    psi = np.zeros((n, 2) + shape, dtype=complex)
    for a in range(3):
        for b in range(3):
            for c in range(3):                                  # modes -1, 0, 1 on every axis
                ph = np.multiply.outer(np.multiply.outer(np.exp(1j * k[0][a - 1] * x[0]), np.exp(1j * k[1][b - 1] * x[1])),
                                       np.exp(1j * k[2][c - 1] * x[2]))
                psi += (rng_u[:, :, a, b, c, 0] + 1j * rng_u[:, :, a, b, c, 1])[:, :, None, None, None] * ph
    psi /= np.sqrt(np.sum(np.abs(psi) ** 2, axis=(1, 2, 3, 4), keepdims=True) * dV)
    wa, wb = 0.2 + 0.8 * wl.uniform01(222, 0, n), 0.1 + 0.3 * wl.uniform01(223, 0, n)      # rho_a != rho_b: alpha != 1
    q = np.array([k[0][2], k[1][1], -k[2][1]])
    boost = np.exp(1j * (np.multiply.outer(np.multiply.outer(q[0] * x[0], np.ones(shape[1])), np.ones(shape[2]))
                         + np.multiply.outer(np.multiply.outer(np.ones(shape[0]), q[1] * x[1]), np.ones(shape[2]))
                         + np.multiply.outer(np.multiply.outer(np.ones(shape[0]), np.ones(shape[1])), q[2] * x[2])))
    psi_b = psi.copy()
    psi_b[:, 0] *= boost
    psi_b[:, 1] *= boost.conj()
    res = []
    for s in (psi, psi_b):
        o = _aslda(shape, dx, n)
        o.set_weights(wa, wb)
        o.densities(s)
        o.update_potentials()
        res.append((o.energy(), {f: o.get_field(f) for f in ("rho_a", "rho_b", "ja_x", "ja_y", "ja_z", "jb_x", "jb_y", "jb_z",
                                                              "alpha_a", "alpha_b", "Aa_x", "Ab_y")}))
    (e0, f0), (e1, f1) = res
    assert relerr(f1["rho_a"], f0["rho_a"]) < 1e-12 and relerr(f1["alpha_a"], f0["alpha_a"]) < 1e-12
    assert relerr(f1["ja_x"], f0["ja_x"] + q[0] * f0["rho_a"]) < 1e-11 and relerr(f1["jb_z"], f0["jb_z"] + q[2] * f0["rho_b"]) < 1e-11
    assert np.abs(f0["alpha_a"] - 1).mean() > 0.02              # the (1 - alpha) terms carry weight
    J = sum(q[d] * (f0["ja_" + "xyz"[d]].sum() + f0["jb_" + "xyz"[d]].sum()) for d in range(3)) * dV
    N = e0["N_a"] + e0["N_b"]
    kin0 = e0["E_kin"] + e0["E_curr"]
    kin1 = e1["E_kin"] + e1["E_curr"]
    assert abs((kin1 - kin0) - (J + 0.5 * q @ q * N)) < 1e-10 * abs(kin1)
    assert abs(e1["E_pot"] - e0["E_pot"]) < 1e-12 * abs(e0["E_pot"])
    # the current potential follows A = (1 - alpha) j / rho (PAPER.md:148 with Eqs. 9b-c)
    assert relerr(f1["Aa_x"], (1 - f1["alpha_a"]) * f1["ja_x"] / f1["rho_a"]) < 1e-12
    assert relerr(f1["Ab_y"], (1 - f1["alpha_b"]) * f1["jb_y"] / f1["rho_b"]) < 1e-12


def test_c4_potentials_are_derivatives_of_the_energy_density_with_currents():
    """V_sigma = dE/drho_sigma and A_sigma = dE/dj_sigma by centred finite differences of the
    oracle's energy density at fixed tau, nu, frozen Lambda_c, for polarised densities with currents."""
    o = _aslda((4, 4, 4), (1.0, 1.0, 1.0), 1)
    ra, rb, ta, tb, nu = 0.031, 0.017, 0.021, 0.009, 0.004 + 0.002j
    ja, jb = np.array([0.004, -0.002, 0.001]), np.array([-0.001, 0.003, 0.002])
    base = o.functional_point(ra, rb, ta, tb, nu, j_a=ja, j_b=jb)
    lam = base["lambda_c"]

    def E(ra_=ra, rb_=rb, ja_=ja, jb_=jb):
        return o.functional_point(ra_, rb_, ta, tb, nu, lambda_in=lam, j_a=ja_, j_b=jb_)["edens"]

    ref = o.functional_point(ra, rb, ta, tb, nu, lambda_in=lam, j_a=ja, j_b=jb)
    h = 1e-6
    # g_eff depends on rho through rho^(1/3)/C: the pairing part of V is -|Delta|^2/(3 C rho^(2/3)) (P14); the j-part is new
    Va = (E(ra_=ra + h) - E(ra_=ra - h)) / (2 * h)
    Vb = (E(rb_=rb + h) - E(rb_=rb - h)) / (2 * h)
    assert abs(Va - ref["V_a"]) < 2e-7 * abs(ref["V_a"]) and abs(Vb - ref["V_b"]) < 2e-7 * abs(ref["V_b"])
    for d in range(3):
        e = np.zeros(3); e[d] = 1e-6
        Aa = (E(ja_=ja + e) - E(ja_=ja - e)) / 2e-6
        Ab = (E(jb_=jb + e) - E(jb_=jb - e)) / 2e-6
        assert abs(Aa - ref["A_a"][d]) < 1e-8 * np.abs(ref["A_a"]).max() + 1e-12
        assert abs(Ab - ref["A_b"][d]) < 1e-8 * np.abs(ref["A_b"]).max() + 1e-12
    # and the j-terms are not a rounding matter: without currents V differs visibly
    o0 = orc.Oracle(3, (4, 4, 4), (1.0, 1.0, 1.0), 1, func_id=2, kin_form=1)
    o0.set_mu(0.5, 0.4)
    v0 = o0.functional_point(ra, rb, ta, tb, nu, lambda_in=lam)
    assert abs(v0["V_a"] - ref["V_a"]) > 1e-5 * abs(ref["V_a"])


def test_c5_bdg_has_no_current_coupling_and_flow_energies():
    """alpha = 1 (BdG): A = 0 and E_0's -j^2/rho cancels E_CM inside the functional (Eqs. 9b, 9c), while the reported
    E_kin (33a) and E_curr (33d) move j^2/2rho between them; E_vel.ext = -int v.j (33g)."""
    shape, dx = (8, 4, 4), (1.0, 1.0, 1.0)
    n = 4
    o = orc.Oracle(3, shape, dx, n, func_id=1, kin_form=0, four_pi_as=-4.0, current_terms=1)
    o.set_mu(0.5, 0.5)
    va, vb = _vel(231, shape, 0.1), _vel(232, shape, 0.1)
    o.set_velocity(va, vb)
    psi = wl.random_spinors(233, n, shape)
    wa, wb = wl.uniform01(234, 0, n), wl.uniform01(235, 0, n)
    o.set_weights(wa, wb)
    o.densities(psi)
    o.update_potentials()
    for f in ("Aa_x", "Aa_z", "Ab_y"):
        assert np.abs(o.get_field(f)).max() == 0.0
    e = o.energy()
    fld = {f: o.get_field(f) for f in ("rho_a", "rho_b", "tau_a", "tau_b", "ja_x", "ja_y", "ja_z", "jb_x", "jb_y", "jb_z")}
    ja2 = sum(fld["ja_" + c] ** 2 for c in "xyz"); jb2 = sum(fld["jb_" + c] ** 2 for c in "xyz")
    assert abs(e["E_kin"] + e["E_curr"] - 0.5 * (fld["tau_a"] + fld["tau_b"]).sum()) < 1e-12 * abs(e["E_kin"])
    assert abs(e["E_curr"] - 0.5 * (ja2 / fld["rho_a"] + jb2 / fld["rho_b"]).sum()) < 1e-12 * e["E_curr"]
    want = -sum((va[d] * fld["ja_" + "xyz"[d]] + vb[d] * fld["jb_" + "xyz"[d]]).sum() for d in range(3))
    assert abs(e["E_vel_ext"] - want) < 1e-12 * abs(want)
