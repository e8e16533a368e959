"""GPU-vs-oracle parity through the C-ABI (run with -m gpu on a B200).

Tolerances are north_star's: one H-apply 1e-12, densities 1e-11, 100 ABM steps 1e-9, all as
max|x - ref| / max|ref| over the returned array.
"""
import numpy as np
import pytest

import paper_2602_08982_b200 as ws
import workloads as wl
from harness import make_gpu, make_oracle, relerr, to_gpu, to_np

pytestmark = pytest.mark.gpu

TOL_H, TOL_D, TOL_ABM = 1e-12, 1e-11, 1e-9
DENS = ["rho_a", "rho_b", "tau_a", "tau_b", "nu", "ja_x", "ja_y", "ja_z", "jb_x", "jb_y", "jb_z"]
POTS = ["alpha_a", "alpha_b", "V_a", "V_b", "U_a", "U_b", "delta", "lambda_c", "g_eff", "lap_alpha_a", "lap_alpha_b"]


def random_fields(seed, shape):
    M = int(np.prod(shape))
    z = wl.normal(seed, 0, 6 * M).reshape(6, *shape)
    return dict(alpha_a=1.1 + 0.2 * np.tanh(z[0]), alpha_b=0.9 + 0.2 * np.tanh(z[1]), U_a=0.3 * z[2], U_b=0.3 * z[3],
                delta=0.2 + 0.1 * (z[4] + 1j * z[5]))


def generic(shape, dx, n_wf, kin_form, func_id=0, seed=5, n_modes=1, full_dims=None, **kw):
    """A small random workload on an arbitrary lattice (fixed random fields, random weights, random modes)."""
    mode = len(shape)
    dims = tuple(shape) + (1,) * (3 - mode) if full_dims is None else full_dims
    dxs = tuple(dx) + (1.0,) * (3 - mode)
    u = wl.uniform01(seed + 1, 0, 2 * n_wf)
    base = dict(ab_order=4, am_order=5, dt=0.004, n_steps=10, mu=(0.4, 0.3))
    base.update(kw)
    w = wl.Workload(f"generic{shape}", mode, dims, dxs, n_wf, func_id, base.pop("force_a1", 0),
                    base.pop("spin_symmetric", 0), kin_form, base.pop("ab_order"), base.pop("am_order"), base.pop("dt"),
                    base.pop("n_steps"), base.pop("mu"), w_a=u[:n_wf], w_b=u[n_wf:], **base)
    if func_id == 0:
        w.fixed = random_fields(seed + 2, shape)
    if n_modes > 1 or mode < 3:
        n_modes = max(n_modes, 1)
        kp = 0.3 * wl.normal(seed + 3, 0, 2 * n_modes).reshape(n_modes, 2)
        if mode == 2:
            kp[:, 1] = 0.0
        w.kperp, w.mult = kp, 1.0 + np.arange(n_modes) % 2
        w.first = np.linspace(0, n_wf, n_modes + 1).astype(np.int64)
    return w


def spinors(w, seed=9):
    return wl.random_spinors(seed, w.n_wf, w.shape, w.dV)


SHAPES = [((8, 4, 8), (1.0, 0.9, 1.1)), ((16, 8), (1.0, 1.2)), ((32,), (0.8,)), ((2, 2, 4), (1.0, 1.0, 1.0)),
          ((32, 16, 16), (1.0, 1.0, 0.9)),      # 8192 points: the multi-pass (large lattice) regime
          ((128, 64), (1.0, 1.1)),              # 2-D lattice in the large regime
          ((8, 32, 32), (1.0, 1.1, 0.9)),       # Ny = Nz = 32: the fused register-FFT path (fast3d.cuh)
          ((16, 32, 32), (0.9, 1.0, 1.0))]


@pytest.mark.parametrize("kin_form", [0, 1, 2])
@pytest.mark.parametrize("shape,dx", SHAPES)
def test_apply_h_matches_oracle(shape, dx, kin_form):
    n_wf = 7 if np.prod(shape) > 4096 else 19            # ragged against every chunk / group size
    w = generic(shape, dx, n_wf, kin_form, n_modes=3)
    psi = spinors(w)
    o, g = make_oracle(w), make_gpu(w)
    ref, eref = o.apply_h(psi)
    h, e = g.apply_h(to_gpu(psi))
    assert relerr(to_np(h), ref) < TOL_H
    assert relerr(to_np(e), eref) < TOL_H
    # sub-range call leaves the other spinors untouched
    h2, _ = g.apply_h(to_gpu(psi), n_first=2, n_count=3)
    h2 = to_np(h2)
    assert relerr(h2[2:5], ref[2:5]) < TOL_H and not h2[:2].any() and not h2[5:].any()


@pytest.mark.parametrize("shape,dx", SHAPES)
@pytest.mark.parametrize("sym", [0, 1])
def test_densities_match_oracle(shape, dx, sym):
    n_wf = 9 if np.prod(shape) > 4096 else 37
    w = generic(shape, dx, n_wf, 0, n_modes=4, spin_symmetric=sym)
    psi = spinors(w)
    o, g = make_oracle(w), make_gpu(w)
    o.densities(psi)
    gp = to_gpu(psi)
    g.densities(gp)
    names = DENS[:5] + [f"j{s}_{'xyz'[d]}" for s in "ab" for d in range(len(shape))]
    for name in names:
        assert relerr(to_np(g.get_field(name)), o.get_field(name)) < TOL_D, name
    # batch streaming: two accumulating calls give the same sums
    g.densities(gp, 0, 4, accumulate=0)
    g.densities(gp, 4, n_wf - 4, accumulate=1)
    for name in names:
        assert relerr(to_np(g.get_field(name)), o.get_field(name)) < TOL_D, name


@pytest.mark.parametrize("func_id,force_a1,sym", [(1, 0, 0), (2, 0, 0), (2, 1, 0), (2, 0, 1), (2, 1, 1)])
@pytest.mark.parametrize("kin_form", [0, 1])
def test_potentials_match_oracle(func_id, force_a1, sym, kin_form):
    shape, dx = (8, 8, 4), (1.0, 1.0, 1.0)
    n_wf = 64
    w = generic(shape, dx, n_wf, kin_form, func_id=func_id, force_a1=force_a1, spin_symmetric=sym, mu=(0.5, 0.35))
    X = np.meshgrid(*[np.arange(s) - s // 2 for s in shape], indexing="ij")
    w.vext_a = 0.02 * sum(x * x for x in X).astype(float)
    w.vext_b = w.vext_a * 1.1
    # realistic density scale: 64 spinors on 256 points, weights of order one, times 1/dV
    psi = spinors(w) * 1.5
    o, g = make_oracle(w), make_gpu(w)
    o.densities(psi); o.update_potentials()
    g.densities(to_gpu(psi)); g.update_potentials()
    for name in POTS:
        if name.startswith("lap_alpha") and kin_form != 1:
            continue                      # lap(alpha) is only built (and consumed) by the Eq. 40 form
        ref = o.get_field(name)
        got = to_np(g.get_field(name))
        scale = max(np.max(np.abs(ref)), 1e-300)
        assert np.max(np.abs(got - ref)) / scale < TOL_D or np.max(np.abs(got - ref)) < 1e-13, name
    # frozen Lambda_c: second update with lambda_mode = 1 reuses the field
    o2, g2 = make_oracle(w, lambda_mode=1), make_gpu(w, lambda_mode=1)
    lam = np.abs(wl.normal(3, 0, int(np.prod(shape)))).reshape(shape) * 0.05
    o2.set_field("lambda_c", lam); g2.set_field("lambda_c", lam)
    o2.densities(psi); o2.update_potentials()
    g2.densities(to_gpu(psi)); g2.update_potentials()
    assert relerr(to_np(g2.get_field("delta")), o2.get_field("delta")) < TOL_D
    assert relerr(to_np(g2.get_field("lambda_c")), lam) == 0.0


def run_both(w, psi0, n_steps, selfstart=1, n_wf=None):
    """abm_init + n_steps abm_steps on both sides; returns (phi_gpu, phi_oracle, f0_gpu, f0_oracle, o, g)."""
    import torch
    o, g = make_oracle(w, n_wf), make_gpu(w, n_wf)
    phi_o = psi0.copy()
    hist_o = [np.zeros_like(psi0) for _ in range(o.m)]
    phi_g = to_gpu(psi0)
    hist_g = [torch.zeros_like(phi_g) for _ in range(g.m)]
    assert g.m == o.m
    hist_o = o.abm_init(phi_o, hist_o, w.dt, selfstart)
    hist_g = g.abm_init(phi_g, hist_g, w.dt, selfstart)
    for _ in range(n_steps):
        hist_o = o.abm_step(phi_o, hist_o, w.dt)
        hist_g = g.abm_step(phi_g, hist_g, w.dt)
    return to_np(phi_g), phi_o, to_np(hist_g[0]), hist_o[0], o, g


def test_cfg1_100_steps_bdg_8cubed():
    """configs[0]: full basis of 1024 spinors on 8^3, AB4AM4, 100 steps (3 Taylor + 97 ABM), fixed potentials."""
    w = wl.cfg1()
    psi0 = w.spinors()
    pg, po, fg, fo, o, g = run_both(w, psi0, w.n_steps - (w.history - 1))
    assert relerr(pg, po) < TOL_ABM
    assert relerr(fg, fo) < TOL_ABM


@pytest.mark.parametrize("ab,am", [(3, 4), (4, 4), (4, 5), (5, 5)])
@pytest.mark.parametrize("selfstart,normalize,shift", [(1, 1, 1), (0, 1, 1), (1, 0, 0), (1, 1, 0)])
def test_abm_fixed_potentials_all_orders(ab, am, selfstart, normalize, shift):
    w = generic((8, 4, 8), (1.0, 0.9, 1.1), 21, 1, ab_order=ab, am_order=am, normalize=normalize,
                subtract_mean_energy=shift, dt=0.004)
    pg, po, fg, fo, _, _ = run_both(w, spinors(w), 12, selfstart)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4_sym40", "cfg4_divgrad", "bdg_large", "aslda_polarised"])
def test_abm_selfconsistent_reduced_configs(name):
    """Self-consistent stepping on reduced versions of configs[1..3] (same recipes, fewer modes / points)."""
    if name == "cfg2":
        w = wl.cfg2(n_modes_side=4, nx=32, n_steps=20)              # 16 modes x 64 spinors, quasi-1D
    elif name == "cfg3":
        w = wl.cfg3(n_side=16, n_kz=3, nz=8, n_steps=20)            # 3 kz x 256 spinors, quasi-2D, vortex
    elif name == "cfg4_sym40":
        w = wl.cfg4(n_side=8, kin_form=1, n_steps=20)               # 256 spinors on 8^3, trap, general alpha
    elif name == "cfg4_divgrad":
        w = wl.cfg4(n_side=8, kin_form=2, n_steps=20)
    elif name == "bdg_large":
        w = generic((32, 16, 16), (1.0, 1.0, 1.0), 24, 0, func_id=1, four_pi_as=-2.0, dt=0.005)
        w.n_steps = 6
    else:
        w = generic((8, 8, 8), (1.0, 1.0, 1.0), 96, 1, func_id=2, mu=(0.5, 0.3), dt=0.005)
        w.n_steps = 12
    psi0 = w.spinors() if w.kidx is not None else spinors(w)
    pg, po, fg, fo, o, g = run_both(w, psi0, w.n_steps)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    for f in ("delta", "U_a", "U_b", "alpha_a"):
        assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-8, f


def test_run_to_run_bit_reproducible():
    w = wl.cfg3(n_side=16, n_kz=2, nz=8, n_steps=5)
    psi0 = w.spinors()
    a = run_both(w, psi0, 5)[0]
    b = run_both(w, psi0, 5)[0]
    assert np.array_equal(a, b)


# ---- the fused 3-D path (Ny = Nz = 32): ragged chunks over several concurrent streams ---------------------------
SMALL = dict(fused_chunk=3, fused_streams=3, group=3)     # ragged last chunk / group, more groups than ring slots


@pytest.fixture
def tuning():
    """tuning(**fields): process-wide wslda_set_tuning for the contexts the test creates; defaults restored afterwards."""
    yield ws.set_tuning
    ws.set_tuning()


@pytest.fixture
def small_fast_chunks(tuning):
    tuning(**SMALL)


@pytest.mark.parametrize("kin_form", [0, 1])
@pytest.mark.parametrize("nx", [8, 32])
def test_fast3d_apply_h_ragged_chunks(small_fast_chunks, nx, kin_form):
    w = generic((nx, 32, 32), (1.0, 0.95, 1.05), 11, kin_form, n_modes=2)
    psi = spinors(w)
    o, g = make_oracle(w), make_gpu(w)
    ref, eref = o.apply_h(psi)
    h, e = g.apply_h(to_gpu(psi))
    assert relerr(to_np(h), ref) < TOL_H and relerr(to_np(e), eref) < TOL_H
    assert any(k.startswith("k_f3") for k in _kernels_of(g, lambda: g.apply_h(to_gpu(psi))))


def _kernels_of(g, fn):
    g.profile(True)
    fn()
    rep = g.profile_report()
    g.profile(False)
    return list(rep)


def test_fast3d_multikernel_fallback(tuning):
    """disable_persistent: the three-pass chunk pipeline on concurrent streams (fast3d.cuh kernels) instead of the persistent kernel."""
    tuning(disable_persistent=1, **SMALL)
    w = wl.cfg4(n_side=32, n_wf=10, kin_form=1, n_steps=3)
    psi0 = w.spinors()
    pg, po, fg, fo, o, g = run_both(w, psi0, w.n_steps)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    assert "k_f3_pass_c" in _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))


@pytest.mark.parametrize("sep,pm,em", [("0", 0, 0), ("1", 1, 1), ("1", 8, 4), ("1", 2, 2)])
def test_axis_by_axis_stage_kernel_32cubed(tuning, sep, pm, em):
    """The default 32^3 Eq. 40 stage kernels (mega3s.cuh: Laplacian axis by axis) for several item sizes, ragged groups
    of 3 spinors, and the three-pass kernels they replace (disable_axis_split): H psi and self-consistent steps."""
    tuning(disable_axis_split=int(sep == "0"), dmma_stage=-1, p_planes=pm, x_rows=em, **SMALL)
    w = wl.cfg4(n_side=32, n_wf=10, kin_form=1, n_steps=3)
    psi0 = w.spinors()
    o, g = make_oracle(w), make_gpu(w)
    ref, eref = o.apply_h(psi0)
    h, e = g.apply_h(to_gpu(psi0))
    assert relerr(to_np(h), ref) < TOL_H and relerr(to_np(e), eref) < TOL_H
    pg, po, fg, fo, o, g = run_both(w, psi0, w.n_steps)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    for f in ("delta", "U_a", "rho_a", "nu"):
        assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-8, f
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    names = _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))
    assert ("k_f3s_mega_corr" in names) == (sep == "1") and ("k_f3_mega_corr" in names) == (sep == "0")


@pytest.mark.parametrize("nwf,group,block,ring,lag", [(10, 4, 2, 4, 1), (21, 8, 2, 20, 5), (7, 8, 4, 6, 2)])
def test_tma_stage_kernel_32cubed(tuning, nwf, group, block, ring, lag):
    """The opt-in TMA-fed, warp-specialised 32^3 Eq. 40 stage kernel (mega3t.cuh, enable_tma_stage): H psi with eps_n,
    self-consistent steps with ragged groups / blocks and more blocks than ring slots, and the kernels really ran."""
    tuning(enable_tma_stage=1, tma_group=group, tma_block=block, tma_ring=ring, tma_lag=lag, fused_chunk=3, fused_streams=3)
    w = wl.cfg4(n_side=32, n_wf=nwf, kin_form=1, n_steps=3)
    psi0 = w.spinors()
    o, g = make_oracle(w), make_gpu(w)
    ref, eref = o.apply_h(psi0)
    h, e = g.apply_h(to_gpu(psi0))
    assert relerr(to_np(h), ref) < TOL_H and relerr(to_np(e), eref) < TOL_H
    h2, _ = g.apply_h(to_gpu(psi0), n_first=1, n_count=3)
    h2 = to_np(h2)
    assert relerr(h2[1:4], ref[1:4]) < TOL_H and not h2[:1].any() and not h2[4:].any()
    pg, po, fg, fo, o, g = run_both(w, psi0, w.n_steps)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    for f in ("delta", "U_a", "rho_a", "nu"):
        assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-8, f
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    names = _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))
    assert "k_t3_mega_corr" in names and "k_t3_mega_rhs" in names and "k_f3s_mega_corr" not in names


@pytest.mark.parametrize("nwf,pm,em,ctas", [(10, 4, 2, 3), (37, 1, 1, 2), (7, 8, 4, 1)])
def test_dmma_stage_kernel_32cubed(tuning, nwf, pm, em, ctas):
    """The matrix-form (Eq. 28b) 32^3 Eq. 40 stage kernel on FP64 tensor instructions (mega3m.cuh, dmma_stage): H psi with
    eps_n, a sub-range, self-consistent steps with ragged groups and more groups than ring slots; the kernels really ran."""
    tuning(dmma_stage=1, dmma_ctas=ctas, p_planes=pm, x_rows=em, group=(5 if nwf > 30 else 0), fused_chunk=3, fused_streams=3)
    w = wl.cfg4(n_side=32, n_wf=nwf, kin_form=1, n_steps=3)
    psi0 = w.spinors()
    o, g = make_oracle(w), make_gpu(w)
    ref, eref = o.apply_h(psi0)
    h, e = g.apply_h(to_gpu(psi0))
    assert relerr(to_np(h), ref) < TOL_H and relerr(to_np(e), eref) < TOL_H
    h2, _ = g.apply_h(to_gpu(psi0), n_first=1, n_count=3)
    h2 = to_np(h2)
    assert relerr(h2[1:4], ref[1:4]) < TOL_H and not h2[:1].any() and not h2[4:].any()
    pg, po, fg, fo, o, g = run_both(w, psi0, w.n_steps)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    for f in ("delta", "U_a", "rho_a", "nu"):
        assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-8, f
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    names = _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))
    assert "k_f3m_mega_corr" in names and "k_f3m_mega_rhs" in names and "k_f3s_mega_corr" not in names


def test_dmma_stage_kernel_anisotropic_spacings(tuning):
    """mega3m with three different lattice spacings (each axis has its own folded matrices: a swapped pair would pass every
    isotropic test) and fixed random fields with alpha_a != alpha_b: H psi, eps_n and ABM steps against the oracle."""
    tuning(dmma_stage=1)
    w = generic((32, 32, 32), (1.0, 0.85, 1.2), 9, 1, func_id=0, dt=0.004)
    psi0 = spinors(w)
    o, g = make_oracle(w), make_gpu(w)
    ref, eref = o.apply_h(psi0)
    h, e = g.apply_h(to_gpu(psi0))
    assert relerr(to_np(h), ref) < TOL_H and relerr(to_np(e), eref) < TOL_H
    pg, po, fg, fo, o, g = run_both(w, psi0, 3)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    names = _kernels_of(g, lambda: g.apply_h(to_gpu(psi0)))
    assert "k_f3m_mega_apply" in names


@pytest.mark.parametrize("shape,dx,nwf", [((128,), (0.9,), 5), ((128,), (1.0,), 19), ((128,), (1.1,), 37), ((64, 64), (1.0, 0.9), 3)])
@pytest.mark.parametrize("dmma", [0, -1])
def test_onchip_matrix_form_cores_with_ragged_batches(tuning, shape, dx, nwf, dmma):
    """The on-chip stage kernels with the matrix-form (Eq. 28b, DMMA) core and with the FFT core (dmma_stage = -1) on the two
    shapes the matrix form covers, with batches that do not fill the CTA (lines of 128: 16 spinors per batch): H psi with
    eps_n, a sub-range, self-consistent steps; the kernels really ran."""
    tuning(dmma_stage=dmma)
    w = generic(shape, dx, nwf, 0, func_id=2, force_a1=1, n_modes=3, dt=0.004)     # SLDA with alpha = 1: the step rebuilds rho and nu only
    psi0 = spinors(w)
    o, g = make_oracle(w), make_gpu(w)
    ref, eref = o.apply_h(psi0)
    h, e = g.apply_h(to_gpu(psi0))
    assert relerr(to_np(h), ref) < TOL_H and relerr(to_np(e), eref) < TOL_H
    h2, _ = g.apply_h(to_gpu(psi0), n_first=1, n_count=2)
    h2 = to_np(h2)
    assert relerr(h2[1:3], ref[1:3]) < TOL_H and not h2[:1].any() and not h2[3:].any()
    pg, po, fg, fo, o, g = run_both(w, psi0, 3)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    for f in ("delta", "U_a", "rho_a", "rho_b", "nu"):
        assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-8, f
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    names = _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))
    assert "k_onchip_corr" in names and "k_onchip_rhs" in names and "k_onchip_pred" in names


@pytest.mark.parametrize("which", ["mega3s_32", "mega3d_16", "mega64", "tma_32", "dmma_32"])
def test_persistent_kernels_bit_reproducible(tuning, which):
    """The ticketed persistent kernels hand items to whichever CTA is free, but every sum is taken in a fixed order
    (partial sums per item, densities per ring slot in group order): two runs give identical bits."""
    if which == "mega3s_32":
        tuning(group=5, dmma_stage=-1); w = wl.cfg4(n_side=32, n_wf=23, kin_form=1, n_steps=3)
    elif which == "mega3d_16":
        tuning(group=3); w = generic((16, 32, 32), (1.0, 1.0, 1.0), 11, 1, func_id=2, dt=0.004)
    elif which == "mega64":
        w = wl.cfg4(n_side=64, n_wf=5, kin_form=1, n_steps=2)
    elif which == "dmma_32":
        tuning(dmma_stage=1, group=5); w = wl.cfg4(n_side=32, n_wf=23, kin_form=1, n_steps=3)
    else:
        tuning(enable_tma_stage=1, tma_group=4, tma_ring=6, tma_lag=2); w = wl.cfg4(n_side=32, n_wf=13, kin_form=1, n_steps=3)
    psi0 = w.spinors() if w.kidx is not None else spinors(w)
    import torch
    outs = []
    for _ in range(2):
        g = make_gpu(w)
        phi = to_gpu(psi0)
        hist = [torch.zeros_like(phi) for _ in range(g.m)]
        hist = g.abm_init(phi, hist, w.dt, 0)
        for _ in range(3):
            hist = g.abm_step(phi, hist, w.dt)
        outs.append((to_np(phi).copy(), to_np(hist[0]).copy(), to_np(g.get_field("rho_a")).copy(), to_np(g.get_field("nu")).copy()))
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


def test_device_wait_timeout_is_reported(tuning):
    """A device-side dependency wait that runs out must not pass silently: with a bound of one poll the
    persistent kernel flags the launch, the flag travels to the host behind it, and every later call fails with
    WSLDA_ECUDA and a message naming the cause."""
    tuning(spin_limit=1, group=2)
    w = wl.cfg4(n_side=32, n_wf=64, kin_form=1, n_steps=1)
    g = make_gpu(w)
    import torch
    psi = to_gpu(w.spinors())
    failed = None
    for _ in range(6):                                   # a wait has to be hit; a handful of launches make it certain
        try:
            g.apply_h(psi)
            torch.cuda.synchronize()
        except ws.WsldaError as e:
            failed = str(e)
            break
    assert failed is not None and "timed out" in failed
    with pytest.raises(ws.WsldaError):
        g.get_field("rho_a")


@pytest.mark.parametrize("case", ["fixed_sym40", "fixed_laplace_noshift", "bdg", "slda_trap_32", "fixed_ab5am5_nonorm"])
def test_fast3d_abm_matches_oracle(small_fast_chunks, case):
    if case == "fixed_sym40":
        w = generic((8, 32, 32), (1.0, 1.0, 1.1), 10, 1, dt=0.004); n = 8
    elif case == "fixed_laplace_noshift":
        w = generic((16, 32, 32), (1.0, 1.0, 1.0), 7, 0, dt=0.004, subtract_mean_energy=0); n = 6
    elif case == "fixed_ab5am5_nonorm":
        w = generic((8, 32, 32), (1.0, 1.0, 1.0), 8, 1, dt=0.004, ab_order=5, am_order=5, normalize=0); n = 6
    elif case == "bdg":
        w = generic((8, 32, 32), (1.0, 1.0, 1.0), 20, 0, func_id=1, four_pi_as=-2.0, dt=0.005); n = 6
    else:
        w = wl.cfg4(n_side=32, n_wf=20, kin_form=1, n_steps=5); n = 5      # configs[3] recipe, full lattice, 20 spinors
    psi0 = w.spinors() if w.kidx is not None else spinors(w)
    pg, po, fg, fo, o, g = run_both(w, psi0, n)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    if w.func_id:
        for f in ("delta", "U_a", "rho_a", "nu"):
            assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-8, f
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    assert any(k.startswith("k_f3") for k in _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt)))


# ---- full size, in the launch configuration bench.py times (configs[3]: 32^3, 16384 spinors, 86 GB resident) ------
def test_cfg4_full_size_sampled_against_oracle():
    """The whole-batch calls run at BASELINE.json's full size; the oracle follows a seeded sample of spinors.
    Only the sampled spinors carry occupation weight, so the densities (hence the self-consistent potentials) of
    the full-size GPU run depend on the sample alone and the oracle can reproduce them with n_wf = len(sample);
    every other spinor is still evolved by the same launches (spinors are independent given the potentials)."""
    import torch
    import copy
    w = wl.cfg4()
    shape = (w.n_wf, 2) + w.shape
    need = 5 * w.n_wf * 32 * w.M + 2e9
    if torch.cuda.mem_get_info()[0] < need:
        pytest.skip("needs 90 GB of free device memory")
    u = wl.uniform01(4242, 0, 250)
    sample = sorted(set([0, 1, 3, 4, 15, 16, w.n_wf - 1, w.n_wf - 2] + [int(x * w.n_wf) for x in u]))
    S = len(sample)
    wa, wb = np.zeros(w.n_wf), np.zeros(w.n_wf)
    wb[sample] = w.w_b[sample]
    wf = copy.copy(w); wf.w_a, wf.w_b = wa, wb
    g = make_gpu(wf)
    phi = torch.empty(shape, dtype=torch.complex128, device="cuda")
    wl.spinors_device(w, 0, w.n_wf, phi)
    psi_s = to_np(phi[sample])                                    # inputs of the oracle: the generator's output
    ws_ = copy.copy(w); ws_.n_wf = S; ws_.w_a, ws_.w_b = wa[sample], wb[sample]
    o = make_oracle(ws_)
    # densities -> potentials -> H psi
    o.densities(psi_s); o.update_potentials()
    g.densities(phi); g.update_potentials()
    for f in DENS:                                                # all eleven density fields, 250+ weighted spinors
        assert relerr(to_np(g.get_field(f)), o.get_field(f)) < TOL_D, f
    for f in ("delta", "U_a", "alpha_a"):
        assert relerr(to_np(g.get_field(f)), o.get_field(f)) < TOL_D, f
    hist = [torch.zeros(shape, dtype=torch.complex128, device="cuda") for _ in range(g.m)]
    h, e = g.apply_h(phi, hpsi=hist[0])
    href, eref = o.apply_h(psi_s)
    assert relerr(to_np(h[sample]), href) < TOL_H
    assert relerr(to_np(e[sample]), eref) < TOL_H
    hist[0].zero_()
    # two full Alg. 2 steps from a zero history (exactly what bench.py times)
    phi_o = psi_s.copy()
    hist_o = [np.zeros_like(psi_s) for _ in range(o.m)]
    hist_o = o.abm_init(phi_o, hist_o, w.dt, 0)
    hist = g.abm_init(phi, hist, w.dt, 0)
    for _ in range(2):
        hist_o = o.abm_step(phi_o, hist_o, w.dt)
        hist = g.abm_step(phi, hist, w.dt)
    assert relerr(to_np(phi[sample]), phi_o) < TOL_ABM
    assert relerr(to_np(hist[0][sample]), hist_o[0]) < TOL_ABM
    for f in ("delta", "U_a", "rho_a"):
        assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-9, f
    nrm = torch.sum(phi.real ** 2 + phi.imag ** 2, dim=(1, 2, 3, 4)) * w.dV
    assert float(torch.max(torch.abs(nrm - 1.0))) < 1e-12          # property at any size: every spinor normalised
    del phi, hist
    torch.cuda.empty_cache()


# ---- 64^3: pair-of-threads lines, component-granular persistent kernels (mega64.cuh) -------------------------------
def test_mega64_apply_h():
    w = generic((64, 64, 64), (1.0, 0.95, 1.05), 3, 1, n_modes=1)
    psi = spinors(w)
    o, g = make_oracle(w), make_gpu(w)
    ref, eref = o.apply_h(psi)
    h, e = g.apply_h(to_gpu(psi))
    assert relerr(to_np(h), ref) < TOL_H and relerr(to_np(e), eref) < TOL_H
    assert any(k.startswith("k_f6") for k in _kernels_of(g, lambda: g.apply_h(to_gpu(psi))))
    h2, _ = g.apply_h(to_gpu(psi), n_first=1, n_count=2)
    h2 = to_np(h2)
    assert relerr(h2[1:3], ref[1:3]) < TOL_H and not h2[:1].any()


@pytest.mark.parametrize("case", ["cfg5_fixed", "slda_selfconsistent"])
def test_mega64_abm_matches_oracle(case):
    if case == "cfg5_fixed":
        w = wl.cfg5(n_wf=7, n_steps=3)                       # configs[4] recipe: h_a != h_b, fixed smooth fields
    else:
        w = wl.cfg4(n_side=64, n_wf=6, kin_form=1, n_steps=2)  # self-consistent SLDA on 64^3 (densities in the D items)
    psi0 = w.spinors()
    pg, po, fg, fo, o, g = run_both(w, psi0, w.n_steps)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    if w.func_id:
        for f in ("delta", "U_a", "rho_a", "nu"):
            assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-8, f


# ---- the other configs at BASELINE.json's full size, on seeded samples (same technique as configs[3] above) ----------
def _full_size_sampled(w, n_sample, n_steps, seed):
    import copy
    import torch
    shape = (w.n_wf, 2) + w.shape
    need = (2 + w.history) * w.n_wf * 32 * w.M + 3e9
    if torch.cuda.mem_get_info()[0] < need:
        pytest.skip("not enough free device memory for the full-size batch")
    u = wl.uniform01(seed, 0, n_sample)
    sample = sorted(set([0, 1, w.n_wf - 1] + [int(x * w.n_wf) for x in u]))
    S = len(sample)
    wa, wb = np.zeros(w.n_wf), np.zeros(w.n_wf)
    wa[sample], wb[sample] = w.w_a[sample], w.w_b[sample]
    if not (wa[sample].any() or wb[sample].any()):
        wb[sample] = 1.0                                           # make sure the sample carries density
    wf = copy.copy(w); wf.w_a, wf.w_b = wa, wb
    g = make_gpu(wf)
    phi = torch.empty(shape, dtype=torch.complex128, device="cuda")
    wl.spinors_device(w, 0, w.n_wf, phi)
    psi_s = to_np(phi[sample])
    ws_ = copy.copy(w); ws_.n_wf = S; ws_.w_a, ws_.w_b = wa[sample], wb[sample]
    if w.kperp is not None:                                        # one mode entry per sampled spinor
        mo = np.asarray(w.mode_of)[sample]
        ws_.kperp, ws_.mult = np.asarray(w.kperp)[mo], np.asarray(w.mult)[mo]
        ws_.first = np.arange(S + 1, dtype=np.int64)
        ws_.mode_of = np.arange(S)
    o = make_oracle(ws_)
    hist = [torch.zeros(shape, dtype=torch.complex128, device="cuda") for _ in range(g.m)]
    o.densities(psi_s)                                             # every density field at full size
    g.densities(phi)
    held = "xyz"[: len(w.shape)]
    for f in [x for x in DENS if not x.startswith("j") or x[-1] in held]:
        ref = o.get_field(f)
        if np.abs(ref).max() > 0:
            assert relerr(to_np(g.get_field(f)), ref) < TOL_D, f
    if w.func_id:
        o.update_potentials(); g.update_potentials()
        for f in ("delta", "U_a"):
            assert relerr(to_np(g.get_field(f)), o.get_field(f)) < TOL_D, f
    h, e = g.apply_h(phi, hpsi=hist[0])
    href, eref = o.apply_h(psi_s)
    assert relerr(to_np(h[sample]), href) < TOL_H
    assert relerr(to_np(e[sample]), eref) < TOL_H
    hist[0].zero_()
    phi_o = psi_s.copy()
    hist_o = [np.zeros_like(psi_s) for _ in range(o.m)]
    hist_o = o.abm_init(phi_o, hist_o, w.dt, 0)
    hist = g.abm_init(phi, hist, w.dt, 0)
    for _ in range(n_steps):
        hist_o = o.abm_step(phi_o, hist_o, w.dt)
        hist = g.abm_step(phi, hist, w.dt)
    assert relerr(to_np(phi[sample]), phi_o) < TOL_ABM
    assert relerr(to_np(hist[0][sample]), hist_o[0]) < TOL_ABM
    if w.func_id:
        for f in ("delta", "U_a", "rho_a"):
            assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-9, f
    nd = len(w.shape)
    nrm = torch.sum(phi.real ** 2 + phi.imag ** 2, dim=tuple(range(1, nd + 2))) * w.dV
    assert float(torch.max(torch.abs(nrm - 1.0))) < 1e-12
    del phi, hist, h
    torch.cuda.empty_cache()


def test_cfg2_full_size_sampled_against_oracle():
    """configs[1]: quasi-1D, 262144 spinors over 1024 transverse modes, self-consistent (fused on-chip stages)."""
    _full_size_sampled(wl.cfg2(), 256, 10, 5151)


def test_cfg3_full_size_sampled_against_oracle():
    """configs[2]: quasi-2D 64^2, 65536 spinors over 16 k_z modes, vortex imprint, self-consistent."""
    _full_size_sampled(wl.cfg3(), 256, 10, 5252)


def test_cfg5_full_size_sampled_against_oracle():
    """configs[4]: 64^3, 2048 resident spinors, fixed smooth h_a != h_b fields (64^3 persistent kernels)."""
    _full_size_sampled(wl.cfg5(n_wf=2048), 64, 2, 5353)


# ---- NEXT-2: the spinor index sharded over ranks, one density sum per build (include/wslda.h: wslda_set_reduce_hook) --
def _run_sharded(w, psi0, n_steps, n_shards, selfstart=1, pre_all=False, fields=("rho_a", "nu", "delta", "U_a")):
    """n_shards contexts on this GPU, each over its own share of the spinors and stepped by its own host thread;
    the reduce hook is a host rendezvous that sums the density blocks of all shards (what ncclAllReduce does across
    GPUs).  Nothing on the device waits on another launch.  Returns (phi, f_hist[0]) gathered in spinor order."""
    import threading
    import torch
    bounds = [wl.shard_range(w.n_wf, r, n_shards) for r in range(n_shards)]
    blocks, tmp, out, errs = [None] * n_shards, [None] * n_shards, [None] * n_shards, []
    bar = threading.Barrier(n_shards)
    calls = [0] * n_shards

    def worker(r):
        try:
            n0, n1 = bounds[r]
            g = make_gpu(wl.shard(w, n0, n1))

            def hook(block, stream):
                calls[r] += 1
                torch.cuda.synchronize()
                blocks[r] = block
                bar.wait(timeout=120)
                tmp[r] = torch.stack([blocks[q] for q in range(n_shards)]).sum(0)      # same order on every shard
                torch.cuda.synchronize()
                bar.wait(timeout=120)
                block.copy_(tmp[r])
                torch.cuda.synchronize()

            g.set_reduce_hook(hook)
            phi = to_gpu(psi0[n0:n1])
            if pre_all:                                   # every density plane (tau, j too) built once, before the steps
                g.densities(phi)
            hist = [torch.zeros_like(phi) for _ in range(g.m)]
            hist = g.abm_init(phi, hist, w.dt, selfstart)
            for _ in range(n_steps):
                hist = g.abm_step(phi, hist, w.dt)
            out[r] = (to_np(phi), to_np(hist[0]), {f: to_np(g.get_field(f)) for f in fields})
        except BaseException as e:                     # release the other threads, then report
            errs.append(e)
            bar.abort()

    th = [threading.Thread(target=worker, args=(r,)) for r in range(n_shards)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    if errs:
        raise errs[0]
    assert len(set(calls)) == 1 and calls[0] > 0          # every shard made the same number of reductions
    return (np.concatenate([o[0] for o in out]), np.concatenate([o[1] for o in out]), [o[2] for o in out])


@pytest.mark.parametrize("case", ["mega32_sym40", "onchip_cfg3", "general_divgrad"])
def test_sharded_contexts_match_unsharded_oracle(case, small_fast_chunks):
    if case == "mega32_sym40":
        w = wl.cfg4(n_side=32, n_wf=11, kin_form=1, n_steps=2)
    elif case == "onchip_cfg3":
        w = wl.cfg3(n_side=16, n_kz=3, nz=8, n_steps=2)           # three k_z modes: the split cuts through a mode
    else:
        w = wl.cfg4(n_side=8, n_wf=9, kin_form=2, n_steps=2)
    psi0 = w.spinors()
    o = make_oracle(w)
    phi_o = psi0.copy()
    hist_o = [np.zeros_like(psi0) for _ in range(o.m)]
    hist_o = o.abm_init(phi_o, hist_o, w.dt, 1)
    for _ in range(w.n_steps):
        hist_o = o.abm_step(phi_o, hist_o, w.dt)
    for n_shards in (2, 3):
        phi, f0, fields = _run_sharded(w, psi0, w.n_steps, n_shards)
        assert relerr(phi, phi_o) < TOL_ABM and relerr(f0, hist_o[0]) < TOL_ABM
        for fl in fields:                                          # every shard ends with the whole-system fields
            for f in ("rho_a", "nu", "delta", "U_a"):
                assert relerr(fl[f], o.get_field(f)) < 1e-8, f


@pytest.mark.parametrize("case", ["mega32_sym40", "general_8"])
def test_sharded_steps_do_not_resum_planes_they_did_not_rebuild(case, small_fast_chunks):
    """a step rebuilds rho and nu only; the tau and j planes left by an earlier wslda_densities(D_ALL) are
    already whole-system sums and must not go through the all-reduce again (they grew by world_size per reduction).
    densities(all) -> steps with the hook: rho, nu, delta equal the unsharded oracle's after the steps, and tau, j --
    which wslda_abm_step does not refresh (DESIGN R25; the oracle rebuilds every plane) -- still equal the unsharded
    oracle's densities of the INITIAL spinors, however many reductions went by."""
    w = wl.cfg4(n_side=32, n_wf=9, kin_form=1, n_steps=3) if case == "mega32_sym40" else wl.cfg4(n_side=8, n_wf=9, kin_form=1, n_steps=3)
    psi0 = w.spinors()
    o = make_oracle(w)
    phi_o = psi0.copy()
    o.densities(phi_o)
    stale = {f: o.get_field(f).copy() for f in ("tau_a", "tau_b", "ja_x", "jb_z")}
    hist_o = [np.zeros_like(psi0) for _ in range(o.m)]
    hist_o = o.abm_init(phi_o, hist_o, w.dt, 0)
    for _ in range(w.n_steps):
        hist_o = o.abm_step(phi_o, hist_o, w.dt)
    names = ("rho_a", "nu", "tau_a", "tau_b", "ja_x", "jb_z", "delta")
    for n_shards in (2, 3):
        phi, f0, fields = _run_sharded(w, psi0, w.n_steps, n_shards, selfstart=0, pre_all=True, fields=names)
        assert relerr(phi, phi_o) < TOL_ABM
        for fl in fields:
            for f in names:
                ref = stale[f] if f in stale else o.get_field(f)
                scale = max(np.abs(ref).max(), 1e-30)
                assert np.abs(fl[f] - ref).max() <= 1e-8 * scale + 1e-13, (f, n_shards)


def test_density_allreduce_through_nccl_single_rank():
    """The torch.distributed plumbing of Context.set_density_allreduce on a 1-rank NCCL group: the hook runs inside
    the step, on the step's stream, and a sum over one rank changes nothing."""
    import torch
    import torch.distributed as dist
    if not dist.is_available() or not dist.is_nccl_available():
        pytest.skip("no NCCL in this torch build")
    created = False
    if not dist.is_initialized():
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:29613", rank=0, world_size=1)
        created = True
    try:
        w = wl.cfg4(n_side=32, n_wf=6, kin_form=1, n_steps=2)
        psi0 = w.spinors()
        res = []
        for hooked in (False, True):
            g = make_gpu(w)
            if hooked:
                g.set_density_allreduce()
            phi = to_gpu(psi0)
            hist = [torch.zeros_like(phi) for _ in range(g.m)]
            s = torch.cuda.Stream()
            s.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(s):                          # a non-default stream: the collective must follow it
                hist = g.abm_init(phi, hist, w.dt, 1)
                for _ in range(w.n_steps):
                    hist = g.abm_step(phi, hist, w.dt)
            s.synchronize()
            res.append((to_np(phi), to_np(g.get_field("delta"))))
        assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])
    finally:
        if created:
            dist.destroy_process_group()


@pytest.mark.parametrize("case", ["fused32", "mega3d16", "onchip", "general"])
def test_reduce_hook_fires_on_the_callers_stream_with_complete_sums(case, tuning):
    """The density block handed to the hook is complete when the hook's work runs: the hook is given the
    CALLER's stream -- never one of the library-owned stage-1 streams --, twice per self-consistent step; a copy of the block
    enqueued there by the hook equals the block after a full device synchronisation (nothing writes it after the last hook),
    and a hook that only copies leaves the step bit-identical to an unhooked one."""
    import torch
    if case == "fused32":
        tuning(fused_chunk=3, fused_streams=3); w = wl.cfg4(n_side=32, n_wf=11, kin_form=1, n_steps=2)
    elif case == "mega3d16":
        tuning(fused_chunk=2, fused_streams=3, group=3); w = generic((16, 32, 32), (1.0, 1.0, 1.0), 7, 1, func_id=2, dt=0.004)
    elif case == "onchip":
        w = generic((64, 64), (1.0, 1.0), 6, 0, func_id=2, dt=0.004)
    else:
        w = generic((16, 8, 8), (1.0, 1.0, 1.0), 9, 2, func_id=2, dt=0.004)
    psi0 = w.spinors() if getattr(w, "kidx", None) is not None else spinors(w)
    final = {}
    for hooked in (True, False):
        g = make_gpu(w)
        s = torch.cuda.Stream()
        calls = []
        if hooked:
            def hook(block, stream, calls=calls):
                with torch.cuda.stream(torch.cuda.ExternalStream(stream)):
                    calls.append((stream, block, block.clone()))
            g.set_reduce_hook(hook)
        phi = to_gpu(psi0)
        hist = [torch.zeros_like(phi) for _ in range(g.m)]
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            hist = g.abm_init(phi, hist, w.dt, 0)
            n0 = len(calls)
            hist = g.abm_step(phi, hist, w.dt)
        torch.cuda.synchronize()
        if hooked:
            step_calls = calls[n0:]
            assert len(step_calls) == 2, len(step_calls)                 # after the predictor's and after the corrector's densities
            for stream, block, snap in step_calls:
                assert stream == s.cuda_stream                            # the caller's stream, not a library-owned one
                assert block.numel() % g.M == 0 and 4 <= block.numel() // g.M <= 14
            stream, block, snap = step_calls[-1]
            assert torch.equal(snap, block) and float(block.abs().max()) > 0.0
        final[hooked] = (to_np(phi).copy(), to_np(g.get_field("rho_a")).copy(), to_np(g.get_field("nu")).copy())
    for a, b in zip(final[True], final[False]):
        assert np.array_equal(a, b)


# ---- NEXT-1: current / velocity coupling (Eq. 4c, Eqs. 9b-c), general path ---------------
def _with_currents(w, seed, amp=0.2):
    M = int(np.prod(w.shape))
    nd = len(w.shape)
    v = amp * wl.normal(seed, 0, 6 * M).reshape(2, 3, *w.shape)
    w.current_terms = 1
    w.vel = (v[0, :nd], v[1, :nd])
    return w


@pytest.mark.parametrize("kin_form", [0, 1, 2])
@pytest.mark.parametrize("shape,dx", [((8, 4, 8), (1.0, 0.9, 1.1)), ((16, 8), (1.0, 1.2)), ((32,), (0.8,)),
                                      ((32, 16, 16), (1.0, 1.0, 0.9)), ((8, 32, 32), (1.0, 1.1, 0.9))])
def test_current_coupling_apply_h_matches_oracle(shape, dx, kin_form):
    """H psi with rough external velocity fields on every lattice regime of the general path (on-chip, multi-pass, and
    a Ny = Nz = 32 lattice, where the fused kernels step aside for the coupling term)."""
    n_wf = 5 if np.prod(shape) > 4096 else 13
    w = _with_currents(generic(shape, dx, n_wf, kin_form, n_modes=2), 401)
    psi = spinors(w)
    o, g = make_oracle(w), make_gpu(w)
    ref, eref = o.apply_h(psi)
    h, e = g.apply_h(to_gpu(psi))
    assert relerr(to_np(h), ref) < TOL_H and relerr(to_np(e), eref) < TOL_H
    w0 = generic(shape, dx, n_wf, kin_form, n_modes=2)            # and the term is not a rounding matter
    assert relerr(make_oracle(w0).apply_h(psi)[0], ref) > 1e-3


@pytest.mark.parametrize("shape,dx,nwf", [((64, 64), (1.0, 0.9), 5), ((128,), (0.9,), 19)])
@pytest.mark.parametrize("func_id,force_a1", [(0, 0), (2, 1), (1, 0)])
def test_current_coupling_on_the_fused_onchip_paths(shape, dx, nwf, func_id, force_a1):
    """NEXT-1 on fused paths: on 64 x 64 lattices and on lines of 128 points the on-chip stage kernels take the coupling
    -(i/2){W, grad} inside their matrix-form core (first-derivative matrices on DMMA; W = -v_ext whenever the step rebuilds rho
    and nu only: fixed fields, SLDA with alpha = 1, BdG): H psi with eps_n and ABM steps against the oracle (ragged batches on
    the lines), and the on-chip kernels really ran."""
    kw = dict(four_pi_as=-3.0) if func_id == 1 else {}
    w = _with_currents(generic(shape, dx, nwf, 0, func_id=func_id, force_a1=force_a1, n_modes=2, dt=0.004, **kw), 461, amp=0.3)
    psi0 = spinors(w)
    o, g = make_oracle(w), make_gpu(w)
    if func_id:
        o.densities(psi0); o.update_potentials(); g.densities(to_gpu(psi0)); g.update_potentials()
    ref, eref = o.apply_h(psi0)
    names = _kernels_of(g, lambda: g.apply_h(to_gpu(psi0)))
    assert "k_onchip_apply" in names
    h, e = g.apply_h(to_gpu(psi0))
    assert relerr(to_np(h), ref) < TOL_H and relerr(to_np(e), eref) < TOL_H
    w0 = generic(shape, dx, nwf, 0, func_id=func_id, force_a1=force_a1, n_modes=2, dt=0.004, **kw)
    o0 = make_oracle(w0)
    if func_id:
        o0.densities(psi0); o0.update_potentials()
    assert relerr(o0.apply_h(psi0)[0], ref) > 1e-3                     # the term is not a rounding matter
    pg, po, fg, fo, o, g = run_both(w, psi0, 3)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    names = _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))
    assert "k_onchip_corr" in names and "k_onchip_rhs" in names


@pytest.mark.parametrize("func_id,force_a1,nwf", [(0, 0, 9), (2, 1, 37), (1, 0, 5)])
def test_current_coupling_on_the_fused_32cubed_path(tuning, func_id, force_a1, nwf):
    """NEXT-1 on the persistent 32^3 Eq. 40 kernels: the matrix-form stage kernels (mega3m.cuh, own instantiation) take the
    coupling -(i/2){W, grad}: its y and z parts ride on the alpha-w field of the P items, its x part on the XE items' x-derivative
    (2 D_d matrices on DMMA).  Fixed random fields with alpha_a != alpha_b, SLDA with alpha = 1, BdG; three lattice spacings;
    ragged groups; H psi with eps_n and ABM steps against the oracle; the fused kernels really ran."""
    tuning(group=(5 if nwf > 30 else 0), fused_chunk=3, fused_streams=3)
    kw = dict(four_pi_as=-3.0) if func_id == 1 else {}
    mk = lambda: generic((32, 32, 32), (1.0, 0.85, 1.2), nwf, 1, func_id=func_id, force_a1=force_a1, dt=0.004, **kw)
    w = _with_currents(mk(), 471, amp=0.3)
    psi0 = spinors(w)
    o, g = make_oracle(w), make_gpu(w)
    if func_id:
        o.densities(psi0); o.update_potentials(); g.densities(to_gpu(psi0)); g.update_potentials()
    ref, eref = o.apply_h(psi0)
    names = _kernels_of(g, lambda: g.apply_h(to_gpu(psi0)))
    assert "k_f3m_mega_apply" in names
    h, e = g.apply_h(to_gpu(psi0))
    assert relerr(to_np(h), ref) < TOL_H and relerr(to_np(e), eref) < TOL_H
    o0 = make_oracle(mk())
    if func_id:
        o0.densities(psi0); o0.update_potentials()
    assert relerr(o0.apply_h(psi0)[0], ref) > 1e-3                     # the term is not a rounding matter
    pg, po, fg, fo, o, g = run_both(w, psi0, 3)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    names = _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))
    assert "k_f3m_mega_corr" in names and "k_f3m_mega_rhs" in names


def test_fused_64cubed_step_polarised_aslda():
    """Polarised ASLDA on 64^3: the persistent 64^3 stage kernels do the stages, tau comes from the axis-by-axis gradient
    densities after each of them.  Two steps and the fields against the oracle; the fused kernels and k_gdens really ran."""
    w = wl.cfg4(n_side=64, n_wf=4, kin_form=1, n_steps=2)
    w.spin_symmetric = 0
    w.w_a = 0.6 * np.asarray(w.w_b)
    psi0 = w.spinors()
    pg, po, fg, fo, o, g = run_both(w, psi0, 2, selfstart=0)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    for f in ("rho_a", "rho_b", "nu", "delta", "U_a", "U_b", "alpha_a", "alpha_b", "tau_a", "tau_b"):
        assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-8, f
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    names = _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))
    assert "k_f6_mega_corr" in names and "k_f6_mega_rhs" in names and "k_gdens" in names


@pytest.mark.parametrize("case", ["polarised", "polarised_currents", "symmetric_currents"])
def test_fused_32cubed_step_with_gradient_densities(tuning, case):
    """Functionals that consume tau and j inside the step on the fused 32^3 path: polarised ASLDA (alpha_sigma depends on p, so tau
    enters V_sigma) and ASLDA with the current coupling (A_sigma = (1 - alpha_sigma) j_sigma / rho_sigma rebuilt at both stages):
    the persistent stage kernels do the stages, the axis-by-axis gradient densities (gdens.cuh) follow each of them.  Steps and
    fields against the oracle; the fused kernels and k_gdens really ran."""
    tuning(group=5, fused_chunk=3, fused_streams=3)
    w = wl.cfg4(n_side=32, n_wf=14, kin_form=1, n_steps=3)
    if case.startswith("polarised"):
        w.spin_symmetric = 0
        w.w_a = 0.6 * np.asarray(w.w_b)                         # both spin densities populated, p != 0: alpha_a != alpha_b != 1
    if case.endswith("currents"):
        w = _with_currents(w, 481, amp=0.05)
    psi0 = w.spinors()
    pg, po, fg, fo, o, g = run_both(w, psi0, 3, selfstart=0)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    names_f = ["rho_a", "nu", "delta", "U_a", "U_b", "alpha_a"] + (["tau_a", "tau_b"] if case.startswith("polarised") else [])
    names_f += ["ja_x", "jb_z", "Aa_x", "Ab_y", "V_a"] if case.endswith("currents") else []
    for f in names_f:
        ref = o.get_field(f)
        assert relerr(to_np(g.get_field(f)), ref) < 1e-8, f
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    names = _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))
    assert "k_f3m_mega_corr" in names and "k_f3m_mega_rhs" in names and "k_gdens" in names


@pytest.mark.parametrize("case", ["aslda_polarised", "aslda_symmetric", "bdg_moving_frame", "fixed"])
def test_current_coupling_selfconsistent_steps(case):
    """Self-consistent steps with the coupling: A_sigma = (1 - alpha_sigma) j_sigma / rho_sigma rebuilt at both stages of
    Alg. 2 (j joins the densities the step refreshes), the j-terms of V_sigma, a uniform frame velocity for BdG."""
    shape, dx = (8, 8, 8), (1.0, 1.0, 1.0)
    if case == "fixed":
        w = _with_currents(generic(shape, dx, 12, 1, dt=0.004), 411)
    else:
        w = wl.cfg4(n_side=8, n_wf=24, kin_form=1, n_steps=4)
        if case == "aslda_polarised":
            w.spin_symmetric = 0
            w.w_a = 0.6 * np.asarray(w.w_b)                     # both spin densities populated, p != 0: alpha_a != alpha_b != 1
        elif case == "bdg_moving_frame":
            w.func_id, w.kin_form, w.four_pi_as = 1, 0, -3.0
        w = _with_currents(w, 412, amp=0.05)
        if case == "bdg_moving_frame":
            v = np.zeros((3,) + shape); v[0] = 0.1
            w.vel = (v, v)
    psi0 = w.spinors() if w.kidx is not None else spinors(w)
    pg, po, fg, fo, o, g = run_both(w, psi0, 4, selfstart=1)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    if case != "fixed":
        for f in ("rho_a", "nu", "delta", "U_a", "U_b", "alpha_a"):
            assert relerr(to_np(g.get_field(f)), o.get_field(f)) < 1e-8, f
    if case.startswith("aslda"):
        for f in ("ja_x", "jb_z", "Aa_x", "Ab_y", "V_a"):
            ref = o.get_field(f)
            assert np.abs(ref).max() > 0
            assert relerr(to_np(g.get_field(f)), ref) < 1e-8, f


# ---- NEXT-4: on-device observables (Eqs. 33a-g) and the conservation watchdog -----
OBS_ORACLE = ["N_a", "N_b", "E_kin", "E_pot", "E_pair", "E_pot_ext", "E_pair_ext", "E_total", "E_curr", "E_vel_ext"]


@pytest.mark.parametrize("case", ["cfg4_32", "cfg3_q2d", "polarised_currents", "bdg_8", "cfg4_64"])
def test_energy_matches_oracle(case):
    import torch
    if case == "cfg4_32":
        w = wl.cfg4(n_side=32, n_wf=9, kin_form=1, n_steps=1)
    elif case == "cfg4_64":
        w = wl.cfg4(n_side=64, n_wf=3, kin_form=1, n_steps=1)
    elif case == "cfg3_q2d":
        w = wl.cfg3(n_side=16, n_kz=3, nz=8, n_steps=1)             # multiplicities 1, 2, 2; Delta_ext; L_perp != 1
    elif case == "bdg_8":
        w = wl.cfg4(n_side=8, n_wf=20, kin_form=0, n_steps=1); w.func_id, w.four_pi_as = 1, -3.0
    else:
        w = wl.cfg4(n_side=8, n_wf=24, kin_form=1, n_steps=1)
        w.spin_symmetric = 0; w.w_a = 0.6 * np.asarray(w.w_b)
        w = _with_currents(w, 431, amp=0.05)
    psi0 = w.spinors()
    o, g = make_oracle(w), make_gpu(w)
    o.densities(psi0); o.update_potentials()
    g.densities(to_gpu(psi0)); g.update_potentials()
    ref = o.energy()
    got = to_np(g.energy())
    scale = max(abs(ref[k]) for k in OBS_ORACLE[2:])
    for i, k in enumerate(OBS_ORACLE):
        assert abs(got[i] - ref[k]) <= 1e-11 * (abs(ref[k]) if i < 2 else scale), (k, got[i], ref[k])
    assert np.array_equal(got, to_np(g.energy()))                   # fixed summation order
    assert abs(ref["E_kin"]) > 0 and abs(ref["E_pair"]) > 0


def test_watchdog_passes_a_conserving_run_and_stops_a_violating_one():
    """The conservation check of the time-dependent codes on the device: a self-consistent BdG run within tolerance
    passes silently; the same check with an impossible tolerance poisons the context (every later call WSLDA_ESTATE)."""
    import torch
    w = wl.cfg4(n_side=8, n_wf=32, kin_form=0, n_steps=1)
    w.func_id, w.four_pi_as, w.lambda_mode = 1, -3.0, 1
    psi0 = w.spinors()
    g = make_gpu(w)
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 1)
    g.densities(phi); g.update_potentials()
    ref = g.energy()
    for _ in range(5):
        hist = g.abm_step(phi, hist, w.dt)
    g.densities(phi); g.update_potentials()
    now = g.watchdog(ref, 1e-6, 1e-3)
    torch.cuda.synchronize()
    g.get_field("rho_a")                                            # still alive
    r, n = to_np(ref), to_np(now)
    assert abs(n[0] - r[0]) < 1e-8 * abs(r[0]) and abs(n[7] - r[7]) < 1e-3 * abs(r[7]) and n[7] != r[7]
    g.watchdog(ref, 1e-6, 1e-16)                                    # nobody conserves energy to 1e-16 over 5 steps
    torch.cuda.synchronize()
    with pytest.raises(ws.WsldaError, match="conservation"):
        g.get_field("rho_a")
    with pytest.raises(ws.WsldaError):
        g.abm_step(phi, hist, w.dt)


# ---- NEXT-3: quantum friction (Eqs. 66-70), general path --------------------------------------------
@pytest.mark.parametrize("shape,dx", [((8, 4, 8), (1.0, 0.9, 1.1)), ((16, 8), (1.0, 1.2)), ((32,), (0.8,)), ((32, 16, 16), (1.0, 1.0, 0.9))])
@pytest.mark.parametrize("sym", [0, 1])
def test_kinetic_anomalous_density_matches_oracle(shape, dx, sym):
    """B' of Eq. 68 (mask WSLDA_D_BP) on on-chip and multi-pass lattices, with transverse modes and multiplicities,
    overwritten and accumulated over batches."""
    n_wf = 7 if np.prod(shape) > 4096 else 19
    w = generic(shape, dx, n_wf, 1, n_modes=3, spin_symmetric=sym)
    psi = spinors(w)
    o, g = make_oracle(w), make_gpu(w)
    o.densities(psi)
    dev = to_gpu(psi)
    g.densities(dev, which=ws.D_BP | ws.D_NU)
    assert relerr(to_np(g.get_field("bp")), o.get_field("bp")) < TOL_D
    assert relerr(to_np(g.get_field("nu")), o.get_field("nu")) < TOL_D
    g.densities(dev, n_first=0, n_count=3, which=ws.D_BP)
    g.densities(dev, n_first=3, n_count=n_wf - 3, which=ws.D_BP, accumulate=1)
    assert relerr(to_np(g.get_field("bp")), o.get_field("bp")) < TOL_D


@pytest.mark.parametrize("side,nwf", [(32, 21), (64, 3)])
def test_kinetic_anomalous_density_axis_by_axis(side, nwf):
    """B' on cubic 32^3 / 64^3 lattices comes from second derivatives taken axis by axis (k_gdens_bp): against the oracle, with
    both spins populated, overwritten and accumulated over batches; the kernel really ran."""
    w = wl.cfg4(n_side=side, n_wf=nwf, kin_form=1)
    w.spin_symmetric = 0
    w.w_a = 0.3 * np.asarray(w.w_b) + 0.1
    psi = w.spinors()
    o, g = make_oracle(w), make_gpu(w)
    o.densities(psi)
    dev = to_gpu(psi)
    names = _kernels_of(g, lambda: g.densities(dev, which=ws.D_BP | ws.D_NU))
    assert "k_gdens_bp" in names
    ref = o.get_field("bp")
    assert np.abs(ref).max() > 0
    assert relerr(to_np(g.get_field("bp")), ref) < TOL_D and relerr(to_np(g.get_field("nu")), o.get_field("nu")) < TOL_D
    g.densities(dev, n_first=0, n_count=2, which=ws.D_BP)
    g.densities(dev, n_first=2, n_count=nwf - 2, which=ws.D_BP, accumulate=1)
    assert relerr(to_np(g.get_field("bp")), ref) < TOL_D


@pytest.mark.parametrize("case", ["symmetric", "polarised"])
def test_quantum_friction_on_the_fused_32cubed_path(tuning, case):
    """NEXT-3 on a fused path: on cubic 32^3 lattices the persistent stage kernels do the stages and j, B' (and tau) come from the
    axis-by-axis density kernels after each of them; the friction terms are applied by the potential update as everywhere."""
    tuning(group=5, fused_chunk=3, fused_streams=3)
    w = wl.cfg4(n_side=32, n_wf=13, kin_form=1, n_steps=3)
    if case == "polarised":
        w.spin_symmetric = 0; w.w_a = 0.6 * np.asarray(w.w_b)
    w.friction = dict(qf_alpha=6.0, qf_beta=5.0, qf_gamma=0.1, qf_rho0=0.03, qf_nreq=1.7)
    psi0 = w.spinors()
    pg, po, fg, fo, o, g = run_both(w, psi0, 3, selfstart=0)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    for f in ("rho_a", "nu", "bp", "ja_x", "jb_z", "delta", "V_a", "U_b"):
        ref = o.get_field(f)
        assert np.abs(ref).max() > 0
        assert relerr(to_np(g.get_field(f)), ref) < 1e-8, f
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    names = _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))
    assert "k_f3m_mega_corr" in names and "k_gdens" in names and "k_gdens_bp" in names and "k_qf" in names


def test_quantum_friction_on_the_fused_64cubed_path():
    """The same on 64^3: the persistent 64^3 stage kernels + k_gdens (j) + k_gdens_bp (B') + k_qf."""
    w = wl.cfg4(n_side=64, n_wf=3, kin_form=1, n_steps=2)
    w.friction = dict(qf_alpha=6.0, qf_beta=5.0, qf_gamma=0.1, qf_rho0=0.03, qf_nreq=1.7)
    psi0 = w.spinors()
    pg, po, fg, fo, o, g = run_both(w, psi0, 2, selfstart=0)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    for f in ("rho_a", "nu", "bp", "ja_x", "delta", "V_a", "U_b"):
        ref = o.get_field(f)
        assert np.abs(ref).max() > 0
        assert relerr(to_np(g.get_field(f)), ref) < 1e-8, f
    import torch
    phi = to_gpu(psi0)
    hist = [torch.zeros_like(phi) for _ in range(g.m)]
    hist = g.abm_init(phi, hist, w.dt, 0)
    names = _kernels_of(g, lambda: g.abm_step(phi, hist, w.dt))
    assert "k_f6_mega_corr" in names and "k_gdens" in names and "k_gdens_bp" in names and "k_qf" in names


@pytest.mark.parametrize("case", ["bdg", "aslda_polarised", "slda_symmetric_32"])
def test_quantum_friction_steps_match_oracle(case):
    """Dissipative self-consistent steps: V^(d) from div j, Delta^(d) from the phases of nu and B' and from N - N_req,
    rebuilt at both stages of Alg. 2 and in the Taylor starter."""
    if case == "slda_symmetric_32":
        w = wl.cfg4(n_side=32, n_wf=6, kin_form=1, n_steps=2)          # a Ny = Nz = 32 lattice: the fused kernels step aside
        steps = 2
    else:
        w = wl.cfg4(n_side=8, n_wf=24, kin_form=1, n_steps=4)
        steps = 4
        if case == "bdg":
            w.func_id, w.kin_form, w.four_pi_as = 1, 0, -3.0
        else:
            w.spin_symmetric = 0; w.w_a = 0.6 * np.asarray(w.w_b)
    w.friction = dict(qf_alpha=6.0, qf_beta=5.0, qf_gamma=0.1, qf_rho0=0.03, qf_nreq=1.7)
    psi0 = w.spinors()
    pg, po, fg, fo, o, g = run_both(w, psi0, steps, selfstart=1)
    assert relerr(pg, po) < TOL_ABM and relerr(fg, fo) < TOL_ABM
    for f in ("rho_a", "nu", "bp", "ja_x", "delta", "V_a", "U_b"):
        ref = o.get_field(f)
        assert np.abs(ref).max() > 0
        assert relerr(to_np(g.get_field(f)), ref) < 1e-8, f
    w0 = wl.cfg4(n_side=8, n_wf=24, kin_form=1, n_steps=4)             # friction is not a rounding matter
    if case == "aslda_polarised":
        w0.spin_symmetric = 0; w0.w_a = 0.6 * np.asarray(w0.w_b)
        o0 = make_oracle(w0); o0.densities(psi0); o0.update_potentials()
        o1 = make_oracle(w); o1.densities(psi0); o1.update_potentials()
        assert relerr(o1.get_field("delta"), o0.get_field("delta")) > 1e-3
