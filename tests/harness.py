"""Builds an oracle context and a CUDA context from the same seeded Workload (tests only)."""
import numpy as np

import oracle as orc
import paper_2602_08982_b200 as ws


def relerr(x, ref):
    x, ref = np.asarray(x), np.asarray(ref)
    d = np.max(np.abs(ref))
    return float(np.max(np.abs(x - ref)) / (d if d > 0 else 1.0))


def _kw(w, n_wf, over):
    kw = dict(func_id=w.func_id, force_a1=w.force_a1, spin_symmetric=w.spin_symmetric, kin_form=w.kin_form,
              ab_order=w.ab_order, am_order=w.am_order, subtract_mean_energy=w.subtract_mean_energy,
              normalize=w.normalize, four_pi_as=w.four_pi_as, E_cut=w.E_cut, lambda_mode=w.lambda_mode)
    kw.update(over)
    return kw


def _modes(w, n_wf):
    """Mode table restricted to the first n_wf spinors."""
    if w.kperp is None:
        return None
    first = np.minimum(np.asarray(w.first), n_wf)
    return w.kperp, w.mult, first


def make_oracle(w, n_wf=None, **over):
    n_wf = w.n_wf if n_wf is None else n_wf
    o = orc.Oracle(w.mode, w.dims, w.dx, n_wf, **_kw(w, n_wf, over))
    _configure(o, w, n_wf, np.asarray)
    return o


def make_gpu(w, n_wf=None, **over):
    n_wf = w.n_wf if n_wf is None else n_wf
    g = ws.Context(w.mode, w.dims, w.dx, n_wf, **_kw(w, n_wf, over))
    _configure(g, w, n_wf, np.asarray)
    return g


def _configure(c, w, n_wf, conv):
    c.set_mu(*w.mu)
    md = _modes(w, n_wf)
    if md is not None:
        c.set_modes(*md)
    c.set_weights(conv(w.w_a[:n_wf]), conv(w.w_b[:n_wf]))
    if w.vext_a is not None or w.delta_ext is not None:
        shp = w.shape
        va = None if w.vext_a is None else np.broadcast_to(w.vext_a.reshape(shp), shp).copy()
        vb = None if w.vext_b is None else np.broadcast_to(w.vext_b.reshape(shp), shp).copy()
        c.set_external(va, vb, w.delta_ext)
    if w.fixed:
        c.set_potentials(**w.fixed)


def to_gpu(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def to_np(t):
    return t.detach().cpu().numpy()
